// vlasov_gs.cuh -- the GLOBAL SPLINE variant of the shifts (system (15);
// the paper's accuracy comparator "GS" of Tables 1-2), as CUDA kernels for sm_100a.
//
// The paper solves the tridiagonal system (15) for f'' on the CPU and calls it "not effective enough" in parallel
// (L104).  Here it is not solved at all.  The system has constant coefficients (1/6, 2/3, 1/6; DESIGN.md reading
// D22), so its inverse on a periodic (or infinite, zero-extended) line is the convolution with the two-sided
// geometric sequence
//         G_q = sqrt(3) r^|q|,   r = sqrt(3) - 2 = -0.2679...,        (1/6) G_{q-1} + (2/3) G_q + (1/6) G_{q+1} = [q == 0]
// which falls below 1e-16 at |q| = GS_Q = 28 (|r|^28 = 9.6e-17).  With the second difference folded in,
//         f''_k h^2 = sum_m H_m f_{k+m},   H_m = G_{m-1} - 2 G_m + G_{m+1}   (|m| <= GS_Q + 1, G_q = 0 for |q| > GS_Q)
// and substituting in eq (13) the h^2 cancels, exactly as for eq (16): one shift of a line is the GS_NT = 60 tap filter
//         f_new[i] = sum_{m=-29}^{30} w_m(a) f[i + s + m],   w_m = [m==0](1-a) + [m==1] a + (A H_m + B H_{m-1})/6,
// A = (1-a)^3 - (1-a), B = a^3 - a.  The truncation changes f_new by < 4e-17 max|f|, below the rounding of the sum.
// On a periodic line of N >= 32 nodes the images the exact inverse contains (r^N) are below 5e-19; the taps that
// wrap around the line are summed by the wrapped indexing itself.  vlasov_set_param refuses GS on shorter axes.
//
// 60 FMAs per point and shift instead of 10: these kernels are bound by the fp64 pipe, not by HBM (540 fp64 FMAs
// per 16 bytes moved).  Both keep a window of R values and R accumulators in registers and slide it tap by tap, so
// that a tap costs one shared-memory (or L1) load of data and one of a weight per R FMAs.
//   gs_theta_sweep_kernel: a CTA owns a chunk of blockDim * 9 columns and walks down a band of rows; each lane owns 9
//       consecutive columns (lane stride 9: conflict-free) and keeps their column sums (density partials, eq (10));
//       the next row's window is prefetched into registers while the current one is computed.  One wave of CTAs.
//   gs_p_sweep_kernel: a thread owns one column and produces 8 consecutive rows at a time; the 60 weights of a
//       column (they depend on the force there, eq (11)) sit in shared memory [tap][column] and serve 4 row groups.
// Arithmetic is fp64 for both storage precisions.
#pragma once
#include "vlasov_fused.cuh"  // ptx::cp_async
#include "vlasov_kernels.cuh"

namespace vl {

constexpr int GS_Q = 28;             // half width of the truncated inverse
constexpr int GS_NT = 2 * GS_Q + 4;  // taps of one shift: m = -(GS_Q+1) .. GS_Q+2
constexpr int GS_M0 = GS_Q + 1;      // w[n] multiplies f[k + n - GS_M0]
constexpr int GS_MIN_N = 32;         // shortest axis the truncation argument covers

__host__ __device__ inline double gs_G(int q) {
    const double r = 1.7320508075688772 - 2.0;
    if (q < 0) q = -q;
    if (q > GS_Q) return 0.0;
    double v = 1.7320508075688772;
    for (int k = 0; k < q; ++k) v *= r;
    return v;
}

// H_m / 6, m = -(GS_Q+1) .. GS_Q+1, index m + GS_Q + 1; 2 GS_Q + 3 entries
__host__ __device__ inline void gs_H_over_6(double* H) {
    for (int m = -(GS_Q + 1); m <= GS_Q + 1; ++m) H[m + GS_Q + 1] = (gs_G(m - 1) - 2.0 * gs_G(m) + gs_G(m + 1)) / 6.0;
}

// the GS_NT weights of a shift with fraction a from the table H/6 (host: rows; device: columns)
// taps n = n0, n0 + nstep, ..
__host__ __device__ inline void gs_weights(double a, const double* H6, double* w, int stride = 1, int n0 = 0,
                                           int nstep = 1) {
    const double al = 1.0 - a;
    const double A = al * (al * al - 1.0);
    const double B = a * (a * a - 1.0);
    for (int n = n0; n < GS_NT; n += nstep) {
        const int m = n - GS_M0;  // -(Q+1) .. Q+2
        double v = 0.0;
        if (m <= GS_Q + 1) v += A * H6[m + GS_Q + 1];
        if (m - 1 >= -(GS_Q + 1)) v += B * H6[m - 1 + GS_Q + 1];
        if (m == 0) v += al;
        if (m == 1) v += a;
        w[(size_t)n * stride] = v;
    }
}

// ------------------------------------------------------------------------------------------------
// theta shift, eq (9) / (12) with the global spline
// ------------------------------------------------------------------------------------------------
#ifndef VL_GS_TR
#define VL_GS_TR 9
#endif
constexpr int GS_TR = VL_GS_TR;                // consecutive outputs per thread (odd: conflict-free lane stride)
constexpr int GS_TMAXT = 256;                  // most threads per CTA (the host picks 64 .. 256 by the row length)
#ifndef VL_GS_TMINB
#define VL_GS_TMINB 3  // <= 85 registers: 8 CTAs of 96 threads per SM (sweep in profiles/README.md)
#endif
constexpr int GS_TKPRE = GS_TR + 1;            // window values a thread prefetches: ceil((9 bd + 59) / bd), bd >= 64

template <typename T>
struct GsThetaArgs {
    const T* fin;
    T* fout;
    const int* srow;     // [Np] integer cell shift of one half step
    const double* gsw;   // [Np][GS_NT] weights of one half step
    double* colpart;     // [nbands][Ntheta] or null
    int ntheta, np, bc_x, rows_per_band;
};

// Arithmetic is fp64 whatever the storage type T (60 taps in fp32 would not keep 1e-4 over 100 steps).
template <typename T>
__global__ void __launch_bounds__(GS_TMAXT, VL_GS_TMINB) gs_theta_sweep_kernel(const GsThetaArgs<T> arg) {
    __shared__ double xs[GS_TR * GS_TMAXT + GS_NT];
    __shared__ double ws[GS_NT];
    const int tid = threadIdx.x, bd = blockDim.x;
    const int ntheta = arg.ntheta;
    const int chunk = GS_TR * bd, win = chunk + GS_NT - 1;
    const int c0 = blockIdx.x * chunk;
    const int j0 = blockIdx.y * arg.rows_per_band;
    const int j1 = min(arg.np, j0 + arg.rows_per_band);
    const bool periodic = (arg.bc_x == BC_PERIODIC);
    const int q0 = tid * GS_TR;
    const int i0 = c0 + q0;

    double csum[GS_TR];
#pragma unroll
    for (int r = 0; r < GS_TR; ++r) csum[r] = 0.0;

    // the window of the next row (and its weights) travel through registers while this row is computed
    T pre[GS_TKPRE];
    double wpre = 0.0;
    auto prefetch = [&](int j) {
        const T* __restrict__ row = arg.fin + (size_t)j * ntheta;
        int base = c0 + arg.srow[j] - GS_M0;
        if (periodic) base = wrap_index(base, ntheta);
#pragma unroll
        for (int k = 0; k < GS_TKPRE; ++k) {
            const int q = tid + k * bd;
            T v = T(0);
            if (q < win) {
                int src = base + q;
                if (periodic) {
                    if (src >= ntheta) src %= ntheta;
                    v = __ldg(row + src);
                } else if ((unsigned)src < (unsigned)ntheta) {
                    v = __ldg(row + src);
                }
            }
            pre[k] = v;
        }
        if (tid < GS_NT) wpre = arg.gsw[(size_t)j * GS_NT + tid];
    };

    if (j0 < j1) prefetch(j0);
    for (int j = j0; j < j1; ++j) {
        __syncthreads();  // the previous row's window and weights are no longer read
#pragma unroll
        for (int k = 0; k < GS_TKPRE; ++k) {
            const int q = tid + k * bd;
            if (q < win) xs[q] = (double)pre[k];
        }
        if (tid < GS_NT) ws[tid] = wpre;
        __syncthreads();
        if (j + 1 < j1) prefetch(j + 1);

        double x[GS_TR], out[GS_TR];
#pragma unroll
        for (int r = 0; r < GS_TR - 1; ++r) x[r] = xs[q0 + r];
#pragma unroll
        for (int r = 0; r < GS_TR; ++r) out[r] = 0.0;
#pragma unroll
        for (int n = 0; n < GS_NT; ++n) {
            // window slot (n + r) % GS_TR holds xs[q0 + n + r]
            x[(n + GS_TR - 1) % GS_TR] = xs[q0 + n + GS_TR - 1];
            const double w = ws[n];
#pragma unroll
            for (int r = 0; r < GS_TR; ++r) out[r] = fma(w, x[(n + r) % GS_TR], out[r]);
        }
        T* __restrict__ orow = arg.fout + (size_t)j * ntheta;
#pragma unroll
        for (int r = 0; r < GS_TR; ++r) {
            if (i0 + r < ntheta) {
                const T o = (T)out[r];
                orow[i0 + r] = o;
                csum[r] += (double)o;
            }
        }
    }
    if (arg.colpart != nullptr) {
        double* cp = arg.colpart + (size_t)blockIdx.y * ntheta;
#pragma unroll
        for (int r = 0; r < GS_TR; ++r)
            if (i0 + r < ntheta) cp[i0 + r] = csum[r];
    }
}

// ------------------------------------------------------------------------------------------------
// momentum shift, eq (11) with the global spline
//
// A CTA owns GS_PTX = 32 adjacent columns and a segment of GS_PSEG = 256 rows.  The source rows of the segment go
// through a shared-memory tile ONCE (per-thread cp.async, one commit group per chunk of 128 output rows): tile[k][c] = f[jA + s_c - 29 + k][i0 + c], k < GS_PSEG + 59, each column at its own
// integer shift s_c, so that inside the tile every column's window starts at the same k.  (Re-reading the window
// from global memory through L1 does not work: rows are a power-of-two stride apart and evict each other.)
// Thread (column c, row group g) produces GS_PR consecutive rows at a time from a sliding register window.
// ------------------------------------------------------------------------------------------------
#ifndef VL_GS_PG
#define VL_GS_PG 8
#endif
#ifndef VL_GS_PR
#define VL_GS_PR 16
#endif
#ifndef VL_GS_PSEGMUL
#define VL_GS_PSEGMUL 2
#endif
#ifndef VL_GS_PMINB
#define VL_GS_PMINB 1
#endif
#ifndef VL_GS_PTX
#define VL_GS_PTX 32
#endif
constexpr int GS_PTX = VL_GS_PTX;   // columns per CTA
constexpr int GS_PG = VL_GS_PG;     // row groups per CTA
constexpr int GS_PR = VL_GS_PR;     // consecutive output rows per thread and block
constexpr int GS_PSEG = VL_GS_PSEGMUL * GS_PG * GS_PR;  // rows per CTA
constexpr int GS_PROWS = GS_PSEG + GS_NT - 1;           // rows of the tile
template <typename T>
constexpr size_t gs_p_smem() {
    return sizeof(double) * ((size_t)GS_NT * GS_PTX + 2 * GS_Q + 4) + sizeof(T) * (size_t)GS_PROWS * GS_PTX;
}

template <typename T>
struct GsPArgs {
    const T* fin;
    T* fout;
    const double* force;  // [Ntheta]
    const double* H6;     // [2 GS_Q + 3]
    int ntheta, np, bc_p;
    double dt, dp;
};

template <typename T>
__global__ void __launch_bounds__(GS_PTX * GS_PG, VL_GS_PMINB) gs_p_sweep_kernel(const GsPArgs<T> arg) {
    extern __shared__ __align__(16) unsigned char gs_smem[];
    double* wsm = reinterpret_cast<double*>(gs_smem);       // [GS_NT][GS_PTX]
    double* H6s = wsm + (size_t)GS_NT * GS_PTX;             // [2 GS_Q + 3] (+ 1 pad)
    T* tile = reinterpret_cast<T*>(H6s + 2 * GS_Q + 4);     // [GS_PROWS][GS_PTX], storage type
    const int tid = threadIdx.x, c = tid % GS_PTX, g = tid / GS_PTX;
    const int ntheta = arg.ntheta, np = arg.np;
    const int i = blockIdx.x * GS_PTX + c;
    const bool act = i < ntheta;
    const bool periodic = (arg.bc_p == BC_PERIODIC);
    if (tid < 2 * GS_Q + 3) H6s[tid] = arg.H6[tid];
    const int jA = blockIdx.y * GS_PSEG;
    const int jB = min(np, jA + GS_PSEG);
    const size_t pitch = (size_t)ntheta;

    // integer shift and fraction of the column: eta = F dt / dp cells; the foot of row j is row j + s + a
    double sf, a;
    split_shift(-((act ? arg.force[i] : 0.0) * arg.dt) / arg.dp, &sf, &a);
    int s;
    if (periodic) {
        sf = fmod(sf, (double)np);
        s = (int)sf;
    } else {
        const double lim = (double)np + 64.0;
        s = (int)fmin(fmax(sf, -lim), lim);
    }

    // the tile: rows jA + s - 29 + k of this thread's column, k = g, g + GS_PG, ..  All copies are issued at once, in
    // one commit group per chunk of GS_PG * GS_PR output rows (chunk 0 also carries the 59 halo rows), so that the
    // first chunk can be computed while the others are still in flight.
    constexpr int CH = GS_PG * GS_PR, NCH = VL_GS_PSEGMUL;
    {
        const T* __restrict__ col = arg.fin + (act ? i : 0);
        const int nrows = (jB - jA) + GS_NT - 1;
        int y = jA + s - GS_M0 + g;
        if (periodic) y = wrap_index(y, np);
        uint32_t dst = ptx::smem_u32(tile + g * GS_PTX + c);
        int k = g;
#pragma unroll
        for (int m = 0; m < NCH; ++m) {
            const int hi = min(nrows, (m + 1) * CH + GS_NT - 1);
            for (; k < hi; k += GS_PG) {
                const bool ok = act && (periodic || (unsigned)y < (unsigned)np);
                const T* src = ok ? col + (size_t)y * pitch : arg.fin;
                ptx::cp_async_zfill<(int)sizeof(T)>(dst, src, ok ? (unsigned)sizeof(T) : 0u);
                dst += (uint32_t)(GS_PG * GS_PTX * sizeof(T));
                y += GS_PG;
                if (periodic && y >= np) y -= np;
            }
            ptx::cp_async_commit();
        }
    }
    __syncthreads();  // H6s
    gs_weights(a, H6s, wsm + c, GS_PTX, g, GS_PG);  // while the copies fly: group g takes the taps g, g + GS_PG, ..

    T* __restrict__ ocol = arg.fout + (act ? i : 0);
    const double* __restrict__ wc = wsm + c;
#pragma unroll 1
    for (int m = 0; m < NCH; ++m) {
        const int jb = jA + m * CH + g * GS_PR;
        // this thread's copies of chunks 0..m have landed; after the barrier everybody's have (and the weights)
        switch (NCH - 1 - m) {
            case 0: ptx::cp_async_wait<0>(); break;
            case 1: ptx::cp_async_wait<1>(); break;
            case 2: ptx::cp_async_wait<2>(); break;
            case 3: ptx::cp_async_wait<3>(); break;
            case 4: ptx::cp_async_wait<4>(); break;
            case 5: ptx::cp_async_wait<5>(); break;
            case 6: ptx::cp_async_wait<6>(); break;
            default: ptx::cp_async_wait<7>(); break;
        }
        __syncthreads();
        if (!act || jb >= jB) continue;
        const T* __restrict__ tc = tile + (size_t)(jb - jA) * GS_PTX + c;
        double x[GS_PR], out[GS_PR];
#pragma unroll
        for (int r = 0; r < GS_PR - 1; ++r) x[r] = (double)tc[r * GS_PTX];
#pragma unroll
        for (int r = 0; r < GS_PR; ++r) out[r] = 0.0;
#pragma unroll
        for (int n = 0; n < GS_NT; ++n) {
            // rows past the end of a short last block read stale tile rows: their outputs are not stored
            x[(n + GS_PR - 1) % GS_PR] = (double)tc[(n + GS_PR - 1) * GS_PTX];
            const double w = wc[n * GS_PTX];
#pragma unroll
            for (int r = 0; r < GS_PR; ++r) out[r] = fma(w, x[(n + r) % GS_PR], out[r]);
        }
#pragma unroll
        for (int r = 0; r < GS_PR; ++r)
            if (jb + r < jB) ocol[(size_t)(jb + r) * pitch] = (T)out[r];
    }
}

}  // namespace vl
