// vlasov_gs.cuh -- the GLOBAL SPLINE variant of the shifts (system (15);
// the paper's accuracy comparator "GS" of Tables 1-2), as CUDA kernels for sm_100a.
//
// Two sets of kernels: the RECURSIVE ones (gs_theta_rec_kernel, gs_p_rec_kernel: the default, further down) and the
// 60-TAP FILTER ones (gs_theta_sweep_kernel, gs_p_sweep_kernel: tune_gsfir = 1, the A/B partner), described first.
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
//   gs_p_sweep_kernel: a thread owns one column and produces 16 consecutive rows at a time; the 60 weights of a
//       column (they depend on the force there, eq (11)) sit in shared memory [tap][column] and serve 8 row groups.
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
// theta shift with the global spline, RECURSIVE form (default).  Beyond its centre the inverse is geometric, so
//     f''_k h^2 = sqrt(3) (P_k + N_k - d_k),   d_k = f_{k+1} - 2 f_k + f_{k-1},
//     P_k = d_k + r P_{k-1}  (causal),   N_k = d_k + r N_{k+1}  (anti-causal),   r = sqrt(3) - 2,
// two first-order recursions instead of the 60-tap sum, and eq (13) is evaluated as printed:
//     f_new[i] = (1-a) f_k + a f_{k+1} + (A/6) f''_k h^2 + (B/6) f''_{k+1} h^2,  k = i + s.
// A WARP owns 32 x 9 consecutive nodes of a row; a lane runs both recursions over its 9 nodes from a zero start and
// the carries travel between lanes by shuffles: the true carry into a lane is C(l) = P0_8(l-1) + r^9 C(l-1), and
// four rounds of shuffle resolve it to r^36 = 1e-21.  The first and last four lanes (36 nodes) are warm-up only:
// lanes 4..27 produce the warp's 216 outputs.  About 17 fp64 operations per output instead of 60, 11 shared-memory
// loads per lane and row instead of 98; no block-wide barrier: every warp has its own ring of three row windows in
// shared memory, filled by per-lane cp.async two rows ahead (the pass is bound by bytes in flight, not by flops).
// ------------------------------------------------------------------------------------------------
constexpr int GS_RL = 9;                       // nodes per lane
constexpr int GS_RWL = 4;                      // warm-up lanes on each side (4 * 9 = 36 nodes, r^36 = 1e-21)
constexpr int GS_ROUT = (32 - 2 * GS_RWL) * GS_RL;   // outputs per warp and row: 216
constexpr int GS_RWIN = 32 * GS_RL + 2;        // window of a warp: 288 nodes + one more on each side for d
constexpr int GS_RWARPS = 4;                   // warps per CTA
constexpr int GS_RKPRE = (GS_RWIN + 31) / 32;  // window values a lane prefetches: 10

template <typename T>
struct GsThetaRecArgs {
    const T* fin;
    T* fout;
    const int* srow;     // [Np] integer cell shift of one half step
    const double* gsab;  // [Np][4]: 1-a, a, A/6, B/6 of the row
    double* colpart;     // [nbands][Ntheta] or null
    int ntheta, np, bc_x, rows_per_band;
};

#ifndef VL_GS_RSTG
#define VL_GS_RSTG 3
#endif
#ifndef VL_GS_RMINB
#define VL_GS_RMINB 5  // <= 102 registers: 20 warps per SM (sweep: 4 -> 0.337 ms, 5 -> 0.322)
#endif
constexpr int GS_RSTG = VL_GS_RSTG;            // rows in flight per warp (cp.async ring of windows)
constexpr int GS_RWINP = GS_RWIN + 6;          // padded window: a multiple of 16 bytes for both storage types

template <typename T>
__global__ void __launch_bounds__(GS_RWARPS * 32, VL_GS_RMINB) gs_theta_rec_kernel(const GsThetaRecArgs<T> arg) {
    __shared__ __align__(16) T ring[GS_RWARPS][GS_RSTG][GS_RWINP];
    __shared__ __align__(16) double abring[GS_RWARPS][GS_RSTG][4];
    __shared__ __align__(16) T obuf[GS_RWARPS][GS_ROUT];
    constexpr unsigned FULL = 0xffffffffu;
    constexpr double SQ3 = 1.7320508075688772;
    constexpr double r = SQ3 - 2.0;
    constexpr double r2 = r * r, r3 = r2 * r, r4 = r2 * r2, r5 = r4 * r, r6 = r3 * r3, r7 = r6 * r, r8 = r4 * r4, r9 = r8 * r;
    const double rp[GS_RL] = {r, r2, r3, r4, r5, r6, r7, r8, r9};  // r^(k+1)
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int ntheta = arg.ntheta;
    const int o0 = (blockIdx.x * GS_RWARPS + warp) * GS_ROUT;  // first output column of the warp
    if (o0 >= ntheta) return;                                  // whole warp; there is no block-wide barrier
    const int j0 = blockIdx.y * arg.rows_per_band;
    const int j1 = min(arg.np, j0 + arg.rows_per_band);
    const bool periodic = (arg.bc_x == BC_PERIODIC);
    const bool owner = lane >= GS_RWL && lane < 32 - GS_RWL;
    const int icol = o0 + (lane - GS_RWL) * GS_RL;  // first output column of the lane (owners only)
    const int nout = min(GS_ROUT, ntheta - o0);     // outputs of the warp that exist
    T* const O = obuf[warp];

    double csum[GS_RL];
#pragma unroll
    for (int k = 0; k < GS_RL; ++k) csum[k] = 0.0;

    // the window of row j (position q holds source column o0 + s - 36 - 1 + q) and its four coefficients -> slot
    auto issue = [&](int j, int slot) {
        const T* __restrict__ row = arg.fin + (size_t)j * ntheta;
        int base = o0 + arg.srow[j] - GS_RWL * GS_RL - 1;
        if (periodic) base = wrap_index(base, ntheta);
        const uint32_t dst0 = ptx::smem_u32(&ring[warp][slot][0]);
#pragma unroll
        for (int m = 0; m < GS_RKPRE; ++m) {
            const int q = lane + 32 * m;
            if (q < GS_RWIN) {
                int src = base + q;
                bool ok = true;
                if (periodic) {
                    if (src >= ntheta) src %= ntheta;
                } else {
                    ok = (unsigned)src < (unsigned)ntheta;
                }
                ptx::cp_async_zfill<(int)sizeof(T)>(dst0 + (uint32_t)(q * sizeof(T)), ok ? row + src : arg.fin,
                                                    ok ? (unsigned)sizeof(T) : 0u);
            }
        }
        if (lane < 2)
            ptx::cp_async<16>(ptx::smem_u32(&abring[warp][slot][2 * lane]), arg.gsab + (size_t)j * 4 + 2 * lane);
    };

#pragma unroll
    for (int st = 0; st < GS_RSTG - 1; ++st) {
        if (j0 + st < j1) issue(j0 + st, st);
        ptx::cp_async_commit();
    }
    int slot = 0;
    for (int j = j0; j < j1; ++j) {
        ptx::cp_async_wait<GS_RSTG - 2>();  // this lane's copies of row j have landed
        __syncwarp();                       // everybody's have; the slot of row j - 1 and the output tile are free
        {
            int ns = slot + GS_RSTG - 1;
            if (ns >= GS_RSTG) ns -= GS_RSTG;
            if (j + GS_RSTG - 1 < j1) issue(j + GS_RSTG - 1, ns);
            ptx::cp_async_commit();
        }
        const T* __restrict__ W = ring[warp][slot];
        const double al = abring[warp][slot][0], be = abring[warp][slot][1], A6 = abring[warp][slot][2],
                     B6 = abring[warp][slot][3];

        // xv[t] = node 9 lane - 1 + t, t = 0..10
        double xv[GS_RL + 2];
#pragma unroll
        for (int t = 0; t < GS_RL + 2; ++t) xv[t] = (double)W[lane * GS_RL + t];
        double d[GS_RL], P[GS_RL], N[GS_RL];
#pragma unroll
        for (int k = 0; k < GS_RL; ++k) d[k] = (xv[k + 2] - 2.0 * xv[k + 1]) + xv[k];
        P[0] = d[0];
#pragma unroll
        for (int k = 1; k < GS_RL; ++k) P[k] = fma(r, P[k - 1], d[k]);
        N[GS_RL - 1] = d[GS_RL - 1];
#pragma unroll
        for (int k = GS_RL - 2; k >= 0; --k) N[k] = fma(r, N[k + 1], d[k]);
        // carries: C(l) = P0_8(l-1) + r^9 C(l-1), Cb(l) = N0_0(l+1) + r^9 Cb(l+1); zero at the ends of the warp
        double C = 0.0, Cb = 0.0;
#pragma unroll
        for (int it = 0; it < 4; ++it) {
            const double up = __shfl_up_sync(FULL, fma(r9, C, P[GS_RL - 1]), 1);
            const double dn = __shfl_down_sync(FULL, fma(r9, Cb, N[0]), 1);
            C = lane == 0 ? 0.0 : up;
            Cb = lane == 31 ? 0.0 : dn;
        }
        double D[GS_RL + 1];
#pragma unroll
        for (int k = 0; k < GS_RL; ++k) {
            const double Pk = fma(rp[k], C, P[k]);
            const double Nk = fma(rp[GS_RL - 1 - k], Cb, N[k]);
            D[k] = SQ3 * ((Pk + Nk) - d[k]);
        }
        D[GS_RL] = __shfl_down_sync(FULL, D[0], 1);

        // outputs through the warp's tile (lane stride 9: conflict-free) so that the row is stored coalesced
        if (owner) {
#pragma unroll
            for (int k = 0; k < GS_RL; ++k) {
                const T o = (T)fma(B6, D[k + 1], fma(A6, D[k], fma(be, xv[k + 2], al * xv[k + 1])));
                O[(lane - GS_RWL) * GS_RL + k] = o;
                if (icol + k < ntheta) csum[k] += (double)o;
            }
        }
        __syncwarp();
        T* __restrict__ orow = arg.fout + (size_t)j * ntheta + o0;
#pragma unroll
        for (int m = 0; m < (GS_ROUT + 31) / 32; ++m) {
            const int q = lane + 32 * m;
            if (q < nout) orow[q] = O[q];
        }
        if (++slot == GS_RSTG) slot = 0;
    }
    ptx::cp_async_wait<0>();
    if (arg.colpart != nullptr && owner) {
        double* cp = arg.colpart + (size_t)blockIdx.y * ntheta;
#pragma unroll
        for (int k = 0; k < GS_RL; ++k)
            if (icol + k < ntheta) cp[icol + k] = csum[k];
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

// ------------------------------------------------------------------------------------------------
// momentum shift with the global spline, RECURSIVE form (default): same tile as gs_p_sweep_kernel (each column at
// its own integer shift, 37 halo rows on each side), but a thread runs the two recursions of gs_theta_rec_kernel
// down and up its column over a run of GS_PRUN = 24 rows: 36 warm-up rows, the causal values P of the run kept in
// registers, then the anti-causal pass from 36 rows below the run upwards, which emits eq (13) row by row.
// About 18 fp64 operations per point instead of 60; no weight table.
// ------------------------------------------------------------------------------------------------
#ifndef VL_GS_PRUN
#define VL_GS_PRUN 24
#endif
#ifndef VL_GS_PRG
#define VL_GS_PRG 8
#endif
#ifndef VL_GS_PRMINB
#define VL_GS_PRMINB 2
#endif
constexpr int GS_PRUN = VL_GS_PRUN;              // rows per thread
constexpr int GS_PRG = VL_GS_PRG;                // row groups per CTA
constexpr int GS_PRX = 32;                       // columns per CTA
constexpr int GS_PRW = GS_RWL * GS_RL;           // warm-up rows: 36
constexpr int GS_PRSEG = GS_PRUN * GS_PRG;       // rows per CTA
constexpr int GS_PRROWS = GS_PRSEG + 2 * (GS_PRW + 1) + 1;  // rows of the tile: t = -37 .. SEG + 37
template <typename T>
constexpr size_t gs_p_rec_smem() {
    return sizeof(T) * (size_t)GS_PRROWS * GS_PRX;
}

template <typename T>
__global__ void __launch_bounds__(GS_PRX * GS_PRG, VL_GS_PRMINB) gs_p_rec_kernel(const GsPArgs<T> arg) {
    extern __shared__ __align__(16) unsigned char gs_smem[];
    T* tile = reinterpret_cast<T*>(gs_smem);  // [GS_PRROWS][GS_PRX]; row 0 is source row jA + s - 37 of the column
    constexpr double SQ3 = 1.7320508075688772;
    constexpr double r = SQ3 - 2.0;
    const int tid = threadIdx.x, c = tid % GS_PRX, g = tid / GS_PRX;
    const int ntheta = arg.ntheta, np = arg.np;
    const int i = blockIdx.x * GS_PRX + c;
    const bool act = i < ntheta;
    const bool periodic = (arg.bc_p == BC_PERIODIC);
    const int jA = blockIdx.y * GS_PRSEG;
    const int jB = min(np, jA + GS_PRSEG);
    const size_t pitch = (size_t)ntheta;

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
    {
        const T* __restrict__ col = arg.fin + (act ? i : 0);
        const int nrows = (jB - jA) + 2 * (GS_PRW + 1) + 1;  // rows past it (ragged last segment) are zero-filled
        int y = jA + s - (GS_PRW + 1) + g;
        if (periodic) y = wrap_index(y, np);
        uint32_t dst = ptx::smem_u32(tile + g * GS_PRX + c);
        const int ylast = y + (GS_PRROWS - 1 - g) / GS_PRG * GS_PRG;  // last row this thread copies
        if (act && nrows == GS_PRROWS && y >= 0 && ylast < np) {       // every row exists: no per-row tests
            const T* __restrict__ src = col + (size_t)y * pitch;
            const size_t step = (size_t)GS_PRG * pitch;
#pragma unroll 4
            for (int k = g; k < GS_PRROWS; k += GS_PRG) {
                ptx::cp_async<(int)sizeof(T)>(dst, src);
                dst += (uint32_t)(GS_PRG * GS_PRX * sizeof(T));
                src += step;
            }
        } else
        for (int k = g; k < GS_PRROWS; k += GS_PRG) {
            const bool ok = act && k < nrows && (periodic || (unsigned)y < (unsigned)np);
            const T* src = ok ? col + (size_t)y * pitch : arg.fin;
            ptx::cp_async_zfill<(int)sizeof(T)>(dst, src, ok ? (unsigned)sizeof(T) : 0u);
            dst += (uint32_t)(GS_PRG * GS_PRX * sizeof(T));
            y += GS_PRG;
            if (periodic && y >= np) y -= np;
        }
        ptx::cp_async_commit();
    }
    const double al = 1.0 - a, be = a;
    const double A6 = al * (al * al - 1.0) / 6.0, B6 = a * (a * a - 1.0) / 6.0;
    ptx::cp_async_wait<0>();
    __syncthreads();
    const int jlo = jA + g * GS_PRUN;
    if (!act || jlo >= jB) return;

    // x(t) = value at the foot cell of output row jlo + t: tile row g * GS_PRUN + 37 + t
    const T* __restrict__ xcol = tile + (size_t)(g * GS_PRUN + GS_PRW + 1) * GS_PRX + c;
    auto X = [&](int t) -> double { return (double)xcol[t * GS_PRX]; };

    // causal pass: warm-up over t = -36 .. -1, then the run
    double xm = X(-GS_PRW - 1), x0 = X(-GS_PRW), P = 0.0;
#pragma unroll 6
    for (int t = -GS_PRW; t < 0; ++t) {
        const double xp = X(t + 1);
        P = fma(r, P, (xp - 2.0 * x0) + xm);
        xm = x0;
        x0 = xp;
    }
    double Pv[GS_PRUN];
#pragma unroll
    for (int t = 0; t < GS_PRUN; ++t) {
        const double xp = X(t + 1);
        P = fma(r, P, (xp - 2.0 * x0) + xm);
        Pv[t] = P;
        xm = x0;
        x0 = xp;
    }
    // here x0 = x(RUN), xm = x(RUN - 1): P at RUN for the f'' that the last row needs
    const double dR = (X(GS_PRUN + 1) - 2.0 * x0) + xm;
    const double PR = fma(r, P, dR);

    // anti-causal pass: warm-up over t = RUN + 36 .. RUN + 1, then upwards through the run
    double xp = X(GS_PRUN + GS_PRW + 1), N = 0.0;
    x0 = X(GS_PRUN + GS_PRW);
#pragma unroll 6
    for (int t = GS_PRUN + GS_PRW; t > GS_PRUN; --t) {
        const double xl = X(t - 1);
        N = fma(r, N, (xp - 2.0 * x0) + xl);
        xp = x0;
        x0 = xl;
    }
    // here x0 = x(RUN), xp = x(RUN + 1)
    N = fma(r, N, dR);
    double Dn = SQ3 * ((PR + N) - dR);  // f'' h^2 at RUN
    T* __restrict__ ocol = arg.fout + i + (size_t)jlo * pitch;
    double xh = x0, xc = xm;  // x(t + 1), x(t) for t = RUN - 1 (xm is still x(RUN - 1) from the causal pass)
#pragma unroll
    for (int t = GS_PRUN - 1; t >= 0; --t) {
        const double xl = X(t - 1);
        const double d = (xh - 2.0 * xc) + xl;
        N = fma(r, N, d);
        const double D = SQ3 * ((Pv[t] + N) - d);
        const double o = fma(B6, Dn, fma(A6, D, fma(be, xh, al * xc)));
        if (jlo + t < jB) ocol[(size_t)t * pitch] = (T)o;
        Dn = D;
        xh = xc;
        xc = xl;
    }
}

}  // namespace vl
