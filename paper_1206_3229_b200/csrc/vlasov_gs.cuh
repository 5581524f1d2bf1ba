// vlasov_gs.cuh -- the GLOBAL SPLINE variant of the shifts (system (15);
// the paper's accuracy comparator "GS" of Tables 1-2), as CUDA kernels for sm_100a.
//
// The paper solves the tridiagonal system (15) for f'' on the CPU and calls it "not effective enough" in parallel
// (L104).  Here it is not solved at all.  The system has constant coefficients (1/6, 2/3, 1/6; DESIGN.md reading
// D22), so its inverse on a periodic (or infinite, zero-extended) line is the convolution with the two-sided
// geometric sequence
//         G_q = sqrt(3) r^|q|,   r = sqrt(3) - 2 = -0.2679...,        (1/6) G_{q-1} + (2/3) G_q + (1/6) G_{q+1} = [q == 0]
// and a convolution with a two-sided geometric sequence is one causal and one anti-causal first-order recursion
// (gs_theta_rec_kernel, gs_p_rec_kernel below).  The recursions are started from zero 36 nodes before the first
// output (|r|^36 = 1e-21); on a periodic line of N >= 32 nodes the images the exact inverse contains (r^N) are below
// 5e-19.  vlasov_set_param refuses GS on shorter axes.  Arithmetic is fp64 for both storage precisions.
// (Round 1 also carried the truncated inverse as a 60-tap filter per shift, fp64-ALU bound at 46 Gpts/s against the
// 75 Gpts/s of the recursions; it was the A/B partner and has been removed.)
#pragma once
#include "vlasov_fused.cuh"  // ptx::cp_async
#include "vlasov_kernels.cuh"

namespace vl {

constexpr int GS_MIN_N = 32;         // shortest axis the zero-start argument covers

// ------------------------------------------------------------------------------------------------
// theta shift with the global spline, RECURSIVE form.  Beyond its centre the inverse is geometric, so
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

template <typename T>
struct GsPArgs {
    const T* fin;
    T* fout;
    const double* force;  // [Ntheta]
    int ntheta, np, bc_p;
    double dt, dp;
};

// ------------------------------------------------------------------------------------------------
// momentum shift with the global spline, RECURSIVE form: a CTA owns 32 adjacent columns and a segment of
// rows; the source rows (+37 halo rows on each side) go ONCE through a shared-memory tile, each column at its own integer
// shift (per-thread cp.async; re-reading the window from global memory through L1 does not work: rows are a power-of-two
// stride apart and evict each other); a thread runs the two recursions of gs_theta_rec_kernel
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
