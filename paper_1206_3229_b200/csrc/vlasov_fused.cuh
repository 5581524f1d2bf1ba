// vlasov_fused.cuh -- ONE pass per Strang step: momentum shift, then the theta half shift(s), then the density.
//
// Method (section 3): a step is  theta(dt/2) -> rho, F -> p(dt) -> theta(dt/2).  The density
// (eq (10)) is a reduction over all rows, so theta(dt/2) -> p cannot share a pass; but
//     p(dt) of step k  ->  theta(dt/2) of step k  ->  theta(dt/2) of step k+1  ->  rho of step k+1
// can: the force of step k is known before the pass starts and the density of step k+1 is its epilogue.
// n steps = n + 1 passes over f (16 B per grid point per step in fp64) instead of the 2n + 1 of separate
// p and theta kernels.  Every shift is still the spline of eqs (13)-(14) (L89-L98) with f'' from eq (16)
// (L106-L111), folded into ten weights per line (see vlasov_kernels.cuh).
//
// Geometry.  A CTA owns TI + NTAP - 1 consecutive SOURCE columns and a band of rows and marches down the band:
//   p stage      one thread per source column; a register window slides down the column (one new value and ten
//                FMAs per row, exactly p_sweep_kernel); the new values of the next rows are prefetched with
//                per-thread cp.async into a shared-memory ring (no registers held by loads in flight).  The
//                shifted row g goes to shared memory.
//   theta stage  one warp per row of the phase: lane l produces R consecutive values from a register window of
//                its shared-memory row.  In source-column coordinates the theta shift is shift-free:
//                out'[q] = sum_n W_n g'[q + n]; the integer part of the shift only decides WHERE the row is
//                written: column i0 + q - NST*s_j (mod Ntheta).  The output region of a CTA is therefore a
//                parallelogram that drifts with the row, and the source columns stay fixed (which is what the
//                register window of the p stage needs).  NST = 2 applies both half shifts at once with the 19
//                composite weights W = w * w of the row (periodic theta only); NST = 1 applies one.
//   store stage  one thread per OUTPUT column (fixed for the whole band): coalesced stores from the shared
//                output tile and the column sums of the band in registers (density partials, eq (10)).
// At the end of the band the column sums are added to colpart[band][column]; at most two CTAs (neighbouring
// column blocks whose parallelograms overlap) contribute to an entry that starts at zero, and x + y = y + x
// in IEEE arithmetic, so the result does not depend on their order.
#pragma once
#include "vlasov_kernels.cuh"

namespace vl {

template <typename T>
struct FusedArgs {
    const T* fin;
    T* fout;
    const double* force;     // [Ntheta] force of this step's momentum shift
    const int* srow;         // [Np] integer part of ONE half theta shift (reduced mod Ntheta when periodic)
    const double* wtab;      // [Np][wstride] theta weights of the row: NST = 1: w_0..w_9; NST = 2: W_0..W_18
    const int* band_s;       // [nbands][2] {min, max} of NST * srow over the rows of the band
    double* colpart;         // [nbands][Ntheta], zero on entry; column sums are ADDED (may be null)
    int ntheta, np, bc_p, rows_per_band, wstride;
    double dt, dp;
};

template <typename T, int NST, int NT, int R, int NSTG>
struct FusedCfg {
    static constexpr int NW = NT / 32;
    static constexpr int RB = NW;                       // rows per phase: one per warp in the theta stage
    static constexpr int NTAP = NST == 2 ? 19 : 10;
    static constexpr int TI = 32 * R;                   // output columns per CTA and row
    static constexpr int NTA = TI + NTAP - 1;           // source columns = active threads of the p stage
    static constexpr int NCS = 2;                       // output columns owned per thread (drift <= NCS*NT - TI)
    static constexpr int MAX_DRIFT = (NCS * NT - TI) < TI ? (NCS * NT - TI) : TI;
    static constexpr size_t STAGE_ELEMS = (size_t)NSTG * RB * NT;
    static constexpr size_t G_ELEMS = (size_t)RB * NT;
    static constexpr size_t O_ELEMS = (size_t)RB * TI;
    static constexpr size_t SMEM_BYTES = (STAGE_ELEMS + G_ELEMS + O_ELEMS) * sizeof(T) + 4 * RB * sizeof(int);
    static_assert(NT % 32 == 0 && NTA <= NT, "one thread per source column");
    static_assert(R & 1, "lane stride R must be odd (shared-memory banks)");
    static_assert(RB == 12, "the p-stage register ring is written for 12 rows per phase");
};

namespace ptx {
// per-thread asynchronous copy global -> shared of sizeof(T) bytes; src_bytes = 0 writes zeros instead
template <int BYTES>
__device__ __forceinline__ void cp_async_zfill(void* dst_smem, const void* src_gmem, unsigned src_bytes) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], %2, %3;" ::"r"(smem_u32(dst_smem)), "l"(src_gmem), "n"(BYTES),
                 "r"(src_bytes)
                 : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() {
    asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory");
}
__device__ __forceinline__ void red_add_f64(double* addr, double v) {
    asm volatile("red.global.add.f64 [%0], %1;" ::"l"(addr), "d"(v) : "memory");
}
}  // namespace ptx

template <typename T, int NST, int NT, int R, int NSTG>
__global__ void __launch_bounds__(NT, 1) strang_fused_kernel(const FusedArgs<T> arg) {
    using C = FusedCfg<T, NST, NT, R, NSTG>;
    constexpr int RB = C::RB, NTAP = C::NTAP, TI = C::TI, NTA = C::NTA, NCS = C::NCS;

    extern __shared__ __align__(16) unsigned char smem_raw[];
    T* stage = reinterpret_cast<T*>(smem_raw);                 // [NSTG][RB][NT] new taps of the p stage
    T* gt = stage + C::STAGE_ELEMS;                            // [RB][NT]      rows after the momentum shift
    T* ot = gt + C::G_ELEMS;                                   // [RB][TI]      rows after the theta shift(s)
    int* rinfo = reinterpret_cast<int*>(ot + C::O_ELEMS);      // [2][RB][2]    {first output column, drift offset}

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int ntheta = arg.ntheta, np = arg.np;
    const int i0 = blockIdx.x * TI;
    const int band = blockIdx.y;
    const int jA = band * arg.rows_per_band;
    const int jB = min(np, jA + arg.rows_per_band);
    if (jA >= jB) return;  // whole CTA
    const int nph = (jB - jA + RB - 1) / RB;
    const bool p_periodic = (arg.bc_p == BC_PERIODIC);
    const int smin2 = arg.band_s[2 * band + 0], smax2 = arg.band_s[2 * band + 1];

    // ---- p stage set-up: this thread's source column, its shift and ten weights (eq (11))
    const bool active = tid < NTA;
    const int c = wrap_index(i0 - 4 * NST + tid, ntheta);
    double sf, a;
    split_shift(-((active ? arg.force[c] : 0.0) * arg.dt) / arg.dp, &sf, &a);
    int s;
    if (p_periodic) {
        sf = fmod(sf, (double)np);
        s = (int)sf;
        if (s < 0) s += np;
    } else {
        const double lim = (double)np + 64.0;
        s = (int)fmin(fmax(sf, -lim), lim);
    }
    T w[10];
    {
        double wd[10];
        spline_fd8_weights(a, wd);
#pragma unroll
        for (int m = 0; m < 10; ++m) w[m] = (T)wd[m];
    }
    const T* __restrict__ col = arg.fin + c;
    const size_t pitch = (size_t)ntheta;

    // row of tap m of output row j is j + s + m - 4; rn = row of the next value the window has not seen yet
    int rn = jA + s - 4;
    if (p_periodic) rn = wrap_index(rn, np);
    T v[12];  // register ring: taps of output row r of a phase are v[(r + m) % 12]
#pragma unroll
    for (int k = 0; k < 9; ++k) {
        const bool ok = active && (p_periodic || (unsigned)rn < (unsigned)np);
        v[k] = ok ? __ldg(col + (size_t)rn * pitch) : T(0);
        ++rn;
        if (p_periodic && rn >= np) rn = 0;
    }
    v[9] = v[10] = v[11] = T(0);

    auto issue_stage = [&](int ph) {  // new taps of the RB rows of phase ph -> ring slot ph % NSTG
        T* dst = stage + (size_t)(ph % NSTG) * RB * NT + tid;
#pragma unroll
        for (int r = 0; r < RB; ++r) {
            const bool ok = active && (p_periodic || (unsigned)rn < (unsigned)np);
            const T* src = ok ? col + (size_t)rn * pitch : arg.fin;
            ptx::cp_async_zfill<(int)sizeof(T)>(dst + r * NT, src, ok ? (unsigned)sizeof(T) : 0u);
            ++rn;
            if (p_periodic && rn >= np) rn = 0;
        }
    };

#pragma unroll
    for (int st = 0; st < NSTG - 1; ++st) {
        if (st < nph) issue_stage(st);
        ptx::cp_async_commit();
    }

    double csum[NCS];
#pragma unroll
    for (int k = 0; k < NCS; ++k) csum[k] = 0.0;

    for (int ph = 0; ph < nph; ++ph) {
        const int jph = jA + ph * RB;
        if (ph + NSTG - 1 < nph) issue_stage(ph + NSTG - 1);
        ptx::cp_async_commit();
        ptx::cp_async_wait<NSTG - 1>();  // this thread's taps of phase ph have landed (only it reads them)

        int* ri = rinfo + (ph & 1) * 2 * RB;
        if (tid < RB && jph + tid < jB) {
            const int S = NST * __ldg(arg.srow + jph + tid);
            ri[2 * tid + 0] = wrap_index(i0 - S, ntheta);  // output column of q = 0
            ri[2 * tid + 1] = smax2 - S;                   // >= 0: position of q = 0 among the CTA's output columns
        }

        // ---- p stage: ten FMAs per row from the register ring
        {
            const T* src = stage + (size_t)(ph % NSTG) * RB * NT + tid;
            T* g = gt + tid;
#pragma unroll
            for (int r = 0; r < RB; ++r) {
                v[(r + 9) % 12] = src[r * NT];
                T acc = w[0] * v[r % 12];
#pragma unroll
                for (int m = 1; m < 10; ++m) acc = fma(w[m], v[(r + m) % 12], acc);
                g[r * NT] = acc;
            }
        }
        __syncthreads();

        // ---- theta stage: warp = row; shift-free in source-column coordinates
        if (jph + warp < jB) {
            const double* __restrict__ wr = arg.wtab + (size_t)(jph + warp) * arg.wstride;
            T W[NTAP];
#pragma unroll
            for (int n = 0; n < NTAP; ++n) W[n] = (T)__ldg(wr + n);
            const T* grow = gt + warp * NT + lane * R;
            T x[R + NTAP - 1];
#pragma unroll
            for (int k = 0; k < R + NTAP - 1; ++k) x[k] = grow[k];
            T* orow = ot + warp * TI + lane * R;
#pragma unroll
            for (int r = 0; r < R; ++r) {
                T acc = W[0] * x[r];
#pragma unroll
                for (int n = 1; n < NTAP; ++n) acc = fma(W[n], x[r + n], acc);
                orow[r] = acc;
            }
        }
        __syncthreads();

        // ---- store stage: thread = output column (fixed over the band); coalesced stores + column sums
        {
            const int nr = min(RB, jB - jph);
            for (int r = 0; r < nr; ++r) {
                const int base = ri[2 * r + 0], d = ri[2 * r + 1];
                T* __restrict__ orow_g = arg.fout + (size_t)(jph + r) * pitch;
#pragma unroll
                for (int k = 0; k < NCS; ++k) {
                    const int q = tid + k * NT - d;
                    if (q >= 0 && q < TI && i0 + q < ntheta) {
                        const T val = ot[r * TI + q];
                        int i = base + q;
                        if (i >= ntheta) i -= ntheta;
                        orow_g[i] = val;
                        csum[k] += (double)val;
                    }
                }
            }
        }
    }

    if (arg.colpart != nullptr) {
        double* __restrict__ cp = arg.colpart + (size_t)band * ntheta;
        const int ext = TI + (smax2 - smin2);
#pragma unroll
        for (int k = 0; k < NCS; ++k) {
            const int e = tid + k * NT;
            // position e is output column i0 + e - smax2; only positions some row really wrote carry a sum
            if (e < ext && csum[k] != 0.0) ptx::red_add_f64(cp + wrap_index(i0 + e - smax2, ntheta), csum[k]);
        }
    }
}

}  // namespace vl
