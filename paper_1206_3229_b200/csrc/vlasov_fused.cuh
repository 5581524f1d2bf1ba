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
// Geometry.  A CTA owns NTA = TI + NTAP - 1 consecutive SOURCE columns (one per thread) and a band of rows and
// marches down the band in phases of RB = 12 rows; one block-wide barrier per phase.
//   p stage      thread = source column.  A register window slides down the column (one new value and ten FMAs
//                per row, as in p_sweep_kernel).  The new values of the next two phases are in flight as
//                per-thread cp.async copies into a three-slot shared-memory ring (no registers held by loads);
//                the shifted value overwrites the tap in place, so a slot turns from "taps" into "rows after the
//                momentum shift".
//   theta stage  warp = row of the phase (no further block-wide barrier: each warp finishes its row alone).
//                In source-column coordinates the theta shift is shift-free: out'[q] = sum_n W_n g'[q + n]; the
//                integer part S of the shift only decides WHERE the row is written: column i0 + q - S (mod
//                Ntheta).  The output region of a CTA is a parallelogram that drifts with the row while the
//                source columns stay fixed (which is what the register window of the p stage needs).  Lane l
//                makes R consecutive values from a window of its shared-memory row (lane stride R, odd:
//                conflict-free), the weights of the row come from shared memory (they travel with the taps).
//                NST = 2 applies both half shifts at once with the 19 composite weights W = w * w of the row
//                (periodic theta only); NST = 1 applies one.
//   store        the warp writes its row to a private shared tile and lane 0 hands it to the bulk-copy engine
//                (cp.async.bulk shared -> global, 16-byte aligned body; the 0..EPV-1 elements before and after
//                the aligned body are stored by lanes).  Rows that are not a multiple of 16 bytes use plain
//                coalesced stores instead.
//   density      each lane keeps the column sums of its R outputs in registers.  When the integer shift of the
//                warp's next row is smaller by one, every sum moves one register to the left (the leftmost of a
//                lane comes from its right neighbour by shuffle) and the sum that leaves lane 0 is final for
//                this warp: it is added to colpart[band][warp][column].  At the end of the band all sums are
//                added.  An entry receives at most two contributions (this CTA and the neighbouring column
//                block whose parallelogram overlaps) onto zero, and x + y = y + x in IEEE arithmetic: the
//                density does not depend on the order of arrival.
#pragma once
#include "vlasov_kernels.cuh"

namespace vl {

template <typename T>
struct FusedArgs {
    const T* fin;
    T* fout;
    const double* force;     // [Ntheta] force of this step's momentum shift
    const double* wtab;      // [Np + RB][WST] theta weights of the row, then its integer shift as a double:
                             //   NST = 1: w_0..w_9, s;  NST = 2: W_0..W_18, 2 s   (s non-increasing with the row)
    double* colpart;         // [nbands * NW][Ntheta], zero on entry; column sums are ADDED (may be null)
    int ntheta, np, bc_p, rows_per_band, bulk_ok, gran;
    double dt, dp;
};

template <typename T, int NST, int NT, int R, int NSTG>
struct FusedCfg {
    static constexpr int NW = NT / 32;
    static constexpr int RB = 12;                       // rows per phase = length of the p-stage register ring
    static constexpr int NTAP = NST == 2 ? 19 : 10;
    static constexpr int WST = NST == 2 ? 20 : WROW_STRIDE;
    static constexpr int TI = 32 * R;                   // output columns per CTA and row (at most)
    static constexpr int NTA = TI + NTAP - 1;           // source columns = active threads of the p stage
    static constexpr int EPV = 16 / (int)sizeof(T);     // elements per 16 bytes
    static constexpr int OB = (TI + EPV + EPV - 1) / EPV * EPV;
    static constexpr size_t SLOT_ELEMS = (size_t)RB * NT;
    static constexpr size_t SLOTS_BYTES = (size_t)NSTG * SLOT_ELEMS * sizeof(T);
    static constexpr size_t W_BYTES = (size_t)NSTG * RB * WST * sizeof(double);
    static constexpr size_t O_BYTES = (size_t)NW * 2 * OB * sizeof(T);
    static constexpr size_t SMEM_BYTES = SLOTS_BYTES + W_BYTES + O_BYTES;
    static constexpr int W_COPIES = RB * WST * 8 / 16;  // 16-byte copies of the weight rows of one phase
    static_assert(NT % 32 == 0 && NTA <= NT, "one thread per source column");
    static_assert(R & 1, "lane stride R must be odd (shared-memory banks)");
    static_assert(NW == RB, "one warp per row of a phase");
    static_assert(W_COPIES <= NT && NSTG >= 2, "");
    static_assert(SLOTS_BYTES % 16 == 0 && W_BYTES % 16 == 0, "");
};

namespace ptx {
// per-thread asynchronous copy global -> shared of BYTES (4, 8 or 16) bytes; src_bytes = 0 writes zeros instead
template <int BYTES>
__device__ __forceinline__ void cp_async_zfill(uint32_t dst_smem, const void* src_gmem, unsigned src_bytes) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], %2, %3;" ::"r"(dst_smem), "l"(src_gmem), "n"(BYTES),
                 "r"(src_bytes)
                 : "memory");
}
template <int BYTES>
__device__ __forceinline__ void cp_async(uint32_t dst_smem, const void* src_gmem) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], %2;" ::"r"(dst_smem), "l"(src_gmem), "n"(BYTES) : "memory");
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

// Column blocks.  The Ntheta columns are cut into granules of gran * R columns (gran lanes of the theta stage; gran =
// elements per 16 bytes makes every block start on a 16-byte boundary, gran = 1 is the finest split) and the
// granules are dealt out evenly: block c of `cols` gets granules [c U / cols, (c + 1) U / cols), at most 32 lanes.
// Only the last block can end inside a lane.
__host__ __device__ inline int fused_block_cols(int ntheta, int R, int gran) {
    const int U = (ntheta + R * gran - 1) / (R * gran);
    const int per = 32 / gran;
    return (U + per - 1) / per;
}
__host__ __device__ inline void fused_block_range(int c, int cols, int ntheta, int R, int gran, int* i0, int* width) {
    const long long U = (ntheta + R * gran - 1) / (R * gran);
    const int u0 = (int)((long long)c * U / cols), u1 = (int)((long long)(c + 1) * U / cols);
    const int e = u1 * R * gran < ntheta ? u1 * R * gran : ntheta;
    *i0 = u0 * R * gran;
    *width = e - u0 * R * gran;
}

template <typename T, int NST, int NT, int R, int NSTG>
__global__ void __launch_bounds__(NT, 1) strang_fused_kernel(const FusedArgs<T> arg) {
    using C = FusedCfg<T, NST, NT, R, NSTG>;
    constexpr int RB = C::RB, NTAP = C::NTAP, NTA = C::NTA, WST = C::WST, EPV = C::EPV, OB = C::OB, NW = C::NW;
    constexpr unsigned FULL = 0xffffffffu;

    extern __shared__ __align__(128) unsigned char smem_raw[];
    T* slots = reinterpret_cast<T*>(smem_raw);                                        // [NSTG][RB][NT]
    double* wsm = reinterpret_cast<double*>(smem_raw + C::SLOTS_BYTES);               // [NSTG][RB][WST]
    T* obuf = reinterpret_cast<T*>(smem_raw + C::SLOTS_BYTES + C::W_BYTES);           // [NW][2][OB]

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int ntheta = arg.ntheta, np = arg.np;
    int i0, qmax;
    fused_block_range((int)blockIdx.x, (int)gridDim.x, ntheta, R, arg.gran, &i0, &qmax);
    const int band = blockIdx.y;
    const int jA = band * arg.rows_per_band;
    const int jB = min(np, jA + arg.rows_per_band);
    if (jA >= jB || qmax <= 0) return;  // whole CTA
    const int nph = (jB - jA + RB - 1) / RB;
    const bool p_periodic = (arg.bc_p == BC_PERIODIC);

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
    const unsigned pitch = (unsigned)ntheta;

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

    const uint32_t slots_u32 = ptx::smem_u32(slots) + (uint32_t)tid * (uint32_t)sizeof(T);
    const uint32_t wsm_u32 = ptx::smem_u32(wsm) + (uint32_t)tid * 16u;

    // new taps of the RB rows of phase ph (and the weight rows of its theta stage) -> ring slot `slot`
    auto issue_stage = [&](int ph, int slot) {
        const uint32_t dst = slots_u32 + (uint32_t)slot * (uint32_t)(C::SLOT_ELEMS * sizeof(T));
        if (active) {
            if (rn >= 0 && rn + RB <= np) {  // all RB rows exist: no per-row tests
                const T* src = col + (long long)rn * (long long)pitch;
#pragma unroll
                for (int r = 0; r < RB; ++r)
                    ptx::cp_async<(int)sizeof(T)>(dst + (uint32_t)(r * NT * sizeof(T)),
                                                  src + (size_t)((unsigned)r * pitch));
                rn += RB;
                if (p_periodic && rn >= np) rn = 0;
            } else {
#pragma unroll
                for (int r = 0; r < RB; ++r) {
                    const bool ok = p_periodic || (unsigned)rn < (unsigned)np;
                    const T* src = ok ? col + (size_t)rn * pitch : arg.fin;
                    ptx::cp_async_zfill<(int)sizeof(T)>(dst + (uint32_t)(r * NT * sizeof(T)), src,
                                                        ok ? (unsigned)sizeof(T) : 0u);
                    ++rn;
                    if (p_periodic && rn >= np) rn = 0;
                }
            }
        }
        if (tid < C::W_COPIES) {  // the table has RB rows of padding after row Np - 1
            const char* wsrc = reinterpret_cast<const char*>(arg.wtab + (size_t)(jA + ph * RB) * WST) + tid * 16;
            ptx::cp_async<16>(wsm_u32 + (uint32_t)slot * (uint32_t)(RB * WST * sizeof(double)), wsrc);
        }
    };

#pragma unroll
    for (int st = 0; st < NSTG - 1; ++st) {
        if (st < nph) issue_stage(st, st);
        ptx::cp_async_commit();
    }

    double csum[R];
#pragma unroll
    for (int k = 0; k < R; ++k) csum[k] = 0.0;
    const int nv = max(0, min(R, qmax - lane * R));  // valid outputs of this lane
    int curS = 0;
    bool have = false;
    int ob = 0;
    double* __restrict__ cpw = arg.colpart ? arg.colpart + ((size_t)band * NW + warp) * (size_t)ntheta : nullptr;

    int slot = 0;
    for (int ph = 0; ph < nph; ++ph) {
        const int jph = jA + ph * RB;
        ptx::cp_async_wait<NSTG - 2>();  // this thread's copies of phase ph have landed

        // ---- p stage: ten FMAs per row from the register ring, result in place
        if (active) {
            T* sl = slots + (size_t)slot * C::SLOT_ELEMS + tid;
#pragma unroll
            for (int r = 0; r < RB; ++r) {
                v[(r + 9) % 12] = sl[r * NT];
                T acc = w[0] * v[r % 12];
#pragma unroll
                for (int m = 1; m < 10; ++m) acc = fma(w[m], v[(r + m) % 12], acc);
                sl[r * NT] = acc;
            }
        }
        __syncthreads();  // rows of phase ph complete; every warp has finished the theta stage of phase ph - 1

        {
            int nslot = slot + NSTG - 1;
            if (nslot >= NSTG) nslot -= NSTG;  // the slot of phase ph - 1
            if (ph + NSTG - 1 < nph) issue_stage(ph + NSTG - 1, nslot);
            ptx::cp_async_commit();
        }

        // ---- theta stage + store + column sums: warp = row
        const int j = jph + warp;
        if (j < jB) {
            const double* Wr = wsm + ((size_t)slot * RB + warp) * WST;
            const int S = (int)Wr[NTAP];
            if (!have) {
                curS = S;
                have = true;
            }
            while (curS > S) {  // the output window moves one column to the right
                const double first = csum[0];
                if (lane == 0 && cpw != nullptr) ptx::red_add_f64(cpw + wrap_index(i0 - curS, ntheta), first);
                double in = __shfl_down_sync(FULL, first, 1);
                if (lane == 31) in = 0.0;
#pragma unroll
                for (int k = 0; k + 1 < R; ++k) csum[k] = csum[k + 1];
                csum[R - 1] = in;
                --curS;
            }

            const T* grow = slots + (size_t)slot * C::SLOT_ELEMS + warp * NT + lane * R;
            T x[R + NTAP - 1];
#pragma unroll
            for (int k = 0; k < R + NTAP - 1; ++k) x[k] = grow[k];
            T out[R];
            {
                const T W0 = (T)Wr[0];
#pragma unroll
                for (int r = 0; r < R; ++r) out[r] = W0 * x[r];
            }
#pragma unroll
            for (int n = 1; n < NTAP; ++n) {
                const T Wn = (T)Wr[n];
#pragma unroll
                for (int r = 0; r < R; ++r) out[r] = fma(Wn, x[r + n], out[r]);
            }

            if (nv == R) {
#pragma unroll
                for (int r = 0; r < R; ++r) csum[r] += (double)out[r];
            } else if (nv > 0) {
#pragma unroll
                for (int r = 0; r < R; ++r)
                    if (r < nv) csum[r] += (double)out[r];
            }

            // the tile used two rows ago must have been read by the copy engine
            if (lane == 0) ptx::bulk_wait_read<1>();
            __syncwarp();
            T* O = obuf + (size_t)(warp * 2 + (ob & 1)) * OB;
            ++ob;
            const int base = wrap_index(i0 - S, ntheta);  // output column of q = 0
            T* __restrict__ orow = arg.fout + (size_t)j * pitch;
            if (arg.bulk_ok) {
                const int al = base & (EPV - 1);
#pragma unroll
                for (int r = 0; r < R; ++r) O[al + lane * R + r] = out[r];
                ptx::fence_proxy_async_smem();
                __syncwarp();
                // q in [qb, qb + len) -> columns [gcol, gcol + len): aligned body by the copy engine, edges by lanes
                auto store_piece = [&](int qb, int len, int gcol) {
                    T* dst = orow + gcol;
                    const T* src = O + al + qb;
                    const int h = min(len, (EPV - (gcol & (EPV - 1))) & (EPV - 1));
                    const int nb = (len - h) & ~(EPV - 1);
                    const int t0 = h + nb;
                    if (lane < h) dst[lane] = src[lane];
                    if (lane < len - t0) dst[t0 + lane] = src[t0 + lane];
                    if (lane == 0 && nb > 0) ptx::bulk_s2g(dst + h, src + h, (unsigned)(nb * sizeof(T)));
                };
                const int qa = min(qmax, ntheta - base);
                store_piece(0, qa, base);
                if (qa < qmax) store_piece(qa, qmax - qa, 0);
                if (lane == 0) ptx::bulk_commit();
            } else {
#pragma unroll
                for (int r = 0; r < R; ++r) O[lane * R + r] = out[r];
                __syncwarp();
                for (int q = lane; q < qmax; q += 32) {
                    int i = base + q;
                    if (i >= ntheta) i -= ntheta;
                    orow[i] = O[q];
                }
            }
        }
        if (++slot == NSTG) slot = 0;
    }
    if (lane == 0) ptx::bulk_wait_read<0>();

    if (cpw != nullptr && have) {
#pragma unroll
        for (int r = 0; r < R; ++r)
            if (r < nv && csum[r] != 0.0) ptx::red_add_f64(cpw + wrap_index(i0 + lane * R + r - curS, ntheta), csum[r]);
    }
}

}  // namespace vl
