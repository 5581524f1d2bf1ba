// vlasov_tile.cuh -- the one-pass Strang step (vlasov_fused.cuh: momentum shift, NST theta half shifts, density) for
// SMALL grids, whose state lives in L2 (cfg 1: 256^2, cfg 2: 1024^2; at small sizes the run time is
// latency, not work).
//
// strang_fused_ws_kernel marches one CTA per SM down a long band through a three-deep ring: on a 256^2 or 1024^2 grid that
// is a chain of latencies (first taps, two copy groups, three groups of twelve rows, ...) of about 19 us per pass whatever
// the size.  Here a CTA owns a TILE of NR = 16 (or 8, or 12) rows x (32 lanes x R = 7 (or 11)) output columns and does the pass in three short
// phases with two block-wide barriers; a grid of several hundred such CTAs covers the grid in one or two waves:
//   p stage      thread = source column (TC + NTAP - 1 of them).  All NR + 9 taps of the column are loaded at once (they
//                come from L2; adjacent lanes read adjacent columns), then NR outputs of ten FMAs each (eq (11))
//                go to shared memory.
//   theta stage  warp = row, lane = R consecutive outputs from a window of R + NTAP - 1 values (lane stride R, odd:
//                conflict-free), the NTAP weights of the row (W = w * w for NST = 2, eqs (12) and (9) at once) from the
//                same tables as the big kernel; the row overwrites its source in shared memory and is stored with plain
//                coalesced stores at column i0 + q - S (mod Ntheta), S the integer shift of the row.
//   density      thread = output column of the tile: adds the NR rows (each at its own offset S_first - S_r) and adds the
//                sum to colpart[band][column] (red.global.add: at most two tiles touch an entry, onto zero, so the result
//                does not depend on the order; eq (10)).
// The arithmetic of both shifts is the same sequence of operations as in strang_fused_ws_kernel (the results agree bit
// for bit, fp32 in difference form included); only periodic theta axes are built.
#pragma once
#include "vlasov_fused.cuh"

namespace vl {

template <typename T, int NST, int NR_, int R_>
struct TileCfg {
    static constexpr int NR = NR_;                 // rows per tile: 16, or 8 on the smallest grids (more CTAs: cfg 1 10.3 -> 9.3 us
                                                   // per step; sweep of 8 / 16 / 24 / 32 in profiles/README.md)
    static constexpr int MINB = R_ <= 7 ? 3 : 2;   // CTAs per SM the register budget is set for (256 threads x 3, 384 x 2: <= 85 registers)
    static constexpr int R = R_;                   // outputs per lane: 7 (256 threads), or 11 (384 threads) on grids of about 1024^2,
                                                   // where fewer, larger tiles win (cfg 2 14.4 -> 13.4 us per step; 2048^2: 35.1 against 32.8)
    static constexpr int TC = 32 * R;              // output columns per tile (at most)
    static constexpr int NTAP = NST == 2 ? 19 : 10;
    static constexpr int NTA = TC + NTAP - 1;      // source columns
    static constexpr int NT = (TC + NTAP - 1 + 31) / 32 * 32;  // threads: one per source column (256 for R = 7)
    static constexpr int NW = NT / 32;
    static constexpr int GP = NTA | 1;             // row pitch of the tile in shared memory
    static constexpr int WST = NST == 2 ? 20 : WROW_STRIDE;
    static constexpr size_t W_OFF = ((size_t)NR * GP * sizeof(T) + 15) / 16 * 16;  // weight rows behind the tile
    static constexpr size_t SMEM_BYTES = W_OFF + (size_t)NR * WST * sizeof(double);
    static_assert(NTA <= NT, "one thread per source column");
    // (NR need not be a multiple of NW: warps beyond the rows idle in the theta stage)
};

template <typename T, int NST, int NR_, int R_>
__global__ void __launch_bounds__(TileCfg<T, NST, NR_, R_>::NT, TileCfg<T, NST, NR_, R_>::MINB) strang_tile_kernel(const FusedArgs<T> arg) {
    using C = TileCfg<T, NST, NR_, R_>;
    constexpr int NR = C::NR, R = C::R, NTAP = C::NTAP, NTA = C::NTA, GP = C::GP, WST = C::WST;
    extern __shared__ __align__(16) unsigned char tile_smem[];
    T* g = reinterpret_cast<T*>(tile_smem);                    // [NR][GP] rows after the momentum shift, then the outputs
    double* wsm = reinterpret_cast<double*>(tile_smem + C::W_OFF);  // [NR][WST] weight rows
    __shared__ int delta[NR];                                  // S_first - S_r

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int ntheta = arg.ntheta, np = arg.np;
    int i0, qmax;
    fused_block_range((int)blockIdx.x, (int)gridDim.x, arg.xw, R, arg.gran, &i0, &qmax, 100);
    const int jA = (int)blockIdx.y * NR;
    const int nrows = min(NR, np - jA);
    const unsigned pitch = (unsigned)ntheta;

    ptx::pdl_launch_dependents();
    // weight rows of the tile: constants of the run, fetched while the density / force kernel this pass was launched behind
    // still runs (programmatic dependent launch)
    for (int e = tid; e < nrows * WST; e += C::NT) wsm[e] = __ldg(arg.wtab + (size_t)jA * WST + e);
    ptx::pdl_wait();  // the force and f are read from here on

    // ---- p stage ----
    if (tid < NTA) {
        const int c = wrap_index(i0 - 4 * NST + tid, ntheta);
        double sf, a;
        split_shift(-(arg.force[c] * arg.dt) / arg.dp, &sf, &a);
        const bool p_periodic = (arg.bc_p == BC_PERIODIC);
        int s;
        if (p_periodic) {
            sf = fmod(sf, (double)np);
            s = (int)sf;
            if (s < 0) s += np;
        } else {
            const double lim = (double)np + 64.0;
            s = (int)fmin(fmax(sf, -lim), lim);
        }
        double wd[10];
        spline_fd8_weights(a, wd);
        T w[10];
        if constexpr (sizeof(T) == 4) {  // fp32 arithmetic: difference form (diff_form_weights), as in the big kernel
            double U[9];
            diff_form_weights(wd, 10, FD_C, U);
#pragma unroll
            for (int m = 0; m < 9; ++m) w[m] = (T)U[m];
            w[9] = T(0);
        } else {
#pragma unroll
            for (int m = 0; m < 10; ++m) w[m] = (T)wd[m];
        }
        const T* col = arg.fin + c;
        int rn = jA + s - 4;
        if (p_periodic) rn = wrap_index(rn, np);
        T v[NR + 9];
        if (rn >= 0 && rn + NR + 9 <= np) {  // all taps exist and do not wrap (the usual column): no per-row tests
            const T* p0 = col + (size_t)rn * pitch;
#pragma unroll
            for (int m = 0; m < NR + 9; ++m) v[m] = __ldg(p0 + (size_t)((unsigned)m * pitch));
        } else {
#pragma unroll
            for (int m = 0; m < NR + 9; ++m) {
                const bool ok = p_periodic || (unsigned)rn < (unsigned)np;
                v[m] = ok ? __ldg(col + (size_t)rn * pitch) : T(0);
                ++rn;
                if (p_periodic && rn >= np) rn = 0;
            }
        }
        if constexpr (sizeof(T) == 4) {
            T e[NR + 8];
#pragma unroll
            for (int m = 0; m < NR + 8; ++m) e[m] = v[m + 1] - v[m];
#pragma unroll
            for (int r = 0; r < NR; ++r) {
                T acc = v[r + FD_C];
#pragma unroll
                for (int m = 0; m < 9; ++m) acc = fma(w[m], e[r + m], acc);
                g[r * GP + tid] = acc;
            }
        } else {
#pragma unroll
            for (int r = 0; r < NR; ++r) {
                T acc = w[0] * v[r];
#pragma unroll
                for (int m = 1; m < 10; ++m) acc = fma(w[m], v[r + m], acc);
                g[r * GP + tid] = acc;
            }
        }
    }
    __syncthreads();

    // ---- theta stage ----
    const int S0 = (int)wsm[NTAP];  // shift of the first row (the largest: S does not increase with the row)
    double* const rowmom = arg.rowmom;
    const double* const cos_t = arg.cos_t;
    const double* const sin_t = arg.sin_t;
    T* const fout = arg.fout;
    int base0 = wrap_index(i0 - S0, ntheta);  // output column of q = 0 in the first row; later rows: + (S0 - S)
    for (int r = warp; r < nrows; r += C::NW) {
        const double* Wr = wsm + r * WST;
        T* grow = g + r * GP;
        T x[R + NTAP - 1];
#pragma unroll
        for (int k = 0; k < R + NTAP - 1; ++k) x[k] = grow[lane * R + k];
        T out[R];
        if constexpr (sizeof(T) == 4) {  // difference form: the table holds U_0 .. U_{NTAP-2}, centre tap CT
            constexpr int CT = NST == 2 ? 2 * FD_C + 1 : FD_C;
            T d[R + NTAP - 2];
#pragma unroll
            for (int k = 0; k < R + NTAP - 2; ++k) d[k] = x[k + 1] - x[k];
#pragma unroll
            for (int q = 0; q < R; ++q) out[q] = x[q + CT];
#pragma unroll
            for (int n = 0; n < NTAP - 1; ++n) {
                const T Wn = (T)Wr[n];
#pragma unroll
                for (int q = 0; q < R; ++q) out[q] = fma(Wn, d[q + n], out[q]);
            }
        } else {
            {
                const T W0 = (T)Wr[0];
#pragma unroll
                for (int q = 0; q < R; ++q) out[q] = W0 * x[q];
            }
#pragma unroll
            for (int n = 1; n < NTAP; ++n) {
                const T Wn = (T)Wr[n];
#pragma unroll
                for (int q = 0; q < R; ++q) out[q] = fma(Wn, x[q + n], out[q]);
            }
        }
        const int S = (int)Wr[NTAP];
        __syncwarp();  // every lane has its window
#pragma unroll
        for (int q = 0; q < R; ++q) grow[lane * R + q] = out[q];
        if (lane == 0) delta[r] = S0 - S;
        __syncwarp();
        int base = base0 + (S0 - S);  // = wrap(i0 - S): S0 - S >= 0 stays below one turn inside a tile (configure_tile)
        if (base >= ntheta) base -= ntheta;
        T* orow = fout + (size_t)(jA + r) * pitch;
        double r0 = 0.0, rc = 0.0, rs = 0.0;
#pragma unroll
        for (int k = 0; k < R; ++k) {
            const int q = lane + 32 * k;
            if (q < qmax) {
                int i = base + q;
                if (i >= ntheta) i -= ntheta;
                const T vo = grow[q];
                orow[i] = vo;
                const double v = (double)vo;
                if (rowmom != nullptr) {  // history on the one-pass path: the row's sum and first Fourier sums
                    r0 += v;
                    rc = fma(v, __ldg(cos_t + i), rc);
                    rs = fma(v, __ldg(sin_t + i), rs);
                }
            }
        }
        if (rowmom != nullptr) {
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                r0 += __shfl_down_sync(0xffffffffu, r0, o);
                rc += __shfl_down_sync(0xffffffffu, rc, o);
                rs += __shfl_down_sync(0xffffffffu, rs, o);
            }
            if (lane == 0) {
                double* rm = rowmom + ((size_t)blockIdx.x * (size_t)np + (size_t)(jA + r)) * 3;
                rm[0] = r0;
                rm[1] = rc;
                rm[2] = rs;
            }
        }
    }
    if (arg.colpart == nullptr) return;
    __syncthreads();

    // ---- density partials of the tile: output column u (relative to i0 - S0) sums row r at q = u - delta[r] ----
    const int dmax = delta[nrows - 1];
    double* cp = arg.colpart + (size_t)blockIdx.y * (size_t)ntheta;
    const int cb = wrap_index(i0 - S0, ntheta);
    for (int u = tid; u < qmax + dmax; u += C::NT) {
        double acc = 0.0;
        for (int r = 0; r < nrows; ++r) {
            const int q = u - delta[r];
            if (q >= 0 && q < qmax) acc += (double)g[r * GP + q];
        }
        ptx::red_add_f64(cp + wrap_index(cb + u, ntheta), acc);
    }
}

}  // namespace vl
