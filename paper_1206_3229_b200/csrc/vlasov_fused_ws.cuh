// vlasov_fused_ws.cuh -- the one-pass Strang kernel (see vlasov_fused.cuh for the method and the geometry) with
// WARP SPECIALISATION: the momentum shift and the theta shifts run concurrently on different warps of the CTA.
//
//   p warps (4, one warpgroup, setmaxnreg 152)
//       thread t owns the three source columns t, t + 128, t + 256 of the CTA.  For each column a register window
//       slides down (one new value + ten FMAs per row, eq (11)); new values arrive by per-thread cp.async
//       into a ring of NSTG groups of 12 rows; the shifted value overwrites the tap in place.  After every 2 rows
//       ("sub-slot") the warp arrives on the sub-slot's READY mbarrier.  Before refilling a group it waits for
//       the EMPTY mbarriers of its three sub-slots.
//   theta warps (NTW = 12, three warpgroups, setmaxnreg 120; 8 at 176 registers also builds)
//       warp w takes the rows r = w (mod NTW) of the band: waits READY of the row's sub-slot, pulls its window of
//       the row into registers (in two halves: fewer values alive), arrives on EMPTY (the ring row is free again),
//       applies the NTAP composite theta weights (eqs (12), (9)), keeps the column sums (eq (10)) and hands the row
//       to the bulk-copy engine through a private tile.  The weights of its next row are prefetched (cp.async)
//       into a private two-entry buffer.
// No block-wide barrier after the set-up: the fp64 pipe sees a p warp and three theta warps per scheduler instead
// of warps that all load, all multiply and all store in step.
//
// Tried and measured slower on B200 (8192^2 fp64, us per pass; this version: 258): plain coalesced stores instead
// of the bulk copy (289); ring depth 2 (285) / 4 and 5 with > 186 KB of shared memory (316, 369: less L1 for the
// copies in flight); the theta threads issuing the tap copies with a FULL mbarrier (265: the theta warps are the
// critical path, the p warps have slack); that plus pairs of columns per 16-byte copy (313: the fallback path of a
// pair with different shifts diverges the warp); column sums in a rotating register ring instead of moving them
// (280: the dispatch on the rotation costs more than the moves).  Without the theta FMAs the pass takes 203 us,
// without the p FMAs 255 us: the theta warps' serial work per row is what bounds the kernel.
#pragma once
#include <type_traits>

#include "vlasov_fused.cuh"

namespace vl {

#ifndef VL_FW_NOB
#define VL_FW_NOB 1
#endif
template <typename T, int NST, int R, int NSTG, int NTW_ = 8, bool ZX = false>
struct FusedWsCfg {
    static constexpr int NOB = VL_FW_NOB;               // output tiles per theta warp
#ifndef VL_FW_NPW
#define VL_FW_NPW 4
#endif
    static constexpr int NPW = VL_FW_NPW, NTW = NTW_;    // p warps (whole warpgroups), theta warps (two or three warpgroups)
    static constexpr int NT = (NPW + NTW) * 32;
    static constexpr int NPT = NPW * 32;                // p threads
    // columns per p thread: three register rings of doubles fit the p warps' 152 registers, four of floats (a ring row of 512
    // columns then feeds R = 15 outputs per theta lane: fewer window loads and less per-row work per grid point)
#ifdef VL_FW_CPT
    static constexpr int CPT = VL_FW_CPT;
#else
    static constexpr int CPT = sizeof(T) == 4 ? 4 : 3;
#endif
    static constexpr int PITCH = NPT * CPT;             // columns of a ring row
    static constexpr int RG = 12;                       // rows per group = length of the register ring
#ifndef VL_FW_SUB
#define VL_FW_SUB 2
#endif
    static constexpr int SUB = VL_FW_SUB;               // rows per sub-slot (granularity of READY / EMPTY)
    static constexpr int SPG = RG / SUB;                // sub-slots per group
    static constexpr int NSUB = NSTG * SPG;
    static constexpr int NTAP = NST == 2 ? 19 : 10;
    // weight row: NST = 1: w_0..w_9, s, -;  NST = 2: W_0..W_18, 2 s, and for a zero-extended theta axis (ZX) also the ten
    // weights of ONE half shift and its s (entries 20..30): the rows near the ends of the axis apply the two half shifts
    // one after the other, because the first one is cropped to [0, Ntheta) before the second reads it
    static constexpr int WST = NST == 2 ? (ZX ? 32 : 20) : WROW_STRIDE;
    static constexpr int TI = 32 * R;
    static constexpr int NTA = TI + NTAP - 1;
    static constexpr int EPV = 16 / (int)sizeof(T);
    static constexpr int OB = (TI + EPV + EPV - 1) / EPV * EPV;
    static constexpr size_t RING_BYTES = (size_t)NSTG * RG * PITCH * sizeof(T);
    static constexpr size_t O_BYTES = (size_t)NTW * NOB * OB * sizeof(T);
    static constexpr size_t W_BYTES = (size_t)NTW * 2 * WST * sizeof(double);
    static constexpr size_t BAR_BYTES = (size_t)2 * NSUB * sizeof(uint64_t);
    static constexpr size_t SMEM_BYTES = RING_BYTES + O_BYTES + W_BYTES + BAR_BYTES;
    static constexpr int W_COPIES = WST * 8 / 16;
    static_assert(NTA <= PITCH, "source columns must fit the ring row");
    static_assert(R & 1, "lane stride R must be odd (shared-memory banks)");
    static_assert(NTW % SUB == 0 && NTW <= RG, "a sub-slot is released by SUB different theta warps");
    // registers per thread after setmaxnreg: 128*152 + 384*120 = 65536; 128*152 + 256*176 = 64512
#ifndef VL_FW_PREGS
#define VL_FW_PREGS 152
#define VL_FW_TREGS 120
#endif
    static constexpr int P_REGS = VL_FW_PREGS, T_REGS = VL_FW_TREGS;
    static constexpr int LAUNCH_REGS = 65536 / NT / 8 * 8;
    static_assert(NPW * 32 * P_REGS + NTW * 32 * T_REGS <= 65536 && P_REGS % 8 == 0 && T_REGS % 8 == 0, "");
    static_assert(RING_BYTES % 16 == 0 && O_BYTES % 16 == 0 && W_BYTES % 16 == 0, "");
    static_assert(NSTG >= 2 && W_COPIES <= 32, "");
};

template <typename T, int NST, int R, int NSTG, int NTW_, bool ZX>
__global__ void __launch_bounds__(FusedWsCfg<T, NST, R, NSTG, NTW_, ZX>::NT, 1) strang_fused_ws_kernel(const FusedArgs<T> arg) {
    using C = FusedWsCfg<T, NST, R, NSTG, NTW_, ZX>;
    constexpr int NTAP = C::NTAP, NTA = C::NTA, WST = C::WST, EPV = C::EPV, OB = C::OB, PITCH = C::PITCH, RG = C::RG,
                  SUB = C::SUB, SPG = C::SPG, NSUB = C::NSUB, CPT = C::CPT, NPT = C::NPT, NTW = C::NTW;
    constexpr unsigned FULL = 0xffffffffu;

    extern __shared__ __align__(128) unsigned char smem_raw[];
    T* ring = reinterpret_cast<T*>(smem_raw);                                                  // [NSTG][RG][PITCH]
    T* obuf = reinterpret_cast<T*>(smem_raw + C::RING_BYTES);                                  // [NTW][2][OB]
    double* wbuf = reinterpret_cast<double*>(smem_raw + C::RING_BYTES + C::O_BYTES);           // [NTW][2][WST]
    uint64_t* ready = reinterpret_cast<uint64_t*>(smem_raw + C::RING_BYTES + C::O_BYTES + C::W_BYTES);  // [NSUB]
    uint64_t* empty = ready + NSUB;                                                            // [NSUB]

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int ntheta = arg.ntheta, np = arg.np;
    int i0, qmax;
    fused_block_range((int)blockIdx.x, (int)gridDim.x, arg.xw, R, arg.gran, &i0, &qmax, arg.edge_w);
    i0 += arg.x0;  // ZX: may be negative or reach beyond Ntheta (source columns out there are zeros)
    const int band = blockIdx.y;
    const int jA = band * arg.rows_per_band;
    const int nrows = min(np, jA + arg.rows_per_band) - jA;
    if (nrows <= 0 || qmax <= 0) return;  // whole CTA
    const int ngroups = (nrows + RG - 1) / RG;
    const unsigned pitch = (unsigned)ntheta;

    ptx::pdl_launch_dependents();  // the density / force kernel that follows may be scheduled while this pass runs
    if (tid == 0) {
#pragma unroll
        for (int k = 0; k < NSUB; ++k) {
            ptx::mbar_init(&ready[k], C::NPW);
            ptx::mbar_init(&empty[k], SUB);
        }
        ptx::fence_mbar_init();
    }
    if constexpr (ZX) {
        // zero extension in theta: the source columns of this CTA outside [0, Ntheta) are zeros.  Their ring columns are
        // zero-filled here, once, by everybody; the p threads that own them issue no copies and compute 0 from 0.
        const int cl = i0 - 4 * NST;  // column of q = 0
        const int nlo = min(NTA, max(0, -cl)), nhi = min(NTA, max(0, cl + NTA - ntheta));
        for (int e = tid; e < NSTG * RG * (nlo + nhi); e += C::NT) {
            const int r = e / (nlo + nhi), qq = e - r * (nlo + nhi);
            ring[(size_t)r * PITCH + (qq < nlo ? qq : NTA - nhi + (qq - nlo))] = T(0);
        }
    }
    __syncthreads();
    // everything above is independent of the force and of f; from here on both are read (and the density partials
    // written): wait for the density / force kernel this pass was launched behind (programmatic dependent launch)
    ptx::pdl_wait();
    const uint32_t ready_u32 = ptx::smem_u32(ready), empty_u32 = ptx::smem_u32(empty);

    if (warp < C::NPW) {
        if (C::P_REGS > C::LAUNCH_REGS) asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(C::P_REGS));
        else asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(C::P_REGS));
        // =========================== p warps: momentum shift (eq (11)) ===========================
        const bool p_periodic = (arg.bc_p == BC_PERIODIC);
        bool act[CPT];
        const T* col[CPT];
        int rn[CPT];
        T w[CPT][10];
        T v[CPT][12];  // register rings: taps of output row r of a group are v[k][(r + m) % 12]
        // SC (fp64): the rings hold PARTIAL SUMS instead: v[k][(r + j) % 12], j = 0..8, is output row r + j with its taps
        // m = 0..8-j added.  A new tap then feeds ten independent FMAs that share it as an operand (no dependent chain, one
        // operand from the reuse cache), in the same order per output as the gather form: bit-identical results, 3 % off
        // the pass (8192^2: 0.2667 -> 0.2581 ms per step in the same session)
        constexpr bool SC = sizeof(T) == 8;
        T e[sizeof(T) == 4 ? CPT : 1][12];  // fp32 arithmetic (difference form): e[k][i] = v[k][i + 1] - v[k][i]
#pragma unroll
        for (int k = 0; k < CPT; ++k) {
            const int q = tid + k * NPT;
            act[k] = q < NTA;
            int c = i0 - 4 * NST + q;
            if constexpr (ZX) {  // zero extension in theta: columns outside [0, Ntheta) are zeros and stay zeros
                if ((unsigned)c >= (unsigned)ntheta) act[k] = false;
                c = act[k] ? c : 0;
            } else {
                c = wrap_index(c, ntheta);
            }
            double sf, a;
            split_shift(-((act[k] ? arg.force[c] : 0.0) * arg.dt) / arg.dp, &sf, &a);
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
            if (sizeof(T) == 4) {  // difference-form weights U_0..U_8 (diff_form_weights)
                double U[9];
                diff_form_weights(wd, 10, FD_C, U);
#pragma unroll
                for (int m = 0; m < 9; ++m) w[k][m] = (T)U[m];
                w[k][9] = T(0);
            } else {
#pragma unroll
                for (int m = 0; m < 10; ++m) w[k][m] = (T)wd[m];
            }
            col[k] = arg.fin + c;
            // row of tap m of output row j is j + s + m - 4; rn = row of the next value the window has not seen
            rn[k] = jA + s - 4;
            if (p_periodic) rn[k] = wrap_index(rn[k], np);
        }
#pragma unroll
        for (int k = 0; k < CPT; ++k) {
#pragma unroll
            for (int m = 0; m < 9; ++m) {
                const bool ok = act[k] && (p_periodic || (unsigned)rn[k] < (unsigned)np);
                v[k][m] = ok ? __ldg(col[k] + (size_t)rn[k] * pitch) : T(0);
                ++rn[k];
                if (p_periodic && rn[k] >= np) rn[k] = 0;
            }
            v[k][9] = v[k][10] = v[k][11] = T(0);
            if constexpr (SC) {  // scatter form: turn the nine taps into the partial sums of output rows 0..8
                T t[9];
#pragma unroll
                for (int i = 0; i < 9; ++i) t[i] = v[k][i];
#pragma unroll
                for (int i = 0; i < 9; ++i) {
#pragma unroll
                    for (int j = 0; j <= i; ++j) v[k][j] = (i == j) ? w[k][0] * t[i] : fma(w[k][i - j], t[i], v[k][j]);
                }
            }
            if constexpr (sizeof(T) == 4) {
#pragma unroll
                for (int m = 0; m < 12; ++m) e[k][m] = m < 8 ? v[k][m + 1] - v[k][m] : T(0);
            }
        }

        const uint32_t ring_u32 = ptx::smem_u32(ring) + (uint32_t)tid * (uint32_t)sizeof(T);
        // new taps of the RG rows of a group -> ring slot `slot`
        auto issue_group = [&](int slot) {
            const uint32_t dst0 = ring_u32 + (uint32_t)slot * (uint32_t)(RG * PITCH * sizeof(T));
#pragma unroll
            for (int k = 0; k < CPT; ++k) {
                if (!act[k]) continue;
                const uint32_t dst = dst0 + (uint32_t)(k * NPT * sizeof(T));
                if (rn[k] >= 0 && rn[k] + RG <= np) {  // all RG rows exist: no per-row tests
                    const T* src = col[k] + (long long)rn[k] * (long long)pitch;
#pragma unroll
                    for (int r = 0; r < RG; ++r)
                        ptx::cp_async<(int)sizeof(T)>(dst + (uint32_t)(r * PITCH * sizeof(T)),
                                                      src + (size_t)((unsigned)r * pitch));
                    rn[k] += RG;
                    if (p_periodic && rn[k] >= np) rn[k] = 0;
                } else {
#pragma unroll
                    for (int r = 0; r < RG; ++r) {
                        const bool ok = p_periodic || (unsigned)rn[k] < (unsigned)np;
                        const T* src = ok ? col[k] + (size_t)rn[k] * pitch : arg.fin;
                        ptx::cp_async_zfill<(int)sizeof(T)>(dst + (uint32_t)(r * PITCH * sizeof(T)), src,
                                                            ok ? (unsigned)sizeof(T) : 0u);
                        ++rn[k];
                        if (p_periodic && rn[k] >= np) rn[k] = 0;
                    }
                }
            }
        };

#pragma unroll
        for (int st = 0; st < NSTG - 1; ++st) {
            if (st < ngroups) issue_group(st);
            ptx::cp_async_commit();
        }

        int slot = 0;
        for (int g = 0; g < ngroups; ++g) {
            ptx::cp_async_wait<NSTG - 2>();  // this thread's copies of group g have landed
            T* sl = ring + (size_t)slot * (RG * PITCH) + tid;
#pragma unroll
            for (int sub = 0; sub < SPG; ++sub) {
#pragma unroll
                for (int rr = 0; rr < SUB; ++rr) {
                    const int r = sub * SUB + rr;
#pragma unroll
                    for (int k = 0; k < CPT; ++k) {  // columns beyond NTA compute on whatever the ring holds: never read
                        // (ZX: a column outside [0, Ntheta) has no copies and a zero-filled ring column: it computes 0)
                        if constexpr (SC) {
                            const T t = sl[r * PITCH + k * NPT];
#pragma unroll
                            for (int j = 0; j < 9; ++j) v[k][(r + j) % 12] = fma(w[k][9 - j], t, v[k][(r + j) % 12]);
                            v[k][(r + 9) % 12] = w[k][0] * t;
                            sl[r * PITCH + k * NPT] = v[k][r % 12];
                            continue;
                        }
                        v[k][(r + 9) % 12] = sl[r * PITCH + k * NPT];
                        T acc;
                        if constexpr (sizeof(T) == 4) {
                            e[k][(r + 8) % 12] = v[k][(r + 9) % 12] - v[k][(r + 8) % 12];
                            acc = v[k][(r + FD_C) % 12];
#pragma unroll
                            for (int m = 0; m < 9; ++m) acc = fma(w[k][m], e[k][(r + m) % 12], acc);
                        } else {
                            acc = w[k][0] * v[k][r % 12];
#pragma unroll
                            for (int m = 1; m < 10; ++m) acc = fma(w[k][m], v[k][(r + m) % 12], acc);
                        }
                        sl[r * PITCH + k * NPT] = acc;
                    }
                }
                __syncwarp();
                if (lane == 0) ptx::mbar_arrive_u32(ready_u32 + (uint32_t)((slot * SPG + sub) * 8));
            }
            // refill the slot of group g - 1 with group g + NSTG - 1 once the theta warps have let go of it
            const int gn = g + NSTG - 1;
            int nslot = slot + NSTG - 1;
            if (nslot >= NSTG) nslot -= NSTG;
            if (gn < ngroups) {
                if (gn >= NSTG) {
                    const unsigned par = (unsigned)((gn / NSTG) - 1) & 1u;
#pragma unroll
                    for (int sub = 0; sub < SPG; ++sub)
                        ptx::mbar_wait_u32(empty_u32 + (uint32_t)((nslot * SPG + sub) * 8), par);
                }
                issue_group(nslot);
            }
            ptx::cp_async_commit();
            if (++slot == NSTG) slot = 0;
        }
        ptx::cp_async_wait<0>();
        return;
    }

    // =========================== theta warps: eqs (12), (9), (10) ===========================
    if (C::T_REGS > C::LAUNCH_REGS) asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(C::T_REGS));
    else asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(C::T_REGS));
    const int tw = warp - C::NPW;  // this warp takes the band rows r = tw + NTW * it

    // everything that changes from row to row is advanced, not recomputed
    const uint32_t wb_u32 = ptx::smem_u32(wbuf) + (uint32_t)(tw * 2 * WST * 8 + lane * 16);
    const double* wb = wbuf + (size_t)tw * 2 * WST;
    const char* wsrc = reinterpret_cast<const char*>(arg.wtab + (size_t)(jA + tw) * WST) + lane * 16;  // weight row of r
    constexpr size_t WSRC_STEP = (size_t)NTW * WST * sizeof(double);
    const T* xrow0 = ring + lane * R;
    T* const O0 = obuf + (size_t)tw * C::NOB * OB;
    const uint32_t O0_u32 = ptx::smem_u32(obuf) + (uint32_t)(tw * C::NOB * OB * sizeof(T));
    T* orow = arg.fout + (size_t)(jA + tw) * pitch;
    const size_t orow_step = (size_t)NTW * pitch;
    const bool wlane = lane < C::W_COPIES;

    double csum[R];
#pragma unroll
    for (int k = 0; k < R; ++k) csum[k] = 0.0;
    const int nv = max(0, min(R, qmax - lane * R));  // valid outputs of this lane
    int curS = 0, cbase = 0;                         // shift of the rows summed so far, output column of q = 0
    bool have = false;
    double* __restrict__ cpw = arg.colpart ? arg.colpart + ((size_t)band * NTW + tw) * (size_t)ntheta : nullptr;

    // K columns leave on the left (their sums are final for this warp), K columns enter on the right
    auto shift_sums = [&](auto kc) {
        constexpr int K = decltype(kc)::value;
#pragma unroll
        for (int u = 0; u < K; ++u) {
            if (lane == 0 && cpw != nullptr) {
                int cidx = cbase + u;
                if (!ZX && cidx >= ntheta) cidx -= ntheta;
                if (!ZX || (unsigned)cidx < (unsigned)ntheta) ptx::red_add_f64(cpw + cidx, csum[u]);  // ZX: outside = dropped
            }
        }
        double in[K];
#pragma unroll
        for (int u = 0; u < K; ++u) {
            in[u] = __shfl_down_sync(FULL, csum[u], 1);
            if (lane == 31) in[u] = 0.0;
        }
#pragma unroll
        for (int k = 0; k + K < R; ++k) csum[k] = csum[k + K];
#pragma unroll
        for (int u = 0; u < K; ++u) csum[R - K + u] = in[u];
        curS -= K;
        cbase += K;
        if (!ZX && cbase >= ntheta) cbase -= ntheta;
    };

    if (tw < nrows && wlane) ptx::cp_async<16>(wb_u32, wsrc);
    ptx::cp_async_commit();

    int slot = 0, wsel = 0, rin = tw;  // row r is row `rin` of the group in ring slot `slot`
    unsigned par = 0;
    for (int r = tw; r < nrows; r += NTW) {
        wsrc += WSRC_STEP;
        if (r + NTW < nrows && wlane) ptx::cp_async<16>(wb_u32 + (uint32_t)((wsel ^ 1) * WST * 8), wsrc);
        ptx::cp_async_commit();
        ptx::cp_async_wait<1>();
        __syncwarp();  // the weight row of r is visible to every lane
        const double* Wr = wb + wsel * WST;

        const uint32_t boff = (uint32_t)((slot * SPG + rin / SUB) * 8);
        ptx::mbar_wait_u32(ready_u32 + boff, par);
        const T* grow = xrow0 + (size_t)(slot * RG + rin) * PITCH;
        // the window of the row in two halves (fewer values alive at a time): taps 0..NH-1 need x[0 .. R+NH-2]
        constexpr int NH = (NTAP + 1) / 2;
        T x[R + NTAP - 1];
#pragma unroll
        for (int k = 0; k < R + NH - 1; ++k) x[k] = grow[k];

        const int S = (int)Wr[NTAP];
        if (!have) {
            curS = S;
            cbase = ZX ? i0 - S : wrap_index(i0 - S, ntheta);
            have = true;
        }
        while (curS - S >= 2) shift_sums(std::integral_constant<int, 2>());
        if (curS > S) shift_sums(std::integral_constant<int, 1>());

        T out[R];
        bool edge_row = false;
        if constexpr (ZX && NST == 2) {
            // Zero-extended theta axis: the first half shift is cropped to [0, Ntheta) before the second reads it (the
            // oracle stores f_I on the grid), so the composite weights W = w * w are right only where no intermediate
            // value the row needs lies outside.  Intermediate column of the warp's h[j]: cbase + lane R + j + s - 4.
            const int h0 = cbase + (int)Wr[30] - FD_C;
            edge_row = h0 < 0 || h0 + 32 * R + 8 >= ntheta;
            if (edge_row) {  // warp-uniform: the two half shifts one after the other (eqs (12), (9)), cropped in between
#pragma unroll
                for (int k = R + NH - 1; k < R + NTAP - 1; ++k) x[k] = grow[k];
                __syncwarp();
                if (lane == 0) ptx::mbar_arrive_u32(empty_u32 + boff);
                T w1[10];
#pragma unroll
                for (int m = 0; m < 10; ++m) w1[m] = (T)Wr[20 + m];
                T h[R + 9];
#pragma unroll
                for (int j = 0; j < R + 9; ++j) {
                    T acc = w1[0] * x[j];
#pragma unroll
                    for (int m = 1; m < 10; ++m) acc = fma(w1[m], x[j + m], acc);
                    h[j] = (unsigned)(h0 + lane * R + j) < (unsigned)ntheta ? acc : T(0);
                }
#pragma unroll
                for (int q = 0; q < R; ++q) {
                    T acc = w1[0] * h[q];
#pragma unroll
                    for (int m = 1; m < 10; ++m) acc = fma(w1[m], h[q + m], acc);
                    out[q] = acc;
                }
            }
        }
        if (edge_row) {
        } else if constexpr (sizeof(T) == 4) {
            // fp32 arithmetic: difference form (diff_form_weights; the table holds U_0 .. U_{NTAP-2}), centre tap CT
            constexpr int CT = NST == 2 ? 2 * FD_C + 1 : FD_C;
#pragma unroll
            for (int k = R + NH - 1; k < R + NTAP - 1; ++k) x[k] = grow[k];
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive_u32(empty_u32 + boff);  // the ring row may be refilled
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
            for (int n = 1; n < NH; ++n) {
                const T Wn = (T)Wr[n];
#pragma unroll
                for (int q = 0; q < R; ++q) out[q] = fma(Wn, x[q + n], out[q]);
            }
#pragma unroll
            for (int k = R + NH - 1; k < R + NTAP - 1; ++k) x[k] = grow[k];
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive_u32(empty_u32 + boff);  // the ring row may be refilled
#pragma unroll
            for (int n = NH; n < NTAP; ++n) {
                const T Wn = (T)Wr[n];
#pragma unroll
                for (int q = 0; q < R; ++q) out[q] = fma(Wn, x[q + n], out[q]);
            }
        }

        if (nv == R) {
#pragma unroll
            for (int q = 0; q < R; ++q) csum[q] += (double)out[q];
        } else if (nv > 0) {
#pragma unroll
            for (int q = 0; q < R; ++q)
                if (q < nv) csum[q] += (double)out[q];
        }

        // hand the row to the bulk-copy engine through one of the warp's two private tiles (shared -> global,
        // 16-byte aligned body; the 0..EPV-1 elements before and after an aligned body are stored by lanes)
        if (lane == 0) ptx::bulk_wait_read<C::NOB - 1>();  // the tile about to be overwritten has been read
        __syncwarp();
        const int osel = C::NOB == 2 ? wsel : 0;
        T* O = O0 + osel * OB;
        const int base = cbase;  // output column of q = 0: wrap(i0 - S)
        if (arg.bulk_ok) {
            const int al = base & (EPV - 1);
#pragma unroll
            for (int q = 0; q < R; ++q) O[al + lane * R + q] = out[q];
            ptx::fence_proxy_async_smem();
            __syncwarp();
            const uint32_t O_u32 = O0_u32 + (uint32_t)((osel * OB + al) * sizeof(T));
            // q in [qb, qb + len) -> columns [gcol, gcol + len)
            auto store_piece = [&](int qb, int len, int gcol) {
                const int h = min(len, (EPV - (gcol & (EPV - 1))) & (EPV - 1));
                const int nb = (len - h) & ~(EPV - 1);
                const int t0 = h + nb;
                if (h | (len - t0)) {  // warp-uniform: some elements outside the aligned body
                    if (lane < h) orow[gcol + lane] = O[al + qb + lane];
                    if (lane < len - t0) orow[gcol + t0 + lane] = O[al + qb + t0 + lane];
                }
                if (lane == 0 && nb > 0)
                    ptx::bulk_s2g_u32(orow + gcol + h, O_u32 + (uint32_t)((qb + h) * sizeof(T)), (unsigned)(nb * sizeof(T)));
            };
            if constexpr (ZX) {  // the part of the row inside [0, Ntheta): one piece, the rest is dropped
                const int qlo = max(0, -base), qhi = min(qmax, ntheta - base);
                if (qhi > qlo) store_piece(qlo, qhi - qlo, base + qlo);
            } else {
                const int qa = min(qmax, ntheta - base);
                store_piece(0, qa, base);
                if (qa < qmax) store_piece(qa, qmax - qa, 0);
            }
            if (lane == 0) ptx::bulk_commit();
        } else {
#pragma unroll
            for (int q = 0; q < R; ++q) O[lane * R + q] = out[q];
            __syncwarp();
#pragma unroll
            for (int k = 0; k < R; ++k) {
                const int q = lane + 32 * k;
                if (q < qmax) {
                    int i = base + q;
                    if (!ZX && i >= ntheta) i -= ntheta;
                    if (!ZX || (unsigned)i < (unsigned)ntheta) orow[i] = O[q];
                }
            }
        }
        __syncwarp();  // every lane is done with the tile and with this row's weights
        orow += orow_step;
        wsel ^= 1;
        rin += NTW;
        if (rin >= RG) {
            rin -= RG;
            if (++slot == NSTG) {
                slot = 0;
                par ^= 1u;
            }
        }
    }
    ptx::cp_async_wait<0>();
    if (lane == 0) ptx::bulk_wait_read<0>();

    if (cpw != nullptr && have) {
#pragma unroll
        for (int q = 0; q < R; ++q) {
            if (q < nv && csum[q] != 0.0) {
                int cidx = cbase + lane * R + q;
                if (!ZX && cidx >= ntheta) cidx -= ntheta;
                if (!ZX || (unsigned)cidx < (unsigned)ntheta) ptx::red_add_f64(cpw + cidx, csum[q]);
            }
        }
    }
}

}  // namespace vl
