// vlasov_kernels.cuh -- CUDA kernels (sm_100a) of the Strang semi-Lagrangian Vlasov step.
//
// Method: arXiv 1206.3229.  One shift of a grid line by a constant displacement evaluates the
// cubic spline of eqs (13)-(14) (L89-L98) with f'' from the 9-point difference of eq (16) (L106-L111).
// Substituting (16) into (13) the h^2 cancels and the value at the foot becomes a 10-tap filter
//     f_new[i] = sum_{m=-4}^{5} w_m(a) f[i + s + m],
//     w_m = [m==0](1-a) + [m==1] a + (A c_m + B c_{m-1})/6,  A = (1-a)^3-(1-a),  B = a^3-a,
// with s the integer part and a in [0,1) the fractional part of -displacement/h.  The weights depend only on
// the line (row for the theta shift, column for the p shift), never on the position along it.
//
// Layout (L115): f[j*Ntheta + i], theta contiguous.  No transposes (the paper's steps (i), (iii), L117-L119,
// are not needed): the theta shift runs along the contiguous axis through shared memory, the p shift lets
// adjacent threads own adjacent columns and march down p with a register window.
#pragma once
#include <cooperative_groups.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "vlasov_ptx.cuh"

namespace vl {

enum { BC_PERIODIC = 0, BC_ZERO = 1 };

// per-row table of the theta half shift: {w_0..w_9, (double) s, e}; 96 bytes = one 16-byte-aligned bulk copy.
// For fp32 storage the ten entries are the nine difference-form weights U_0..U_8 (diff_form_weights) and a 0.
constexpr int WROW_STRIDE = 12;
constexpr int FD_C = 4;  // centre tap of the ten: w[FD_C] multiplies f[k]

// eq (16), divided by 6 (the 1/6 of gamma, delta in eq (14)); index m+4, m = -4..4
__host__ __device__ inline double c16_over_6(int m) {
    switch (m < 0 ? -m : m) {
        case 0: return (-205.0 / 72.0) / 6.0;
        case 1: return (8.0 / 5.0) / 6.0;
        case 2: return (-1.0 / 5.0) / 6.0;
        case 3: return (8.0 / 315.0) / 6.0;
        case 4: return (-1.0 / 560.0) / 6.0;
        default: return 0.0;
    }
}

// ten filter weights for fraction a; w[mm] multiplies f[k + mm - 4]
__host__ __device__ inline void spline_fd8_weights(double a, double w[10]) {
    const double al = 1.0 - a;
    const double A = al * (al * al - 1.0);  // alpha^3 - alpha
    const double B = a * (a * a - 1.0);     // beta^3 - beta
#pragma unroll
    for (int mm = 0; mm < 10; ++mm) {
        const int m = mm - 4;
        double v = A * c16_over_6(m) + B * c16_over_6(m - 1);
        if (m == 0) v += al;
        if (m == 1) v += a;
        w[mm] = v;
    }
}

// fp32 arithmetic runs every filter in DIFFERENCE FORM.  With n weights that add up to 1 and centre tap c,
//     sum_m w_m x_m = x_c + sum_{j=0}^{n-2} U_j (x_{j+1} - x_j),   U_j = -sum_{m<=j} w_m (j < c),  U_j = sum_{m>j} w_m (j >= c).
// Why: in the plain form the partial sums of a float accumulation are of the size of f itself and their rounding
// errors add up to more than half an ulp; on a plateau of f (the water-bags of cfg 1, 3, 4, 5) every point of a line
// then gets the SAME error, step after step (the weights of a row never change), so the mass of the line, the moments
// (M_x, M_y), the force and the feet of all characteristics drift coherently: at 8192^2 the fp32 path left north_star's
// 1e-4 max|f| after 30 steps (7.6e-4 after 100; measured in round 2).  In difference form a plateau is reproduced
// exactly (all differences are 0) and elsewhere the rounding errors scale with the local variation of f, not with f.
// fp64 keeps the plain ten-tap form (its rounding is 1e-9 of the tolerance).  U has n - 1 entries.
__host__ __device__ inline void diff_form_weights(const double* w, int n, int c, double* U) {
    double acc = 0.0;
    for (int j = 0; j < c; ++j) {
        acc -= w[j];
        U[j] = acc;
    }
    acc = 0.0;
    for (int j = n - 2; j >= c; --j) {
        acc += w[j + 1];
        U[j] = acc;
    }
}

// R consecutive outputs of an NT-tap filter from the window x[0 .. R + NT - 1): out[r] = sum_m w[m] x[r + m] (fp64), or
// in difference form with w[0 .. NT - 1) = U and centre tap C (fp32)
template <typename T, int R, int NT, int C>
__device__ __forceinline__ void fir_window(const T* w, const T* x, T* out) {
    if constexpr (sizeof(T) == 4) {
        T e[R + NT - 2];
#pragma unroll
        for (int k = 0; k < R + NT - 2; ++k) e[k] = x[k + 1] - x[k];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            T acc = x[r + C];
#pragma unroll
            for (int jj = 0; jj < NT - 1; ++jj) acc = fma(w[jj], e[r + jj], acc);
            out[r] = acc;
        }
    } else {
#pragma unroll
        for (int r = 0; r < R; ++r) {
            T acc = w[0] * x[r];
#pragma unroll
            for (int m = 1; m < NT; ++m) acc = fma(w[m], x[r + m], acc);
            out[r] = acc;
        }
    }
}

// split u = -displacement/h into integer cell shift and fraction in [0,1)
__host__ __device__ inline void split_shift(double u, double* s_out, double* a_out) {
    double sf = floor(u);
    double a = u - sf;
    if (a >= 1.0) {  // u = -tiny: floor = -1 and u + 1 rounds to 1
        sf += 1.0;
        a = 0.0;
    }
    *s_out = sf;
    *a_out = a;
}

__device__ __forceinline__ int wrap_index(int k, int n) {
    int r = k % n;
    return r < 0 ? r + n : r;
}

// ------------------------------------------------------------------------------------------------
// GENERIC theta shift (any Ntheta, any alignment; used when a row is not a multiple of 16 bytes).
// theta shift (rows, contiguous axis).  NSTAGE = 1: one half shift (eq (9) or (12)).  NSTAGE = 2: the
// half shift that ends step k followed by the one that opens step k+1, same row, same (s, w), the
// intermediate row kept in registers (halo exchanged with warp shuffles).
//
// A CTA owns a chunk of NW warp tiles of one row and walks down a band of rows, so that each thread owns
// the same R consecutive COLUMNS for every row of the band and can keep their column sums (the density
// partials, eq (10)) in registers.  Each lane reads its R+9 window from shared memory with lane stride R
// (R odd: conflict-free for 8-byte words) and produces R consecutive values with R*10 FMAs.
// ------------------------------------------------------------------------------------------------
template <typename T>
struct ThetaArgs {
    const T* fin;
    T* fout;
    const int* srow;      // [Np] integer cell shift of one half step
    const double* wrow;   // [Np][WROW_STRIDE]: ten weights of one half step, then s as a double
    double* colpart;      // [nbands][Ntheta] column sums of the OUTPUT over the band's rows (may be null)
    int ntheta, np, bc_x, rows_per_band;
};

template <typename T, int NSTAGE, int R>
__global__ void __launch_bounds__(384) theta_sweep_generic_kernel(const ThetaArgs<T> arg) {
    constexpr int LANES = (NSTAGE == 2) ? 31 : 32;  // lanes that own outputs
    constexpr int TILE = LANES * R;                 // outputs per warp
    constexpr int HALO = 9 * NSTAGE;
    constexpr int KPRE = R + 1;                     // >= ceil((NW*TILE + HALO) / (32*NW))

    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, NW = blockDim.x >> 5;
    const int chunk = NW * TILE;
    const int lenA = chunk + HALO;
    T* A = reinterpret_cast<T*>(smem_raw);
    T* O = A + ((lenA + 1) & ~1);

    const int ntheta = arg.ntheta;
    const int c0 = blockIdx.x * chunk;
    const int j0 = blockIdx.y * arg.rows_per_band;
    const int j1 = min(arg.np, j0 + arg.rows_per_band);
    const int myq = warp * TILE + lane * R;
    const int i0 = c0 + myq;
    const bool owner = (lane < LANES);
    const bool periodic = (arg.bc_x == BC_PERIODIC);

    double csum[R];
#pragma unroll
    for (int r = 0; r < R; ++r) csum[r] = 0.0;

    T pre[KPRE];
    auto prefetch = [&](int j) {
        const int S = NSTAGE * arg.srow[j];
        const T* __restrict__ row = arg.fin + (size_t)j * ntheta;
        int base = c0 + S - 4 * NSTAGE;
        if (periodic) base = wrap_index(base, ntheta);
#pragma unroll
        for (int k = 0; k < KPRE; ++k) {
            const int q = tid + k * blockDim.x;
            T v = T(0);
            if (q < lenA) {
                int src = base + q;
                if (periodic) {
                    while (src >= ntheta) src -= ntheta;
                    v = __ldg(row + src);
                } else if ((unsigned)src < (unsigned)ntheta) {
                    v = __ldg(row + src);
                }
            }
            pre[k] = v;
        }
    };
    auto stash = [&]() {
#pragma unroll
        for (int k = 0; k < KPRE; ++k) {
            const int q = tid + k * blockDim.x;
            if (q < lenA) A[q] = pre[k];
        }
    };

    if (j0 < j1) {
        prefetch(j0);
        stash();
    }
    __syncthreads();

    for (int j = j0; j < j1; ++j) {
        if (j + 1 < j1) prefetch(j + 1);  // global loads of the next row fly during this row's arithmetic

        T w[10];
        {
            const double* __restrict__ wr = arg.wrow + (size_t)j * WROW_STRIDE;
#pragma unroll
            for (int m = 0; m < 10; ++m) w[m] = (T)__ldg(wr + m);
        }
        T v[R + 9];
#pragma unroll
        for (int k = 0; k < R + 9; ++k) v[k] = A[myq + k];

        T g[R];
        fir_window<T, R, 10, FD_C>(w, v, g);

        T out[R];
        if (NSTAGE == 2) {
            if (!periodic) {  // the intermediate row is zero outside [0, Ntheta) (two separate cropped shifts)
                const int x0 = i0 + arg.srow[j] - 4;
#pragma unroll
                for (int r = 0; r < R; ++r)
                    if ((unsigned)(x0 + r) >= (unsigned)ntheta) g[r] = T(0);
            }
            T h[R + 9];
#pragma unroll
            for (int r = 0; r < R; ++r) {
                h[r] = g[r];
                h[R + r] = __shfl_down_sync(0xffffffffu, g[r], 1);
            }
            fir_window<T, R, 10, FD_C>(w, h, out);
        } else {
#pragma unroll
            for (int r = 0; r < R; ++r) out[r] = g[r];
        }

        if (owner) {
#pragma unroll
            for (int r = 0; r < R; ++r) {
                O[myq + r] = out[r];
                csum[r] += (double)out[r];
            }
        }
        __syncthreads();  // O complete, all reads of A done

        {
            T* __restrict__ orow = arg.fout + (size_t)j * ntheta;
            const int lim = min(chunk, ntheta - c0);
            for (int q = tid; q < lim; q += blockDim.x) orow[c0 + q] = O[q];
        }
        if (j + 1 < j1) stash();
        __syncthreads();
    }

    if (arg.colpart != nullptr && owner) {
        double* __restrict__ cp = arg.colpart + (size_t)blockIdx.y * ntheta;
#pragma unroll
        for (int r = 0; r < R; ++r)
            if (i0 + r < ntheta) cp[i0 + r] = csum[r];
    }
}

// ------------------------------------------------------------------------------------------------
// p shift (columns, strided axis), eq (11): f_II(x_i, p_j) = f_I(x_i, p_j - F_i dt).
// One thread = one column x one segment of rows.  Adjacent lanes own adjacent columns, so every load and
// store of a warp is one contiguous 256-byte piece of a row: coalesced without any transpose.  The ten
// taps live in a register window that slides down the column: one new load and ten FMAs per output.
// ------------------------------------------------------------------------------------------------
template <typename T>
struct PArgs {
    const T* fin;
    T* fout;
    const double* force;  // [Ntheta]
    int ntheta, np, bc_p, seg_len;
    double dt, dp;
};

template <typename T>
__device__ __forceinline__ T load_row(const T* __restrict__ col, int r, int np, size_t pitch, bool periodic) {
    if (periodic) {
        while (r >= np) r -= np;  // callers keep r >= 0; np may be smaller than the ten-tap window
        return __ldg(col + (size_t)r * pitch);
    }
    return ((unsigned)r < (unsigned)np) ? __ldg(col + (size_t)r * pitch) : T(0);
}

template <typename T>
__global__ void __launch_bounds__(256) p_sweep_kernel(const PArgs<T> arg) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= arg.ntheta) return;
    const int np = arg.np;
    const int j0 = blockIdx.y * arg.seg_len;
    const int j1 = min(np, j0 + arg.seg_len);
    if (j0 >= j1) return;
    const bool periodic = (arg.bc_p == BC_PERIODIC);
    const size_t pitch = (size_t)arg.ntheta;

    // foot of the characteristic: u = -(F dt)/dp cells  (D18)
    double sf, a;
    split_shift(-(arg.force[i] * arg.dt) / arg.dp, &sf, &a);
    int s;
    if (periodic) {
        sf = fmod(sf, (double)np);
        s = (int)sf;
        if (s < 0) s += np;  // s in [0, np)
    } else {
        const double lim = (double)np + 64.0;
        s = (int)fmin(fmax(sf, -lim), lim);
    }
    double wd[10];
    spline_fd8_weights(a, wd);
    T w[10];
    if (sizeof(T) == 4) {  // fp32 arithmetic: difference form (diff_form_weights)
        double U[9];
        diff_form_weights(wd, 10, FD_C, U);
#pragma unroll
        for (int m = 0; m < 9; ++m) w[m] = (T)U[m];
        w[9] = T(0);
    } else {
#pragma unroll
        for (int m = 0; m < 10; ++m) w[m] = (T)wd[m];
    }

    const T* __restrict__ col = arg.fin + i;
    T* __restrict__ ocol = arg.fout + i;

    // row index of tap mm for output j is j + s + mm - 4.  In periodic mode keep an offset in [0, np).
    int rbase = j0 + s - 4;
    if (periodic) rbase = wrap_index(rbase, np);

    T v[10], e[10];  // e (fp32 only): e[k] = v[k + 1] - v[k] of the window, kept as a ring like v
#pragma unroll
    for (int k = 0; k < 9; ++k) {
        v[k] = load_row(col, rbase + k, np, pitch, periodic);
    }
    v[9] = T(0);
#pragma unroll
    for (int k = 0; k < 10; ++k) e[k] = k < 8 ? v[k + 1] - v[k] : T(0);
    int rnext = rbase + 9;  // row of the next new tap
    if (periodic) rnext = rnext % np;

    T nv[10];
    auto fetch = [&](int jb) {  // the ten new taps of outputs jb .. jb+9
#pragma unroll
        for (int k = 0; k < 10; ++k) {
            int r = rnext + k;
            nv[k] = (jb + k < j1) ? load_row(col, r, np, pitch, periodic) : T(0);
        }
        rnext += 10;
        if (periodic) rnext %= np;
    };

    fetch(j0);
    for (int jb = j0; jb < j1; jb += 10) {
        T cur[10];
#pragma unroll
        for (int k = 0; k < 10; ++k) cur[k] = nv[k];
        if (jb + 10 < j1) fetch(jb + 10);  // loads of the next ten rows fly during these 100 FMAs
#pragma unroll
        for (int k = 0; k < 10; ++k) {
            v[(k + 9) % 10] = cur[k];
            T acc;
            if (sizeof(T) == 4) {
                e[(k + 8) % 10] = v[(k + 9) % 10] - v[(k + 8) % 10];
                acc = v[(k + FD_C) % 10];
#pragma unroll
                for (int m = 0; m < 9; ++m) acc = fma(w[m], e[(k + m) % 10], acc);
            } else {
                acc = w[0] * v[k % 10];
#pragma unroll
                for (int m = 1; m < 10; ++m) acc = fma(w[m], v[(k + m) % 10], acc);
            }
            if (jb + k < j1) ocol[(size_t)(jb + k) * pitch] = acc;
        }
    }
}

// ------------------------------------------------------------------------------------------------
// density and forces (eq (10); per model eqs (2), (4), (7)-(8))
// ------------------------------------------------------------------------------------------------
template <int NT>
__device__ __forceinline__ double block_sum(double v, double* red /* NT/32 doubles */) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    __syncthreads();
    if (lane == 0) red[warp] = v;
    __syncthreads();
    double t = 0.0;
    if (warp == 0) {
        t = (lane < NT / 32) ? red[lane] : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) t += __shfl_down_sync(0xffffffffu, t, o);
    }
    return t;  // valid in thread 0
}

// sheet, eq (4) (L41-L45), reading D11: F_i = -dx (sum_{k<i} rho_k - sum_{k>i} rho_k) = -dx (2 C_i + rho_i - S)
// with C the exclusive prefix sum and S the total.  One CTA of 1024 threads scans the whole vector.
// With mode = 1 writes instead the potential phi_i = dx sum_k |x_i - x_k| rho_k (for the energy):
// phi_i = dx * dxnode * (i (2 C_i - S + rho_i) ... ) evaluated from the two prefix sums of rho_k and k rho_k.
// (device body: also the tail of rho_force_kernel's last CTA; rho is read through L2, it may just have been written
// by other CTAs)
__device__ __forceinline__ void sheet_scan_body(const double* rho, int n, double dx, int mode, double* out) {
    __shared__ double wsum0[32], wsum1[32];
    __shared__ double carry0, carry1, tot0, tot1;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    // pass 1: totals S0 = sum rho_k, S1 = sum k rho_k
    {
        double a0 = 0.0, a1 = 0.0;
        for (int k = threadIdx.x; k < n; k += 1024) {
            const double rk = __ldcg(rho + k);
            a0 += rk;
            a1 += (double)k * rk;
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            a0 += __shfl_down_sync(0xffffffffu, a0, o);
            a1 += __shfl_down_sync(0xffffffffu, a1, o);
        }
        if (lane == 0) {
            wsum0[warp] = a0;
            wsum1[warp] = a1;
        }
        __syncthreads();
        if (threadIdx.x == 0) {
            double t0 = 0.0, t1 = 0.0;
            for (int q = 0; q < 32; ++q) {
                t0 += wsum0[q];
                t1 += wsum1[q];
            }
            tot0 = t0;
            tot1 = t1;
            carry0 = 0.0;
            carry1 = 0.0;
        }
        __syncthreads();
    }
    // pass 2: chunked inclusive scan with carry
    for (int base = 0; base < n; base += 1024) {
        const int k = base + threadIdx.x;
        const double r = (k < n) ? __ldcg(rho + k) : 0.0;
        double x0 = r, x1 = (double)k * r;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const double y0 = __shfl_up_sync(0xffffffffu, x0, o);
            const double y1 = __shfl_up_sync(0xffffffffu, x1, o);
            if (lane >= o) {
                x0 += y0;
                x1 += y1;
            }
        }
        __syncthreads();
        if (lane == 31) {
            wsum0[warp] = x0;
            wsum1[warp] = x1;
        }
        __syncthreads();
        if (warp == 0) {
            double z0 = wsum0[lane], z1 = wsum1[lane];
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const double y0 = __shfl_up_sync(0xffffffffu, z0, o);
                const double y1 = __shfl_up_sync(0xffffffffu, z1, o);
                if (lane >= o) {
                    z0 += y0;
                    z1 += y1;
                }
            }
            wsum0[lane] = z0;
            wsum1[lane] = z1;
        }
        __syncthreads();
        const double inc0 = carry0 + (warp > 0 ? wsum0[warp - 1] : 0.0) + x0;  // inclusive prefix of rho
        const double inc1 = carry1 + (warp > 0 ? wsum1[warp - 1] : 0.0) + x1;  // inclusive prefix of k rho
        if (k < n) {
            const double C0 = inc0 - r;                  // sum_{q<k} rho_q
            const double C1 = inc1 - (double)k * r;      // sum_{q<k} q rho_q
            if (mode == 0) {
                out[k] = -dx * (2.0 * C0 + r - tot0);
            } else {
                // sum_q |k - q| rho_q = k C0 - C1 + (S1 - C1 - k r) - k (S0 - C0 - r)
                const double right0 = tot0 - C0 - r, right1 = tot1 - C1 - (double)k * r;
                out[k] = dx * dx * (((double)k * C0 - C1) + (right1 - (double)k * right0));
            }
        }
        __syncthreads();
        if (threadIdx.x == 1023) {
            carry0 = inc0;
            carry1 = inc1;
        }
        __syncthreads();
    }
}

__global__ void __launch_bounds__(1024) sheet_scan_kernel(const double* rho, int n, double dx, int mode, double* out) {
    sheet_scan_body(rho, n, dx, mode, out);
}

// rho_i = dp * sum_b colpart[b][i]; for HMF also per-CTA partial sums of cos(theta_i) rho_i, sin(theta_i) rho_i.
// zero_after: the partials of the one-pass kernel are accumulated by atomic adds and must be zero for the next pass.
// 32 columns x 32 groups of bands per CTA, and for the HMF model fused
// with the force: the last CTA to finish (ticket counter) adds the per-CTA moment partials over a fixed tree --
// the tree is fixed, so the result does not depend on which CTA is last -- and writes F_i = -M_x sin(theta_i) + M_y cos(theta_i)
// (eqs (7)-(8), L56-L63) for every column.
constexpr int RR_COLS = 32, RR_GROUPS = 32;
__global__ void __launch_bounds__(RR_COLS* RR_GROUPS)
    rho_force_kernel(double* __restrict__ colpart, int nbands, int ntheta, double dp, double* __restrict__ rho,
                     const double* __restrict__ cos_t, const double* __restrict__ sin_t,
                     double* __restrict__ mpart /* [gridDim.x][2] or null */, int zero_after,
                     unsigned* __restrict__ ticket, double dtheta, double* __restrict__ force /* null: no force */,
                     int sheet /* 1: the last CTA writes the sheet force (prefix scan of rho) instead */) {
    __shared__ double part[RR_GROUPS][RR_COLS];
    __shared__ double2 mp[RR_COLS * RR_GROUPS];
    __shared__ bool last;
    ptx::pdl_launch_dependents();  // the next pass may be scheduled (its set-up does not depend on the force)
    ptx::pdl_wait();               // the pass whose column sums are read here has completed
    const int tid = threadIdx.x, c = tid & (RR_COLS - 1), g = tid / RR_COLS;
    const int i = blockIdx.x * RR_COLS + c;
    double a0 = 0.0, a1 = 0.0;
    if (i < ntheta) {
        // batches of eight independent loads (the kernel is latency-bound); the order of the additions is fixed
        constexpr int NB = 4;
        for (int b0 = g; b0 < nbands; b0 += NB * RR_GROUPS) {
            double v[NB];
#pragma unroll
            for (int k = 0; k < NB; ++k) {
                const int b = b0 + k * RR_GROUPS;
                v[k] = (b < nbands) ? __ldcg(colpart + (size_t)b * ntheta + i) : 0.0;
            }
            if (zero_after) {
#pragma unroll
                for (int k = 0; k < NB; ++k) {
                    const int b = b0 + k * RR_GROUPS;
                    if (b < nbands) __stcg(colpart + (size_t)b * ntheta + i, 0.0);
                }
            }
#pragma unroll
            for (int k = 0; k < NB; k += 2) {
                a0 += v[k];
                a1 += v[k + 1];
            }
        }
    }
    part[g][c] = a0 + a1;
    __syncthreads();
    if (g == 0) {  // one warp
        double acc = 0.0;
        if (i < ntheta) {
#pragma unroll
            for (int q = 0; q < RR_GROUPS; ++q) acc += part[q][c];
            acc *= dp;
            rho[i] = acc;
            __threadfence();  // every lane's rho is released before thread 0 takes the ticket
        }
        __syncwarp();
        if (mpart != nullptr) {
            double cs = (i < ntheta) ? cos_t[i] * acc : 0.0;
            double ss = (i < ntheta) ? sin_t[i] * acc : 0.0;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                cs += __shfl_down_sync(0xffffffffu, cs, o);
                ss += __shfl_down_sync(0xffffffffu, ss, o);
            }
            if (tid == 0) {
                mpart[2 * blockIdx.x + 0] = cs;
                mpart[2 * blockIdx.x + 1] = ss;
            }
        }
        if (tid == 0) {
            bool l = false;
            if (force != nullptr) {
                __threadfence();
                l = (atomicAdd(ticket, 1u) == gridDim.x - 1);
                if (l) *ticket = 0u;
            }
            last = l;
        }
    }
    if (force == nullptr) return;
    __syncthreads();
    if (!last) return;
    __threadfence();
    if (sheet) {  // eq (4), D11: F_i = -dx (2 C_i + rho_i - S) from the prefix sums of the rho every CTA has written
        sheet_scan_body(rho, ntheta, dtheta, 0, force);
        return;
    }
    // last CTA: M = dtheta * (sum of the partials over a fixed tree: thread t adds partials t, t + 1024, ...; then
    // shuffles inside each warp, then across the warps), the same whichever CTA happens to be last; then the force
    double mx = 0.0, my = 0.0;
    for (unsigned b = tid; b < gridDim.x; b += RR_COLS * RR_GROUPS) {
        mx += __ldcg(mpart + 2 * b);
        my += __ldcg(mpart + 2 * b + 1);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        mx += __shfl_down_sync(0xffffffffu, mx, o);
        my += __shfl_down_sync(0xffffffffu, my, o);
    }
    if ((tid & 31) == 0) mp[tid >> 5] = make_double2(mx, my);
    __syncthreads();
    if (tid < 32) {
        double2 t = mp[tid];  // RR_COLS * RR_GROUPS / 32 == 32 warps
        mx = t.x;
        my = t.y;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            mx += __shfl_down_sync(0xffffffffu, mx, o);
            my += __shfl_down_sync(0xffffffffu, my, o);
        }
        if (tid == 0) mp[32] = make_double2(mx * dtheta, my * dtheta);
    }
    __syncthreads();
    mx = mp[32].x;
    my = mp[32].y;
#pragma unroll 8
    for (int k = tid; k < ntheta; k += RR_COLS * RR_GROUPS) force[k] = -sin_t[k] * mx + cos_t[k] * my;
}

// Short theta axes (Ntheta <= 1024: cfg 1, cfg 2), HMF model: density, Fourier moments and force by ONE THREAD-BLOCK CLUSTER
// of up to eight CTAs, each with 128 columns.  rho_force_kernel above is a chain of six dependent round trips through L2
// (partials, rho + fence, ticket, moment partials, tables, force) whatever the size: 5 us on a 256-column grid whose
// whole pass takes 4.5 us.  Here thread (column c, group g) adds the partials of bands g, g + 8, ... of its column (all
// loads in flight at once), the eight groups are added in order, the CTA adds its moments over a fixed tree, the CTAs
// read one another's moment partials through distributed shared memory in rank order (one cluster barrier instead of a
// ticket in global memory) and every CTA writes the force of its own columns.  eqs (10), (7)-(8) (L75-L78, L56-L63).
// With HISTORY = 1 on the one-pass path the cluster has one more CTA, the last, which meanwhile turns the per-row sums of the pass
// that just ended into the moments of that step (history_rows_body below): the history costs no launch of its own.
struct HistArgs {
    const double* rowmom;  // null: no history CTA
    const double* invT;
    double* out;
    int nblk, np, ident;
    double pmin, t;
};
__device__ __forceinline__ void history_rows_body(const double* __restrict__ rowmom, int nblk, int np, const double* __restrict__ invT,
                                                  int ident, double pmin, double dp, double dtheta, double t,
                                                  double* __restrict__ out, double* red);
constexpr int RC_COLS = 128, RC_GROUPS = 8;
__global__ void __launch_bounds__(RC_COLS* RC_GROUPS)
    rho_force_cluster_kernel(double* __restrict__ colpart, int nbands, int ntheta, double dp, double* __restrict__ rho,
                             const double* __restrict__ cos_t, const double* __restrict__ sin_t, int zero_after,
                             double dtheta, double* __restrict__ force, const HistArgs hist) {
    namespace cg = cooperative_groups;
    cg::cluster_group cluster = cg::this_cluster();
    __shared__ double part[RC_GROUPS][RC_COLS];
    __shared__ double2 red[RC_COLS / 32];
    __shared__ double2 mine;  // this CTA's (sum cos theta_i rho_i, sum sin theta_i rho_i)
    ptx::pdl_launch_dependents();
    const int tid = threadIdx.x, c = tid & (RC_COLS - 1), g = tid / RC_COLS, lane = tid & 31, warp = tid >> 5;
    const unsigned ndens = gridDim.x - (hist.rowmom != nullptr ? 1u : 0u);  // CTAs that own columns
    if (blockIdx.x >= ndens) {  // the history CTA: no columns, but it keeps the cluster's two barriers
        ptx::pdl_wait();
        history_rows_body(hist.rowmom, hist.nblk, hist.np, hist.invT, hist.ident, hist.pmin, dp, dtheta, hist.t, hist.out, &part[0][0]);
        cluster.sync();
        cluster.sync();
        return;
    }
    const int i = blockIdx.x * RC_COLS + c;
    const bool in = i < ntheta;
    const bool own = in && g == 0;
    const double ct = own ? cos_t[i] : 0.0, st = own ? sin_t[i] : 0.0;  // constants of the run: fetched before the wait
    ptx::pdl_wait();                                                    // the pass whose column sums are read has completed
    double acc = 0.0;
    if (in) {
        constexpr int NB = 4;
        for (int b0 = g; b0 < nbands; b0 += NB * RC_GROUPS) {
            double v[NB];
#pragma unroll
            for (int k = 0; k < NB; ++k) {
                const int b = b0 + k * RC_GROUPS;
                v[k] = (b < nbands) ? __ldcg(colpart + (size_t)b * ntheta + i) : 0.0;
            }
            if (zero_after) {
#pragma unroll
                for (int k = 0; k < NB; ++k) {
                    const int b = b0 + k * RC_GROUPS;
                    if (b < nbands) __stcg(colpart + (size_t)b * ntheta + i, 0.0);
                }
            }
#pragma unroll
            for (int k = 0; k < NB; ++k) acc += v[k];
        }
    }
    part[g][c] = acc;
    __syncthreads();
    double r = 0.0;
    if (g == 0) {
#pragma unroll
        for (int q = 0; q < RC_GROUPS; ++q) r += part[q][c];
        r *= dp;
        if (in) rho[i] = r;
    }
    if (warp < RC_COLS / 32) {  // the warps of group 0
        double cs = ct * r, ss = st * r;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            cs += __shfl_down_sync(0xffffffffu, cs, o);
            ss += __shfl_down_sync(0xffffffffu, ss, o);
        }
        if (lane == 0) red[warp] = make_double2(cs, ss);
    }
    __syncthreads();
    if (tid == 0) {
        double2 t = red[0];
#pragma unroll
        for (int w = 1; w < RC_COLS / 32; ++w) {
            t.x += red[w].x;
            t.y += red[w].y;
        }
        mine = t;
    }
    cluster.sync();  // every CTA's partial is written
    if (own) {
        double mx = 0.0, my = 0.0;
        for (unsigned rk = 0; rk < ndens; ++rk) {
            const double2 t = *cluster.map_shared_rank(&mine, rk);
            mx += t.x;
            my += t.y;
        }
        force[i] = -st * (mx * dtheta) + ct * (my * dtheta);
    }
    cluster.sync();  // no CTA leaves while its shared memory may still be read
}

// HMF force from a density vector (eqs (7)-(8), L56-L63), one CTA: M = dtheta sum_i (cos, sin)(theta_i) rho_i over a fixed
// tree, F_i = -M_x sin(theta_i) + M_y cos(theta_i).  Used where rho does not come out of rho_force_kernel: in slab
// mode the density is all-reduced over the ranks between the two.
__global__ void __launch_bounds__(1024) hmf_force_from_rho_kernel(const double* __restrict__ rho, const double* __restrict__ cos_t,
                                                                  const double* __restrict__ sin_t, int ntheta, double dtheta,
                                                                  double* __restrict__ force) {
    __shared__ double red[32];
    __shared__ double msh[2];
    double cx = 0.0, sx = 0.0;
    for (int i = threadIdx.x; i < ntheta; i += 1024) {
        const double r = rho[i];
        cx = fma(cos_t[i], r, cx);
        sx = fma(sin_t[i], r, sx);
    }
    const double CX = block_sum<1024>(cx, red);
    const double SX = block_sum<1024>(sx, red);
    if (threadIdx.x == 0) {
        msh[0] = CX * dtheta;
        msh[1] = SX * dtheta;
    }
    __syncthreads();
    const double mx = msh[0], my = msh[1];
    for (int i = threadIdx.x; i < ntheta; i += 1024) force[i] = -sin_t[i] * mx + cos_t[i] * my;
}

// ring, eq (2) (L33-L35), reading D9: out_i = scale * sum_{m=0}^{N-1} tab[m] rho[(i - m) mod N].
// Used with tab = K (force) and tab = V (potential, for the energy).  The sum over m is cut into chunks of RING_L
// terms: CTA (tile of 256 outputs, chunk c) stages its piece of the table and the matching window of rho in shared
// memory and writes 256 partial sums; the last CTA of a tile to finish (ticket counter per tile) adds the chunks
// in chunk order -- the result does not depend on which CTA that is.  N = 2048: 8 x 16 CTAs of 128 FMAs per thread
// instead of 8 CTAs of 2048.
constexpr int RING_L = 128;
__global__ void __launch_bounds__(256) ring_convolve_kernel(const double* __restrict__ tab,
                                                            const double* __restrict__ rho, int n, double scale,
                                                            double* __restrict__ part /* [chunks][n] */,
                                                            unsigned* __restrict__ tickets /* [tiles], zero */,
                                                            double* __restrict__ out) {
    __shared__ double sK[RING_L];
    __shared__ double sR[RING_L + 256];
    __shared__ bool last;
    const int ib = blockIdx.x * 256, i = ib + threadIdx.x;
    const int m0 = blockIdx.y * RING_L, tm = min(RING_L, n - m0);
    for (int q = threadIdx.x; q < tm; q += 256) sK[q] = tab[m0 + q];
    // sR[q] = rho[(ib - m0 - (tm - 1) + q) mod n], q in [0, tm + 255)
    const int lo = wrap_index(ib - m0 - (tm - 1), n);
    for (int q = threadIdx.x; q < tm + 255; q += 256) sR[q] = rho[(lo + q) % n];
    __syncthreads();
    // rho index i - m  ->  sR[(i - ib) + (tm - 1) - (m - m0)]
    const int off = threadIdx.x + tm - 1;
    double acc0 = 0.0, acc1 = 0.0, acc2 = 0.0, acc3 = 0.0;
    int mm = 0;
    for (; mm + 4 <= tm; mm += 4) {
        acc0 = fma(sK[mm], sR[off - mm], acc0);
        acc1 = fma(sK[mm + 1], sR[off - mm - 1], acc1);
        acc2 = fma(sK[mm + 2], sR[off - mm - 2], acc2);
        acc3 = fma(sK[mm + 3], sR[off - mm - 3], acc3);
    }
    for (; mm < tm; ++mm) acc0 = fma(sK[mm], sR[off - mm], acc0);
    if (i < n) __stcg(part + (size_t)blockIdx.y * n + i, (acc0 + acc1) + (acc2 + acc3));
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) {
        const bool l = (atomicAdd(tickets + blockIdx.x, 1u) == gridDim.y - 1);
        if (l) tickets[blockIdx.x] = 0u;
        last = l;
    }
    __syncthreads();
    if (!last) return;
    __threadfence();
    if (i < n) {
        double t = 0.0;
        for (unsigned c = 0; c < gridDim.y; ++c) t += __ldcg(part + (size_t)c * n + i);
        out[i] = t * scale;
    }
}

// ------------------------------------------------------------------------------------------------
// moments (a7): one read pass over f.  Each thread owns one column over a band of rows.
// ------------------------------------------------------------------------------------------------
template <typename T>
__global__ void __launch_bounds__(256) moments_pass_kernel(const T* __restrict__ f, int ntheta, int np,
                                                           int rows_per_band, double pmin, double dp,
                                                           double* __restrict__ colpart /* [bands][ntheta] */,
                                                           double* __restrict__ pk_part /* [blocks][2] */) {
    __shared__ double red[8];
    const int i = blockIdx.x * 256 + threadIdx.x;
    const int j0 = blockIdx.y * rows_per_band, j1 = min(np, j0 + rows_per_band);
    double c0 = 0.0, c1 = 0.0, c2 = 0.0;
    if (i < ntheta) {
        for (int j = j0; j < j1; ++j) {
            const double v = (double)f[(size_t)j * ntheta + i];
            const double p = pmin + (double)j * dp;
            c0 += v;
            c1 = fma(p, v, c1);
            c2 = fma(0.5 * p * p, v, c2);
        }
        colpart[(size_t)blockIdx.y * ntheta + i] = c0;
    }
    const double s1 = block_sum<256>(c1, red);
    const double s2 = block_sum<256>(c2, red);
    if (threadIdx.x == 0) {
        const int b = blockIdx.y * gridDim.x + blockIdx.x;
        pk_part[2 * b + 0] = s1;
        pk_part[2 * b + 1] = s2;
    }
}

// HISTORY on the one-pass path (HMF model, periodic theta axis of length 2 pi): the eight moments of the END-OF-STEP state
// f^{n+1} from per-row sums of the state the one-pass path stores, h = theta(dt/2) f^{n+1} (the leading half shift of the
// next step is already applied).  A half shift of a periodic row is a circular convolution, h_i = sum_m w_m f_{i+s+m-4},
// so it multiplies the row's first Fourier sum by a number that depends on the row only:
//     sum_i h_i e^{i theta_i} = T_j sum_l f_l e^{i theta_l},   T_j = e^{-i s_j dtheta} sum_m w_m e^{-i (m-4) dtheta},
// and leaves the row's sum alone.  So with R0_j, Rc_j, Rs_j the sums of row j of h (times 1, cos theta_i, sin theta_i; from
// strang_tile_kernel, per column block) and 1/T_j from the host:  mass, P, K from R0 (eq (6) discretised, D6), and
// M_x + i M_y = dtheta dp sum_j (Rc_j + i Rs_j) / T_j (eq (8)); U = (m^2 - M^2) / 2 (D10).  ident = 1: the stored state IS
// f^{n+1} (last pass of a call: one half shift only).  One CTA, fixed order.  out = {t, mass, P, K, U, Mx, My, E}
__device__ __forceinline__ void history_rows_body(const double* __restrict__ rowmom /* [nblk][np][3] */, int nblk, int np,
                                                  const double* __restrict__ invT /* [np][2] */, int ident, double pmin,
                                                  double dp, double dtheta, double t, double* __restrict__ out,
                                                  double* red /* 32 doubles of shared memory */) {
    double m = 0.0, pp = 0.0, kk = 0.0, mx = 0.0, my = 0.0;
    for (int j = threadIdx.x; j < np; j += 1024) {
        double r0 = 0.0, rc = 0.0, rs = 0.0;
        for (int b = 0; b < nblk; ++b) {
            const double* rm = rowmom + ((size_t)b * np + j) * 3;
            r0 += __ldcg(rm);
            rc += __ldcg(rm + 1);
            rs += __ldcg(rm + 2);
        }
        const double p = pmin + (double)j * dp;
        m += r0;
        pp = fma(p, r0, pp);
        kk = fma(0.5 * p * p, r0, kk);
        if (ident) {
            mx += rc;
            my += rs;
        } else {  // (rc + i rs) (a + i b), a + i b = 1 / T_j
            const double a = invT[2 * j], b = invT[2 * j + 1];
            mx += rc * a - rs * b;
            my += rc * b + rs * a;
        }
    }
    const double M = block_sum<1024>(m, red);
    const double PP = block_sum<1024>(pp, red);
    const double KK = block_sum<1024>(kk, red);
    const double MX = block_sum<1024>(mx, red);
    const double MY = block_sum<1024>(my, red);
    if (threadIdx.x == 0) {
        const double w = dtheta * dp;
        const double mass = M * w, Mx = MX * w, My = MY * w, K = KK * w;
        const double U = 0.5 * (mass * mass - Mx * Mx - My * My);
        out[0] = t;
        out[1] = mass;
        out[2] = PP * w;
        out[3] = K;
        out[4] = U;
        out[5] = Mx;
        out[6] = My;
        out[7] = K + U;
    }
}

// the three sums of every row of f (times 1, cos theta_i, sin theta_i) by a read pass: what strang_tile_kernel leaves behind on
// small grids, for the grids of the warp-specialised kernel (HISTORY = 1 on the one-pass path at any size).  One warp per row.
template <typename T>
__global__ void __launch_bounds__(256) row_moments_kernel(const T* __restrict__ f, int ntheta, int np,
                                                          const double* __restrict__ cos_t, const double* __restrict__ sin_t,
                                                          double* __restrict__ rowmom /* [np][3] */) {
    const int lane = threadIdx.x & 31;
    const int j = (int)blockIdx.x * 8 + (int)(threadIdx.x >> 5);
    if (j >= np) return;  // whole warp
    const T* __restrict__ row = f + (size_t)j * ntheta;
    double r0 = 0.0, rc = 0.0, rs = 0.0;
    int i = lane;
    for (; i + 7 * 32 < ntheta; i += 8 * 32) {  // eight loads in flight per lane; the order of the additions is fixed
        double v[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) v[k] = (double)__ldcs(row + i + 32 * k);
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            r0 += v[k];
            rc = fma(v[k], __ldg(cos_t + i + 32 * k), rc);
            rs = fma(v[k], __ldg(sin_t + i + 32 * k), rs);
        }
    }
    for (; i < ntheta; i += 32) {
        const double v = (double)__ldcs(row + i);
        r0 += v;
        rc = fma(v, __ldg(cos_t + i), rc);
        rs = fma(v, __ldg(sin_t + i), rs);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        r0 += __shfl_down_sync(0xffffffffu, r0, o);
        rc += __shfl_down_sync(0xffffffffu, rc, o);
        rs += __shfl_down_sync(0xffffffffu, rs, o);
    }
    if (lane == 0) {
        rowmom[3 * (size_t)j + 0] = r0;
        rowmom[3 * (size_t)j + 1] = rc;
        rowmom[3 * (size_t)j + 2] = rs;
    }
}

__global__ void __launch_bounds__(1024) history_rows_kernel(const double* __restrict__ rowmom, int nblk, int np,
                                                            const double* __restrict__ invT, int ident, double pmin, double dp,
                                                            double dtheta, double t, double* __restrict__ out) {
    __shared__ double red[32];
    history_rows_body(rowmom, nblk, np, invT, ident, pmin, dp, dtheta, t, out, red);
}

// final: one CTA.  rho must already hold dp * column sums; phi (ring / sheet potential) may be null.
// out = {t, mass, P, K, U, Mx, My, E}
__global__ void __launch_bounds__(1024) moments_final_kernel(const double* __restrict__ rho,
                                                             const double* __restrict__ phi, int ntheta,
                                                             const double* __restrict__ pk_part, int nparts,
                                                             const double* __restrict__ cos_t,
                                                             const double* __restrict__ sin_t, double dtheta,
                                                             double dp, int model, double t,
                                                             double* __restrict__ out) {
    __shared__ double red[32];
    double m = 0.0, cx = 0.0, sx = 0.0, u = 0.0, pp = 0.0, kk = 0.0;
    for (int i = threadIdx.x; i < ntheta; i += 1024) {
        const double r = rho[i];
        m += r;
        cx = fma(cos_t[i], r, cx);
        sx = fma(sin_t[i], r, sx);
        if (phi != nullptr) u = fma(r, phi[i], u);
    }
    for (int b = threadIdx.x; b < nparts; b += 1024) {
        pp += pk_part[2 * b + 0];
        kk += pk_part[2 * b + 1];
    }
    const double M = block_sum<1024>(m, red);
    const double CX = block_sum<1024>(cx, red);
    const double SX = block_sum<1024>(sx, red);
    const double UU = block_sum<1024>(u, red);
    const double PP = block_sum<1024>(pp, red);
    const double KK = block_sum<1024>(kk, red);
    if (threadIdx.x == 0) {
        const double mass = M * dtheta, Mx = CX * dtheta, My = SX * dtheta;
        const double P = PP * dtheta * dp, K = KK * dtheta * dp;
        double U = 0.0;
        if (model == 1) U = 0.5 * (mass * mass - Mx * Mx - My * My);
        else if (model == 2 || model == 3) U = 0.5 * UU * dtheta;
        out[0] = t;
        out[1] = mass;
        out[2] = P;
        out[3] = K;
        out[4] = U;
        out[5] = Mx;
        out[6] = My;
        out[7] = K + U;
    }
}

// ------------------------------------------------------------------------------------------------
// Casimir invariants, eq (18): C[s] = int s(f) dp dx by the rectangle rule.
//   s(f) = -f log f (entropy of Fig. 2; nodes with f <= 0 contribute 0, D20),  s(f) = f^2,
//   negative mass sum min(f, 0), max f.  One read pass over f; block partials, then one CTA adds them over a fixed
//   tree (deterministic).
// ------------------------------------------------------------------------------------------------
template <int NT>
__device__ __forceinline__ double block_max(double v, double* red /* NT/32 doubles */) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_down_sync(0xffffffffu, v, o));
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    __syncthreads();
    if (lane == 0) red[warp] = v;
    __syncthreads();
    double t = v;
    if (warp == 0) {
        t = (lane < NT / 32) ? red[lane] : red[0];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) t = fmax(t, __shfl_down_sync(0xffffffffu, t, o));
    }
    return t;  // valid in thread 0
}

template <typename T>
__global__ void __launch_bounds__(256) casimir_pass_kernel(const T* __restrict__ f, int ntheta, int np,
                                                           int rows_per_band,
                                                           double* __restrict__ part /* [blocks][4] */) {
    __shared__ double red[8];
    const int i = blockIdx.x * 256 + threadIdx.x;
    const int j0 = blockIdx.y * rows_per_band, j1 = min(np, j0 + rows_per_band);
    double s = 0.0, c2 = 0.0, neg = 0.0, mx = (double)f[0];
    if (i < ntheta) {
        for (int j = j0; j < j1; ++j) {
            const double v = (double)f[(size_t)j * ntheta + i];
            if (v > 0.0) s -= v * log(v);
            if (v < 0.0) neg += v;
            c2 = fma(v, v, c2);
            mx = fmax(mx, v);
        }
    }
    const double S = block_sum<256>(s, red);
    const double C = block_sum<256>(c2, red);
    const double N = block_sum<256>(neg, red);
    const double M = block_max<256>(mx, red);
    if (threadIdx.x == 0) {
        const int b = blockIdx.y * gridDim.x + blockIdx.x;
        part[4 * b + 0] = S;
        part[4 * b + 1] = C;
        part[4 * b + 2] = N;
        part[4 * b + 3] = M;
    }
}

__global__ void __launch_bounds__(1024) casimir_final_kernel(const double* __restrict__ part, int nparts, double cell,
                                                             double* __restrict__ out) {
    __shared__ double red[32];
    double s = 0.0, c2 = 0.0, neg = 0.0, mx = part[3];
    for (int b = threadIdx.x; b < nparts; b += 1024) {
        s += part[4 * b + 0];
        c2 += part[4 * b + 1];
        neg += part[4 * b + 2];
        mx = fmax(mx, part[4 * b + 3]);
    }
    const double S = block_sum<1024>(s, red);
    const double C = block_sum<1024>(c2, red);
    const double N = block_sum<1024>(neg, red);
    const double M = block_max<1024>(mx, red);
    if (threadIdx.x == 0) {
        out[0] = S * cell;
        out[1] = C * cell;
        out[2] = N * cell;
        out[3] = M;
    }
}

__global__ void fill_zero_kernel(double* __restrict__ p, int n) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) p[i] = 0.0;
}

}  // namespace vl
