// vlasov_theta_bulk.cuh -- theta shift (contiguous axis) for sm_100a with the bulk asynchronous copy engine.
//
// Arithmetic: exactly that of theta_sweep_generic_kernel (vlasov_kernels.cuh): the spline of eqs (13)-(14)
// with f'' from eq (16) (L106-L111) folded into ten weights per row, one (NSTAGE = 1) or
// two (NSTAGE = 2, steps (12) of step k and (9) of step k+1, L71-L87) half shifts per pass.
//
// Organisation: every WARP is its own pipeline -- no block-wide barrier anywhere.  A warp owns CHUNK
// consecutive columns and walks down the rows of its band:
//   * lane 0 asks the copy engine (cp.async.bulk, global -> shared, completion on an mbarrier) for the
//     source window of row j + NS while the warp works on row j: NS rows of every warp are always in flight,
//     independent of registers and of the arithmetic.  The integer part of the shift only moves the start of
//     the window; the copy starts at the 16-byte boundary below it and the lanes add the 0..AL-1 elements of
//     misalignment to their shared-memory index.  A periodic wrap is two copies; for zero extension the part
//     of the window outside the row is filled with zeros by the lanes.
//   * the ten weights and the shift of the row travel in the same stage (one 96-byte copy of the row table).
//   * each lane reads its R + 9 window from shared memory (lane stride R, odd: conflict-free), produces R
//     consecutive values with 10 FMAs each from registers, passes nine of them to its neighbour by shuffles
//     for the second shift, writes the R results to a shared output tile, and lane 0 hands the tile to the
//     copy engine (shared -> global).  Loads and stores are full 16-byte-aligned runs: no partial sectors.
//   * the column sums of the OUTPUT rows (the density of eq (10)) stay in registers for the band.
#pragma once
#include "vlasov_kernels.cuh"

namespace vl {

template <typename T, int NSTAGE, int R, int NS, int WARPS>
struct ThetaBulk {
    static constexpr int LANES = NSTAGE == 2 ? 31 : 32;     // lanes that own outputs
    static constexpr int AL = 16 / (int)sizeof(T);          // elements per 16 bytes
    static constexpr int TILE = LANES * R;
    static constexpr int CHUNK = TILE & ~(AL - 1);          // columns per warp (keeps every store 16-byte aligned)
    static constexpr int HALO = 9 * NSTAGE;
    static constexpr int IN_ALLOC = (32 * R + 9 + 2 * (AL - 1)) & ~(AL - 1);
    static constexpr int OUT_ALLOC = (32 * R + AL - 1) & ~(AL - 1);
    static constexpr int HDR_BYTES = WROW_STRIDE * 8;
    static constexpr int IN_BYTES = (IN_ALLOC * (int)sizeof(T) + 127) / 128 * 128;
    static constexpr int STAGE_BYTES = IN_BYTES + 128;      // window + row header
    static constexpr int OUT_BYTES = (OUT_ALLOC * (int)sizeof(T) + 127) / 128 * 128;
    static constexpr int WARP_BYTES = NS * STAGE_BYTES + 2 * OUT_BYTES + 128;  // + mbarriers
    static constexpr int SMEM_BYTES = WARPS * WARP_BYTES;
    static_assert(NS * 8 <= 128, "mbarriers must fit their slot");
    static_assert(R >= 9 && (R & 1), "R odd (bank conflicts) and >= 9 (one neighbour provides the halo)");
};

struct ThetaBulkGrid {
    int nchunks, nbands, rows_per_band;
};

template <typename T, int NSTAGE, int R, int NS, int WARPS, int MINB>
__global__ void __launch_bounds__(WARPS * 32, MINB)
    theta_sweep_bulk_kernel(const ThetaArgs<T> arg, const ThetaBulkGrid gr) {
    using C = ThetaBulk<T, NSTAGE, R, NS, WARPS>;
    constexpr int AL = C::AL, HALO = C::HALO, CHUNK = C::CHUNK;

    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int gw = blockIdx.x * WARPS + warp;
    const int band = gw / gr.nchunks, chunk = gw - band * gr.nchunks;
    if (band >= gr.nbands) return;  // whole warp; there is no block-wide barrier below

    unsigned char* wbase = smem_raw + (size_t)warp * C::WARP_BYTES;
    auto stage_in = [&](int st) { return reinterpret_cast<T*>(wbase + st * C::STAGE_BYTES); };
    auto stage_hdr = [&](int st) { return reinterpret_cast<double*>(wbase + st * C::STAGE_BYTES + C::IN_BYTES); };
    auto out_buf = [&](int k) { return reinterpret_cast<T*>(wbase + NS * C::STAGE_BYTES + k * C::OUT_BYTES); };
    uint64_t* full = reinterpret_cast<uint64_t*>(wbase + NS * C::STAGE_BYTES + 2 * C::OUT_BYTES);

    const int ntheta = arg.ntheta;
    const int c0 = chunk * CHUNK;
    const int nvalid = min(CHUNK, ntheta - c0);
    const int j0 = band * gr.rows_per_band;
    const int nrows = min(arg.np, j0 + gr.rows_per_band) - j0;
    const bool periodic = (arg.bc_x == BC_PERIODIC);
    const int myq = lane * R;
    const bool owner = (lane < C::LANES);
    if (nrows <= 0 || nvalid <= 0) return;

    if (lane == 0) {
#pragma unroll
        for (int st = 0; st < NS; ++st) ptx::mbar_init(&full[st], 1);
        ptx::fence_mbar_init();
    }
    __syncwarp();

    // ask the copy engine for the window of row j (shift s) into stage st; all lanes call
    auto issue_load = [&](int j, int st, int s) {
        const int start = c0 + NSTAGE * s - 4 * NSTAGE;
        const int off = start & (AL - 1);
        const int e0 = start - off;  // 16-byte boundary at or below the first tap
        const int len = (off + nvalid + HALO + AL - 1) & ~(AL - 1);
        T* A = stage_in(st);
        const T* row = arg.fin + (size_t)j * ntheta;
        const double* hsrc = arg.wrow + (size_t)j * WROW_STRIDE;
        if (periodic) {
            if (lane == 0) {
                ptx::mbar_arrive_expect_tx(&full[st], (unsigned)(len * sizeof(T)) + C::HDR_BYTES);
                ptx::bulk_g2s(stage_hdr(st), hsrc, C::HDR_BYTES, &full[st]);
                int pos = e0 % ntheta;
                if (pos < 0) pos += ntheta;
                int done = 0;
                while (done < len) {
                    const int n = min(len - done, ntheta - pos);
                    ptx::bulk_g2s(A + done, row + pos, (unsigned)(n * sizeof(T)), &full[st]);
                    done += n;
                    pos = 0;
                }
            }
        } else {
            const int lo = min(len, max(0, -e0)), hi = max(lo, min(len, ntheta - e0));  // part inside the row
            if (lo > 0 || hi < len) {  // the line is zero outside [0, Ntheta) (D4)
                for (int q = lane; q < len; q += 32)
                    if (q < lo || q >= hi) A[q] = T(0);
                ptx::fence_proxy_async_smem();
                __syncwarp();
            }
            if (lane == 0) {
                const unsigned bytes = (unsigned)((hi - lo) * sizeof(T));
                ptx::mbar_arrive_expect_tx(&full[st], bytes + C::HDR_BYTES);
                ptx::bulk_g2s(stage_hdr(st), hsrc, C::HDR_BYTES, &full[st]);
                if (bytes) ptx::bulk_g2s(A + lo, row + (e0 + lo), bytes, &full[st]);
            }
        }
    };

    // prologue: NS rows in flight
    int s_pref = 0;
#pragma unroll
    for (int st = 0; st < NS; ++st)
        if (st < nrows) issue_load(j0 + st, st, __ldg(arg.srow + j0 + st));
    if (NS < nrows) s_pref = __ldg(arg.srow + j0 + NS);

    double csum[R];
#pragma unroll
    for (int r = 0; r < R; ++r) csum[r] = 0.0;

    int st = 0;
    unsigned parity = 0;
    for (int it = 0; it < nrows; ++it) {
        const int j = j0 + it;
        ptx::mbar_wait(&full[st], parity);

        const double* hdr = stage_hdr(st);
        T w[10];
#pragma unroll
        for (int m = 0; m < 10; ++m) w[m] = (T)hdr[m];
        const int s = (int)hdr[10];
        const int off = (c0 + NSTAGE * s - 4 * NSTAGE) & (AL - 1);
        const T* A = stage_in(st) + off + myq;
        T v[R + 9];
#pragma unroll
        for (int k = 0; k < R + 9; ++k) v[k] = A[k];
        __syncwarp();  // every lane has its window: the stage can be refilled

        if (it + NS < nrows) {
            issue_load(j + NS, st, s_pref);
            if (it + NS + 1 < nrows) s_pref = __ldg(arg.srow + j + NS + 1);
        }

        T g[R];
        fir_window<T, R, 10, FD_C>(w, v, g);

        T out[R];
        if (NSTAGE == 2) {
            if (!periodic) {  // the intermediate row is zero outside [0, Ntheta): two separate cropped shifts
                const int x0 = c0 + myq + s - 4;
#pragma unroll
                for (int r = 0; r < R; ++r)
                    if ((unsigned)(x0 + r) >= (unsigned)ntheta) g[r] = T(0);
            }
            T h[R + 9];
#pragma unroll
            for (int r = 0; r < R; ++r) h[r] = g[r];
#pragma unroll
            for (int r = 0; r < 9; ++r) h[R + r] = __shfl_down_sync(0xffffffffu, g[r], 1);
            fir_window<T, R, 10, FD_C>(w, h, out);
        } else {
#pragma unroll
            for (int r = 0; r < R; ++r) out[r] = g[r];
        }

        // the output tile used two rows ago must have been read by the copy engine
        if (lane == 0) ptx::bulk_wait_read<1>();
        __syncwarp();
        T* O = out_buf(it & 1);
        if (owner) {
#pragma unroll
            for (int r = 0; r < R; ++r) {
                O[myq + r] = out[r];
                csum[r] += (double)out[r];
            }
        }
        ptx::fence_proxy_async_smem();
        __syncwarp();
        if (lane == 0) {
            ptx::bulk_s2g(arg.fout + (size_t)j * ntheta + c0, O, (unsigned)(nvalid * sizeof(T)));
            ptx::bulk_commit();
        }

        if (++st == NS) {
            st = 0;
            parity ^= 1u;
        }
    }
    if (lane == 0) ptx::bulk_wait_read<0>();

    if (arg.colpart != nullptr && owner) {
        double* __restrict__ cp = arg.colpart + (size_t)band * ntheta + c0;
#pragma unroll
        for (int r = 0; r < R; ++r)
            if (myq + r < nvalid) cp[myq + r] = csum[r];
    }
}

}  // namespace vl
