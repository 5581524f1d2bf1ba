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
// Geometry (the kernel itself is in vlasov_fused_ws.cuh; this header holds what it shares with the host: the argument
// block, the column-block split and the per-thread asynchronous copies).  A CTA owns NTA = TI + NTAP - 1 consecutive
// SOURCE columns and a band of rows and marches down the band in groups of 12 rows.
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
                             //   NST = 1: w_0..w_9, s, e;  NST = 2: W_0..W_18, 2 s, e   (s non-increasing with the row;
                             //   e: fp32 residual of the row's weights, weight_residual)
    double* colpart;         // [nbands * NW][Ntheta], zero on entry; column sums are ADDED (may be null)
    int ntheta, np, bc_p, rows_per_band, bulk_ok, gran;
    int edge_w;              // relative width (percent) of the first and last column block (fused_block_range)
    int x0, xw;              // the column blocks tile the source positions [x0, x0 + xw): [0, Ntheta) on a periodic axis; on a
                             // zero-extended one (ZX) also what the rows drift beyond the ends (x0 <= 0, even)
    double dt, dp;
    // tile kernel only (history on the one-pass path, vlasov_tile.cuh): per (column block, row) the sums of the output row and
    // of the row times cos theta_i, sin theta_i -> rowmom[block][row][3]; null: not wanted
    double* rowmom;
    const double *cos_t, *sin_t;
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
// edge_w (percent, 100 = like the others): relative width of the first and the last block.  On a zero-extended axis
// the rows of those two blocks apply the two half shifts one after the other (half as many FMAs again), and with one
// CTA per SM the pass takes as long as its slowest block: they get fewer columns.
__host__ __device__ inline long long fused_block_cum(int c, int cols, int edge_w) {  // weight of the blocks before c
    if (cols < 3 || edge_w == 100) return 100LL * c;
    if (c == 0) return 0;
    if (c == cols) return 100LL * (cols - 2) + 2LL * edge_w;
    return edge_w + 100LL * (c - 1);
}
__host__ __device__ inline int fused_block_cols(int ntheta, int R, int gran, int edge_w = 100) {
    const int U = (ntheta + R * gran - 1) / (R * gran);
    const int per = 32 / gran;
    int cols = (U + per - 1) / per;
    if (edge_w != 100 && cols >= 3) {  // smallest count whose widest (inner) block still fits the 32 lanes
        for (;; ++cols) {
            const long long tot = fused_block_cum(cols, cols, edge_w);
            bool ok = true;
            for (int c = 0; c < cols && ok; ++c) {
                const long long u0 = (long long)U * fused_block_cum(c, cols, edge_w) / tot,
                                u1 = (long long)U * fused_block_cum(c + 1, cols, edge_w) / tot;
                ok = (u1 - u0) <= per;
            }
            if (ok) break;
        }
    }
    return cols;
}
__host__ __device__ inline void fused_block_range(int c, int cols, int ntheta, int R, int gran, int* i0, int* width,
                                                  int edge_w = 100) {
    const long long U = (ntheta + R * gran - 1) / (R * gran);
    const long long tot = fused_block_cum(cols, cols, edge_w);
    const int u0 = (int)(U * fused_block_cum(c, cols, edge_w) / tot), u1 = (int)(U * fused_block_cum(c + 1, cols, edge_w) / tot);
    const int e = u1 * R * gran < ntheta ? u1 * R * gran : ntheta;
    *i0 = u0 * R * gran;
    *width = e - u0 * R * gran;
}

}  // namespace vl
