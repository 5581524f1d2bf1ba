// vlasov_api.cu -- host side of the C ABI declared in include/vlasov.h.
//
// Singleton context, tables computed once on the host (PAPER.md L210 stores sin/cos of the nodes once; the
// per-row shift of the theta half step is constant for the whole run because p_j and dt never change),
// launch sequencing of one Strang step (L71-L87):
//     theta(dt/2) -> rho -> F -> p(dt) -> theta(dt/2)
// with the trailing and leading half shifts of consecutive steps merged into one pass (a6).
#include <cuda_runtime.h>
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <algorithm>
#include <vector>

#include "../../include/vlasov.h"
#include "vlasov_kernels.cuh"
#include "vlasov_theta_bulk.cuh"
#include "vlasov_fused.cuh"
#include "vlasov_fused_ws.cuh"
#include "vlasov_tile.cuh"
#include "vlasov_gs.cuh"

namespace {

constexpr int R_THETA = 9;       // consecutive outputs per lane in the theta kernel (odd: bank-conflict-free)
constexpr int TB_NS = 3;         // rows in flight per warp in the bulk-copy theta kernel
constexpr int TB_WARPS = 4;      // warps per CTA (independent pipelines)
constexpr int TB_MINB = 3;       // CTAs per SM the register budget is set for
#ifndef VL_FW_NTW_
#define VL_FW_NTW_ 12
#endif
// consecutive outputs per lane in the theta stage of the one-pass kernel (odd): fp64 11 of a ring row of 384 columns,
// fp32 15 of a ring row of 512 (FusedWsCfg::CPT; 8192^2 fp32: 286 -> 302 Gpts/s)
#ifdef VL_FU_R
template <typename T> constexpr int FU_R = VL_FU_R;
#else
template <typename T> constexpr int FU_R = sizeof(T) == 4 ? 15 : 11;
#endif
#ifndef VL_FW_NSTG
#define VL_FW_NSTG 3
#endif
constexpr int FW_NSTG = VL_FW_NSTG;       // ring depth (groups of 12 rows) of the one-pass kernel
constexpr int FW_NTW = VL_FW_NTW_;       // its theta warps = density partial rows per band
constexpr int KEY_TUNE_GRAPH = 109, KEY_TUNE_PDL = 110, KEY_TUNE_FEDGE = 108;
constexpr int FU_PAD = 12;       // rows of padding of the theta weight tables (the last phase of a band reads on)
constexpr int NCLS = 6;          // profiled kernel classes: theta x1, theta x2, p, rho+force, p+theta x2, p+theta x1
constexpr int KEY_TUNE_FBANDS = 107, KEY_TUNE_TILE = 111, KEY_TUNE_RC = 112, KEY_TUNE_HIST = 113;
constexpr double TILE_MAX_POINTS = 4.5e6;  // grids up to 2048^2 take the tile kernel (sweep in profiles/README.md: it wins up to there)
constexpr int KEY_TUNE_NW1 = 101, KEY_TUNE_NW2 = 102, KEY_TUNE_BANDS = 103, KEY_TUNE_PSEG = 104,
              KEY_TUNE_PTX = 105, KEY_TUNE_GENERIC = 106;

thread_local char g_err[512] = "";

struct Ctx {
    bool ready = false, prepared = false, cuda_failed = false;
    int model = 0, ntheta = 0, np = 0;
    double xmin = 0, xmax = 0, pmin = 0, pmax = 0, dt = 0, eps = 0.01, t = 0;
    int bc_x = 0, bc_p = 1, prec = 64;
    int spline = 0;  // 0: f'' by eq (16) (the paper's method), 1: global spline, system (15) (vlasov_gs.cuh)
    int halo_lo = 0, halo_hi = 0;  // slab mode (p-slab sharding): halo rows below / above the Np owned rows
    int np_ext() const { return np + halo_lo + halo_hi; }
    void* owned(int k) const;      // first owned row of state buffer k
    int order = 2;   // 2: the paper's time split; 4: its triple-jump composition S2(g1 dt) S2(g2 dt) S2(g1 dt) (L238)
    double dt_sub = 0;                                 // time step of the sub-step being enqueued (= dt for order 2)
    int* srow_sub[2] = {nullptr, nullptr};            // order 4: row tables of the sub-steps g1 dt, g2 dt
    double* wrow_sub[2] = {nullptr, nullptr};
    double* gsab = nullptr;          // [Np][4] = 1-a, a, A/6, B/6 of a half theta shift
    int gs_rbands = 0, gs_rrpb = 0;  // bands of the global-spline theta kernel
    bool history = false;
    int fuse = 2;  // 0: p and theta passes apart, 1: adjacent half theta shifts in one pass, 2: p + theta in one pass
    cudaStream_t stream = nullptr;
    int sm_count = 148;

    void* f[2] = {nullptr, nullptr};  // ping-pong copies of the state
    int cur = 0;
    bool own_f = false, own_work = false, attached = false;
    void* work = nullptr;
    double* colpart = nullptr;  // inside work
    int cp_bands = 0;

    // small library-owned device buffers
    int* srow = nullptr;
    double *wrow = nullptr, *cos_t = nullptr, *sin_t = nullptr, *ringK = nullptr, *ringV = nullptr;
    double *rho = nullptr, *force = nullptr, *rho_m = nullptr, *phi = nullptr, *mpart = nullptr, *pkpart = nullptr,
           *mom_dev = nullptr, *hist = nullptr;
    int hist_cap = 0, hist_count = 0;
    // one-pass kernel: composite theta weights, band shift ranges, its own density partials
    double *wrow2 = nullptr, *colpart_f = nullptr;
    unsigned* ticket = nullptr;    // last-CTA counter of rho_force_kernel
    double* ringpart = nullptr;    // [Ntheta / RING_L][Ntheta] chunk partials of the ring convolution
    unsigned* ringtick = nullptr;  // [Ntheta / 256] last-CTA counters of its tiles
    double* caspart = nullptr;     // [mbands * column blocks][4] partials of the Casimir pass, then 4 results
    // CUDA graph of two consecutive steady-state steps of the one-pass path (density/force + pass, twice), one
    // per parity of the ping-pong; captured on a private stream, launched on the attached one
    bool graphs = true;
    bool pdl = true;  // programmatic dependent launch between the pass and the density / force kernels (KEY_TUNE_PDL)
    cudaGraphExec_t gexec[2] = {nullptr, nullptr};
    unsigned graph_kernels[2] = {0, 0};
    cudaStream_t cap_stream = nullptr;
    int fbands[3] = {0, 0, 0}, frpb[3] = {0, 0, 0}, fcols[3] = {0, 0, 0};
    int fedge = 100;       // relative width (percent) of the first / last column block (KEY_TUNE_FEDGE)
    int tune_fedge = 0;
    int fx0 = 0, fxw = 0;  // source positions the column blocks of the one-pass kernel tile: [fx0, fx0 + fxw)
    bool onepass = false;
    int tune_fbands = 0;
    // small grids (state in L2): the tile kernel instead of the warp-specialised one (vlasov_tile.cuh); KEY_TUNE_TILE:
    // 0 = by size, 1 = whenever its conditions hold, 2 = never
    // history on the one-pass path (history_rows_kernel): per-row sums of the tile kernel, 1 / T_j of every row
    double *rowmom = nullptr, *hist_invT = nullptr;
    bool want_rowmom = false;
    vl::HistArgs hist_pending = {};  // history of the step that just ended, to ride along with the next density / force launch
    int rc_max_cluster = 8;  // largest cluster rho_force_cluster_kernel may be launched with (16 where the GPU can place it)
    int tune_hist = 0;       // KEY_TUNE_HIST: 2 = history always by the separate passes (theta, p + theta, moments pass)
    int tune_rc = 0;         // KEY_TUNE_RC: 2 = never the cluster kernel (the ticketed rho_force_kernel on every grid)
    bool tile = false;
    int tune_tile = 0, tile_nr = 16;
    int fnw() const { return tile ? 1 : FW_NTW; }  // rows of density partials per band of the one-pass kernel
    int fgran(size_t elem) const { return (int)(16 / elem); }  // lanes per column-block granule
    std::vector<int> h_srow;

    // launch configuration
    int nw[3] = {0, 6, 6};         // warps per theta CTA for NSTAGE = 1, 2
    int nchunks[3] = {0, 0, 0};
    int nbands[3] = {0, 0, 0}, rpb[3] = {0, 0, 0};
    bool theta_bulk = false;       // rows are multiples of 16 bytes: bulk-copy kernel (else the generic one)
    vl::ThetaBulkGrid bgrid[3] = {};
    int bctas[3] = {0, 0, 0};
    int mbands = 0, mrpb = 0;      // moments pass
    int p_tx = 128, p_seg = 0, p_nseg = 0;
    int tune_nw1 = 0, tune_nw2 = 0, tune_bands = 0, tune_pseg = 0, tune_ptx = 0;
    bool force_generic = false;    // KEY_TUNE_GENERIC: use the generic theta kernel even when rows are aligned
    unsigned long long launches = 0;

    // optional per-kernel timing with CUDA events on the launch stream (KEY_PROFILE)
    bool profile = false;
    std::vector<cudaEvent_t> ev[NCLS][2];  // class: 0 theta x1, 1 theta x2, 2 p, 3 rho+force, 4 p+theta x2, 5 p+theta x1
    size_t ev_used[NCLS] = {0, 0, 0, 0, 0, 0};
};

Ctx G;
void* Ctx::owned(int k) const {
    return static_cast<char*>(f[k]) + (size_t)halo_lo * (size_t)ntheta * (size_t)(prec == 32 ? 4 : 8);
}
constexpr size_t EV_CAP = 2048;

void prof_begin(int cls) {
    if (!G.profile || G.ev_used[cls] >= EV_CAP) return;
    if (G.ev[cls][0].size() <= G.ev_used[cls]) {
        cudaEvent_t a, b;
        if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) return;
        G.ev[cls][0].push_back(a);
        G.ev[cls][1].push_back(b);
    }
    cudaEventRecord(G.ev[cls][0][G.ev_used[cls]], G.stream);
}
void prof_end(int cls) {
    if (!G.profile || G.ev_used[cls] >= EV_CAP || G.ev[cls][1].size() <= G.ev_used[cls]) return;
    cudaEventRecord(G.ev[cls][1][G.ev_used[cls]], G.stream);
    G.ev_used[cls]++;
}
void prof_free() {
    for (int c = 0; c < NCLS; ++c)
        for (int k = 0; k < 2; ++k) {
            for (cudaEvent_t e : G.ev[c][k]) cudaEventDestroy(e);
            G.ev[c][k].clear();
        }
}

int fail(int code, const char* fmt, const char* a = "") {
    snprintf(g_err, sizeof(g_err), fmt, a);
    return code;
}

#define CU(call)                                                                                 \
    do {                                                                                         \
        cudaError_t e_ = (call);                                                                 \
        if (e_ != cudaSuccess) {                                                                 \
            G.cuda_failed = true;                                                                \
            snprintf(g_err, sizeof(g_err), "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_), \
                     __FILE__, __LINE__);                                                        \
            return VLASOV_ECUDA;                                                                 \
        }                                                                                        \
    } while (0)

#define LAUNCH_CHECK()                 \
    do {                               \
        G.launches++;                  \
        CU(cudaGetLastError());        \
    } while (0)

size_t elem_bytes() { return G.prec == 32 ? 4 : 8; }
size_t state_bytes() { return (size_t)G.ntheta * (size_t)G.np_ext() * elem_bytes(); }  // owned rows + halos
size_t owned_bytes() { return (size_t)G.ntheta * (size_t)G.np * elem_bytes(); }
size_t round256(size_t b) { return (b + 255) & ~(size_t)255; }
int cdiv(int a, int b) { return (a + b - 1) / b; }

void free_small() {
    void* ptrs[] = {G.srow, G.wrow, G.cos_t, G.sin_t, G.ringK, G.ringV, G.rho, G.force, G.rho_m,
                    G.phi,  G.mpart, G.pkpart, G.mom_dev, G.hist, G.wrow2, G.colpart_f, G.ticket, G.caspart, G.ringpart, G.ringtick,
                    G.gsab, G.srow_sub[0], G.srow_sub[1], G.wrow_sub[0], G.wrow_sub[1], G.rowmom, G.hist_invT};
    for (void* p : ptrs)
        if (p) cudaFree(p);
    G.srow = nullptr;
    G.wrow = G.cos_t = G.sin_t = G.ringK = G.ringV = G.rho = G.force = G.rho_m = G.phi = G.mpart = G.pkpart =
        G.mom_dev = G.hist = G.wrow2 = G.colpart_f = nullptr;
    G.ticket = nullptr;
    G.rowmom = G.hist_invT = nullptr;
    G.gsab = nullptr;
    G.srow_sub[0] = G.srow_sub[1] = nullptr;
    G.wrow_sub[0] = G.wrow_sub[1] = nullptr;
    G.caspart = nullptr;
    G.ringpart = nullptr;
    G.ringtick = nullptr;
    G.hist_cap = G.hist_count = 0;
}

void free_graphs() {
    for (int k = 0; k < 2; ++k) {
        if (G.gexec[k]) cudaGraphExecDestroy(G.gexec[k]);
        G.gexec[k] = nullptr;
    }
}

void free_big() {
    free_graphs();  // they hold the buffer addresses
    if (G.own_f && G.f[0]) cudaFree(G.f[0]);
    if (G.own_work && G.work) cudaFree(G.work);
    G.f[0] = G.f[1] = G.work = nullptr;
    G.colpart = nullptr;
    G.own_f = G.own_work = G.attached = false;
    G.cur = 0;
}

// launch with programmatic stream serialisation (programmatic dependent launch): the kernel may be scheduled while its
// predecessor in the stream still runs and waits for it inside (ptx::pdl_wait).  Works in stream capture too (the
// graph gets a programmatic edge).  G.pdl = false: an ordinary launch.
template <typename... KArgs, typename... Args>
cudaError_t launch_pdl(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = G.stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = G.pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kern, KArgs(args)...);
}

template <typename T, int NSTAGE>
size_t theta_smem_bytes(int nw) {
    constexpr int LANES = (NSTAGE == 2) ? 31 : 32;
    const int chunk = nw * LANES * R_THETA;
    const int lenA = chunk + 9 * NSTAGE;
    return (size_t)(((lenA + 1) & ~1) + chunk) * sizeof(T);
}

// choose warps per CTA so that the ragged last chunk wastes little; bands so that one wave fills the GPU
template <typename T, int NSTAGE>
int configure_theta(int tune_nw) {
    constexpr int LANES = (NSTAGE == 2) ? 31 : 32;
    const int tile = LANES * R_THETA;
    const int tiles = cdiv(G.ntheta, tile);
    int nw = 0;
    if (tune_nw > 0) {
        nw = tune_nw;
    } else {
        int best_nw = 1, best_waste = 1 << 30;
        for (int c = 8; c >= 1; --c) {
            const int waste = cdiv(tiles, c) * c - tiles;
            if (waste * 25 <= tiles) {  // <= 4 %
                nw = c;
                break;
            }
            if (waste < best_waste) {
                best_waste = waste;
                best_nw = c;
            }
        }
        if (nw == 0) nw = best_nw;
    }
    if (nw > 12) nw = 12;
    G.nw[NSTAGE] = nw;
    G.nchunks[NSTAGE] = cdiv(tiles, nw);
    auto kern = vl::theta_sweep_generic_kernel<T, NSTAGE, R_THETA>;
    const size_t smem = theta_smem_bytes<T, NSTAGE>(nw);
    CU(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int occ = 1;
    CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, nw * 32, smem));
    if (occ < 1) occ = 1;
    int bands = G.tune_bands > 0 ? G.tune_bands : (G.sm_count * occ) / G.nchunks[NSTAGE];
    if (bands < 1) bands = 1;
    if (bands > G.np) bands = G.np;
    G.rpb[NSTAGE] = cdiv(G.np, bands);
    G.nbands[NSTAGE] = cdiv(G.np, G.rpb[NSTAGE]);
    return VLASOV_OK;
}

// bulk-copy kernel: every warp is a pipeline over (band of rows) x (chunk of columns); one wave of warps
template <typename T, int NSTAGE>
int configure_theta_bulk() {
    using C = vl::ThetaBulk<T, NSTAGE, R_THETA, TB_NS, TB_WARPS>;
    auto kern = vl::theta_sweep_bulk_kernel<T, NSTAGE, R_THETA, TB_NS, TB_WARPS, TB_MINB>;
    CU(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_BYTES));
    int occ = 1;
    CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, TB_WARPS * 32, C::SMEM_BYTES));
    if (occ < 1) occ = 1;
    const int nchunks = cdiv(G.ntheta, C::CHUNK);
    int bands = G.tune_bands > 0 ? G.tune_bands : (G.sm_count * occ * TB_WARPS) / nchunks;
    const int max_bands = G.np >= 16 ? G.np / 8 : 1;  // at least 8 rows per pipeline
    if (bands > max_bands && G.tune_bands <= 0) bands = max_bands;
    if (bands < 1) bands = 1;
    if (bands > G.np) bands = G.np;
    vl::ThetaBulkGrid g;
    g.nchunks = nchunks;
    g.rows_per_band = cdiv(G.np, bands);
    g.nbands = cdiv(G.np, g.rows_per_band);
    G.bgrid[NSTAGE] = g;
    G.bctas[NSTAGE] = cdiv(g.nchunks * g.nbands, TB_WARPS);
    return VLASOV_OK;
}

// one-pass kernel (p shift + NST theta half shifts): column blocks x bands, one CTA per SM.  Conditions: the
// integer theta shift must not increase with the row (the column sums follow it by moving left), and inside a
// band it may drift by at most the width of the narrowest column block (then at most two CTAs add to an entry
// of the density partials).  Sets G.fbands[NST] = 0 when the grid does not qualify.
template <typename T, int NST>
int configure_fused() {
    CU(cudaFuncSetAttribute(vl::strang_fused_ws_kernel<T, NST, FU_R<T>, FW_NSTG, FW_NTW, false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                            (int)vl::FusedWsCfg<T, NST, FU_R<T>, FW_NSTG, FW_NTW, false>::SMEM_BYTES));
    CU(cudaFuncSetAttribute(vl::strang_fused_ws_kernel<T, NST, FU_R<T>, FW_NSTG, FW_NTW, true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                            (int)vl::FusedWsCfg<T, NST, FU_R<T>, FW_NSTG, FW_NTW, true>::SMEM_BYTES));
    const int np = G.np, nt = G.ntheta;
    G.fbands[NST] = 0;
    for (int j = 1; j < np; ++j)
        if (G.h_srow[j] > G.h_srow[j - 1]) return VLASOV_OK;  // shift wrapped around the circle: not monotonic
    if ((double)nt * sizeof(T) >= 2147483648.0) return VLASOV_OK;
    const int gran = G.fgran(sizeof(T));
    // Zero-extended theta axis: a row's outputs [0, Ntheta) come from the source positions [S, Ntheta + S), S its integer
    // shift, so the blocks tile [min(0, S_min), Ntheta + max(0, S_max)) (S of two half shifts; x0 even: 16-byte starts)
    int x0 = 0, xw = nt;
    if (G.bc_x != vl::BC_PERIODIC) {
        int smin = 0, smax = 0;
        for (int j = 0; j < np; ++j) {
            smin = std::min(smin, 2 * G.h_srow[j]);
            smax = std::max(smax, 2 * G.h_srow[j]);
        }
        if (smax - smin > 4 * nt) return VLASOV_OK;  // shifts of several domain lengths: the separate kernels
        x0 = -((-smin + 1) & ~1);
        xw = nt + smax - x0;
    }
    G.fx0 = x0;
    G.fxw = xw;
    // (narrower edge blocks were measured at 4096^2, 40 .. 100 %: no effect on the pass, so 100 unless tuned)
    G.fedge = (G.bc_x != vl::BC_PERIODIC && NST == 2 && G.tune_fedge > 0) ? G.tune_fedge : 100;
    const int edge_w = NST == 2 ? G.fedge : 100;
    const int cols = vl::fused_block_cols(xw, FU_R<T>, gran, edge_w);
    int wmin = nt;
    for (int c = 0; c < cols; ++c) {
        int i0, wd;
        vl::fused_block_range(c, cols, xw, FU_R<T>, gran, &i0, &wd, edge_w);
        wmin = wd < wmin ? wd : wmin;
    }
    if (wmin < 1) return VLASOV_OK;
    // one CTA per SM; but no bands shorter than 32 rows: every band adds 12 rows of density partials for
    // rho_force_kernel to read and a nine-row halo (sweep on 256^2 .. 2048^2 in profiles/README.md)
    int bands = G.sm_count / cols;
    if (bands > np / 32) bands = np / 32;
    if (G.tune_fbands > 0) bands = G.tune_fbands;
    if (bands < 1) bands = 1;
    if (bands > np) bands = np;
    int rpb = cdiv(np, bands);
    for (;;) {
        bands = cdiv(np, rpb);
        int worst = 0;
        for (int b = 0; b < bands; ++b) {
            const int ja = b * rpb, jb = (b + 1) * rpb < np ? (b + 1) * rpb : np;
            const int drift = NST * (G.h_srow[ja] - G.h_srow[jb - 1]);
            worst = drift > worst ? drift : worst;
        }
        if (worst <= wmin || rpb == 1) {
            if (worst > wmin) return VLASOV_OK;
            break;
        }
        rpb = (rpb + 1) / 2;
    }
    if ((size_t)bands * G.fnw() > (size_t)G.sm_count * 64) return VLASOV_OK;  // partials would outgrow the state
    G.fbands[NST] = bands;
    G.frpb[NST] = rpb;
    G.fcols[NST] = cols;
    return VLASOV_OK;
}

// the tile kernel (vlasov_tile.cuh) for NST half shifts: fp64, periodic theta, integer shift not increasing with the row
// and drifting by no more than the narrowest column block inside a tile's rows.  false: the grid does not qualify.
template <typename T, int NST, int NR, int R>
bool configure_tile() {
    using C = vl::TileCfg<T, NST, NR, R>;
    const int np = G.np, nt = G.ntheta;
    for (int j = 1; j < np; ++j)
        if (G.h_srow[j] > G.h_srow[j - 1]) return false;
    const int gran = G.fgran(sizeof(T));
    const int cols = vl::fused_block_cols(nt, C::R, gran, 100);
    int wmin = nt;
    for (int c = 0; c < cols; ++c) {
        int i0, wd;
        vl::fused_block_range(c, cols, nt, C::R, gran, &i0, &wd, 100);
        wmin = wd < wmin ? wd : wmin;
    }
    if (wmin < 1) return false;
    const int bands = cdiv(np, C::NR);
    for (int b = 0; b < bands; ++b) {
        const int ja = b * C::NR, jb = (b + 1) * C::NR < np ? (b + 1) * C::NR : np;
        if (NST * (G.h_srow[ja] - G.h_srow[jb - 1]) > wmin) return false;
    }
    if (cudaFuncSetAttribute(vl::strang_tile_kernel<T, NST, NR, R>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM_BYTES) !=
        cudaSuccess) {
        cudaGetLastError();
        return false;
    }
    G.fbands[NST] = bands;
    G.frpb[NST] = C::NR;
    G.fcols[NST] = cols;
    G.fx0 = 0;
    G.fxw = nt;
    G.fedge = 100;
    return true;
}

template <typename T>
int configure_all() {
    int rc;
    if ((rc = configure_theta<T, 1>(G.tune_nw1)) != 0) return rc;
    if ((rc = configure_theta<T, 2>(G.tune_nw2)) != 0) return rc;
    G.theta_bulk = (G.ntheta % (16 / (int)sizeof(T)) == 0) && !G.force_generic;
    if (G.theta_bulk) {
        if ((rc = configure_theta_bulk<T, 1>()) != 0) return rc;
        if ((rc = configure_theta_bulk<T, 2>()) != 0) return rc;
    }
    {   // clusters of 16 CTAs are not portable: allow them for the density / force kernel and ask whether one can be placed
        G.rc_max_cluster = 8;
        if (cudaFuncSetAttribute(vl::rho_force_cluster_kernel, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) == cudaSuccess) {
            cudaLaunchConfig_t cfg = {};
            cfg.gridDim = dim3(16);
            cfg.blockDim = dim3(vl::RC_COLS * vl::RC_GROUPS);
            cudaLaunchAttribute at[1];
            at[0].id = cudaLaunchAttributeClusterDimension;
            at[0].val.clusterDim.x = 16;
            at[0].val.clusterDim.y = 1;
            at[0].val.clusterDim.z = 1;
            cfg.attrs = at;
            cfg.numAttrs = 1;
            int ncl = 0;
            if (cudaOccupancyMaxActiveClusters(&ncl, vl::rho_force_cluster_kernel, &cfg) == cudaSuccess && ncl >= 1)
                G.rc_max_cluster = 16;
        }
        cudaGetLastError();
    }
    G.onepass = (G.fuse >= 2) && (G.halo_lo + G.halo_hi == 0);
    G.tile = false;
    if (G.onepass && G.bc_x == vl::BC_PERIODIC && G.tune_tile != 2 &&
        (G.tune_tile == 1 || (double)G.ntheta * (double)G.np <= TILE_MAX_POINTS)) {
        G.tile = true;
        // tile shape by size (sweeps in profiles/README.md): 8 rows x 224 columns on the smallest grids (more CTAs), 12 x 352 (384
        // threads) around 1024^2 (fewer, larger tiles), 16 x 224 beyond
        const double npts = (double)G.ntheta * (double)G.np;
        G.tile_nr = npts <= 131072.0 ? 8 : (npts >= 9.5e5 && npts <= 1.2e6 ? 12 : 16);
        G.tile = G.tile_nr == 8    ? (configure_tile<T, 1, 8, 7>() && configure_tile<T, 2, 8, 7>())
                 : G.tile_nr == 12 ? (configure_tile<T, 1, 12, 11>() && configure_tile<T, 2, 12, 11>())
                                   : (configure_tile<T, 1, 16, 7>() && configure_tile<T, 2, 16, 7>());
    }
    if (G.onepass && !G.tile) {
        if ((rc = configure_fused<T, 1>()) != 0) return rc;
        if ((rc = configure_fused<T, 2>()) != 0) return rc;
        G.onepass = G.fbands[1] > 0 && G.fbands[2] > 0;
    }
    // p shift: 128 adjacent columns per CTA; segments so that a bit more than one wave of CTAs exists
    G.p_tx = G.tune_ptx > 0 ? G.tune_ptx : 128;
    if (G.p_tx > 256) G.p_tx = 256;
    int occ = 1;
    CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, vl::p_sweep_kernel<T>, G.p_tx, 0));
    if (occ < 1) occ = 1;
    const int colblocks = cdiv(G.ntheta, G.p_tx);
    int nseg = (G.sm_count * occ) / colblocks;  // floor: every CTA resident at once, no second partial wave
    if (nseg < 1) nseg = 1;
    int seg = G.tune_pseg > 0 ? G.tune_pseg : cdiv(G.np, nseg);
    if (seg < 40 && G.tune_pseg <= 0) seg = 40;  // keep the 9-row halo re-read below ~20 %
    if (seg > G.np) seg = G.np;
    G.p_seg = seg;
    G.p_nseg = cdiv(G.np, seg);
    // moments pass
    G.mbands = cdiv(G.sm_count * 8, cdiv(G.ntheta, 256));
    if (G.mbands > G.np) G.mbands = G.np;
    if (G.mbands < 1) G.mbands = 1;
    G.mrpb = cdiv(G.np, G.mbands);
    G.mbands = cdiv(G.np, G.mrpb);
    return VLASOV_OK;
}

int max_bands_bound() {
    // upper bound of every band count configure_all() can pick: one band per slot of the GPU, or per row
    int b = G.sm_count * 32;
    if (G.tune_bands > b) b = G.tune_bands;
    if (b > G.np) b = G.np;
    return b < 1 ? 1 : b;
}

size_t workspace_bytes() {
    return round256(state_bytes()) + round256((size_t)max_bands_bound() * G.ntheta * sizeof(double));
}

// per-row integer shift and ten weights of a theta shift over the time tau (eq (9): displacement p_j tau)
void row_tables(double tau, std::vector<int>& srow, std::vector<double>& wrow) {
    const int nt = G.ntheta, np = G.np;
    const double dx = (G.xmax - G.xmin) / (double)nt, dp = (G.pmax - G.pmin) / (double)np;
    for (int j = 0; j < np; ++j) {
        const double p = G.pmin + (double)j * dp;
        const double disp = p * tau;
        double sf, a;
        vl::split_shift(-disp / dx, &sf, &a);
        if (G.bc_x == vl::BC_PERIODIC) {
            sf = fmod(sf, (double)nt);
        } else {
            const double lim = (double)nt + 64.0;
            sf = fmin(fmax(sf, -lim), lim);
        }
        srow[j] = (int)sf;
        vl::spline_fd8_weights(a, &wrow[(size_t)j * vl::WROW_STRIDE]);
        wrow[(size_t)j * vl::WROW_STRIDE + 10] = sf;
    }
}

// fp32 arithmetic: the ten weights of every row -> the nine difference-form weights (vl::diff_form_weights)
void row_tables_to_difference_form(std::vector<double>& wrow) {
    for (int j = 0; j < G.np; ++j) {
        double* w = &wrow[(size_t)j * vl::WROW_STRIDE];
        double U[9];
        vl::diff_form_weights(w, 10, vl::FD_C, U);
        for (int m = 0; m < 9; ++m) w[m] = U[m];
        w[9] = 0.0;
    }
}

int prepare_tables() {
    const int nt = G.ntheta, np = G.np;
    const double dx = (G.xmax - G.xmin) / (double)nt, dp = (G.pmax - G.pmin) / (double)np;
    const double tau = 0.5 * G.dt;

    // per-row shift of one half step: displacement p_j tau (eq (9)), u = -disp/dx cells
    std::vector<int> srow(np);
    std::vector<double> wrow((size_t)(np + FU_PAD) * vl::WROW_STRIDE, 0.0);  // FU_PAD rows of padding
    row_tables(tau, srow, wrow);
    G.h_srow = srow;
    // (from the plain weights, before the fp32 tables go to difference form)
    // history on the one-pass path: 1 / T_j, T_j = e^{-i s_j dx} sum_m w_m e^{-i (m - 4) dx} (history_rows_kernel)
    std::vector<double> inv((size_t)np * 2);
    for (int j = 0; j < np; ++j) {
        const double* w = &wrow[(size_t)j * vl::WROW_STRIDE];
        double tr = 0.0, ti = 0.0;
        for (int m = 0; m < 10; ++m) {
            const double ph = -((double)srow[j] + (double)(m - 4)) * dx;
            tr += w[m] * cos(ph);
            ti += w[m] * sin(ph);
        }
        const double n2 = tr * tr + ti * ti;
        inv[2 * j] = tr / n2;
        inv[2 * j + 1] = -ti / n2;
    }
    // composite weights of two equal half shifts, W = w * w (19 taps): the one-pass kernel applies both at once
    const int W2 = G.bc_x == vl::BC_PERIODIC ? 20 : 32;  // FusedWsCfg<T, 2, ..., ZX>::WST
    std::vector<double> wrow2((size_t)(np + FU_PAD) * W2, 0.0);
    for (int j = 0; j < np; ++j) {
        const double* w = &wrow[(size_t)j * vl::WROW_STRIDE];
        double* W = &wrow2[(size_t)j * W2];
        for (int n = 0; n < 19; ++n) {
            double acc = 0.0;
            for (int m = (n > 9 ? n - 9 : 0); m <= (n < 9 ? n : 9); ++m) acc += w[m] * w[n - m];
            W[n] = acc;
        }
        W[19] = 2.0 * (double)srow[j];  // integer part of the two half shifts together
        if (W2 == 32) {  // zero-extended theta axis: the single half shift too (rows near the ends apply it twice)
            for (int m = 0; m < 10; ++m) W[20 + m] = w[m];
            W[30] = (double)srow[j];
        }
        if (G.prec == 32) {  // fp32 arithmetic: both tables hold the difference-form weights (vl::diff_form_weights)
            double U[18];
            vl::diff_form_weights(W, 19, 2 * vl::FD_C + 1, U);
            for (int n = 0; n < 18; ++n) W[n] = U[n];
            W[18] = 0.0;
        }
    }
    if (G.prec == 32) row_tables_to_difference_form(wrow);
    if (G.order == 4) {
        // triple jump: S2(g1 dt) S2(g2 dt) S2(g1 dt), g1 = 1/(2 - 2^(1/3)), g2 = 1 - 2 g1 < 0 (refs [31], [44])
        const double g1 = 1.0 / (2.0 - cbrt(2.0)), g[2] = {g1, 1.0 - 2.0 * g1};
        for (int k = 0; k < 2; ++k) {
            std::vector<int> sr(np);
            std::vector<double> wr((size_t)(np + FU_PAD) * vl::WROW_STRIDE, 0.0);
            row_tables(0.5 * g[k] * G.dt, sr, wr);
            if (G.prec == 32) row_tables_to_difference_form(wr);
            CU(cudaMalloc(&G.srow_sub[k], sizeof(int) * np));
            CU(cudaMalloc(&G.wrow_sub[k], sizeof(double) * wr.size()));
            CU(cudaMemcpy(G.srow_sub[k], sr.data(), sizeof(int) * np, cudaMemcpyHostToDevice));
            CU(cudaMemcpy(G.wrow_sub[k], wr.data(), sizeof(double) * wr.size(), cudaMemcpyHostToDevice));
        }
    }
    CU(cudaMalloc(&G.wrow2, sizeof(double) * wrow2.size()));
    CU(cudaMemcpy(G.wrow2, wrow2.data(), sizeof(double) * wrow2.size(), cudaMemcpyHostToDevice));
    std::vector<double> ct(nt), st(nt);
    for (int i = 0; i < nt; ++i) {
        const double th = G.xmin + (double)i * dx;
        ct[i] = cos(th);
        st[i] = sin(th);
    }
    CU(cudaMalloc(&G.srow, sizeof(int) * np));
    CU(cudaMalloc(&G.wrow, sizeof(double) * wrow.size()));
    CU(cudaMalloc(&G.cos_t, sizeof(double) * nt));
    CU(cudaMalloc(&G.sin_t, sizeof(double) * nt));
    CU(cudaMemcpy(G.srow, srow.data(), sizeof(int) * np, cudaMemcpyHostToDevice));
    CU(cudaMemcpy(G.wrow, wrow.data(), sizeof(double) * wrow.size(), cudaMemcpyHostToDevice));
    CU(cudaMemcpy(G.cos_t, ct.data(), sizeof(double) * nt, cudaMemcpyHostToDevice));
    CU(cudaMemcpy(G.sin_t, st.data(), sizeof(double) * nt, cudaMemcpyHostToDevice));
    if (G.model == VLASOV_MODEL_RING) {
        // eq (2) (L33-L35): V(x) = -1/(sqrt2 sqrt(1 - cos x + eps)); K = -dV/dx; 1 - cos x = 2 sin^2(x/2)
        std::vector<double> K(nt), V(nt);
        for (int m = 0; m < nt; ++m) {
            const double x = (double)m * dx;
            const double h = sin(0.5 * x);
            const double q = 2.0 * h * h + G.eps;
            V[m] = -1.0 / (sqrt(2.0) * sqrt(q));
            K[m] = (m == 0) ? 0.0 : -sin(x) / (2.0 * sqrt(2.0) * q * sqrt(q));
        }
        CU(cudaMalloc(&G.ringK, sizeof(double) * nt));
        CU(cudaMalloc(&G.ringV, sizeof(double) * nt));
        CU(cudaMemcpy(G.ringK, K.data(), sizeof(double) * nt, cudaMemcpyHostToDevice));
        CU(cudaMemcpy(G.ringV, V.data(), sizeof(double) * nt, cudaMemcpyHostToDevice));
        CU(cudaMalloc(&G.ringpart, sizeof(double) * (size_t)cdiv(nt, vl::RING_L) * nt));
        CU(cudaMalloc(&G.ringtick, sizeof(unsigned) * cdiv(nt, 256)));
        CU(cudaMemset(G.ringtick, 0, sizeof(unsigned) * cdiv(nt, 256)));
    }
    CU(cudaMalloc(&G.rho, sizeof(double) * nt));
    CU(cudaMalloc(&G.force, sizeof(double) * nt));
    CU(cudaMalloc(&G.rho_m, sizeof(double) * nt));
    CU(cudaMalloc(&G.phi, sizeof(double) * nt));
    CU(cudaMemset(G.rho, 0, sizeof(double) * nt));
    CU(cudaMemset(G.force, 0, sizeof(double) * nt));
    CU(cudaMalloc(&G.mpart, sizeof(double) * 2 * cdiv(nt, vl::RR_COLS)));
    CU(cudaMalloc(&G.ticket, sizeof(unsigned)));
    CU(cudaMemset(G.ticket, 0, sizeof(unsigned)));
    CU(cudaMalloc(&G.mom_dev, sizeof(double) * 8));

    int rc = (G.prec == 32) ? configure_all<float>() : configure_all<double>();
    if (rc != 0) return rc;
    if (G.spline == 1) {
        // global spline (system (15), L100-L102): per row 1-a, a, A/6, B/6 of a half theta shift
        std::vector<double> gsab((size_t)np * 4);
        for (int j = 0; j < np; ++j) {
            const double p = G.pmin + (double)j * dp;
            double sf, a;
            vl::split_shift(-(p * tau) / dx, &sf, &a);
            const double al = 1.0 - a;
            gsab[(size_t)j * 4 + 0] = al;
            gsab[(size_t)j * 4 + 1] = a;
            gsab[(size_t)j * 4 + 2] = al * (al * al - 1.0) / 6.0;
            gsab[(size_t)j * 4 + 3] = a * (a * a - 1.0) / 6.0;
        }
        CU(cudaMalloc(&G.gsab, sizeof(double) * gsab.size()));
        CU(cudaMemcpy(G.gsab, gsab.data(), sizeof(double) * gsab.size(), cudaMemcpyHostToDevice));
        G.onepass = false;
        {   // theta kernel: 4 warps x 216 columns per CTA, bands of rows for one resident wave
            int occ2 = 1;
            if (G.prec == 32) CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ2, vl::gs_theta_rec_kernel<float>, vl::GS_RWARPS * 32, 0));
            else CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ2, vl::gs_theta_rec_kernel<double>, vl::GS_RWARPS * 32, 0));
            if (occ2 < 1) occ2 = 1;
            const int nchr = cdiv(cdiv(nt, vl::GS_ROUT), vl::GS_RWARPS);
            int b2 = (G.sm_count * occ2) / nchr;
            if (b2 < 1) b2 = 1;
            if (b2 > max_bands_bound()) b2 = max_bands_bound();
            if (b2 > np) b2 = np;
            G.gs_rrpb = cdiv(np, b2);
            G.gs_rbands = cdiv(np, G.gs_rrpb);
        }
        CU(cudaFuncSetAttribute(vl::gs_p_rec_kernel<float>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)vl::gs_p_rec_smem<float>()));
        CU(cudaFuncSetAttribute(vl::gs_p_rec_kernel<double>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)vl::gs_p_rec_smem<double>()));
    }
    CU(cudaMalloc(&G.pkpart, sizeof(double) * 2 * (size_t)G.mbands * cdiv(nt, 256)));
    CU(cudaMalloc(&G.caspart, sizeof(double) * 4 * ((size_t)G.mbands * cdiv(nt, 256) + 1)));
    if (G.onepass && G.bc_x == vl::BC_PERIODIC) {
        CU(cudaMalloc(&G.hist_invT, sizeof(double) * inv.size()));
        CU(cudaMemcpy(G.hist_invT, inv.data(), sizeof(double) * inv.size(), cudaMemcpyHostToDevice));
        // (the tile kernel leaves the row sums per column block; on the large grids a read pass leaves one set per row)
        const size_t nblk = G.tile ? (size_t)(G.fcols[2] > G.fcols[1] ? G.fcols[2] : G.fcols[1]) : 1;
        CU(cudaMalloc(&G.rowmom, sizeof(double) * 3 * nblk * np));
    }
    if (G.onepass) {
        const size_t nb = (size_t)(G.fbands[2] > G.fbands[1] ? G.fbands[2] : G.fbands[1]) * G.fnw();
        CU(cudaMalloc(&G.colpart_f, sizeof(double) * nb * nt));
        CU(cudaMemset(G.colpart_f, 0, sizeof(double) * nb * nt));
    }
    G.cp_bands = max_bands_bound();
    return VLASOV_OK;
}

// Tables, counters and launch shapes, once per context.  The uploads above are blocking copies and memsets on the
// legacy default stream, while the kernels run on the stream handed to vlasov_attach, which may be a non-blocking
// stream that nothing orders after the legacy one: the device-wide synchronisation below makes every table and every
// zeroed counter final before any kernel can be enqueued (a one-time cost).  A failure frees what was allocated, so
// that a retry does not leak.
int prepare() {
    if (G.prepared) return VLASOV_OK;
    if (G.spline == 1 && (G.ntheta < vl::GS_MIN_N || G.np < vl::GS_MIN_N))
        return fail(VLASOV_EINVAL, "SPLINE = 1 (global spline) needs at least 32 nodes on both axes");
    if ((G.halo_lo + G.halo_hi > 0) && (G.order == 4 || G.spline == 1))
        return fail(VLASOV_EINVAL, "slab mode is built for ORDER = 2, SPLINE = 0");
    if (G.order == 4 && G.spline == 1)
        return fail(VLASOV_EINVAL, "ORDER = 4 is built for the eq (16) spline only (SPLINE = 0)");
    const int rc = prepare_tables();
    if (rc != VLASOV_OK) {
        free_small();
        return rc;
    }
    if (cudaDeviceSynchronize() != cudaSuccess) {
        free_small();
        CU(cudaGetLastError());
        return fail(VLASOV_ECUDA, "prepare: device synchronisation failed");
    }
    G.prepared = true;
    return VLASOV_OK;
}

int ensure_buffers() {
    int rc = prepare();
    if (rc != 0) return rc;
    if (G.f[0] != nullptr) return VLASOV_OK;
    // never attached: the library owns both copies
    CU(cudaMalloc(&G.f[0], round256(state_bytes())));
    G.own_f = true;
    CU(cudaMalloc(&G.work, workspace_bytes()));
    G.own_work = true;
    G.f[1] = G.work;
    G.colpart = reinterpret_cast<double*>(static_cast<char*>(G.work) + round256(state_bytes()));
    CU(cudaMemsetAsync(G.f[0], 0, state_bytes(), G.stream));
    G.cur = 0;
    return VLASOV_OK;
}

// ---- launches -----------------------------------------------------------------------------------

template <typename T, int NSTAGE>
int launch_theta(bool want_colsums) {
    vl::ThetaArgs<T> a;
    a.fin = static_cast<const T*>(G.owned(G.cur));
    a.fout = static_cast<T*>(G.owned(G.cur ^ 1));
    a.srow = G.srow;
    a.wrow = G.wrow;
    a.colpart = want_colsums ? G.colpart : nullptr;
    a.ntheta = G.ntheta;
    a.np = G.np;
    a.bc_x = G.bc_x;
    a.rows_per_band = G.rpb[NSTAGE];
    prof_begin(NSTAGE - 1);
    if (G.theta_bulk) {
        using C = vl::ThetaBulk<T, NSTAGE, R_THETA, TB_NS, TB_WARPS>;
        vl::theta_sweep_bulk_kernel<T, NSTAGE, R_THETA, TB_NS, TB_WARPS, TB_MINB>
            <<<G.bctas[NSTAGE], TB_WARPS * 32, C::SMEM_BYTES, G.stream>>>(a, G.bgrid[NSTAGE]);
    } else {
        const int nw = G.nw[NSTAGE];
        dim3 grid(G.nchunks[NSTAGE], G.nbands[NSTAGE]);
        vl::theta_sweep_generic_kernel<T, NSTAGE, R_THETA>
            <<<grid, nw * 32, theta_smem_bytes<T, NSTAGE>(nw), G.stream>>>(a);
    }
    prof_end(NSTAGE - 1);
    LAUNCH_CHECK();
    G.cur ^= 1;
    return VLASOV_OK;
}

template <typename T>
int launch_gs_theta_rec(bool want_colsums) {
    vl::GsThetaRecArgs<T> a;
    a.fin = static_cast<const T*>(G.owned(G.cur));
    a.fout = static_cast<T*>(G.owned(G.cur ^ 1));
    a.srow = G.srow;
    a.gsab = G.gsab;
    a.colpart = want_colsums ? G.colpart : nullptr;
    a.ntheta = G.ntheta;
    a.np = G.np;
    a.bc_x = G.bc_x;
    a.rows_per_band = G.gs_rrpb;
    prof_begin(0);
    vl::gs_theta_rec_kernel<T><<<dim3(cdiv(cdiv(G.ntheta, vl::GS_ROUT), vl::GS_RWARPS), G.gs_rbands), vl::GS_RWARPS * 32, 0, G.stream>>>(a);
    prof_end(0);
    LAUNCH_CHECK();
    G.cur ^= 1;
    return VLASOV_OK;
}

template <typename T>
int launch_gs_theta(bool want_colsums) { return launch_gs_theta_rec<T>(want_colsums); }

int theta_bands(int nstage) {
    if (G.spline == 1) return G.gs_rbands;
    return G.theta_bulk ? G.bgrid[nstage].nbands : G.nbands[nstage];
}

int theta_pass(int nstage, bool want_colsums) {
    if (G.spline == 1) {  // global spline: half shifts one at a time (the composite of two would have 119 taps)
        if (nstage == 2) {
            int rc = G.prec == 32 ? launch_gs_theta<float>(false) : launch_gs_theta<double>(false);
            if (rc != 0) return rc;
        }
        return G.prec == 32 ? launch_gs_theta<float>(want_colsums) : launch_gs_theta<double>(want_colsums);
    }
    if (G.prec == 32)
        return nstage == 2 ? launch_theta<float, 2>(want_colsums) : launch_theta<float, 1>(want_colsums);
    return nstage == 2 ? launch_theta<double, 2>(want_colsums) : launch_theta<double, 1>(want_colsums);
}

template <typename T>
int launch_p() {
    vl::PArgs<T> a;
    a.fin = static_cast<const T*>(G.f[G.cur]);   // slab mode: the momentum shift runs over the owned rows AND the halos
    a.fout = static_cast<T*>(G.f[G.cur ^ 1]);
    a.force = G.force;
    a.ntheta = G.ntheta;
    a.np = G.np_ext();
    a.bc_p = G.bc_p;
    a.seg_len = G.p_seg;
    a.dt = G.dt_sub;
    a.dp = (G.pmax - G.pmin) / (double)G.np;
    dim3 grid(cdiv(G.ntheta, G.p_tx), cdiv(G.np_ext(), G.p_seg));
    prof_begin(2);
    vl::p_sweep_kernel<T><<<grid, G.p_tx, 0, G.stream>>>(a);
    prof_end(2);
    LAUNCH_CHECK();
    G.cur ^= 1;
    return VLASOV_OK;
}

template <typename T>
int launch_gs_p() {
    vl::GsPArgs<T> a;
    a.fin = static_cast<const T*>(G.f[G.cur]);
    a.fout = static_cast<T*>(G.f[G.cur ^ 1]);
    a.force = G.force;
    a.ntheta = G.ntheta;
    a.np = G.np;
    a.bc_p = G.bc_p;
    a.dt = G.dt;
    a.dp = (G.pmax - G.pmin) / (double)G.np;
    prof_begin(2);
    vl::gs_p_rec_kernel<T><<<dim3(cdiv(G.ntheta, vl::GS_PRX), cdiv(G.np, vl::GS_PRSEG)), vl::GS_PRX * vl::GS_PRG, vl::gs_p_rec_smem<T>(), G.stream>>>(a);
    prof_end(2);
    LAUNCH_CHECK();
    G.cur ^= 1;
    return VLASOV_OK;
}

int p_pass() {
    if (G.spline == 1) return G.prec == 32 ? launch_gs_p<float>() : launch_gs_p<double>();
    return G.prec == 32 ? launch_p<float>() : launch_p<double>();
}

// one pass: momentum shift with the stored force, then NST theta half shifts, then (optionally) the density
// partials of the result in colpart_f (eqs (11), (12), (9), (10))
template <typename T, int NST>
int launch_fused(bool want_colsums) {
    using CW = vl::FusedWsCfg<T, NST, FU_R<T>, FW_NSTG, FW_NTW>;
    vl::FusedArgs<T> a;
    a.fin = static_cast<const T*>(G.f[G.cur]);
    a.fout = static_cast<T*>(G.f[G.cur ^ 1]);
    a.force = G.force;
    a.wtab = NST == 2 ? G.wrow2 : G.wrow;  // (a zero-extended axis has the wider rows of FusedWsCfg<.., ZX = true>)
    a.bulk_ok = (G.ntheta % CW::EPV == 0) ? 1 : 0;
    a.gran = G.fgran(sizeof(T));
    a.x0 = G.fx0;
    a.edge_w = NST == 2 ? G.fedge : 100;
    a.xw = G.fxw;
    a.colpart = want_colsums ? G.colpart_f : nullptr;
    a.rowmom = (G.tile && G.want_rowmom) ? G.rowmom : nullptr;
    a.cos_t = G.cos_t;
    a.sin_t = G.sin_t;
    a.ntheta = G.ntheta;
    a.np = G.np;
    a.bc_p = G.bc_p;
    a.rows_per_band = G.frpb[NST];
    a.dt = G.dt;
    a.dp = (G.pmax - G.pmin) / (double)G.np;
    dim3 grid(G.fcols[NST], G.fbands[NST]);
    prof_begin(NST == 2 ? 4 : 5);
    if (G.tile) {
        if (G.tile_nr == 8)
            CU(launch_pdl(vl::strang_tile_kernel<T, NST, 8, 7>, grid, dim3(vl::TileCfg<T, NST, 8, 7>::NT), vl::TileCfg<T, NST, 8, 7>::SMEM_BYTES, a));
        else if (G.tile_nr == 12)
            CU(launch_pdl(vl::strang_tile_kernel<T, NST, 12, 11>, grid, dim3(vl::TileCfg<T, NST, 12, 11>::NT),
                          vl::TileCfg<T, NST, 12, 11>::SMEM_BYTES, a));
        else
            CU(launch_pdl(vl::strang_tile_kernel<T, NST, 16, 7>, grid, dim3(vl::TileCfg<T, NST, 16, 7>::NT), vl::TileCfg<T, NST, 16, 7>::SMEM_BYTES, a));
        prof_end(NST == 2 ? 4 : 5);
        LAUNCH_CHECK();
        G.cur ^= 1;
        return VLASOV_OK;
    }
    if (G.bc_x == vl::BC_PERIODIC)
        CU(launch_pdl(vl::strang_fused_ws_kernel<T, NST, FU_R<T>, FW_NSTG, FW_NTW, false>, grid, dim3(CW::NT), CW::SMEM_BYTES, a));
    else
        CU(launch_pdl(vl::strang_fused_ws_kernel<T, NST, FU_R<T>, FW_NSTG, FW_NTW, true>, grid, dim3(CW::NT),
                      vl::FusedWsCfg<T, NST, FU_R<T>, FW_NSTG, FW_NTW, true>::SMEM_BYTES, a));
    prof_end(NST == 2 ? 4 : 5);
    LAUNCH_CHECK();
    G.cur ^= 1;
    return VLASOV_OK;
}

int fused_pass(int nstage, bool want_colsums) {
    if (G.prec == 32)
        return nstage == 2 ? launch_fused<float, 2>(want_colsums) : launch_fused<float, 1>(want_colsums);
    return nstage == 2 ? launch_fused<double, 2>(want_colsums) : launch_fused<double, 1>(want_colsums);
}

// rho (and for HMF the moment partials) from the column sums left in colpart by `bands` bands; with
// fuse_force (HMF only) the same kernel also writes the force
int rho_from_colpart(int bands, double* rho_out, bool hmf_partials, double* colpart = nullptr, bool zero_after = false,
                     bool fuse_force = false) {
    const double dp = (G.pmax - G.pmin) / (double)G.np;
    const double dx = (G.xmax - G.xmin) / (double)G.ntheta;
    const bool sheet = fuse_force && G.model == VLASOV_MODEL_SHEET;
    // (theta axes of up to 1024 columns: from 2048 on the ticketed kernel is faster -- 33.8 against 36.1 us per step at 2048^2,
    // 259.3 against 264.6 at 8192^2 with four chunks of columns per CTA, profiles/README.md)
    if (fuse_force && hmf_partials && G.tune_rc != 2 && G.ntheta <= 1024 && G.ntheta <= vl::RC_COLS * G.rc_max_cluster &&
        G.halo_lo + G.halo_hi == 0) {
        // short theta axis (cfg 1, cfg 2), HMF: density, moments and force by one thread-block cluster instead of the ticketed
        // kernel (cfg 1: 9.3 -> 7.5 us per step, cfg 2: 15.4 -> 14.4)
        cudaLaunchConfig_t cfg = {};
        vl::HistArgs ha = {};
        unsigned ncta = (unsigned)cdiv(G.ntheta, vl::RC_COLS);
        if (G.hist_pending.rowmom != nullptr && (int)ncta + 1 <= G.rc_max_cluster) {  // one more CTA writes the pending history entry
            ha = G.hist_pending;
            G.hist_pending.rowmom = nullptr;
            ncta += 1;
        }
        cfg.gridDim = dim3(ncta);
        cfg.blockDim = dim3(vl::RC_COLS * vl::RC_GROUPS);
        cfg.stream = G.stream;
        cudaLaunchAttribute attr[2];
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = ncta;
        attr[0].val.clusterDim.y = 1;
        attr[0].val.clusterDim.z = 1;
        attr[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[1].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = attr;
        cfg.numAttrs = G.pdl ? 2 : 1;
        CU(cudaLaunchKernelEx(&cfg, vl::rho_force_cluster_kernel, colpart ? colpart : G.colpart, bands, G.ntheta, dp, rho_out,
                              (const double*)G.cos_t, (const double*)G.sin_t, zero_after ? 1 : 0, dx, G.force, ha));
        LAUNCH_CHECK();
        return VLASOV_OK;
    }
    CU(launch_pdl(vl::rho_force_kernel, dim3(cdiv(G.ntheta, vl::RR_COLS)), dim3(vl::RR_COLS * vl::RR_GROUPS), 0,
                  colpart ? colpart : G.colpart, bands, G.ntheta, dp, rho_out, (const double*)G.cos_t, (const double*)G.sin_t,
                  hmf_partials ? G.mpart : (double*)nullptr, zero_after ? 1 : 0, G.ticket, dx,
                  (fuse_force && (hmf_partials || sheet)) ? G.force : (double*)nullptr, sheet ? 1 : 0));
    LAUNCH_CHECK();
    return VLASOV_OK;
}

// force of the ring, sheet and free models from rho (the HMF force comes out of rho_force_kernel itself)
int force_from_rho() {
    const int nt = G.ntheta;
    const double dx = (G.xmax - G.xmin) / (double)nt;
    switch (G.model) {
        case VLASOV_MODEL_RING:
            // an ordinary launch: behind rho_force_kernel's early trigger its 128 CTAs only sat in the way of the pass
            // (cfg 3: 39.0 -> 41.8 us per step with a programmatic launch here)
            vl::ring_convolve_kernel<<<dim3(cdiv(nt, 256), cdiv(nt, vl::RING_L)), 256, 0, G.stream>>>(
                G.ringK, G.rho, nt, dx, G.ringpart, G.ringtick, G.force);
            break;
        case VLASOV_MODEL_SHEET:
            vl::sheet_scan_kernel<<<1, 1024, 0, G.stream>>>(G.rho, nt, dx, 0, G.force);
            break;
        default:
            vl::fill_zero_kernel<<<cdiv(nt, 256), 256, 0, G.stream>>>(G.force, nt);
            break;
    }
    LAUNCH_CHECK();
    return VLASOV_OK;
}

// density of the pass that just ran, then the force of the next momentum shift (eqs (10), (2)/(4)/(7)-(8))
int rho_and_force(int bands, double* colpart, bool zero_after) {
    const bool hmf = (G.model == VLASOV_MODEL_HMF);
    int rc = rho_from_colpart(bands, G.rho, hmf, colpart, zero_after, true);
    if (rc != 0 || hmf || G.model == VLASOV_MODEL_SHEET) return rc;  // those two forces come out of the same kernel
    return force_from_rho();
}

template <typename T>
int launch_moments_pass() {
    const double dp = (G.pmax - G.pmin) / (double)G.np;
    dim3 grid(cdiv(G.ntheta, 256), G.mbands);
    vl::moments_pass_kernel<T><<<grid, 256, 0, G.stream>>>(static_cast<const T*>(G.owned(G.cur)), G.ntheta, G.np,
                                                           G.mrpb, G.pmin, dp, G.colpart, G.pkpart);
    LAUNCH_CHECK();
    return VLASOV_OK;
}

int moments_pass() { return G.prec == 32 ? launch_moments_pass<float>() : launch_moments_pass<double>(); }

int moments_async(double* dev_out8) {
    int rc;
    const int nt = G.ntheta;
    const double dx = (G.xmax - G.xmin) / (double)nt, dp = (G.pmax - G.pmin) / (double)G.np;
    if ((rc = moments_pass()) != 0) return rc;
    if ((rc = rho_from_colpart(G.mbands, G.rho_m, false)) != 0) return rc;
    const double* phi = nullptr;
    if (G.model == VLASOV_MODEL_RING) {
        vl::ring_convolve_kernel<<<dim3(cdiv(nt, 256), cdiv(nt, vl::RING_L)), 256, 0, G.stream>>>(
            G.ringV, G.rho_m, nt, dx, G.ringpart, G.ringtick, G.phi);
        LAUNCH_CHECK();
        phi = G.phi;
    } else if (G.model == VLASOV_MODEL_SHEET) {
        vl::sheet_scan_kernel<<<1, 1024, 0, G.stream>>>(G.rho_m, nt, dx, 1, G.phi);
        LAUNCH_CHECK();
        phi = G.phi;
    }
    vl::moments_final_kernel<<<1, 1024, 0, G.stream>>>(G.rho_m, phi, nt, G.pkpart, G.mbands * cdiv(nt, 256), G.cos_t,
                                                       G.sin_t, dx, dp, G.model, G.t, dev_out8);
    LAUNCH_CHECK();
    return VLASOV_OK;
}

// two steady-state steps of the one-pass path (each: density/force of the previous pass, then the pass) as one
// graph launch.  After two passes the ping-pong is back where it started, so one graph per starting parity serves
// the whole run.  Captured on a private stream (the attached one may be the legacy default stream, which cannot
// capture) and launched on the attached stream.
int launch_step_pair_graph() {
    const int par = G.cur;
    if (G.gexec[par] == nullptr) {
        if (G.cap_stream == nullptr) CU(cudaStreamCreateWithFlags(&G.cap_stream, cudaStreamNonBlocking));
        cudaStream_t user = G.stream;
        const unsigned long long l0 = G.launches;
        G.stream = G.cap_stream;
        int rc = VLASOV_OK;
        cudaGraph_t graph = nullptr;
        cudaError_t e = cudaStreamBeginCapture(G.cap_stream, cudaStreamCaptureModeThreadLocal);
        if (e == cudaSuccess) {
            for (int q = 0; q < 2 && rc == VLASOV_OK; ++q) {
                rc = rho_and_force(G.fbands[2] * G.fnw(), G.colpart_f, true);
                if (rc == VLASOV_OK) rc = fused_pass(2, true);
            }
            e = cudaStreamEndCapture(G.cap_stream, &graph);
        }
        G.stream = user;
        G.graph_kernels[par] = (unsigned)(G.launches - l0);  // kernels inside the graph (the ring model has six)
        G.launches = l0;
        G.cur = par;
        if (rc != VLASOV_OK) return rc;
        CU(e);
        e = cudaGraphInstantiate(&G.gexec[par], graph, 0);
        cudaGraphDestroy(graph);
        CU(e);
    }
    CU(cudaGraphLaunch(G.gexec[par], G.stream));
    G.launches += G.graph_kernels[par];
    return VLASOV_OK;
}

int check_ready() {
    if (!G.ready) return fail(VLASOV_ENOTINIT, "vlasov_init has not been called");
    if (G.cuda_failed) return VLASOV_ECUDA;
    return VLASOV_OK;
}

}  // namespace

// ---- exported -----------------------------------------------------------------------------------

extern "C" {

const char* vlasov_last_error(void) { return g_err; }

void vlasov_free(void) {
    if (G.ready) cudaStreamSynchronize(G.stream);
    prof_free();
    free_small();
    free_big();
    if (G.cap_stream) cudaStreamDestroy(G.cap_stream);
    G = Ctx();
}

int vlasov_init(int model, const int grid[2], const double domain[4], double dt) {
    if (model < 0 || model > 3 || !grid || !domain) return fail(VLASOV_EINVAL, "vlasov_init: bad model or null argument");
    if (grid[0] < 1 || grid[1] < 1) return fail(VLASOV_EINVAL, "vlasov_init: grid sizes must be >= 1");
    if (!(domain[1] > domain[0]) || !(domain[3] > domain[2]) || !isfinite(dt))
        return fail(VLASOV_EINVAL, "vlasov_init: empty domain or non-finite dt");
    if ((double)grid[0] * (double)grid[1] > 4.0e9) return fail(VLASOV_EINVAL, "vlasov_init: grid too large");
    vlasov_free();
    int dev = 0, count = 0;
    if (cudaGetDeviceCount(&count) != cudaSuccess || count < 1) {
        cudaGetLastError();
        return fail(VLASOV_ECUDA, "vlasov_init: no CUDA device (there is no CPU fallback)");
    }
    CU(cudaGetDevice(&dev));
    CU(cudaDeviceGetAttribute(&G.sm_count, cudaDevAttrMultiProcessorCount, dev));
    G.model = model;
    G.ntheta = grid[0];
    G.np = grid[1];
    G.xmin = domain[0];
    G.xmax = domain[1];
    G.pmin = domain[2];
    G.pmax = domain[3];
    G.dt = dt;
    G.dt_sub = dt;
    G.bc_x = (model == VLASOV_MODEL_SHEET) ? vl::BC_ZERO : vl::BC_PERIODIC;
    G.bc_p = vl::BC_ZERO;
    G.ready = true;
    g_err[0] = 0;
    return VLASOV_OK;
}

int vlasov_set_param(int key, double value) {
    int rc = check_ready();
    if (rc != 0) return rc;
    if (key == VLASOV_KEY_PROFILE) {
        G.profile = (value != 0.0);
        return VLASOV_OK;
    }
    if (G.prepared) return fail(VLASOV_EINVAL, "vlasov_set_param: must precede attach/upload/step");
    switch (key) {
        case VLASOV_KEY_EPS:
            if (!(value > 0.0)) return fail(VLASOV_EINVAL, "EPS must be > 0");
            G.eps = value;
            break;
        case VLASOV_KEY_PRECISION:
            if (value != 64.0 && value != 32.0) return fail(VLASOV_EINVAL, "PRECISION must be 64 or 32");
            G.prec = (int)value;
            break;
        case VLASOV_KEY_BC_X:
            if (value != 0.0 && value != 1.0) return fail(VLASOV_EINVAL, "BC_X must be 0 or 1");
            G.bc_x = (int)value;
            break;
        case VLASOV_KEY_BC_P:
            if (value != 0.0 && value != 1.0) return fail(VLASOV_EINVAL, "BC_P must be 0 or 1");
            G.bc_p = (int)value;
            break;
        case VLASOV_KEY_HISTORY: G.history = (value != 0.0); break;
        case VLASOV_KEY_SPLINE:
            if (value != 0.0 && value != 1.0) return fail(VLASOV_EINVAL, "SPLINE must be 0 (eq 16) or 1 (system 15)");
            if (value == 1.0 && (G.ntheta < vl::GS_MIN_N || G.np < vl::GS_MIN_N))
                return fail(VLASOV_EINVAL, "SPLINE = 1 (global spline) needs at least 32 nodes on both axes");
            G.spline = (int)value;
            break;
        case VLASOV_KEY_HALO_LO:
        case VLASOV_KEY_HALO_HI:
            if (value < 0.0 || value > 1.0e6 || value != floor(value)) return fail(VLASOV_EINVAL, "HALO_LO / HALO_HI must be a row count >= 0");
            (key == VLASOV_KEY_HALO_LO ? G.halo_lo : G.halo_hi) = (int)value;
            break;
        case VLASOV_KEY_ORDER:
            if (value != 2.0 && value != 4.0) return fail(VLASOV_EINVAL, "ORDER must be 2 or 4");
            G.order = (int)value;
            break;
        case VLASOV_KEY_FUSE:
            if (value != 0.0 && value != 1.0 && value != 2.0) return fail(VLASOV_EINVAL, "FUSE must be 0, 1 or 2");
            G.fuse = (int)value;
            break;
        case KEY_TUNE_FBANDS: G.tune_fbands = (int)value; break;
        case KEY_TUNE_TILE: G.tune_tile = (int)value; break;
        case KEY_TUNE_RC: G.tune_rc = (int)value; break;
        case KEY_TUNE_HIST: G.tune_hist = (int)value; break;
        case KEY_TUNE_GRAPH: G.graphs = (value != 0.0); break;
        case KEY_TUNE_PDL: G.pdl = (value != 0.0); break;
        case KEY_TUNE_FEDGE: G.tune_fedge = (int)value; break;
        case VLASOV_KEY_PROFILE: G.profile = (value != 0.0); break;
        case KEY_TUNE_NW1: G.tune_nw1 = (int)value; break;
        case KEY_TUNE_NW2: G.tune_nw2 = (int)value; break;
        case KEY_TUNE_BANDS: G.tune_bands = (int)value; break;
        case KEY_TUNE_PSEG: G.tune_pseg = (int)value; break;
        case KEY_TUNE_PTX: G.tune_ptx = (int)value; break;
        case KEY_TUNE_GENERIC: G.force_generic = (value != 0.0); break;
        default: return fail(VLASOV_EINVAL, "vlasov_set_param: unknown key");
    }
    return VLASOV_OK;
}

size_t vlasov_state_bytes(void) { return G.ready ? state_bytes() : 0; }
size_t vlasov_workspace_bytes(void) { return G.ready ? workspace_bytes() : 0; }

int vlasov_attach(void* f_dev, void* work_dev, size_t work_bytes, void* cuda_stream) {
    int rc = check_ready();
    if (rc != 0) return rc;
    if (!f_dev || !work_dev) return fail(VLASOV_EINVAL, "vlasov_attach: null buffer");
    if (((uintptr_t)f_dev & 15) || ((uintptr_t)work_dev & 255))
        return fail(VLASOV_EINVAL, "vlasov_attach: f_dev must be 16-byte and work_dev 256-byte aligned");
    if (work_bytes < workspace_bytes()) return fail(VLASOV_ENOMEM, "vlasov_attach: work buffer too small");
    G.stream = static_cast<cudaStream_t>(cuda_stream);
    if ((rc = prepare()) != 0) return rc;
    free_big();
    G.f[0] = f_dev;
    G.work = work_dev;
    G.f[1] = work_dev;
    G.colpart = reinterpret_cast<double*>(static_cast<char*>(work_dev) + round256(state_bytes()));
    G.cur = 0;
    G.attached = true;
    return VLASOV_OK;
}

int vlasov_state_ptr(void** out) {
    int rc = check_ready();
    if (rc != 0) return rc;
    if (!out) return fail(VLASOV_EINVAL, "vlasov_state_ptr: null");
    if ((rc = ensure_buffers()) != 0) return rc;
    *out = G.f[G.cur];
    return VLASOV_OK;
}

int vlasov_upload(const void* f_host) {
    int rc = check_ready();
    if (rc != 0) return rc;
    if (!f_host) return fail(VLASOV_EINVAL, "vlasov_upload: null");
    if ((rc = ensure_buffers()) != 0) return rc;
    G.cur = 0;
    if (G.halo_lo + G.halo_hi > 0) CU(cudaMemsetAsync(G.f[0], 0, state_bytes(), G.stream));  // halos start as zeros
    CU(cudaMemcpyAsync(G.owned(0), f_host, owned_bytes(), cudaMemcpyHostToDevice, G.stream));
    G.t = 0.0;
    return VLASOV_OK;
}

int vlasov_download(void* f_host) {
    int rc = check_ready();
    if (rc != 0) return rc;
    if (!f_host) return fail(VLASOV_EINVAL, "vlasov_download: null");
    if ((rc = ensure_buffers()) != 0) return rc;
    CU(cudaMemcpyAsync(f_host, G.owned(G.cur), owned_bytes(), cudaMemcpyDeviceToHost, G.stream));
    CU(cudaStreamSynchronize(G.stream));
    return VLASOV_OK;
}

int vlasov_sync(void) {
    int rc = check_ready();
    if (rc != 0) return rc;
    CU(cudaStreamSynchronize(G.stream));
    return VLASOV_OK;
}

int vlasov_step(int n) {
    int rc = check_ready();
    if (rc != 0) return rc;
    if (n <= 0) return fail(VLASOV_EINVAL, "vlasov_step: n must be >= 1");
    if ((rc = ensure_buffers()) != 0) return rc;
    if (G.halo_lo + G.halo_hi > 0)
        return fail(VLASOV_EINVAL, "vlasov_step: a slab (HALO_LO / HALO_HI > 0) is advanced stage by stage with vlasov_substep, the "
                                   "density all-reduce and the halo exchange in between belong to the caller");
    if (G.history) {
        if (G.hist_cap < n) {
            if (G.hist) CU(cudaFree(G.hist));
            G.hist = nullptr;
            CU(cudaMalloc(&G.hist, sizeof(double) * 8 * (size_t)n));
            G.hist_cap = n;
        }
        G.hist_count = 0;
    }
    if (G.order == 4) {
        // fourth order: every step is three of the paper's steps (1)-(4) over g1 dt, g2 dt, g1 dt, each with its own
        // row tables and its own force evaluation; the middle one runs backwards in time (separate passes)
        const double g1 = 1.0 / (2.0 - cbrt(2.0)), g[2] = {g1, 1.0 - 2.0 * g1};
        int* const srow0 = G.srow;
        double* const wrow0 = G.wrow;
        rc = VLASOV_OK;
        for (int k = 0; k < n && rc == VLASOV_OK; ++k) {
            for (int sub = 0; sub < 3 && rc == VLASOV_OK; ++sub) {
                const int q = sub == 1 ? 1 : 0;
                G.srow = G.srow_sub[q];
                G.wrow = G.wrow_sub[q];
                G.dt_sub = g[q] * G.dt;
                if ((rc = theta_pass(1, true)) != 0) break;                                  // eq (9)
                if ((rc = rho_and_force(theta_bands(1), nullptr, false)) != 0) break;        // eq (10)
                if ((rc = p_pass()) != 0) break;                                             // eq (11)
                rc = theta_pass(1, false);                                                   // eq (12)
            }
            G.t += G.dt;
            if (G.history && rc == VLASOV_OK) {
                rc = moments_async(G.hist + 8 * (size_t)k);
                G.hist_count = k + 1;
            }
        }
        G.srow = srow0;
        G.wrow = wrow0;
        G.dt_sub = G.dt;
        if (rc != 0) return rc;
    } else if (G.onepass && G.history && G.model == VLASOV_MODEL_HMF && G.rowmom != nullptr && G.tune_hist != 2 &&
               fabs((G.xmax - G.xmin) - 6.283185307179586) < 1e-9) {
        // HISTORY on the one-pass path (HMF): n + 1 passes as below; the tile kernel also leaves per-row sums of the state it
        // stores (on the large grids a read pass, row_moments_kernel, takes them) and history_rows_kernel turns them into the
        // moments of the end-of-step state (the half shift that opens the next step only multiplies a row's first Fourier
        // sum by a known number)
        const double dp = (G.pmax - G.pmin) / (double)G.np, dx = (G.xmax - G.xmin) / (double)G.ntheta;
        if ((rc = theta_pass(1, true)) != 0) return rc;                           // eq (9)
        G.want_rowmom = true;
        // the history entry of step k rides along with the density / force launch of step k + 1 (one more CTA of its cluster);
        // where that kernel is not the cluster kernel, and after the last step, history_rows_kernel writes it
        auto flush_history = [&]() {
            if (G.hist_pending.rowmom == nullptr) return;
            const vl::HistArgs h = G.hist_pending;
            G.hist_pending.rowmom = nullptr;
            vl::history_rows_kernel<<<1, 1024, 0, G.stream>>>(h.rowmom, h.nblk, h.np, h.invT, h.ident, h.pmin, dp, dx, h.t, h.out);
            G.launches++;
        };
        G.hist_pending.rowmom = nullptr;
        for (int k = 0; k < n; ++k) {
            const bool last = k + 1 == n;
            if (k == 0) rc = rho_and_force(theta_bands(1), nullptr, false);              // eq (10)
            else rc = rho_and_force(G.fbands[2] * G.fnw(), G.colpart_f, true);
            flush_history();                                                             // (if the launch above did not take it)
            if (rc == VLASOV_OK) rc = fused_pass(last ? 1 : 2, !last);                   // eqs (11), (12) [, (9)]
            if (rc != VLASOV_OK) break;
            if (!G.tile) {  // large grids: the row sums by a read pass over the state the pass has just written
                if (G.prec == 32)
                    vl::row_moments_kernel<float><<<cdiv(G.np, 8), 256, 0, G.stream>>>(static_cast<const float*>(G.f[G.cur]), G.ntheta, G.np,
                                                                                       G.cos_t, G.sin_t, G.rowmom);
                else
                    vl::row_moments_kernel<double><<<cdiv(G.np, 8), 256, 0, G.stream>>>(static_cast<const double*>(G.f[G.cur]), G.ntheta,
                                                                                        G.np, G.cos_t, G.sin_t, G.rowmom);
                G.launches++;
            }
            G.hist_pending.rowmom = G.rowmom;
            G.hist_pending.invT = G.hist_invT;
            G.hist_pending.out = G.hist + 8 * (size_t)k;
            G.hist_pending.nblk = G.tile ? G.fcols[last ? 1 : 2] : 1;
            G.hist_pending.np = G.np;
            G.hist_pending.ident = last ? 1 : 0;
            G.hist_pending.pmin = G.pmin;
            G.hist_pending.t = G.t + (double)(k + 1) * G.dt;
            G.hist_count = k + 1;
        }
        flush_history();
        G.want_rowmom = false;
        if (rc != VLASOV_OK) return rc;
        CU(cudaGetLastError());
        G.t += (double)n * G.dt;
    } else if (G.onepass && !G.history) {
        // n + 1 passes: theta(dt/2), then per step ONE pass  p(dt) -> theta(dt/2) [-> theta(dt/2) of the next step]
        if ((rc = theta_pass(1, true)) != 0) return rc;                           // eq (9)
        int k = 0;
        while (k < n) {
            // steps 1 .. n-2 are identical pairs of launches: two of them at a time as one CUDA graph
            if (k >= 1 && k + 2 < n && G.graphs && !G.profile) {
                if ((rc = launch_step_pair_graph()) != 0) return rc;
                k += 2;
                continue;
            }
            prof_begin(3);
            if (k == 0) rc = rho_and_force(theta_bands(1), nullptr, false);              // eq (10)
            else rc = rho_and_force(G.fbands[2] * G.fnw(), G.colpart_f, true);
            if (rc != 0) return rc;
            prof_end(3);
            if ((rc = fused_pass(k + 1 < n ? 2 : 1, k + 1 < n)) != 0) return rc;  // eqs (11), (12) [, (9)]
            ++k;
        }
        G.t += (double)n * G.dt;
    } else if (G.fuse >= 1 && !G.history && G.spline == 0) {
        if ((rc = theta_pass(1, true)) != 0) return rc;                       // eq (9)
        for (int k = 0; k < n; ++k) {
            prof_begin(3);
            if ((rc = rho_and_force(theta_bands(k == 0 ? 1 : 2), nullptr, false)) != 0) return rc;  // eq (10)
            prof_end(3);
            if ((rc = p_pass()) != 0) return rc;                              // eq (11)
            if (k + 1 < n) {
                if ((rc = theta_pass(2, true)) != 0) return rc;               // eq (12) of step k, eq (9) of k+1
            } else {
                if ((rc = theta_pass(1, false)) != 0) return rc;              // eq (12)
            }
        }
        G.t += (double)n * G.dt;
    } else {
        for (int k = 0; k < n; ++k) {
            if ((rc = theta_pass(1, true)) != 0) return rc;
            if ((rc = rho_and_force(theta_bands(1), nullptr, false)) != 0) return rc;
            if (G.onepass) {
                if ((rc = fused_pass(1, false)) != 0) return rc;              // eqs (11), (12) in one pass
            } else {
                if ((rc = p_pass()) != 0) return rc;
                if ((rc = theta_pass(1, false)) != 0) return rc;
            }
            G.t += G.dt;
            if (G.history) {
                if ((rc = moments_async(G.hist + 8 * (size_t)k)) != 0) return rc;
                G.hist_count = k + 1;
            }
        }
    }
    return VLASOV_OK;
}

int vlasov_substep(int which) {
    int rc = check_ready();
    if (rc != 0) return rc;
    if ((rc = ensure_buffers()) != 0) return rc;
    switch (which) {
        case VLASOV_SUB_THETA_HALF: return theta_pass(1, true);
        case VLASOV_SUB_THETA_TWICE: return theta_pass(2, true);
        case VLASOV_SUB_FORCE:
            if ((rc = moments_pass()) != 0) return rc;
            return rho_and_force(G.mbands, nullptr, false);
        case VLASOV_SUB_P_FULL: return p_pass();
        case VLASOV_SUB_RHO:  // density of the owned rows from the column sums the last theta pass left behind
            return rho_from_colpart(theta_bands(1), G.rho, false);
        case VLASOV_SUB_FORCE_FROM_RHO:  // force from the RHO vector as it stands (after the caller's all-reduce)
            if (G.model == VLASOV_MODEL_HMF) {
                const double dx = (G.xmax - G.xmin) / (double)G.ntheta;
                vl::hmf_force_from_rho_kernel<<<1, 1024, 0, G.stream>>>(G.rho, G.cos_t, G.sin_t, G.ntheta, dx, G.force);
                LAUNCH_CHECK();
                return VLASOV_OK;
            }
            return force_from_rho();
        case VLASOV_SUB_P_THETA_HALF:
        case VLASOV_SUB_P_THETA_TWICE: {
            const int nst = which == VLASOV_SUB_P_THETA_TWICE ? 2 : 1;
            if (!G.onepass) {  // grid or shift pattern outside the one-pass kernel's conditions: separate passes
                if ((rc = p_pass()) != 0) return rc;
                if ((rc = theta_pass(nst, true)) != 0) return rc;
                return rho_and_force(theta_bands(nst), nullptr, false);
            }
            if ((rc = fused_pass(nst, true)) != 0) return rc;
            return rho_and_force(G.fbands[nst] * G.fnw(), G.colpart_f, true);
        }
        default: return fail(VLASOV_EINVAL, "vlasov_substep: unknown stage");
    }
}

int vlasov_get_vector(int which, double* host_out) {
    int rc = check_ready();
    if (rc != 0) return rc;
    if (!host_out || (which != VLASOV_VEC_RHO && which != VLASOV_VEC_FORCE))
        return fail(VLASOV_EINVAL, "vlasov_get_vector: bad argument");
    if ((rc = ensure_buffers()) != 0) return rc;
    const double* src = which == VLASOV_VEC_RHO ? G.rho : G.force;
    CU(cudaMemcpyAsync(host_out, src, sizeof(double) * G.ntheta, cudaMemcpyDeviceToHost, G.stream));
    CU(cudaStreamSynchronize(G.stream));
    return VLASOV_OK;
}

int vlasov_vector_ptr(int which, void** dev_out) {
    int rc = check_ready();
    if (rc != 0) return rc;
    if (!dev_out || (which != VLASOV_VEC_RHO && which != VLASOV_VEC_FORCE)) return fail(VLASOV_EINVAL, "vlasov_vector_ptr: bad argument");
    if ((rc = ensure_buffers()) != 0) return rc;
    *dev_out = which == VLASOV_VEC_RHO ? G.rho : G.force;
    return VLASOV_OK;
}

int vlasov_set_vector(int which, const double* host_in) {
    int rc = check_ready();
    if (rc != 0) return rc;
    if (!host_in || which != VLASOV_VEC_FORCE) return fail(VLASOV_EINVAL, "vlasov_set_vector: only FORCE can be set");
    if ((rc = ensure_buffers()) != 0) return rc;
    CU(cudaMemcpyAsync(G.force, host_in, sizeof(double) * G.ntheta, cudaMemcpyHostToDevice, G.stream));
    CU(cudaStreamSynchronize(G.stream));
    return VLASOV_OK;
}

int vlasov_moments(double out[8]) {
    int rc = check_ready();
    if (rc != 0) return rc;
    if (!out) return fail(VLASOV_EINVAL, "vlasov_moments: null");
    if ((rc = ensure_buffers()) != 0) return rc;
    if ((rc = moments_async(G.mom_dev)) != 0) return rc;
    CU(cudaMemcpyAsync(out, G.mom_dev, sizeof(double) * 8, cudaMemcpyDeviceToHost, G.stream));
    CU(cudaStreamSynchronize(G.stream));
    return VLASOV_OK;
}

int vlasov_casimirs(double out[4]) {
    int rc = check_ready();
    if (rc != 0) return rc;
    if (!out) return fail(VLASOV_EINVAL, "vlasov_casimirs: null");
    if ((rc = ensure_buffers()) != 0) return rc;
    const int nblk = G.mbands * cdiv(G.ntheta, 256);
    const double cell = ((G.xmax - G.xmin) / (double)G.ntheta) * ((G.pmax - G.pmin) / (double)G.np);
    dim3 grid(cdiv(G.ntheta, 256), G.mbands);
    if (G.prec == 32)
        vl::casimir_pass_kernel<float><<<grid, 256, 0, G.stream>>>(static_cast<const float*>(G.owned(G.cur)), G.ntheta, G.np,
                                                                   G.mrpb, G.caspart);
    else
        vl::casimir_pass_kernel<double><<<grid, 256, 0, G.stream>>>(static_cast<const double*>(G.owned(G.cur)), G.ntheta,
                                                                    G.np, G.mrpb, G.caspart);
    LAUNCH_CHECK();
    double* res = G.caspart + 4 * (size_t)nblk;
    vl::casimir_final_kernel<<<1, 1024, 0, G.stream>>>(G.caspart, nblk, cell, res);
    LAUNCH_CHECK();
    CU(cudaMemcpyAsync(out, res, sizeof(double) * 4, cudaMemcpyDeviceToHost, G.stream));
    CU(cudaStreamSynchronize(G.stream));
    return VLASOV_OK;
}

int vlasov_history(double* out, int max_steps) {
    int rc = check_ready();
    if (rc != 0) return rc;
    if (!out || max_steps < 0) return fail(VLASOV_EINVAL, "vlasov_history: bad argument");
    const int n = G.hist_count < max_steps ? G.hist_count : max_steps;
    if (n > 0) {
        CU(cudaMemcpyAsync(out, G.hist, sizeof(double) * 8 * (size_t)n, cudaMemcpyDeviceToHost, G.stream));
        CU(cudaStreamSynchronize(G.stream));
    }
    return n;
}

int vlasov_launch_count(unsigned long long* out) {
    if (!out) return fail(VLASOV_EINVAL, "vlasov_launch_count: null");
    *out = G.launches;
    return VLASOV_OK;
}

int vlasov_kernel_times(double out[12]) {
    int rc = check_ready();
    if (rc != 0) return rc;
    if (!out) return fail(VLASOV_EINVAL, "vlasov_kernel_times: null");
    CU(cudaStreamSynchronize(G.stream));
    for (int c = 0; c < NCLS; ++c) {
        double total = 0.0;
        for (size_t k = 0; k < G.ev_used[c]; ++k) {
            float ms = 0.f;
            CU(cudaEventElapsedTime(&ms, G.ev[c][0][k], G.ev[c][1][k]));
            total += (double)ms;
        }
        out[2 * c + 0] = total;
        out[2 * c + 1] = (double)G.ev_used[c];
        G.ev_used[c] = 0;
    }
    return VLASOV_OK;
}

int vlasov_info(double* out, int n) {
    int rc = check_ready();
    if (rc != 0) return rc;
    if (!out || n < 0) return fail(VLASOV_EINVAL, "vlasov_info: bad argument");
    if ((rc = prepare()) != 0) return rc;
    const bool tb = G.theta_bulk;
    const double v[] = {(double)G.sm_count,
                        tb ? (double)G.bctas[2] : (double)G.nchunks[2] * G.nbands[2],
                        (double)cdiv(G.ntheta, G.p_tx) * G.p_nseg,
                        (double)theta_bands(2),
                        tb ? (double)TB_WARPS : (double)G.nw[2],
                        tb ? (double)TB_WARPS : (double)G.nw[1],
                        tb ? (double)G.bctas[1] : (double)G.nchunks[1] * G.nbands[1],
                        (double)G.p_seg,
                        (double)G.p_tx,
                        tb ? 1.0 : 0.0,
                        G.onepass ? 1.0 : 0.0,
                        (double)G.fcols[2] * G.fbands[2],
                        (double)G.fbands[2],
                        (double)G.frpb[2],
                        G.tile ? 1.0 : 0.0,
                        (double)G.rc_max_cluster};
    const int m = (int)(sizeof(v) / sizeof(v[0]));
    const int k = n < m ? n : m;
    for (int q = 0; q < k; ++q) out[q] = v[q];
    return k;
}

}  // extern "C"
