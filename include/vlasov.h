/*
 * vlasov.h -- C ABI of the B200-native Strang semi-Lagrangian Vlasov step.
 *
 * Method: T. M. Rocha Filho, "Solving the Vlasov equation for one-dimensional models with long range
 * interactions on a GPU", arXiv 1206.3229.  Citations below are PAPER.md line numbers.
 *
 * The library advances the one-particle distribution f(theta, p) on an equally spaced grid
 * (section 3) stored as ONE flat row-major array  f[j * Ntheta + i],  i the position index
 * (fastest), j the momentum index (L115), resident in GPU memory for the whole run (L115), by the time-split
 * steps (1)-(4) of section 3 (L71-L87, eqs (9)-(12)):
 *     f_I (x,p) = f(x - p dt/2, p);  F_I = mean-field force of f_I;  f_II(x,p) = f_I(x, p - F_I(x) dt);
 *     f(t+dt)   = f_II(x - p dt/2, p),
 * every value at the foot of a characteristic taken from the cubic spline of eqs (13)-(14) (L89-L98) whose
 * second derivatives are the eighth-order centred difference of eq (16) (L106-L111).
 *
 * Conventions common to all calls
 *   - every function returns 0 on success or a negative VLASOV_E* code; no exception crosses the ABI;
 *     vlasov_last_error() gives a static, thread-local, human-readable message for the last failure;
 *   - one singleton context per process; calls are not thread-safe;
 *   - "host" pointers are ordinary CPU memory (pinned or pageable), "device" pointers are CUDA global memory
 *     of the current device; the library never frees memory it was handed through vlasov_attach;
 *   - all work is enqueued on the attached CUDA stream (default: the legacy default stream); only
 *     vlasov_moments, vlasov_download, vlasov_history, vlasov_get_vector and vlasov_sync block the host;
 *   - there is no CPU fallback: without a CUDA device vlasov_init fails with VLASOV_ECUDA.
 *   - grid nodes: x_i = x_min + i (x_max - x_min)/Ntheta, i = 0..Ntheta-1 (right end excluded), same for p.
 */
#ifndef VLASOV_B200_H
#define VLASOV_B200_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

/* error codes */
#define VLASOV_OK 0
#define VLASOV_EINVAL (-1)   /* bad argument or call order                       */
#define VLASOV_ENOTINIT (-2) /* vlasov_init has not been called                  */
#define VLASOV_ECUDA (-3)    /* a CUDA call failed; sticky until vlasov_init     */
#define VLASOV_ENOMEM (-4)   /* allocation failed / attached workspace too small */

/* model: which pair potential defines the mean-field force, section 2 */
#define VLASOV_MODEL_FREE 0  /* F = 0 (free streaming; tests)                                    */
#define VLASOV_MODEL_HMF 1   /* eq (3); force by the two moments of eqs (7)-(8) L56-L63      */
#define VLASOV_MODEL_RING 2  /* eq (2), softened; direct circulant sum over theta        */
#define VLASOV_MODEL_SHEET 3 /* eq (4), V = |x - x'|; prefix sum of the density          */

/* keys of vlasov_set_param */
#define VLASOV_KEY_EPS 1       /* ring softening epsilon of eq (2); default 0.01                            */
#define VLASOV_KEY_PRECISION 2 /* storage precision of f: 64 (default) or 32; arithmetic of sums is fp64    */
#define VLASOV_KEY_BC_X 3      /* 0 periodic (paper, L113; default for FREE/HMF/RING), 1 zero extension     */
#define VLASOV_KEY_BC_P 4      /* 0 periodic (paper, L113), 1 zero extension "f = 0 beyond" (default)       */
#define VLASOV_KEY_HISTORY 5   /* 1: vlasov_step records the 8 moments after every step (HMF model: still on the
                                  one-pass path, history_rows_kernel; ring and sheet: separate passes)        */
#define VLASOV_KEY_FUSE 6      /* passes over f per step in vlasov_step(n): 0: three (theta, p, theta); 1: two (the
                                  adjacent half theta shifts of steps k, k+1 share a pass); 2 (default): ONE
                                  (p shift, both half theta shifts and the density of the next step share a pass;
                                  needs periodic x, otherwise behaves like 1)                                   */
#define VLASOV_KEY_PROFILE 7   /* 1: bracket every sweep launch of vlasov_step with CUDA events (any time)   */
#define VLASOV_KEY_SPLINE 8    /* which f'' enters eq (13): 0 (default) the local eighth-order difference of eq (16),
                                  L106-L111, the paper's method; 1 the GLOBAL SPLINE, f'' = solution of the
                                  tridiagonal system (15), L100-L102 (the paper's comparator "GS", Tables 1-2;
                                  diagonal 2/3, D22).  Three passes per step; the solve is replaced by
                                  its closed-form inverse (two first-order recursions per line; or, with tuning
                                  key 110, a 60-tap filter); both axes need >= 32 nodes                          */
#define VLASOV_KEY_ORDER 9     /* order of the time splitting: 2 (default) the paper's steps (1)-(4), L71-L87; 4: their
                                  triple-jump composition S2(g1 dt) S2(g2 dt) S2(g1 dt), g1 = 1/(2 - 2^(1/3)), g2 = 1 - 2 g1
                                  ("higher order time split schemes", L238 with refs [31], [44]):
                                  three times the passes and force evaluations of a step, the middle sub-step
                                  backwards in time; eq (16) spline only                                          */
#define VLASOV_KEY_HALO_LO 10  /* slab mode (p-slab sharding over several GPUs): the context   */
#define VLASOV_KEY_HALO_HI 11  /* owns grid[1] rows of the global grid (domain = their p range) and its two state buffers carry
                                  HALO_LO rows before and HALO_HI rows after them: [HALO_LO + Np + HALO_HI][Ntheta].  Theta
                                  shifts, density and moments act on the owned rows, the momentum shift on all rows
                                  (zero extension beyond them), so an owned row is right if the halos hold the
                                  neighbours' rows and are deeper than max|F| dt/dp + 5.  The all-reduce of the density
                                  and the halo exchange happen BETWEEN the stages of vlasov_substep and belong to the
                                  caller (torch.distributed / NCCL); vlasov_step refuses.  upload / download move the
                                  owned rows; vlasov_state_ptr is the start of the buffer (first halo row).           */
/* Tuning keys (tests and sweeps; results never depend on them beyond rounding order).  0 = automatic.
 *   101 TUNE_NW1, 102 TUNE_NW2   warps per CTA of the generic theta kernel (one / two half shifts)
 *   103 TUNE_BANDS               bands of rows of the theta kernels
 *   104 TUNE_PSEG, 105 TUNE_PTX  rows per segment / threads per CTA of the p kernel (two-pass path)
 *   106 TUNE_GENERIC             1: the generic theta kernel even where rows are multiples of 16 bytes
 *   107 TUNE_FBANDS              bands of rows of the one-pass kernel
 *   108 TUNE_FEDGE               zero-extended theta: width (percent) of the first / last column block of the one-pass kernel
 *   109 TUNE_GRAPH               0: plain launches instead of the captured step-pair graphs (default 1)
 *   110 TUNE_PDL                 0: ordinary launches instead of programmatic dependent launch (default 1)
 *   111 TUNE_TILE                one-pass step of small grids (fp64, periodic theta) by the tile kernel strang_tile_kernel instead of
 *                                the warp-specialised one: 0 by size (default: up to 4.5e6 grid points, i.e. 2048^2), 1 whenever its conditions
 *                                hold, 2 never
 *   112 TUNE_RC                  2: never rho_force_cluster_kernel (HMF density / moments / force of theta axes of up to 1024
 *                                columns by one thread-block cluster); the ticketed rho_force_kernel on every grid instead   
 *   113 TUNE_HIST                2: HISTORY = 1 always by the separate passes (theta, p + theta, moments read pass per step);
 *                                default: with the HMF model (theta axis of length 2 pi) the history is recorded on the
 *                                one-pass path (history_rows_kernel)                                                   */

/* sub-steps for vlasov_substep (parity tests of single stages; same kernels as vlasov_step) */
#define VLASOV_SUB_THETA_HALF 0  /* eq (9)/(12): f(x - p dt/2, p), also leaves the column sums for the force */
#define VLASOV_SUB_FORCE 1       /* eq (10): density + force of the CURRENT f (runs its own density pass)    */
#define VLASOV_SUB_P_FULL 2      /* eq (11): f(x, p - F dt) with the force vector currently stored           */
#define VLASOV_SUB_THETA_TWICE 3 /* two half shifts in one pass (the fused a5 o a1 kernel)                   */
#define VLASOV_SUB_P_THETA_HALF 4  /* one-pass kernel: eq (11) with the stored force, then eq (12); then the density
                                      and force of the result are left in the RHO / FORCE vectors (where the
                                      one-pass kernel does not apply -- vlasov_info says -- the separate kernels) */
#define VLASOV_SUB_P_THETA_TWICE 5 /* one-pass kernel: eq (11), eq (12), eq (9) of the next step, then density, force */

#define VLASOV_SUB_RHO 6            /* density of the (owned) rows from the column sums of the preceding THETA_HALF -> RHO */
#define VLASOV_SUB_FORCE_FROM_RHO 7 /* force of the model from the RHO vector as it stands -> FORCE                       */

/* vectors for vlasov_get_vector / vlasov_set_vector (Ntheta doubles each) */
#define VLASOV_VEC_RHO 0   /* density rho_i = dp sum_j f_ij used by the last force evaluation */
#define VLASOV_VEC_FORCE 1 /* force F_i used by (or set for) the next momentum shift           */

/*
 * Create the singleton context (frees a previous one).
 *   model   VLASOV_MODEL_*
 *   grid    {Ntheta, Np}  (host), each >= 1
 *   domain  {x_min, x_max, p_min, p_max} (host), half-open intervals
 *   dt      time step of one full Strang step
 * Computes once: per-row integer shift and the ten interpolation weights of the theta half shift
 * (p_j and dt never change), sin/cos tables of the nodes (L210), ring force/potential tables.
 * Boundary defaults follow BASELINE.json: x periodic (zero extension for SHEET), p zero extension.
 * f is zero until vlasov_upload.  Errors: EINVAL (arguments), ECUDA (no device / CUDA failure), ENOMEM.
 */
int vlasov_init(int model, const int grid[2], const double domain[4], double dt);

/* Change a parameter (VLASOV_KEY_*) after vlasov_init and before the first upload/attach/step. */
int vlasov_set_param(int key, double value);

/* Bytes of ONE copy of f (Ntheta*Np*sizeof(element)) and of the work buffer vlasov_attach expects
 * (second copy of f for the out-of-place passes + per-band column sums).  0 if not initialised. */
size_t vlasov_state_bytes(void);
size_t vlasov_workspace_bytes(void);

/*
 * Hand the library caller-owned device memory and a stream (all three stay owned by the caller):
 *   f_dev       device, vlasov_state_bytes() bytes, row-major [Np][Ntheta]; its content is taken as f(t)
 *   work_dev    device, >= vlasov_workspace_bytes() bytes, 256-byte aligned, content irrelevant
 *   cuda_stream a cudaStream_t cast to void* (NULL = legacy default stream)
 * If vlasov_attach is never called the library allocates both buffers itself at the first upload.
 * After a step the current f lives in EITHER f_dev or the first vlasov_state_bytes() of work_dev (the passes
 * ping-pong); vlasov_state_ptr tells which.  Errors: EINVAL, ENOMEM (work_bytes too small).
 */
int vlasov_attach(void* f_dev, void* work_dev, size_t work_bytes, void* cuda_stream);

/* Device pointer of the current f (one of the two buffers above). */
int vlasov_state_ptr(void** f_dev_out);

/* Host -> device copy of a full state (row-major [Np][Ntheta], element type per PRECISION); sets t = 0.
 * Device -> host copy of the current state (blocks until done).  Together: checkpoint / resume. */
int vlasov_upload(const void* f_host);
int vlasov_download(void* f_host);

/*
 * Enqueue n >= 1 Strang steps (asynchronous).  The state afterwards is f(t0 + n dt) as n single steps give
 * it: theta(dt/2), [force, p(dt), theta(dt/2) theta(dt/2)] x (n-1), force, p(dt), theta(dt/2).  With FUSE = 2
 * (default; periodic x, shift of a half step below one domain length) everything inside the brackets plus the
 * density of the next force is ONE kernel and the two adjacent half shifts of a row are applied as one 19-tap
 * filter (the convolution of the ten weights with themselves: the same map up to rounding order); with FUSE = 1
 * they are evaluated one after the other inside one kernel; FUSE = 0: separate passes.  HISTORY = 1: the HMF model on a
 * theta axis of length 2 pi keeps the one-pass path (the moments of the end-of-step state follow from per-row sums of the
 * stored state, which already carries the next step's leading half shift); the other models take separate passes.
 * Errors: EINVAL (n <= 0), ENOTINIT, ECUDA.
 */
int vlasov_step(int n);

/* One stage on its own (VLASOV_SUB_*); used by the parity tests.  Does not advance t. */
int vlasov_substep(int which);

/* Copy a device vector (VLASOV_VEC_*) of Ntheta doubles to / from host memory (blocking). */
int vlasov_get_vector(int which, double* host_out);
int vlasov_set_vector(int which, const double* host_in);
/* Device pointer of a vector (Ntheta doubles, owned by the library): for collectives on it between two stages. */
int vlasov_vector_ptr(int which, void** dev_out);

/*
 * out (host, 8 doubles) = {t, mass, P, K, U, M_x, M_y, E = K + U} of the current state, rectangle rule:
 *   mass = dx dp sum f, P = dx dp sum p f, K = dx dp sum p^2/2 f, (M_x, M_y) eq (8),
 *   U = (1/2) int rho phi:  HMF (mass^2 - M_x^2 - M_y^2)/2;  ring  phi = dtheta sum_m V(m dtheta) rho_{i-m};
 *   sheet  phi = dx sum_k |x_i - x_k| rho_k;  FREE 0.
 * Runs one extra read pass over f; blocks until done.
 */
int vlasov_moments(double out[8]);

/*
 * Casimir invariants of the current state (eq (18)), rectangle
 * rule on the nodes; synchronises the stream; out (host, caller-owned):
 *   out[0]  S  = -int f log f   (the entropy of Fig. 2; nodes with f <= 0 contribute 0)
 *   out[1]  C2 = int f^2
 *   out[2]  negative mass  int min(f, 0)  (the scheme is not positivity preserving)
 *   out[3]  max f
 * One read pass over f (8 bytes per grid point in fp64), on demand only.  Errors: EINVAL (null), ENOTINIT, ECUDA.
 */
int vlasov_casimirs(double out[4]);

/* With HISTORY = 1: copy the records {t, mass, P, K, U, M_x, M_y, E} written after each of the steps of
 * the LAST vlasov_step call into out (host, 8*max_steps doubles); returns the number of records copied
 * (>= 0) or a negative code. */
int vlasov_history(double* out, int max_steps);

/* Block until everything enqueued so far has finished. */
int vlasov_sync(void);

/* Number of kernels the library has launched since vlasov_init (for bench.py's gpu_launches). */
int vlasov_launch_count(unsigned long long* out);

/* With PROFILE = 1: out (host, 12 doubles) = {ms, launches} summed over the launches recorded since the last
 * call, for the kernel classes {theta x1, theta x2, p, density+force, p+theta x2 (one pass), p+theta x1};
 * CUDA-event times on the launch stream.  Blocks until the stream is idle; resets the records. */
int vlasov_kernel_times(double out[12]);

/* Fill out[0..n) (host) with implementation facts for reports: {SM count, theta-kernel CTAs, p-kernel CTAs,
 * bands, warps per theta CTA (2-shift), warps per theta CTA (1-shift), theta1 CTAs, p segment length, p threads,
 * bulk-copy theta kernel in use, one-pass kernel in use (0/1), its CTAs, bands, rows per band, whether it is the tile
 * kernel of small grids (0/1), the largest thread-block cluster the density / force kernel of short theta axes may use (8 or
 * 16)}; returns how many were written. */
int vlasov_info(double* out, int n);

void vlasov_free(void);
const char* vlasov_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* VLASOV_B200_H */
