/*
 * vlasov_oracle.c -- TEST INFRASTRUCTURE, NOT PART OF THE PRODUCT.
 *
 * A plain, slow, fp64 CPU statement of the time-split semi-Lagrangian Vlasov
 * step of T. M. Rocha Filho, "Solving the Vlasov equation for one-dimensional
 * models with long range interactions on a GPU" (arXiv 1206.3229), written
 * from the paper in the paper's order and notation so that it can
 * be checked against the text by eye.  It shares no code, header, table or
 * constant generator with the CUDA library in paper_1206_3229_b200/csrc and
 * must only be used by tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs.
 *
 * What it computes, per time step (section 3, eqs 9-12):
 *   (1) f_I (x,p) = f(x - p dt/2, p)            eq (9)
 *   (2) F_I (x)   = mean-field force of f_I      eq (10)
 *   (3) f_II(x,p) = f_I(x, p - F_I(x) dt)        eq (11)
 *   (4) f(t+dt)   = f_II(x - p dt/2, p)          eq (12)
 * where every value at the foot of a characteristic comes from the cubic
 * spline of eqs (13)-(14) (L89-L98) whose second derivatives are NOT the
 * solution of the tridiagonal system (15) but the eighth-order centred finite
 * difference of eq (16) (L106-L111).  As in the paper (L115) the second
 * derivatives are materialised as an array before eq (13) is evaluated;
 * nothing is fused, blocked or reordered.
 *
 * Storage (L115): one flat array f[j*n_x + i], i the position index, j the
 * momentum index.  Grid nodes x_i = x_min + i*dx, dx = (x_max-x_min)/n_x,
 * i = 0..n_x-1 (half-open domain; reading D3), same for p.
 *
 * Readings of the paper where it is silent or garbled:
 *   D1  eq (13) prints f''_{i+i}: read f''_{i+1}.
 *   D2  eq (16) omits the 1/h^2 factor: f'' = (sum_m c_m f_{i+m}) / h^2.
 *   D4  boundaries: the paper is periodic in x and p (L113); BASELINE.json
 *       asks for "f = 0 beyond" in p and for the sheet model in x.  Both are
 *       here (bc = 0 periodic, 1 zero extension).  Zero extension: the line
 *       is the infinite sequence that is 0 outside [0,n); f'' is the stencil
 *       applied to that sequence at every index where it is needed.
 *   D5  foot on a knot: s = floor(u), a = u - s, a clamped to [0,1).
 *   D6  integrals are rectangle-rule sums over the nodes.
 *   D9  ring force: circulant sum with K[m] = -V'(m dtheta), K[0] = 0.
 *   D10 energy E = K + U, U = (1/2) int rho phi.
 *   D11 sheet force F_i = -dx (sum_{k<i} rho_k - sum_{k>i} rho_k).
 *
 * Pins (tests/test_oracle_pins.py, all run with -m "not gpu"): polynomial
 * exactness of eq (16), a = 0 identity, cubic exactness and Fourier symbol of
 * one shift, mass / momentum conservation, free streaming against the
 * analytic solution, stationary homogeneous state, HMF linear growth rate and
 * the T = 1/2 threshold, the paper's printed water-bag numbers (L192, L204),
 * sheet and ring closed forms, Strang second order, zero extension == padded
 * periodic.  Parity unpinned: none of the functions below; the long-time
 * nonlinear curves of Figs 1-5 (images absent) are not reproduced.
 *
 * Global-spline variant (the paper's comparator "GS",
 * L100-L104, Tables 1-2): with oracle_set_param(KEY_SPLINE, 1) the second
 * derivatives are the solution of the tridiagonal system (15) of every line
 * instead of eq (16); everything else is unchanged.  Periodic lines: the
 * cyclic system.  Zero extension (D4, D21): the line is the infinite
 * sequence that is 0 outside [0,n) and f'' its bounded solution of (15),
 * obtained as the cyclic solution on the line padded by GS_EXT zeros on each
 * side (the influence of a value decays by |sqrt(3)-2| = 0.268 per node:
 * 0.268^64 = 2.6e-37).  Pins G1-G7 in tests/test_oracle_pins.py.
 *
 * Sums that define integrals are accumulated in long double; everything else
 * is IEEE double.  Optional OpenMP over independent lines (off unless
 * oracle_set_threads(n>1) is called); it does not change any result.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_OK 0
#define ORACLE_EINVAL (-1)
#define ORACLE_ENOTINIT (-2)
#define ORACLE_ENOMEM (-4)

enum { MODEL_FREE = 0, MODEL_HMF = 1, MODEL_RING = 2, MODEL_SHEET = 3 };
enum { BC_PERIODIC = 0, BC_ZERO = 1 };
enum { KEY_EPS = 1, KEY_PRECISION = 2, KEY_BC_X = 3, KEY_BC_P = 4, KEY_HISTORY = 5, KEY_SPLINE = 6, KEY_ORDER = 7 };
enum { SPLINE_FD = 0, SPLINE_GS = 1 };

/* eq (16): coefficients of f(u_{i-4}) ... f(u_{i+4}). */
static const double C16[9] = {
    -1.0 / 560.0, 8.0 / 315.0, -1.0 / 5.0, 8.0 / 5.0, -205.0 / 72.0,
    8.0 / 5.0,    -1.0 / 5.0,  8.0 / 315.0, -1.0 / 560.0};

#define EXT 5 /* zero extension: f'' can be non-zero for -4 <= k < n+4; we keep k in [-5, n+5) */
#define GS_EXT 64 /* zero extension, system (15): f'' decays by 0.268 per node outside [0,n); kept on [-64, n+64) */

static int g_threads = 1;

void oracle_set_threads(int n) { g_threads = n > 0 ? n : 1; }
int oracle_get_threads(void) { return g_threads; }

/* ------------------------------------------------------------------ */
/* line-level pieces (stateless; exported so the pins can reach them)  */
/* ------------------------------------------------------------------ */

static long wrap(long k, long n) {
    long r = k % n;
    return r < 0 ? r + n : r;
}

/* the line as an infinite sequence: periodic image or zero extension (D4) */
static double line_at(const double* u, long n, int bc, long k) {
    if (bc == BC_PERIODIC) return u[wrap(k, n)];
    return (k >= 0 && k < n) ? u[k] : 0.0;
}

/*
 * eq (16) (L110) with the 1/h^2 of reading D2.
 * periodic: d2 has n entries, d2[k] = f''(u_k).
 * zero ext: d2 has n + 2*EXT entries, d2[k + EXT] = f''(u_k), k = -EXT..n+EXT-1.
 */
void oracle_fd8_second_derivative(const double* u, long n, double h, int bc, double* d2) {
    long lo = (bc == BC_PERIODIC) ? 0 : -EXT;
    long hi = (bc == BC_PERIODIC) ? n : n + EXT;
    for (long k = lo; k < hi; ++k) {
        double acc = 0.0;
        for (int m = -4; m <= 4; ++m) acc += C16[m + 4] * line_at(u, n, bc, k + m);
        d2[k - lo] = acc / (h * h);
    }
}

static double d2_at_ext(const double* d2, long n, int bc, long k, long ext) {
    if (bc == BC_PERIODIC) return d2[wrap(k, n)];
    return (k >= -ext && k < n + ext) ? d2[k + ext] : 0.0;
}

/*
 * System (15) (L100-L102) with periodic closure, i = 0..n-1, indices mod n:
 *     (d2[i+1]/6 + (2/3) d2[i] + d2[i-1]/6) = rhs[i],   rhs[i] = (u[i+1] - 2u[i] + u[i-1]) / h^2.
 * Reading D22: the paper prints the middle coefficient as 1/3.  Continuity of the first derivative of
 * eq (13) across the knot x_i (the condition the text states, L100) gives h/6 d2[i-1] + (h/3 + h/3) d2[i] +
 * h/6 d2[i+1]: each of the two intervals that meet at x_i contributes h/3, so the coefficient is 2/3 (the
 * form of ref. [37]).  With 1/3 a constant f'' would come out 3/2 too large and the system is singular
 * on the mode (-1)^i.  Solved directly: Thomas elimination of the tridiagonal part plus the
 * Sherman-Morrison correction for the two corner entries.  n >= 3.  scratch: 3n doubles.
 */
static void cyclic_spline_system(const double* rhs, long n, double* x, double* scratch) {
    const double lo = 1.0 / 6.0, di = 2.0 / 3.0, up = 1.0 / 6.0;
    double* cp = scratch;         /* modified upper diagonal */
    double* y = scratch + n;      /* solution of T y = rhs   */
    double* z = scratch + 2 * n;  /* solution of T z = u     */
    /* A = T + u v^T, T tridiagonal with T[0][0] = di - gamma, T[n-1][n-1] = di - up*lo/gamma,
       u = (gamma, 0, .., 0, up)^T, v = (1, 0, .., 0, lo/gamma)^T;  x = y - z (v.y)/(1 + v.z) */
    const double gamma = -di;
    for (int pass = 0; pass < 2; ++pass) {
        double* out = pass == 0 ? y : z;
        double b0 = di - gamma, bn = di - up * lo / gamma;
        double r0 = pass == 0 ? rhs[0] : gamma;
        cp[0] = up / b0;
        out[0] = r0 / b0;
        for (long i = 1; i < n; ++i) {
            double b = (i == n - 1) ? bn : di;
            double r = pass == 0 ? rhs[i] : (i == n - 1 ? up : 0.0);
            double m = b - lo * cp[i - 1];
            cp[i] = up / m;
            out[i] = (r - lo * out[i - 1]) / m;
        }
        for (long i = n - 2; i >= 0; --i) out[i] -= cp[i] * out[i + 1];
    }
    double vy = y[0] + lo / gamma * y[n - 1];
    double vz = z[0] + lo / gamma * z[n - 1];
    double fac = vy / (1.0 + vz);
    for (long i = 0; i < n; ++i) x[i] = y[i] - fac * z[i];
}

/*
 * Second derivatives of the global cubic spline, system (15).
 * periodic: d2 has n entries.  zero ext: d2 has n + 2*GS_EXT entries, d2[k + GS_EXT] = f''(u_k).
 * Returns 0, or ORACLE_ENOMEM / ORACLE_EINVAL (n < 3).
 */
int oracle_gs_second_derivative(const double* u, long n, double h, int bc, double* d2) {
    long lo = (bc == BC_PERIODIC) ? 0 : -GS_EXT;
    long hi = (bc == BC_PERIODIC) ? n : n + GS_EXT;
    long N = hi - lo;
    if (N < 3) return ORACLE_EINVAL;
    double* rhs = (double*)malloc((size_t)N * 4 * sizeof(double));
    if (!rhs) return ORACLE_ENOMEM;
    for (long k = lo; k < hi; ++k)
        rhs[k - lo] = (line_at(u, n, bc, k + 1) - 2.0 * line_at(u, n, bc, k) + line_at(u, n, bc, k - 1)) / (h * h);
    cyclic_spline_system(rhs, N, d2, rhs + N);
    free(rhs);
    return ORACLE_OK;
}

/*
 * out_i = f(x_i - disp) for every node of one line, by eqs (13)-(14) (L89-L98)
 * with f'' from eq (16).  h is the node spacing, disp the (signed) physical
 * displacement.  The foot x = x_i - disp lies in [x_k, x_{k+1}] with
 * k = i + s, s = floor(-disp/h); in the paper's symbols
 *   alpha = (x_{k+1} - x)/h = 1 - a,  beta = 1 - alpha = a,
 *   gamma = (alpha^3 - alpha) h^2/6,  delta = (beta^3 - beta) h^2/6.
 * kind = SPLINE_FD: f'' from eq (16); SPLINE_GS: f'' from system (15).
 * d2 is scratch of n + 2*GS_EXT doubles.
 */
int oracle_shift_line_kind(const double* in, long n, double h, double disp, int bc, int kind, double* out,
                           double* d2) {
    long ext = EXT;
    if (kind == SPLINE_GS) {
        int rc = oracle_gs_second_derivative(in, n, h, bc, d2);
        if (rc != ORACLE_OK) return rc;
        ext = GS_EXT;
    } else {
        oracle_fd8_second_derivative(in, n, h, bc, d2);
    }
    double u = -disp / h;
    double sf = floor(u);
    double a = u - sf;
    if (a >= 1.0) { /* u = -tiny: floor = -1 and u+1 rounds to 1 (D5) */
        sf += 1.0;
        a = 0.0;
    }
    long s = (long)sf;
    double alpha = 1.0 - a, beta = a;
    double gamma = (alpha * alpha * alpha - alpha) / 6.0 * (h * h);
    double delta = (beta * beta * beta - beta) / 6.0 * (h * h);
    for (long i = 0; i < n; ++i) {
        long k = i + s;
        out[i] = alpha * line_at(in, n, bc, k) + beta * line_at(in, n, bc, k + 1) +
                 gamma * d2_at_ext(d2, n, bc, k, ext) + delta * d2_at_ext(d2, n, bc, k + 1, ext);
    }
    return ORACLE_OK;
}

/* eq (16) variant (the paper's method); d2 is scratch of n + 2*GS_EXT doubles */
void oracle_shift_line(const double* in, long n, double h, double disp, int bc, double* out,
                       double* d2) {
    (void)oracle_shift_line_kind(in, n, h, disp, bc, SPLINE_FD, out, d2);
}

/* convenience for the pins: allocates its own scratch */
int oracle_shift_line_kind_alloc(const double* in, long n, double h, double disp, int bc, int kind,
                                 double* out) {
    double* d2 = (double*)malloc((size_t)(n + 2 * GS_EXT) * sizeof(double));
    double* tmp = (double*)malloc((size_t)n * sizeof(double));
    if (!d2 || !tmp) { free(d2); free(tmp); return ORACLE_ENOMEM; }
    int rc = oracle_shift_line_kind(in, n, h, disp, bc, kind, tmp, d2);
    if (rc == ORACLE_OK) memcpy(out, tmp, (size_t)n * sizeof(double));
    free(d2);
    free(tmp);
    return rc;
}

int oracle_shift_line_alloc(const double* in, long n, double h, double disp, int bc, double* out) {
    return oracle_shift_line_kind_alloc(in, n, h, disp, bc, SPLINE_FD, out);
}

/* pair potentials, eqs (2)-(4) (L33-L45), and K = -dV/dx for the ring */
static double ring_V(double x, double eps) { return -1.0 / (sqrt(2.0) * sqrt(1.0 - cos(x) + eps)); }
static double ring_K(double x, double eps) {
    double q = 1.0 - cos(x) + eps;
    return -sin(x) / (2.0 * sqrt(2.0) * q * sqrt(q));
}

/*
 * Mean-field force on the nodes from the density, eq (6)/(10) (L52-L54,
 * L75-L78) discretised by the rectangle rule (D6):
 *   HMF   eq (7)-(8) (L56-L63): F = -sin(th) Mx + cos(th) My,
 *         Mx = dth sum cos(th_i) rho_i, My = dth sum sin(th_i) rho_i;
 *   ring  eq (2): F_i = dth sum_m K(m dth) rho_{(i-m) mod n}   (D9);
 *   sheet eq (4): F_i = -dx (sum_{k<i} rho_k - sum_{k>i} rho_k) (D11);
 *   free  F = 0.
 */
void oracle_force_from_rho(int model, const double* rho, long n, double xmin, double xmax,
                           double eps, double* F) {
    double dx = (xmax - xmin) / (double)n;
    if (model == MODEL_HMF) {
        long double mx = 0.0L, my = 0.0L;
        for (long i = 0; i < n; ++i) {
            double th = xmin + (double)i * dx;
            mx += (long double)(cos(th) * rho[i]);
            my += (long double)(sin(th) * rho[i]);
        }
        double Mx = (double)(mx * dx), My = (double)(my * dx);
        for (long i = 0; i < n; ++i) {
            double th = xmin + (double)i * dx;
            F[i] = -sin(th) * Mx + cos(th) * My;
        }
    } else if (model == MODEL_RING) {
        double* K = (double*)malloc((size_t)n * sizeof(double));
        for (long m = 0; m < n; ++m) K[m] = (m == 0) ? 0.0 : ring_K((double)m * dx, eps);
        for (long i = 0; i < n; ++i) {
            long double acc = 0.0L;
            for (long m = 0; m < n; ++m) acc += (long double)(K[m] * rho[wrap(i - m, n)]);
            F[i] = (double)(acc * dx);
        }
        free(K);
    } else if (model == MODEL_SHEET) {
        for (long i = 0; i < n; ++i) {
            long double left = 0.0L, right = 0.0L;
            for (long k = 0; k < i; ++k) left += (long double)rho[k];
            for (long k = i + 1; k < n; ++k) right += (long double)rho[k];
            F[i] = (double)(-(left - right) * dx);
        }
    } else {
        for (long i = 0; i < n; ++i) F[i] = 0.0;
    }
}

/* ------------------------------------------------------------------ */
/* the solver state (singleton, mirrors the product's C ABI)           */
/* ------------------------------------------------------------------ */

typedef struct {
    int ready;
    int model;
    long nx, np;
    double xmin, xmax, pmin, pmax, dt, eps, t;
    int bc_x, bc_p;
    int spline; /* SPLINE_FD (eq 16, default) or SPLINE_GS (system 15) */
    int order;  /* 2: the paper's time split (L71-L87); 4: its triple-jump composition (L238, refs [31], [44]) */
    double* f;
} ctx_t;

static ctx_t G = {0};

void oracle_free(void) {
    free(G.f);
    memset(&G, 0, sizeof(G));
}

int oracle_init(int model, const int grid[2], const double domain[4], double dt) {
    if (model < 0 || model > 3 || !grid || !domain) return ORACLE_EINVAL;
    if (grid[0] < 1 || grid[1] < 1 || !(domain[1] > domain[0]) || !(domain[3] > domain[2]))
        return ORACLE_EINVAL;
    oracle_free();
    G.model = model;
    G.nx = grid[0];
    G.np = grid[1];
    G.xmin = domain[0];
    G.xmax = domain[1];
    G.pmin = domain[2];
    G.pmax = domain[3];
    G.dt = dt;
    G.eps = 0.01;
    G.t = 0.0;
    G.bc_x = (model == MODEL_SHEET) ? BC_ZERO : BC_PERIODIC;
    G.bc_p = BC_ZERO;
    G.spline = SPLINE_FD;
    G.order = 2;
    G.f = (double*)calloc((size_t)G.nx * (size_t)G.np, sizeof(double));
    if (!G.f) return ORACLE_ENOMEM;
    G.ready = 1;
    return ORACLE_OK;
}

int oracle_set_param(int key, double value) {
    if (!G.ready) return ORACLE_ENOTINIT;
    switch (key) {
        case KEY_EPS: if (!(value > 0.0)) return ORACLE_EINVAL; G.eps = value; break;
        case KEY_PRECISION: if (value != 64.0) return ORACLE_EINVAL; break; /* the oracle is fp64 only */
        case KEY_BC_X: if (value != 0.0 && value != 1.0) return ORACLE_EINVAL; G.bc_x = (int)value; break;
        case KEY_BC_P: if (value != 0.0 && value != 1.0) return ORACLE_EINVAL; G.bc_p = (int)value; break;
        case KEY_HISTORY: break;
        case KEY_SPLINE: if (value != 0.0 && value != 1.0) return ORACLE_EINVAL; G.spline = (int)value; break;
        case KEY_ORDER: if (value != 2.0 && value != 4.0) return ORACLE_EINVAL; G.order = (int)value; break;
        default: return ORACLE_EINVAL;
    }
    return ORACLE_OK;
}

int oracle_upload(const double* f_host) {
    if (!G.ready) return ORACLE_ENOTINIT;
    memcpy(G.f, f_host, (size_t)G.nx * (size_t)G.np * sizeof(double));
    G.t = 0.0;
    return ORACLE_OK;
}

int oracle_download(double* f_host) {
    if (!G.ready) return ORACLE_ENOTINIT;
    memcpy(f_host, G.f, (size_t)G.nx * (size_t)G.np * sizeof(double));
    return ORACLE_OK;
}

static double dx_(void) { return (G.xmax - G.xmin) / (double)G.nx; }
static double dp_(void) { return (G.pmax - G.pmin) / (double)G.np; }
static double x_at(long i) { return G.xmin + (double)i * dx_(); }
static double p_at(long j) { return G.pmin + (double)j * dp_(); }

/* steps (1) and (4): f(x,p) <- f(x - p tau, p), row by row; eq (9)/(12) */
int oracle_theta_sweep(double tau) {
    if (!G.ready) return ORACLE_ENOTINIT;
    long nx = G.nx, np = G.np;
    double h = dx_();
#pragma omp parallel num_threads(g_threads)
    {
        double* out = (double*)malloc((size_t)nx * sizeof(double));
        double* d2 = (double*)malloc((size_t)(nx + 2 * GS_EXT) * sizeof(double));
#pragma omp for schedule(static)
        for (long j = 0; j < np; ++j) {
            double* row = G.f + (size_t)j * (size_t)nx;
            (void)oracle_shift_line_kind(row, nx, h, p_at(j) * tau, G.bc_x, G.spline, out, d2);
            memcpy(row, out, (size_t)nx * sizeof(double));
        }
        free(out);
        free(d2);
    }
    return ORACLE_OK;
}

/* rho_i = dp sum_j f_ij  (the p-integral in eqs (6), (8), (10); D6) */
int oracle_density(double* rho) {
    if (!G.ready) return ORACLE_ENOTINIT;
    double dp = dp_();
    for (long i = 0; i < G.nx; ++i) {
        long double acc = 0.0L;
        for (long j = 0; j < G.np; ++j) acc += (long double)G.f[(size_t)j * (size_t)G.nx + (size_t)i];
        rho[i] = (double)(acc * dp);
    }
    return ORACLE_OK;
}

/* step (2): force of the current f; eq (10) */
int oracle_force(double* F) {
    if (!G.ready) return ORACLE_ENOTINIT;
    double* rho = (double*)malloc((size_t)G.nx * sizeof(double));
    if (!rho) return ORACLE_ENOMEM;
    oracle_density(rho);
    oracle_force_from_rho(G.model, rho, G.nx, G.xmin, G.xmax, G.eps, F);
    free(rho);
    return ORACLE_OK;
}

/* step (3): f(x,p) <- f(x, p - F(x) dt), column by column; eq (11) */
int oracle_p_sweep_with_force(const double* F, double dt) {
    if (!G.ready) return ORACLE_ENOTINIT;
    long nx = G.nx, np = G.np;
    double h = dp_();
#pragma omp parallel num_threads(g_threads)
    {
        double* col = (double*)malloc((size_t)np * sizeof(double));
        double* out = (double*)malloc((size_t)np * sizeof(double));
        double* d2 = (double*)malloc((size_t)(np + 2 * GS_EXT) * sizeof(double));
#pragma omp for schedule(static)
        for (long i = 0; i < nx; ++i) {
            for (long j = 0; j < np; ++j) col[j] = G.f[(size_t)j * (size_t)nx + (size_t)i];
            (void)oracle_shift_line_kind(col, np, h, F[i] * dt, G.bc_p, G.spline, out, d2);
            for (long j = 0; j < np; ++j) G.f[(size_t)j * (size_t)nx + (size_t)i] = out[j];
        }
        free(col);
        free(out);
        free(d2);
    }
    return ORACLE_OK;
}

int oracle_p_sweep(double dt) {
    if (!G.ready) return ORACLE_ENOTINIT;
    double* F = (double*)malloc((size_t)G.nx * sizeof(double));
    if (!F) return ORACLE_ENOMEM;
    oracle_force(F);
    int rc = oracle_p_sweep_with_force(F, dt);
    free(F);
    return rc;
}

/* one time-split step (1)-(4) of section 3 (L71-L87) over the time h (h may be negative) */
static void strang_step(double h) {
    oracle_theta_sweep(0.5 * h); /* (1) eq (9)  */
    oracle_p_sweep(h);           /* (2)+(3) eqs (10), (11) */
    oracle_theta_sweep(0.5 * h); /* (4) eq (12) */
}

/*
 * n time steps.  order 2 (default): each step is (1)-(4) of section 3 (L71-L87).
 * order 4 ("Higher order time split schemes ... can also be implemented if required",
 * PAPER.md L238 with ref. [31]): the paper gives no formula, so the reading (D23) is the standard
 * fourth-order composition of a symmetric second-order step S2, the "triple jump" of the paper's own ref. [44]
 * (Yoshida 1990, cited at L206 for the N-body integrator):
 *     S4(dt) = S2(g1 dt) S2(g2 dt) S2(g1 dt),   g1 = 1/(2 - 2^(1/3)),  g2 = 1 - 2 g1 = -2^(1/3)/(2 - 2^(1/3)),
 * whose middle sub-step runs backwards in time (g2 < 0).  Each S2 is the unchanged step (1)-(4), force included.
 */
int oracle_step(int n) {
    if (!G.ready) return ORACLE_ENOTINIT;
    if (n <= 0) return ORACLE_EINVAL;
    const double g1 = 1.0 / (2.0 - cbrt(2.0)), g2 = 1.0 - 2.0 * g1;
    for (int it = 0; it < n; ++it) {
        if (G.order == 4) {
            strang_step(g1 * G.dt);
            strang_step(g2 * G.dt);
            strang_step(g1 * G.dt);
        } else {
            strang_step(G.dt);
        }
        G.t += G.dt;
    }
    return ORACLE_OK;
}

/*
 * Casimir invariants (eq (18)): C[s] = int s(f) dp dx by the rectangle rule on the nodes.
 *   out[0]  S  = dx dp sum s(f_ij),  s(f) = -f log f  (the entropy of Fig. 2); s(0) = 0 (its limit); the scheme is
 *           not positivity preserving, and where it has produced f < 0 the entropy density is undefined: those
 *           nodes contribute 0 here and their weight is reported in out[2] (reading D20)
 *   out[1]  C2 = dx dp sum f_ij^2     (s(f) = f^2, the "enstrophy")
 *   out[2]  N- = dx dp sum min(f_ij, 0)  (negative mass; 0 for a non-negative state)
 *   out[3]  max f_ij
 * Exact Vlasov dynamics conserves S and C2; on a grid both drift once filaments reach the mesh size (L188).
 */
int oracle_casimirs(double out[4]) {
    if (!G.ready) return ORACLE_ENOTINIT;
    long nx = G.nx, np = G.np;
    long double S = 0.0L, C2 = 0.0L, neg = 0.0L;
    double fmax = G.f[0];
    for (long j = 0; j < np; ++j) {
        for (long i = 0; i < nx; ++i) {
            double v = G.f[(size_t)j * (size_t)nx + (size_t)i];
            if (v > 0.0) S -= (long double)(v * log(v));
            if (v < 0.0) neg += (long double)v;
            C2 += (long double)(v * v);
            if (v > fmax) fmax = v;
        }
    }
    long double w = (long double)dx_() * (long double)dp_();
    out[0] = (double)(S * w);
    out[1] = (double)(C2 * w);
    out[2] = (double)(neg * w);
    out[3] = fmax;
    return ORACLE_OK;
}

/*
 * out = {t, mass, P, K, U, Mx, My, E}.  Rectangle rule (D6):
 *   mass = dx dp sum f;  P = dx dp sum p_j f;  K = dx dp sum p_j^2/2 f;
 *   Mx, My: eq (8) (L62);  U = (1/2) int rho phi (D10):
 *     HMF   phi = mass - Mx cos - My sin  => U = (mass^2 - Mx^2 - My^2)/2
 *     ring  phi_i = dth sum_m V(m dth) rho_{i-m}
 *     sheet phi_i = dx sum_k |x_i - x_k| rho_k
 *   E = K + U.
 */
int oracle_moments(double out[8]) {
    if (!G.ready) return ORACLE_ENOTINIT;
    long nx = G.nx, np = G.np;
    double dx = dx_(), dp = dp_();
    long double mass = 0.0L, P = 0.0L, K = 0.0L;
    for (long j = 0; j < np; ++j) {
        long double r = 0.0L;
        for (long i = 0; i < nx; ++i) r += (long double)G.f[(size_t)j * (size_t)nx + (size_t)i];
        double p = p_at(j);
        mass += r;
        P += (long double)p * r;
        K += (long double)(0.5 * p * p) * r;
    }
    mass *= (long double)dx * dp;
    P *= (long double)dx * dp;
    K *= (long double)dx * dp;
    double* rho = (double*)malloc((size_t)nx * sizeof(double));
    if (!rho) return ORACLE_ENOMEM;
    oracle_density(rho);
    long double mx = 0.0L, my = 0.0L;
    for (long i = 0; i < nx; ++i) {
        mx += (long double)(cos(x_at(i)) * rho[i]);
        my += (long double)(sin(x_at(i)) * rho[i]);
    }
    double Mx = (double)(mx * dx), My = (double)(my * dx);
    long double U = 0.0L;
    if (G.model == MODEL_HMF) {
        U = 0.5L * (mass * mass - (long double)Mx * Mx - (long double)My * My);
    } else if (G.model == MODEL_RING) {
        for (long i = 0; i < nx; ++i) {
            long double phi = 0.0L;
            for (long m = 0; m < nx; ++m)
                phi += (long double)(ring_V((double)m * dx, G.eps) * rho[wrap(i - m, nx)]);
            U += (long double)rho[i] * (phi * dx);
        }
        U *= 0.5L * dx;
    } else if (G.model == MODEL_SHEET) {
        for (long i = 0; i < nx; ++i) {
            long double phi = 0.0L;
            for (long k = 0; k < nx; ++k) phi += (long double)(fabs(x_at(i) - x_at(k)) * rho[k]);
            U += (long double)rho[i] * (phi * dx);
        }
        U *= 0.5L * dx;
    }
    free(rho);
    out[0] = G.t;
    out[1] = (double)mass;
    out[2] = (double)P;
    out[3] = (double)K;
    out[4] = (double)U;
    out[5] = Mx;
    out[6] = My;
    out[7] = (double)(K + U);
    return ORACLE_OK;
}
