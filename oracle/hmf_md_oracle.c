/*
 * hmf_md_oracle.c -- TEST INFRASTRUCTURE, NOT PART OF THE PRODUCT.
 *
 * A plain, slow, fp64 CPU statement of the molecular-dynamics comparator of the paper:
 * N particles of the Hamiltonian Mean Field model, eq (1) with the pair potential of eq (3) (L29-L39),
 *     H = sum_i p_i^2 / 2 + (1 / 2N) sum_{i,j} [1 - cos(theta_i - theta_j)],
 * integrated with the fourth-order symplectic scheme the paper names for its Fig. 4 run ("a MD simulation with
 * N = 20,000,000 particle using a sympletic integrator with time step dt = 0.1 [44]", L206; ref. [44] = Yoshida 1990).
 * The force on a particle needs only the two sums of eqs (7)-(8) (L56-L63), which is why "molecular dynamics
 * simulation times for the HMF model with N particles scale as N" (L65):
 *     M_x = (1/N) sum_j cos(theta_j),  M_y = (1/N) sum_j sin(theta_j),  F_i = -M_x sin(theta_i) + M_y cos(theta_i).
 *
 * One step of length dt (the paper gives no formula; reading D24: Yoshida's fourth-order composition of the
 * leapfrog in drift-kick-drift form, written out sub-step by sub-step as below, nothing fused or reordered):
 *     g1 = 1 / (2 - 2^(1/3)),  g2 = 1 - 2 g1
 *     drift(g1/2)  kick(g1)  drift((g1+g2)/2)  kick(g2)  drift((g1+g2)/2)  kick(g1)  drift(g1/2)
 *     drift(c): theta_i += c dt p_i          kick(d): (M_x, M_y) from the current theta, p_i += d dt F_i
 * Sums that define M and the energies are accumulated in long double in index order.  Shares no code, header,
 * table or constant generator with paper_1206_3229_b200/csrc.
 *
 * Pins (tests/test_md_oracle_pins.py): N = 2 is a pendulum (period 4 K(sin(phi0/2))); fourth-order convergence of
 * the trajectory and of the energy error; total momentum conserved to round-off (sum_i F_i = 0 identically); the
 * integrator is time reversible; U = (1 - M^2)/2 equals the double sum of eq (1); M(t) of a water-bag follows the
 * Vlasov oracle within the 1/sqrt(N) noise (Fig. 4).
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>

#define MD_OK 0
#define MD_EINVAL (-1)
#define MD_ENOTINIT (-2)
#define MD_ENOMEM (-4)

typedef struct {
    int ready;
    long n;
    double dt, t;
    double *theta, *p;
} md_t;

static md_t S = {0};

void oracle_md_free(void) {
    free(S.theta);
    free(S.p);
    memset(&S, 0, sizeof(S));
}

int oracle_md_init(long n, double dt) {
    if (n < 1 || !isfinite(dt)) return MD_EINVAL;
    oracle_md_free();
    S.theta = (double*)calloc((size_t)n, sizeof(double));
    S.p = (double*)calloc((size_t)n, sizeof(double));
    if (!S.theta || !S.p) {
        oracle_md_free();
        return MD_ENOMEM;
    }
    S.n = n;
    S.dt = dt;
    S.ready = 1;
    return MD_OK;
}

int oracle_md_upload(const double* theta, const double* p) {
    if (!S.ready) return MD_ENOTINIT;
    memcpy(S.theta, theta, (size_t)S.n * sizeof(double));
    memcpy(S.p, p, (size_t)S.n * sizeof(double));
    S.t = 0.0;
    return MD_OK;
}

int oracle_md_download(double* theta, double* p) {
    if (!S.ready) return MD_ENOTINIT;
    memcpy(theta, S.theta, (size_t)S.n * sizeof(double));
    memcpy(p, S.p, (size_t)S.n * sizeof(double));
    return MD_OK;
}

/* eq (8) for particles: M = (1/N) sum (cos theta_j, sin theta_j) */
static void magnetisation(double* mx, double* my) {
    long double cx = 0.0L, sx = 0.0L;
    for (long j = 0; j < S.n; ++j) {
        cx += (long double)cos(S.theta[j]);
        sx += (long double)sin(S.theta[j]);
    }
    *mx = (double)(cx / (long double)S.n);
    *my = (double)(sx / (long double)S.n);
}

static void drift(double c) {
    for (long i = 0; i < S.n; ++i) S.theta[i] += c * S.dt * S.p[i];
}

/* eq (7): F_i = -sin(theta_i) M_x + cos(theta_i) M_y */
static void kick(double d) {
    double mx, my;
    magnetisation(&mx, &my);
    for (long i = 0; i < S.n; ++i) S.p[i] += d * S.dt * (-sin(S.theta[i]) * mx + cos(S.theta[i]) * my);
}

int oracle_md_step(int nsteps) {
    if (!S.ready) return MD_ENOTINIT;
    if (nsteps <= 0) return MD_EINVAL;
    const double g1 = 1.0 / (2.0 - cbrt(2.0)), g2 = 1.0 - 2.0 * g1;
    for (int it = 0; it < nsteps; ++it) {
        drift(0.5 * g1);
        kick(g1);
        drift(0.5 * (g1 + g2));
        kick(g2);
        drift(0.5 * (g1 + g2));
        kick(g1);
        drift(0.5 * g1);
        S.t += S.dt;
    }
    return MD_OK;
}

/* out = {t, M_x, M_y, K/N, U/N, E/N, P/N, 0}:  K/N = (1/N) sum p^2/2;  U/N = (1 - M_x^2 - M_y^2)/2 (eq (1), (3): the
 * double sum (1/2N^2) sum_ij [1 - cos(theta_i - theta_j)] collapses to this);  P/N = (1/N) sum p */
int oracle_md_moments(double out[8]) {
    if (!S.ready) return MD_ENOTINIT;
    double mx, my;
    magnetisation(&mx, &my);
    long double k = 0.0L, pp = 0.0L;
    for (long i = 0; i < S.n; ++i) {
        k += 0.5L * (long double)S.p[i] * (long double)S.p[i];
        pp += (long double)S.p[i];
    }
    out[0] = S.t;
    out[1] = mx;
    out[2] = my;
    out[3] = (double)(k / (long double)S.n);
    out[4] = 0.5 * (1.0 - mx * mx - my * my);
    out[5] = out[3] + out[4];
    out[6] = (double)(pp / (long double)S.n);
    out[7] = 0.0;
    return MD_OK;
}

/* U/N by the definition, eq (1) with eq (3): (1 / 2N^2) sum_{i,j} [1 - cos(theta_i - theta_j)]; O(N^2), tests only */
double oracle_md_potential_double_sum(void) {
    long double u = 0.0L;
    for (long i = 0; i < S.n; ++i)
        for (long j = 0; j < S.n; ++j) u += 1.0L - (long double)cos(S.theta[i] - S.theta[j]);
    return (double)(u / (2.0L * (long double)S.n * (long double)S.n));
}
