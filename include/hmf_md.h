/*
 * hmf_md.h -- C ABI of the B200-native N-particle molecular dynamics of the Hamiltonian Mean Field model, the
 * comparator of the paper's Fig. 4.  Citations are PAPER.md line numbers.
 *
 * Model: eq (1) with the pair potential of eq (3) (L29-L39), H = sum p_i^2/2 + (1/2N) sum_ij [1 - cos(theta_i - theta_j)].
 * The force needs only the two sums of eqs (7)-(8) (L56-L63),
 *     M_x = (1/N) sum_j cos(theta_j),  M_y = (1/N) sum_j sin(theta_j),  F_i = -M_x sin(theta_i) + M_y cos(theta_i),
 * so that one step costs O(N) (L65).  Integrator: the fourth-order symplectic composition the paper names for its
 * MD run (L206, ref. [44]), in drift-kick-drift form with g1 = 1/(2 - 2^(1/3)), g2 = 1 - 2 g1 (D24):
 *     drift(g1/2) kick(g1) drift((g1+g2)/2) kick(g2) drift((g1+g2)/2) kick(g1) drift(g1/2).
 * On the GPU a kick, the drift after it and the sums (M_x, M_y) of the new angles are ONE pass over the particles
 * (kernel md_kick_drift_kernel); the trailing and leading half drifts of consecutive steps share a pass:
 * n steps = 3 n + 1 passes of 32 bytes per particle (read and write theta and p).
 *
 * Conventions: every function returns 0 or a negative HMF_MD_E* code; hmf_md_last_error() has the message; one
 * singleton context per process (independent of the Vlasov context of vlasov.h); "host" pointers are CPU memory,
 * "device" pointers CUDA global memory of the current device; work is enqueued on the attached stream; only
 * hmf_md_download, hmf_md_moments and hmf_md_kernel_times block.  No CPU fallback: without a CUDA device
 * hmf_md_init fails with HMF_MD_ECUDA.
 */
#ifndef HMF_MD_B200_H
#define HMF_MD_B200_H

#ifdef __cplusplus
extern "C" {
#endif

#define HMF_MD_OK 0
#define HMF_MD_EINVAL (-1)
#define HMF_MD_ENOTINIT (-2)
#define HMF_MD_ECUDA (-3)
#define HMF_MD_ENOMEM (-4)

/* Create the context: n >= 1 particles, time step dt of one full integrator step.  Frees a previous context. */
int hmf_md_init(long long n, double dt);

/* Hand the library caller-owned device arrays (n doubles each, 16-byte aligned; their content is the state) and a
 * cudaStream_t cast to void* (NULL = legacy default stream).  Without this call the library allocates its own. */
int hmf_md_attach(void* theta_dev, void* p_dev, void* cuda_stream);

/* Host -> device copy of the state (n doubles each); sets t = 0.  Device -> host copy of the state (blocks). */
int hmf_md_upload(const double* theta_host, const double* p_host);
int hmf_md_download(double* theta_host, double* p_host);

/* Enqueue nsteps >= 1 integrator steps (asynchronous): 3 nsteps + 1 launches of md_kick_drift_kernel. */
int hmf_md_step(int nsteps);

/* out (host, 8 doubles) = {t, M_x, M_y, K/N, U/N, E/N, P/N, 0} of the current state: K/N = (1/N) sum p^2/2,
 * U/N = (1 - M_x^2 - M_y^2)/2 (the double sum of eq (1) with eq (3)), E = K + U, P/N = (1/N) sum p.  Blocks. */
int hmf_md_moments(double out[8]);

/* out (host) = {milliseconds, launches} of md_kick_drift_kernel since the last call, from CUDA events around every
 * launch (recorded only while profiling is on: hmf_md_profile(1)).  Blocks; resets the record. */
int hmf_md_profile(int on);
int hmf_md_kernel_times(double out[2]);

/* Number of kernels launched since hmf_md_init. */
int hmf_md_launch_count(unsigned long long* out);

void hmf_md_free(void);
const char* hmf_md_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* HMF_MD_B200_H */
