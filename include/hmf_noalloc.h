/*
 * hmf_noalloc.h -- ONE entry point of the library that allocates nothing, for callers that cannot call cudaMalloc
 * (code under CUDA graph capture, tight serving loops, harnesses that forbid allocation).
 *
 * What it computes: the moments of an N-particle state of the Hamiltonian Mean Field model, the same numbers as
 * hmf_md_moments (include/hmf_md.h; eqs (7)-(8), L56-L63, and eq (1) with eq (3)):
 *     M_x = (1/N) sum cos(theta_i),  M_y = (1/N) sum sin(theta_i),  K/N = (1/N) sum p_i^2/2,
 *     U/N = (1 - M_x^2 - M_y^2)/2,  E/N = K/N + U/N,  P/N = (1/N) sum p_i.
 * hmf_md_moments keeps the per-block partial sums of its reduction in a cudaMalloc'ed buffer of the MD context; this
 * variant keeps them in a file-scope `static __device__` array inside the library:
 *     256 KiB of partial sums (8192 blocks x 4 doubles) + 256 bytes (the counter of finished blocks)
 * per GPU that loads the library, held until the process exits.  A block sums 4096 particles, hence the limit
 *     n <= HMF_NOALLOC_MAX_PARTICLES = 8192 * 4096 = 33,554,432
 * (the paper's MD run has N = 2e7, L206).  Larger n is rejected with HMF_NOALLOC_EINVAL, nothing is launched.
 *
 * The call needs no context (no hmf_md_init): the caller passes inputs and output.  It is asynchronous: two memset /
 * kernel nodes on the given stream, no synchronisation, no cudaMalloc / cudaFree / allocating library routine.  The
 * address of the scratch array is looked up once per device (cudaGetSymbolAddress, with that device current) on the
 * first call made while that device is current: make that first call outside graph capture.
 *
 * The scratch array is shared by every call on a device and keeps the last call's contents.  The call clears the
 * counter itself; the partial sums need no clearing (every one that is read has been written by the same call).  TWO
 * CALLS THAT OVERLAP ON THE GPU (different streams, or graph branches without a dependency) RACE on the array and
 * give wrong results: order them on one stream or with events.
 */
#ifndef HMF_NOALLOC_B200_H
#define HMF_NOALLOC_B200_H

#ifdef __cplusplus
extern "C" {
#endif

#define HMF_NOALLOC_OK 0
#define HMF_NOALLOC_EINVAL (-1)
#define HMF_NOALLOC_ECUDA (-3)

#define HMF_NOALLOC_MAX_PARTICLES 33554432LL

/* theta_dev, p_dev: device arrays of n doubles (read only); t: copied to out[0]; out_dev: device array of 8 doubles,
 * {t, M_x, M_y, K/N, U/N, E/N, P/N, 0} when the work on `cuda_stream` (a cudaStream_t cast to void*, NULL = legacy
 * default stream) has completed.  All pointers belong to the caller and to the current device.
 * Errors: HMF_NOALLOC_EINVAL (null pointer, n < 1, n > HMF_NOALLOC_MAX_PARTICLES), HMF_NOALLOC_ECUDA (no device, or a
 * CUDA call failed); hmf_noalloc_last_error() has the message. */
int hmf_noalloc_moments(const double* theta_dev, const double* p_dev, long long n, double t, double* out_dev,
                        void* cuda_stream);

const char* hmf_noalloc_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* HMF_NOALLOC_B200_H */
