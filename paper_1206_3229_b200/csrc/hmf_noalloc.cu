// hmf_noalloc.cu -- hmf_noalloc_moments (include/hmf_noalloc.h): the moments of an N-particle HMF state (PAPER.md eqs
// (7)-(8), L56-L63) with the scratch memory of the reduction in a file-scope device array instead of a cudaMalloc'ed
// buffer.  A variant of md_moments_kernel (hmf_md.cu): same sums, the final addition of the block partials on the
// device (last block, fixed order) instead of on the host.  Nothing here allocates.
#include <cuda_runtime.h>
#include <math.h>
#include <stdio.h>

#include "../../include/hmf_noalloc.h"

namespace {

constexpr int NA_NT = 256;                        // threads per block
constexpr int NA_PER_THREAD = 16;                 // particles per thread
constexpr int NA_CHUNK = NA_NT * NA_PER_THREAD;   // particles per block: 4096
constexpr int NA_MAX_BLOCKS = 8192;
constexpr int NA_PART_DOUBLES = NA_MAX_BLOCKS * 4;
constexpr int NA_MAX_DEVICES = 64;
static_assert((long long)NA_MAX_BLOCKS * NA_CHUNK == HMF_NOALLOC_MAX_PARTICLES, "header and kernel disagree");

// [NA_MAX_BLOCKS][4] partial sums (cos, sin, p, p^2/2), then 32 doubles whose first 4 bytes are the counter of finished
// blocks.  In HOST code this name is a stand-in, not a device address: the host passes what cudaGetSymbolAddress
// returns (scratch_of_current_device below).
static __device__ __align__(256) double g_na_scratch[NA_PART_DOUBLES + 32];

// sum over the block in a fixed order: lanes by shuffles, then the warps in index order; result in every thread
__device__ __forceinline__ double2 na_block_sum2(double x, double y, double2* red) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        x += __shfl_down_sync(0xffffffffu, x, o);
        y += __shfl_down_sync(0xffffffffu, y, o);
    }
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    __syncthreads();
    if (lane == 0) red[warp] = make_double2(x, y);
    __syncthreads();
    double2 t = make_double2(0.0, 0.0);
#pragma unroll
    for (int w = 0; w < NA_NT / 32; ++w) {
        t.x += red[w].x;
        t.y += red[w].y;
    }
    return t;
}

// block b: particles [b * 4096, min(n, (b + 1) * 4096)) -> scratch[4 b ..]; the block that finishes last adds the
// partials in index order and writes the eight moments
__global__ void __launch_bounds__(NA_NT) md_moments_noalloc_kernel(const double* __restrict__ theta, const double* __restrict__ p,
                                                                   long long n, double t, double* __restrict__ scratch,
                                                                   double* __restrict__ out) {
    __shared__ double2 red[NA_NT / 32];
    __shared__ bool last;
    double cx = 0.0, sx = 0.0, ps = 0.0, ks = 0.0;
    const long long base = (long long)blockIdx.x * NA_CHUNK + threadIdx.x;
#pragma unroll 4
    for (int k = 0; k < NA_PER_THREAD; ++k) {
        const long long i = base + (long long)k * NA_NT;
        if (i < n) {
            double s, c;
            sincos(theta[i], &s, &c);
            const double pp = p[i];
            cx += c;
            sx += s;
            ps += pp;
            ks = fma(0.5 * pp, pp, ks);
        }
    }
    const double2 a = na_block_sum2(cx, sx, red);
    const double2 b = na_block_sum2(ps, ks, red);
    unsigned* counter = reinterpret_cast<unsigned*>(scratch + NA_PART_DOUBLES);
    if (threadIdx.x == 0) {
        double* mine = scratch + 4 * (size_t)blockIdx.x;
        __stcg(mine + 0, a.x);
        __stcg(mine + 1, a.y);
        __stcg(mine + 2, b.x);
        __stcg(mine + 3, b.y);
        __threadfence();  // the partials are visible before the counter moves
        last = (atomicAdd(counter, 1u) == gridDim.x - 1);
    }
    __syncthreads();
    if (!last) return;
    __threadfence();
    cx = sx = ps = ks = 0.0;
    for (unsigned q = threadIdx.x; q < gridDim.x; q += NA_NT) {
        const double* pq = scratch + 4 * (size_t)q;
        cx += __ldcg(pq + 0);
        sx += __ldcg(pq + 1);
        ps += __ldcg(pq + 2);
        ks += __ldcg(pq + 3);
    }
    const double2 A = na_block_sum2(cx, sx, red);
    const double2 B = na_block_sum2(ps, ks, red);
    if (threadIdx.x == 0) {
        const double inv = 1.0 / (double)n;
        const double mx = A.x * inv, my = A.y * inv, kin = B.y * inv;
        const double pot = 0.5 * (1.0 - mx * mx - my * my);
        out[0] = t;
        out[1] = mx;
        out[2] = my;
        out[3] = kin;
        out[4] = pot;
        out[5] = kin + pot;
        out[6] = B.x * inv;
        out[7] = 0.0;
        *counter = 0u;  // (the host clears it before every launch as well)
    }
}

thread_local char g_na_err[512] = "";

int na_fail(int code, const char* msg) {
    snprintf(g_na_err, sizeof(g_na_err), "%s", msg);
    return code;
}

#define NACU(call)                                                                                                     \
    do {                                                                                                               \
        cudaError_t e_ = (call);                                                                                       \
        if (e_ != cudaSuccess) {                                                                                       \
            snprintf(g_na_err, sizeof(g_na_err), "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_), __FILE__, __LINE__); \
            return HMF_NOALLOC_ECUDA;                                                                                  \
        }                                                                                                              \
    } while (0)

// device address of g_na_scratch on the current device: looked up once per device, with that device current
double* g_na_ptr[NA_MAX_DEVICES] = {};

int scratch_of_current_device(double** out) {
    int dev = -1;
    NACU(cudaGetDevice(&dev));
    if (dev < 0 || dev >= NA_MAX_DEVICES) return na_fail(HMF_NOALLOC_ECUDA, "hmf_noalloc_moments: device ordinal out of range");
    if (g_na_ptr[dev] == nullptr) {
        double* ptr = nullptr;
        NACU(cudaGetSymbolAddress((void**)&ptr, g_na_scratch));
        if (ptr == nullptr) return na_fail(HMF_NOALLOC_ECUDA, "hmf_noalloc_moments: cudaGetSymbolAddress returned null");
        g_na_ptr[dev] = ptr;
    }
    *out = g_na_ptr[dev];
    return HMF_NOALLOC_OK;
}

}  // namespace

extern "C" {

const char* hmf_noalloc_last_error(void) { return g_na_err; }

int hmf_noalloc_moments(const double* theta_dev, const double* p_dev, long long n, double t, double* out_dev,
                        void* cuda_stream) {
    if (!theta_dev || !p_dev || !out_dev) return na_fail(HMF_NOALLOC_EINVAL, "hmf_noalloc_moments: null pointer");
    if (n < 1) return na_fail(HMF_NOALLOC_EINVAL, "hmf_noalloc_moments: n must be >= 1");
    if (n > HMF_NOALLOC_MAX_PARTICLES) {
        snprintf(g_na_err, sizeof(g_na_err),
                 "hmf_noalloc_moments: n = %lld exceeds the maximum of %lld particles that the fixed 256 KiB scratch array "
                 "holds partial sums for (use hmf_md_moments, which allocates)",
                 n, (long long)HMF_NOALLOC_MAX_PARTICLES);
        return HMF_NOALLOC_EINVAL;
    }
    double* scratch = nullptr;
    int rc = scratch_of_current_device(&scratch);
    if (rc != HMF_NOALLOC_OK) return rc;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    const int blocks = (int)((n + NA_CHUNK - 1) / NA_CHUNK);
    // the counter must start at zero whatever an earlier (possibly aborted) call left behind
    NACU(cudaMemsetAsync(scratch + NA_PART_DOUBLES, 0, 256, stream));
    md_moments_noalloc_kernel<<<blocks, NA_NT, 0, stream>>>(theta_dev, p_dev, n, t, scratch, out_dev);
    NACU(cudaGetLastError());
    return HMF_NOALLOC_OK;
}

}  // extern "C"
