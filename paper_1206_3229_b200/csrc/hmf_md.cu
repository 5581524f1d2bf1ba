// hmf_md.cu -- N-particle molecular dynamics of the HMF model on B200 (include/hmf_md.h).
//
// PAPER.md eqs (7)-(8) (L56-L63): the force on a particle needs only M = (1/N) sum (cos theta_j, sin theta_j), so a step
// is O(N) (L65).  Integrator: fourth-order symplectic composition (L206, ref. [44]) in drift-kick-drift form.
// One kernel, md_kick_drift_kernel, is one pass over the particles:
//     [kick]   p_i     += d dt (-M_x sin theta_i + M_y cos theta_i)      with M of the angles as they are read
//     drift    theta_i += c dt p_i
//     sums     (sum cos theta_i, sum sin theta_i) of the NEW angles -> per-block partials for the next pass
// M is not reduced by a kernel of its own: every block of the next pass adds the previous pass's block partials in
// index order (a few thousand doubles from L2), which is the same number in every block and from run to run.
// A step is three such passes (the half drifts that end one step and open the next share a pass): 3 n + 1 launches
// for n steps, 32 bytes per particle and pass (theta and p read and written).  Per particle and pass: one fp64 sincos
// (for the kick) and a rotation of it by the small drift angle (rotate_small) for the sums of the new angles.
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>
#include <stdio.h>

#include <vector>

#include "../../include/hmf_md.h"

namespace {

constexpr int MD_NT = 256;     // threads per block
constexpr int MD_UNROLL = 4;   // particles in flight per thread
constexpr size_t MD_EV_CAP = 4096;

struct MdArgs {
    double* theta;
    double* p;
    long long n;
    const double* part_in;  // [nblk_in][2] sums of cos, sin of the state as it is read (kick != 0 only)
    int nblk_in;
    double* part_out;       // [gridDim.x][2]
    double kick;            // d dt, 0: no kick in this pass
    double drift;           // c dt
    double inv_n;
};

// sum over the block in a fixed order: lanes by shuffles, then the warps in index order; result in every thread
__device__ __forceinline__ double2 block_sum2(double x, double y, double2* red) {
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
    for (int w = 0; w < MD_NT / 32; ++w) {
        t.x += red[w].x;
        t.y += red[w].y;
    }
    return t;
}

// (cos, sin) of theta + d from (c, s) = (cos, sin) of theta by a rotation, with sin d and cos d from their Taylor
// polynomials (|d| <= 1/2: remainders d^17/17! = 2e-20 and d^18/18! = 6e-22): a third of the instructions of a second
// sincos.  The result only enters the sums (M_x, M_y) of this pass -- the angles themselves are advanced by the plain
// addition -- so its rounding (a few 1e-16) does not accumulate over the steps.
__device__ __forceinline__ void rotate_small(double c, double s, double d, double* c2, double* s2) {
    const double z = d * d;
    double ps = -1.0 / 1307674368000.0;           // -1/15!
    ps = fma(ps, z, 1.0 / 6227020800.0);          //  1/13!
    ps = fma(ps, z, -1.0 / 39916800.0);           // -1/11!
    ps = fma(ps, z, 1.0 / 362880.0);              //  1/9!
    ps = fma(ps, z, -1.0 / 5040.0);               // -1/7!
    ps = fma(ps, z, 1.0 / 120.0);                 //  1/5!
    ps = fma(ps, z, -1.0 / 6.0);                  // -1/3!
    const double sd = fma(ps * z, d, d);          // d + d^3 (...)
    double pc = 1.0 / 20922789888000.0;           //  1/16!
    pc = fma(pc, z, -1.0 / 87178291200.0);        // -1/14!
    pc = fma(pc, z, 1.0 / 479001600.0);           //  1/12!
    pc = fma(pc, z, -1.0 / 3628800.0);            // -1/10!
    pc = fma(pc, z, 1.0 / 40320.0);               //  1/8!
    pc = fma(pc, z, -1.0 / 720.0);                // -1/6!
    pc = fma(pc, z, 1.0 / 24.0);                  //  1/4!
    pc = fma(pc, z, -0.5);                        // -1/2!
    const double cdm1 = pc * z;                   // cos d - 1
    *c2 = fma(c, cdm1, c) - s * sd;               // c cos d - s sin d
    *s2 = fma(s, cdm1, s) + c * sd;               // s cos d + c sin d
}

__global__ void __launch_bounds__(MD_NT) md_kick_drift_kernel(const MdArgs a) {
    __shared__ double2 red[MD_NT / 32];
    double mx = 0.0, my = 0.0;
    const bool kick = a.kick != 0.0;
    if (kick) {  // eq (8): M of the state this pass reads = sum of the previous pass's block partials, in index order
        double sx = 0.0, sy = 0.0;
        for (int b = threadIdx.x; b < a.nblk_in; b += MD_NT) {
            sx += __ldcg(a.part_in + 2 * b);
            sy += __ldcg(a.part_in + 2 * b + 1);
        }
        const double2 m = block_sum2(sx, sy, red);
        mx = m.x * a.inv_n * a.kick;  // d dt M_x
        my = m.y * a.inv_n * a.kick;
    }
    double accx = 0.0, accy = 0.0;
    const long long stride = (long long)gridDim.x * MD_NT;
    long long i = (long long)blockIdx.x * MD_NT + threadIdx.x;
    for (; i + (MD_UNROLL - 1) * stride < a.n; i += MD_UNROLL * stride) {
        double th[MD_UNROLL], pp[MD_UNROLL];
#pragma unroll
        for (int u = 0; u < MD_UNROLL; ++u) {
            th[u] = __ldcs(a.theta + i + u * stride);
            pp[u] = __ldcs(a.p + i + u * stride);
        }
#pragma unroll
        for (int u = 0; u < MD_UNROLL; ++u) {
            double s2, c2;
            if (kick) {  // eq (7): F = -sin(theta) M_x + cos(theta) M_y
                double s, c;
                sincos(th[u], &s, &c);
                pp[u] += -s * mx + c * my;
                __stcs(a.p + i + u * stride, pp[u]);
                const double d = a.drift * pp[u];
                th[u] += d;
                if (fabs(d) <= 0.5) rotate_small(c, s, d, &c2, &s2);
                else sincos(th[u], &s2, &c2);
            } else {
                th[u] += a.drift * pp[u];
                sincos(th[u], &s2, &c2);
            }
            accx += c2;
            accy += s2;
            __stcs(a.theta + i + u * stride, th[u]);
        }
    }
    for (; i < a.n; i += stride) {
        double th = __ldcs(a.theta + i), pp = __ldcs(a.p + i);
        double s2, c2;
        if (kick) {
            double s, c;
            sincos(th, &s, &c);
            pp += -s * mx + c * my;
            __stcs(a.p + i, pp);
            const double d = a.drift * pp;
            th += d;
            if (fabs(d) <= 0.5) rotate_small(c, s, d, &c2, &s2);
            else sincos(th, &s2, &c2);
        } else {
            th += a.drift * pp;
            sincos(th, &s2, &c2);
        }
        accx += c2;
        accy += s2;
        __stcs(a.theta + i, th);
    }
    const double2 t = block_sum2(accx, accy, red);
    if (threadIdx.x == 0) {
        a.part_out[2 * blockIdx.x] = t.x;
        a.part_out[2 * blockIdx.x + 1] = t.y;
    }
}

// read-only pass for hmf_md_moments: per-block sums of cos theta, sin theta, p, p^2/2
__global__ void __launch_bounds__(MD_NT) md_moments_kernel(const double* __restrict__ theta, const double* __restrict__ p,
                                                           long long n, double* __restrict__ part /* [blocks][4] */) {
    __shared__ double2 red[MD_NT / 32];
    double cx = 0.0, sx = 0.0, ps = 0.0, ks = 0.0;
    for (long long i = (long long)blockIdx.x * MD_NT + threadIdx.x; i < n; i += (long long)gridDim.x * MD_NT) {
        double s, c;
        sincos(theta[i], &s, &c);
        const double pp = p[i];
        cx += c;
        sx += s;
        ps += pp;
        ks = fma(0.5 * pp, pp, ks);
    }
    const double2 a = block_sum2(cx, sx, red);
    const double2 b = block_sum2(ps, ks, red);
    if (threadIdx.x == 0) {
        part[4 * blockIdx.x + 0] = a.x;
        part[4 * blockIdx.x + 1] = a.y;
        part[4 * blockIdx.x + 2] = b.x;
        part[4 * blockIdx.x + 3] = b.y;
    }
}

thread_local char g_err[512] = "";

struct Md {
    bool ready = false, cuda_failed = false, own = false, profile = false;
    long long n = 0;
    double dt = 0, t = 0;
    double *theta = nullptr, *p = nullptr;
    double* part[2] = {nullptr, nullptr};  // ping-pong block partials of (cos, sin)
    double* mpart = nullptr;               // partials of the moments pass
    int cur = 0;                           // part[cur] holds the sums of the current angles (valid after a pass)
    bool part_valid = false;
    int nblk = 0;
    cudaStream_t stream = nullptr;
    unsigned long long launches = 0;
    std::vector<cudaEvent_t> ev[2];
    size_t ev_used = 0;
};
Md M;

int fail(int code, const char* msg) {
    snprintf(g_err, sizeof(g_err), "%s", msg);
    return code;
}

#define MCU(call)                                                                                              \
    do {                                                                                                       \
        cudaError_t e_ = (call);                                                                               \
        if (e_ != cudaSuccess) {                                                                               \
            M.cuda_failed = true;                                                                              \
            snprintf(g_err, sizeof(g_err), "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_), __FILE__, __LINE__); \
            return HMF_MD_ECUDA;                                                                               \
        }                                                                                                      \
    } while (0)

int check_ready() {
    if (!M.ready) return fail(HMF_MD_ENOTINIT, "hmf_md_init has not been called");
    if (M.cuda_failed) return HMF_MD_ECUDA;
    return HMF_MD_OK;
}

int ensure_state() {
    if (M.theta != nullptr) return HMF_MD_OK;
    MCU(cudaMalloc(&M.theta, sizeof(double) * (size_t)M.n));
    MCU(cudaMalloc(&M.p, sizeof(double) * (size_t)M.n));
    M.own = true;
    MCU(cudaMemsetAsync(M.theta, 0, sizeof(double) * (size_t)M.n, M.stream));
    MCU(cudaMemsetAsync(M.p, 0, sizeof(double) * (size_t)M.n, M.stream));
    return HMF_MD_OK;
}

// one pass: [kick d] then drift c, sums of the new angles
int pass(double d, double c) {
    if (d != 0.0 && !M.part_valid) return fail(HMF_MD_EINVAL, "internal: kick without the sums of the current angles");
    MdArgs a;
    a.theta = M.theta;
    a.p = M.p;
    a.n = M.n;
    a.part_in = M.part[M.cur];
    a.nblk_in = M.nblk;
    a.part_out = M.part[M.cur ^ 1];
    a.kick = d * M.dt;
    a.drift = c * M.dt;
    a.inv_n = 1.0 / (double)M.n;
    const bool prof = M.profile && M.ev_used < MD_EV_CAP;
    if (prof) {
        if (M.ev[0].size() <= M.ev_used) {
            cudaEvent_t e0, e1;
            MCU(cudaEventCreate(&e0));
            MCU(cudaEventCreate(&e1));
            M.ev[0].push_back(e0);
            M.ev[1].push_back(e1);
        }
        MCU(cudaEventRecord(M.ev[0][M.ev_used], M.stream));
    }
    md_kick_drift_kernel<<<M.nblk, MD_NT, 0, M.stream>>>(a);
    if (prof) {
        MCU(cudaEventRecord(M.ev[1][M.ev_used], M.stream));
        M.ev_used++;
    }
    M.launches++;
    MCU(cudaGetLastError());
    M.cur ^= 1;
    M.part_valid = true;
    return HMF_MD_OK;
}

}  // namespace

extern "C" {

const char* hmf_md_last_error(void) { return g_err; }

void hmf_md_free(void) {
    if (M.ready) cudaStreamSynchronize(M.stream);
    for (int k = 0; k < 2; ++k) {
        for (cudaEvent_t e : M.ev[k]) cudaEventDestroy(e);
        if (M.part[k]) cudaFree(M.part[k]);
    }
    if (M.mpart) cudaFree(M.mpart);
    if (M.own) {
        if (M.theta) cudaFree(M.theta);
        if (M.p) cudaFree(M.p);
    }
    M = Md();
}

int hmf_md_init(long long n, double dt) {
    if (n < 1 || !isfinite(dt)) return fail(HMF_MD_EINVAL, "hmf_md_init: n must be >= 1 and dt finite");
    hmf_md_free();
    int count = 0, dev = 0, sms = 148;
    if (cudaGetDeviceCount(&count) != cudaSuccess || count < 1) {
        cudaGetLastError();
        return fail(HMF_MD_ECUDA, "hmf_md_init: no CUDA device (there is no CPU fallback)");
    }
    MCU(cudaGetDevice(&dev));
    MCU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    M.n = n;
    M.dt = dt;
    // one resident wave: 8 blocks of 256 threads per SM; fewer blocks for few particles
    long long want = (n + (long long)MD_NT * MD_UNROLL - 1) / ((long long)MD_NT * MD_UNROLL);
    const long long cap = (long long)sms * 8;
    M.nblk = (int)(want < 1 ? 1 : (want > cap ? cap : want));
    for (int k = 0; k < 2; ++k) MCU(cudaMalloc(&M.part[k], sizeof(double) * 2 * (size_t)M.nblk));
    MCU(cudaMalloc(&M.mpart, sizeof(double) * 4 * (size_t)M.nblk));
    M.ready = true;
    g_err[0] = 0;
    return HMF_MD_OK;
}

int hmf_md_attach(void* theta_dev, void* p_dev, void* cuda_stream) {
    int rc = check_ready();
    if (rc != 0) return rc;
    if (!theta_dev || !p_dev) return fail(HMF_MD_EINVAL, "hmf_md_attach: null buffer");
    if (((uintptr_t)theta_dev & 15) || ((uintptr_t)p_dev & 15)) return fail(HMF_MD_EINVAL, "hmf_md_attach: buffers must be 16-byte aligned");
    if (M.own) {
        cudaFree(M.theta);
        cudaFree(M.p);
        M.own = false;
    }
    M.theta = static_cast<double*>(theta_dev);
    M.p = static_cast<double*>(p_dev);
    M.stream = static_cast<cudaStream_t>(cuda_stream);
    M.part_valid = false;
    return HMF_MD_OK;
}

int hmf_md_upload(const double* theta_host, const double* p_host) {
    int rc = check_ready();
    if (rc != 0) return rc;
    if (!theta_host || !p_host) return fail(HMF_MD_EINVAL, "hmf_md_upload: null");
    if ((rc = ensure_state()) != 0) return rc;
    MCU(cudaMemcpyAsync(M.theta, theta_host, sizeof(double) * (size_t)M.n, cudaMemcpyHostToDevice, M.stream));
    MCU(cudaMemcpyAsync(M.p, p_host, sizeof(double) * (size_t)M.n, cudaMemcpyHostToDevice, M.stream));
    M.t = 0.0;
    M.part_valid = false;
    return HMF_MD_OK;
}

int hmf_md_download(double* theta_host, double* p_host) {
    int rc = check_ready();
    if (rc != 0) return rc;
    if (!theta_host || !p_host) return fail(HMF_MD_EINVAL, "hmf_md_download: null");
    if ((rc = ensure_state()) != 0) return rc;
    MCU(cudaMemcpyAsync(theta_host, M.theta, sizeof(double) * (size_t)M.n, cudaMemcpyDeviceToHost, M.stream));
    MCU(cudaMemcpyAsync(p_host, M.p, sizeof(double) * (size_t)M.n, cudaMemcpyDeviceToHost, M.stream));
    MCU(cudaStreamSynchronize(M.stream));
    return HMF_MD_OK;
}

int hmf_md_step(int nsteps) {
    int rc = check_ready();
    if (rc != 0) return rc;
    if (nsteps <= 0) return fail(HMF_MD_EINVAL, "hmf_md_step: nsteps must be >= 1");
    if ((rc = ensure_state()) != 0) return rc;
    const double g1 = 1.0 / (2.0 - cbrt(2.0)), g2 = 1.0 - 2.0 * g1;
    if ((rc = pass(0.0, 0.5 * g1)) != 0) return rc;                       // drift(g1/2)
    for (int k = 0; k < nsteps; ++k) {
        if ((rc = pass(g1, 0.5 * (g1 + g2))) != 0) return rc;              // kick(g1) drift((g1+g2)/2)
        if ((rc = pass(g2, 0.5 * (g1 + g2))) != 0) return rc;              // kick(g2) drift((g1+g2)/2)
        // kick(g1), then the closing half drift of this step together with the opening one of the next
        if ((rc = pass(g1, k + 1 < nsteps ? g1 : 0.5 * g1)) != 0) return rc;
    }
    M.t += (double)nsteps * M.dt;
    return HMF_MD_OK;
}

int hmf_md_moments(double out[8]) {
    int rc = check_ready();
    if (rc != 0) return rc;
    if (!out) return fail(HMF_MD_EINVAL, "hmf_md_moments: null");
    if ((rc = ensure_state()) != 0) return rc;
    md_moments_kernel<<<M.nblk, MD_NT, 0, M.stream>>>(M.theta, M.p, M.n, M.mpart);
    M.launches++;
    MCU(cudaGetLastError());
    std::vector<double> h(4 * (size_t)M.nblk);
    MCU(cudaMemcpyAsync(h.data(), M.mpart, sizeof(double) * h.size(), cudaMemcpyDeviceToHost, M.stream));
    MCU(cudaStreamSynchronize(M.stream));
    double s[4] = {0, 0, 0, 0};
    for (int b = 0; b < M.nblk; ++b)
        for (int q = 0; q < 4; ++q) s[q] += h[4 * (size_t)b + q];
    const double inv = 1.0 / (double)M.n;
    out[0] = M.t;
    out[1] = s[0] * inv;
    out[2] = s[1] * inv;
    out[3] = s[3] * inv;
    out[4] = 0.5 * (1.0 - out[1] * out[1] - out[2] * out[2]);
    out[5] = out[3] + out[4];
    out[6] = s[2] * inv;
    out[7] = 0.0;
    return HMF_MD_OK;
}

int hmf_md_profile(int on) {
    int rc = check_ready();
    if (rc != 0) return rc;
    M.profile = on != 0;
    return HMF_MD_OK;
}

int hmf_md_kernel_times(double out[2]) {
    int rc = check_ready();
    if (rc != 0) return rc;
    if (!out) return fail(HMF_MD_EINVAL, "hmf_md_kernel_times: null");
    MCU(cudaStreamSynchronize(M.stream));
    double total = 0.0;
    for (size_t k = 0; k < M.ev_used; ++k) {
        float ms = 0.f;
        MCU(cudaEventElapsedTime(&ms, M.ev[0][k], M.ev[1][k]));
        total += (double)ms;
    }
    out[0] = total;
    out[1] = (double)M.ev_used;
    M.ev_used = 0;
    return HMF_MD_OK;
}

int hmf_md_launch_count(unsigned long long* out) {
    if (!out) return fail(HMF_MD_EINVAL, "hmf_md_launch_count: null");
    *out = M.launches;
    return HMF_MD_OK;
}

}  // extern "C"
