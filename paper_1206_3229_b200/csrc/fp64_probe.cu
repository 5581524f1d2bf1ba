// fp64_probe.cu -- stand-alone micro-benchmark of the fp64 FMA pipe (not part of the library): DFMA throughput per SM
// as a function of resident warps per scheduler and independent chains per thread, and the same with one shared-memory
// load + store per ten FMAs (the instruction mix of the p stage).  MEASURED_PEAKS.json has no fp64 entry; DESIGN.md
// section 7 quotes the result (profiles/fp64_probe.txt).
//     nvcc -O3 -gencode arch=compute_100a,code=sm_100a -o fp64_probe fp64_probe.cu && ./fp64_probe
#include <cstdio>
#include <cuda_runtime.h>
template <int ILP>
__global__ void dfma_kernel(double* out, int iters, double a, double b) {
    double x[ILP];
#pragma unroll
    for (int k = 0; k < ILP; ++k) x[k] = threadIdx.x + k;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 4; ++u)
#pragma unroll
            for (int k = 0; k < ILP; ++k) x[k] = fma(x[k], a, b);
    }
    double s = 0;
#pragma unroll
    for (int k = 0; k < ILP; ++k) s += x[k];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}
// mixed: DFMA stream with interleaved LDS/STS like the p stage: per 10 DFMA one LDS.64 and one STS.64
template <int ILP>
__global__ void mixed_kernel(double* out, int iters, double a, double b) {
    __shared__ double sm[1024 * 4];
    double x[ILP];
#pragma unroll
    for (int k = 0; k < ILP; ++k) x[k] = threadIdx.x + k;
    double* p = sm + threadIdx.x;
    p[0] = 1.0; p[1024] = 2.0; p[2048] = 0.5; p[3072] = 0.25;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int k = 0; k < ILP; ++k) {
            double t = p[(k & 3) * 1024];
#pragma unroll
            for (int u = 0; u < 10; ++u) x[k] = fma(x[k], a, t);
            p[(k & 3) * 1024] = x[k] * 1e-30;
        }
    }
    double s = 0;
#pragma unroll
    for (int k = 0; k < ILP; ++k) s += x[k];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}
// fir: the operand pattern of the real kernels, acc[r] = fma(w_n, x[n + r], acc[r]): per DFMA two distinct 64-bit
// register operands (x, acc) and one shared with its neighbours (w); registers only (LDS = 0), or with the window
// value and the weight of every tap loaded from shared memory (LDS = 1) as in gs_p_sweep_kernel / the theta stages.
template <int R, int LDS>
__global__ void fir_kernel(double* out, int iters, const double* src) {
    __shared__ double sm[32 * 128];
    for (int k = threadIdx.x; k < 32 * 128; k += blockDim.x) sm[k] = src[k & 1023];
    __syncthreads();
    const double* p = sm + (threadIdx.x & 127);
    double acc[R], x[R], w[4];
#pragma unroll
    for (int k = 0; k < R; ++k) { acc[k] = 0.0; x[k] = src[threadIdx.x + k]; }
#pragma unroll
    for (int k = 0; k < 4; ++k) w[k] = src[k + 7];
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int n = 0; n < 60; ++n) {
            double wn = w[n & 3];
            if (LDS) {
                x[(n + R - 1) % R] = p[((n + i) & 31) * 128];
                wn = p[((n + 2 * i + 1) & 31) * 128];
            }
#pragma unroll
            for (int r = 0; r < R; ++r) acc[r] = fma(wn, x[(n + r) % R], acc[r]);
        }
    }
    double s = 0;
#pragma unroll
    for (int k = 0; k < R; ++k) s += acc[k];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}
template <int R, int LDS>
void run_fir(double* d, const double* src, int wps) {
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    int threads = 32 * 4 * wps, iters = 400;
    float best = 1e9;
    for (int rep = 0; rep < 3; ++rep) {
        cudaEventRecord(e0);
        fir_kernel<R, LDS><<<148, threads>>>(d, iters, src);
        cudaEventRecord(e1); cudaEventSynchronize(e1);
        float ms; cudaEventElapsedTime(&ms, e0, e1); if (ms < best) best = ms;
    }
    double fmas = 148.0 * threads * R * 60.0 * iters;
    printf("fir%s warps/SMSP=%d R=%d: %.1f FMA/ns/SM = %.2f clk per warp-DFMA per SMSP (at 1.965 GHz)\n", LDS ? "+lds" : "", wps, R,
           fmas / best / 1e6 / 148, 1.965 * 32 * 4 / (fmas / best / 1e6 / 148));
}
template <int ILP>
void run(double* d, int wps, const char* name, bool mixed) {
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    int threads = 32 * 4 * wps, iters = mixed ? 2000 : 20000;
    float best = 1e9;
    for (int rep = 0; rep < 3; ++rep) {
        cudaEventRecord(e0);
        if (mixed) mixed_kernel<ILP><<<148, threads>>>(d, iters, 1.0000001, 1e-9);
        else dfma_kernel<ILP><<<148, threads>>>(d, iters, 1.0000001, 1e-9);
        cudaEventRecord(e1); cudaEventSynchronize(e1);
        float ms; cudaEventElapsedTime(&ms, e0, e1); if (ms < best) best = ms;
    }
    double fmas = 148.0 * threads * ILP * (mixed ? 10.0 : 4.0) * iters;
    printf("%s warps/SMSP=%d ILP=%d: %.1f FMA/ns/SM = %.2f clk per warp-DFMA per SMSP (at 1.965 GHz)\n", name, wps, ILP,
           fmas / best / 1e6 / 148, 1.965 * 32 * 4 / (fmas / best / 1e6 / 148));
}
int main() {
    double* d; cudaMalloc(&d, 148 * 1024 * 8);
    for (int wps = 1; wps <= 4; ++wps) {
        run<1>(d, wps, "dfma", false); run<2>(d, wps, "dfma", false); run<4>(d, wps, "dfma", false);
        run<8>(d, wps, "dfma", false); run<12>(d, wps, "dfma", false);
    }
    for (int wps = 1; wps <= 4; ++wps) { run<4>(d, wps, "mixed", true); run<12>(d, wps, "mixed", true); }
    double* src; cudaMalloc(&src, 2048 * 8);
    {
        double h[2048];
        for (int k = 0; k < 2048; ++k) h[k] = 1e-3 * (k % 17) - 8e-3;
        cudaMemcpy(src, h, sizeof(h), cudaMemcpyHostToDevice);
    }
    for (int wps = 1; wps <= 4; ++wps) {
        run_fir<8, 0>(d, src, wps); run_fir<9, 0>(d, src, wps); run_fir<16, 0>(d, src, wps);
        run_fir<8, 1>(d, src, wps); run_fir<9, 1>(d, src, wps); run_fir<16, 1>(d, src, wps);
    }
    return 0;
}
