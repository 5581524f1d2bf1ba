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
    return 0;
}
