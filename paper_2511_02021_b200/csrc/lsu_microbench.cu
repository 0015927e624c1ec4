// lsu_microbench.cu -- standalone throughput micro-benchmarks of the L1 / shared-memory data pipe on
// sm_100a (cycles per warp-level instruction per SM). They give the secondary (on-chip) roofline of
// DESIGN.md section 6.1. Not part of libicon_dycore.so.
//   nvcc -O3 -gencode arch=compute_100a,code=sm_100a -o lsu_microbench lsu_microbench.cu && ./lsu_microbench
// 8 independent streams per thread, 2 CTAs x 512 threads per SM, inputs L1/shared resident.
#include <cstdio>
#include <cuda_runtime.h>
#define N 2048
#define U 8
template <int MODE>
__global__ void __launch_bounds__(512, 2) kern(const double* __restrict__ in, double* out, int zero) {
    __shared__ __align__(16) double sm[4096];
    for (int i = threadIdx.x; i < 4096; i += blockDim.x) sm[i] = i;
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double a[U];
#pragma unroll
    for (int u = 0; u < U; ++u) a[u] = u;
    const double* g = in + warp * 2048 + lane;
    const double* gb = in + warp * 2048;
    const double2* g2 = reinterpret_cast<const double2*>(in) + warp * 1024 + lane;
    const double2* s2 = reinterpret_cast<const double2*>(sm);
    int o = zero;
    for (int i = 0; i < N; ++i) {
#pragma unroll
        for (int u = 0; u < U; ++u) {
            if (MODE == 0) a[u] += sm[o + u * 32 + lane];                 // LDS.64 lane
            if (MODE == 1) a[u] += sm[o + u * 8];                         // LDS.64 bcast
            if (MODE == 2) { double2 v = s2[o + u * 32 + lane]; a[u] += v.x + v.y; }   // LDS.128 lane
            if (MODE == 3) { double2 v = s2[o + u * 8]; a[u] += v.x + v.y; }            // LDS.128 bcast
            if (MODE == 4) a[u] += g[o + u * 32];                          // LDG.64 lane, L1 hit, aligned
            if (MODE == 5) a[u] += g[o + u * 32 + 1];                      // LDG.64 lane, misaligned
            if (MODE == 6) { double2 v = g2[o + u * 32]; a[u] += v.x + v.y; }            // LDG.128 lane
            if (MODE == 7) a[u] += gb[o + u * 8];                          // LDG.64 bcast
            if (MODE == 8) a[u] += __shfl_xor_sync(0xffffffffu, a[u], 1);  // SHFL x2
            if (MODE == 9) a[u] = a[u] * 1.0000001 + 0.5;                  // DFMA only
            if (MODE == 10) sm[o + u * 32 + lane + warp * 256] = a[u];     // STS.64 lane
            if (MODE == 11) a[u] += sm[o + u * 32 + lane + 1];             // LDS.64 lane shifted
        }
        o = (o + zero) & 1023;
    }
    double s = 0;
#pragma unroll
    for (int u = 0; u < U; ++u) s += a[u];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s + sm[threadIdx.x];
}
template <int MODE>
void run(const char* name, const double* in, double* out) {
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    kern<MODE><<<296, 512>>>(in, out, 0);
    cudaEventRecord(e0); kern<MODE><<<296, 512>>>(in, out, 0); cudaEventRecord(e1); cudaEventSynchronize(e1);
    float ms; cudaEventElapsedTime(&ms, e0, e1);
    printf("%-22s %9.3f us  %.3f cycles per warp-instr per SM (1.965 GHz)\n", name, ms * 1e3, ms * 1e-3 * 1.965e9 / ((double)N * U * 32));
}
int main() {
    double *in, *out;
    cudaMalloc(&in, 1 << 26); cudaMalloc(&out, 1 << 24);
    cudaMemset(in, 0, 1 << 26);
    run<0>("LDS.64 lane", in, out);
    run<11>("LDS.64 lane shifted", in, out);
    run<1>("LDS.64 bcast", in, out);
    run<2>("LDS.128 lane", in, out);
    run<3>("LDS.128 bcast", in, out);
    run<10>("STS.64 lane", in, out);
    run<4>("LDG.64 lane aligned", in, out);
    run<5>("LDG.64 lane misalign", in, out);
    run<6>("LDG.128 lane", in, out);
    run<7>("LDG.64 bcast", in, out);
    run<8>("SHFL.64 (2x SHFL)", in, out);
    run<9>("DFMA", in, out);
    printf("%s\n", cudaGetErrorString(cudaDeviceSynchronize()));
    return 0;
}
