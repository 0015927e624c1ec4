// bulk_copy_microbench.cu -- stand-alone micro-benchmark (not part of libicon_dycore): request rate and
// throughput of cp.async.bulk (1-D TMA) global -> shared for small copies; 148 CTAs whose warps only issue
// copies into a 4-stage shared-memory ring, each stage completing on an mbarrier. Results and the command
// are in profiles/r01_bulk_copy_microbench.md; they are why kernels_cc.cu has four producer warps and merges
// columns with consecutive ids into one copy.
//   nvcc -O3 -gencode arch=compute_100a,code=sm_100a -o bulk_copy_microbench bulk_copy_microbench.cu
//   ./bulk_copy_microbench [source MiB, default 6144; <= 96 keeps the source in L2]
#include <cstdio>
#include <cstdlib>
#include <cstdint>
#include <cuda_runtime.h>
__device__ __forceinline__ uint32_t s32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mwait(uint32_t bar, uint32_t parity) {
    asm volatile("{\n.reg .pred p;\nW_%=:\nmbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n@p bra D_%=;\nbra W_%=;\nD_%=:\n}\n" ::"r"(bar), "r"(parity) : "memory");
}
// each of NW warps: loop over stages; stage = NPS copies of `bytes`; ring of R stages per warp; wait on stage before reuse
template <int R>
__global__ void k(const unsigned char* src, size_t src_bytes, int bytes, int nps, int iters, int stride_mode, unsigned long long* sink) {
    extern __shared__ __align__(128) unsigned char smem[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nw = blockDim.x >> 5;
    uint64_t* bars = (uint64_t*)smem;            // [nw][R]
    unsigned char* buf = smem + 1024;
    const int stage_bytes = ((bytes + 15) & ~15) * nps;
    if (threadIdx.x == 0) for (int i = 0; i < nw * R; ++i) asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(s32(bars + i)));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    __syncthreads();
    unsigned char* mybuf = buf + (size_t)warp * R * stage_bytes;
    const size_t ncols = src_bytes / 768;
    uint64_t rng = 1234567ull * (blockIdx.x * 64 + warp + 1);
    for (int it = 0; it < iters; ++it) {
        const int st = it % R;
        const uint32_t bar = s32(bars + warp * R + st);
        if (it >= R) mwait(bar, ((it / R) - 1) & 1);
        if (lane == 0) asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes * nps) : "memory");
        __syncwarp();
        for (int i = lane; i < nps; i += 32) {
            size_t col;
            if (stride_mode == 0) col = ((size_t)(blockIdx.x * nw + warp) * iters + it) * nps + i;   // sequential columns
            else { uint64_t z = rng + 0x9E3779B97F4A7C15ull * (it * 64 + i + 1); z ^= z >> 30; z *= 0xBF58476D1CE4E5B9ull; z ^= z >> 27; col = z; }
            col %= ncols;
            asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(s32(mybuf + st * stage_bytes + i * ((bytes + 15) & ~15))),
                         "l"(src + col * 768), "r"(bytes), "r"(bar) : "memory");
        }
    }
    for (int it = iters; it < iters + R && it >= R; ++it) mwait(s32(bars + warp * R + it % R), ((it / R) - 1) & 1);
    if (threadIdx.x == 0) sink[blockIdx.x] = buf[0];
}
int main(int argc, char** argv) {
    size_t src_bytes = (size_t)(argc > 1 ? atol(argv[1]) : 6144) << 20;
    unsigned char* src; cudaMalloc(&src, src_bytes); cudaMemset(src, 1, src_bytes);
    unsigned long long* sink; cudaMalloc(&sink, 148 * 8);
    cudaFuncSetAttribute(k<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    cudaEvent_t a, b; cudaEventCreate(&a); cudaEventCreate(&b);
    printf("bytes nps warps mode  GB/s  ns/copy/SM\n");
    for (int mode = 0; mode < 2; ++mode)
    for (int bytes : {720, 1440})
    for (int nw : {1, 4, 8, 16})
    for (int nps : {4, 8, 32}) {
        int stage = ((bytes + 15) & ~15) * nps;
        if ((size_t)stage * 4 * nw + 1024 > 200 * 1024) continue;
        int iters = (int)(((size_t)3 << 30) / 148 / nw / ((size_t)bytes * nps));
        if (iters < 8) continue;
        for (int rep = 0; rep < 2; ++rep) {
            cudaEventRecord(a);
            k<4><<<148, nw * 32, 1024 + (size_t)stage * 4 * nw>>>(src, src_bytes, bytes, nps, iters, mode, sink);
            cudaEventRecord(b); cudaEventSynchronize(b);
            float ms; cudaEventElapsedTime(&ms, a, b);
            double tot = (double)148 * nw * iters * nps * bytes;
            if (rep) printf("%5d %3d %2d %d  %7.1f  %7.1f   (%s)\n", bytes, nps, nw, mode, tot / ms / 1e6, ms * 1e6 / ((double)nw * iters * nps), cudaGetErrorString(cudaGetLastError()));
        }
    }
    return 0;
}
