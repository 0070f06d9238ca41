// L2 -> SMEM bulk-copy bandwidth per SM with several 32 KB copies in flight on every SM (data L2-resident).
#include <cstdio>
#include <cstdint>
#include <cuda_runtime.h>
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ bool try_wait(uint32_t bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}" : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok != 0;
}
__global__ void __launch_bounds__(128, 1) k(const unsigned char* src, size_t span, int iters, int nst, int chunk, long long* out)
{
    extern __shared__ unsigned char raw[];
    unsigned char* sm = (unsigned char*)(((uintptr_t)raw + 1023) & ~(uintptr_t)1023);
    unsigned long long* bars = (unsigned long long*)(sm + 6 * 32768);
    if (threadIdx.x == 0) {
        for (int i = 0; i < nst; ++i) asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_u32(bars + i)));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        long long t0 = clock64();
        size_t off = ((size_t)blockIdx.x * 7919 * 32768) % span;
        for (int i = 0; i < iters + nst; ++i) {
            const int s = i % nst;
            if (i >= nst) { while (!try_wait(smem_u32(bars + s), ((i / nst) - 1) & 1)) {} }
            if (i < iters) {
                asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bars + s)), "r"(32768) : "memory");
                for (int c = 0; c < 32768 / chunk; ++c)
                    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                                 ::"r"(smem_u32(sm + s * 32768 + c * chunk)), "l"(src + off + c * chunk), "r"(chunk), "r"(smem_u32(bars + s)) : "memory");
                off = (off + 32768 * 151) % span;
            }
        }
        long long t1 = clock64();
        out[blockIdx.x] = t1 - t0;
    }
}
int main()
{
    unsigned char* src; long long* out;
    const size_t span = 48u << 20;  // L2-resident
    cudaMalloc(&src, span + (1 << 20)); cudaMemset(src, 1, span + (1 << 20)); cudaMalloc(&out, 148 * 8);
    const int smem = 6 * 32768 + 2048;
    cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    for (int grid : {8, 148})
    for (int chunk : {32768, 16384, 8192, 4096})
    for (int nst : {4}) {
        const int iters = 400;
        k<<<grid, 128, smem>>>(src, span, iters, nst, chunk, out);
        cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
        cudaEventRecord(e0);
        k<<<grid, 128, smem>>>(src, span, iters, nst, chunk, out);
        cudaEventRecord(e1); cudaEventSynchronize(e1);
        float ms; cudaEventElapsedTime(&ms, e0, e1);
        long long h[148]; cudaMemcpy(h, out, 148 * 8, cudaMemcpyDeviceToHost);
        double mean = 0; for (int i = 0; i < grid; ++i) mean += h[i]; mean /= grid;
        printf("grid %3d chunk %5d stages %d: %.1f B/clk/SM (mean %0.f clk), chip %.2f TB/s by events\n", grid, chunk, nst, 32768.0 * iters / mean, mean, (double)grid * 32768 * iters / (ms * 1e-3) / 1e12);
    }
    return 0;
}
