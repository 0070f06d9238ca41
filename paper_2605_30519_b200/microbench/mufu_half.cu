// MUFU packed-half ex2 throughput on sm_100a
#include <cstdio>
#include <cstdint>
#include <cuda_runtime.h>
constexpr int REP = 16;
template <int MODE>
__global__ void k(uint32_t* out, long long* clk, uint32_t seed)
{
    uint32_t s[64];
#pragma unroll
    for (int i = 0; i < 64; ++i) s[i] = seed * (i + threadIdx.x);
    __syncthreads();
    long long t0 = clock64();
#pragma unroll 1
    for (int r = 0; r < REP; ++r) {
#pragma unroll
        for (int i = 0; i < 64; ++i) {
            if (MODE == 0) asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+r"(s[i]));
            if (MODE == 1) asm volatile("ex2.approx.f16x2 %0, %0;" : "+r"(s[i]));
            if (MODE == 2) asm volatile("ex2.approx.ftz.bf16x2 %0, %0;" : "+r"(s[i]));
            if (MODE == 3) asm volatile("{.reg .b16 lo, hi; mov.b32 {lo, hi}, %0; ex2.approx.f16 lo, lo; mov.b32 %0, {lo, hi};}" : "+r"(s[i]));
        }
    }
    long long t1 = clock64();
    uint32_t o = 0;
#pragma unroll
    for (int i = 0; i < 64; ++i) o ^= s[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = o;
    if (threadIdx.x == 0 && blockIdx.x == 0) *clk = (t1 - t0) / REP;
}
template <int MODE> void run(const char* name)
{
    uint32_t* out; long long* clk;
    cudaMalloc(&out, 148 * 256 * 4); cudaMalloc(&clk, 8);
    for (int warps : {4, 8}) {
        k<MODE><<<148, warps * 32>>>(out, clk, 3);
        k<MODE><<<148, warps * 32>>>(out, clk, 3);
        long long h; cudaMemcpy(&h, clk, 8, cudaMemcpyDeviceToHost);
        printf("%-28s warps/SMSP %d: %6lld clk per 64 instr, %.2f clk per warp-instr\n", name, warps / 4, h, (double)h / 64);
    }
    cudaFree(out); cudaFree(clk);
}
int main()
{
    run<0>("ex2.approx.ftz.f32");
    run<1>("ex2.approx.f16x2");
    run<2>("ex2.approx.ftz.bf16x2");
    run<3>("ex2.approx.f16 (scalar)");
    return 0;
}
