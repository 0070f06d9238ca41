// Micro-benchmarks of the softmax instruction mix on sm_100a: clocks per warp-instruction with 1 or 2 warps per SMSP.
#include <cstdio>
#include <cstdint>
#include <cuda_runtime.h>

__device__ __forceinline__ float ex2(float x) { float y; asm volatile("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ uint64_t f2(float lo, float hi) { uint64_t r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ void unf2(uint64_t v, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ uint64_t fma2(uint64_t a, uint64_t b, uint64_t c) { uint64_t r; asm volatile("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }
__device__ __forceinline__ uint64_t add2(uint64_t a, uint64_t b) { uint64_t r; asm volatile("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ uint32_t pack2(float lo, float hi) { uint32_t r; asm volatile("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo)); return r; }

constexpr int REP = 16;

// mode 0: MUFU only (128 per rep); 1: full mix (fma2, 2 ex2, add2, pack) x 64 pairs; 2: fmnmx 128 (4 chains); 3: fmnmx3 ; 4: ffma2 only 64; 5: fadd2 only 64; 6: pack only 64
// 7: ffma (scalar) 128 ; 8: mix without ex2
template <int MODE>
__global__ void k(float* out, long long* clk, float seed)
{
    float s[128];
#pragma unroll
    for (int i = 0; i < 128; ++i) s[i] = seed * (float)(i + threadIdx.x) * 1e-3f;
    float acc = 0.f;
    uint64_t rs[4] = {0, 0, 0, 0};
    uint32_t pk = 0;
    __syncthreads();
    long long t0 = clock64();
#pragma unroll 1
    for (int r = 0; r < REP; ++r) {
        if (MODE == 0) {
#pragma unroll
            for (int i = 0; i < 128; ++i) s[i] = ex2(s[i]);
        } else if (MODE == 1 || MODE == 8) {
            const uint64_t sl2 = f2(seed, seed), nm2 = f2(-seed, -seed);
#pragma unroll
            for (int c = 0; c < 64; ++c) {
                const uint64_t x = fma2(f2(s[2 * c], s[2 * c + 1]), sl2, nm2);
                float x0, x1;
                unf2(x, x0, x1);
                float p0 = MODE == 1 ? ex2(x0) : x0, p1 = MODE == 1 ? ex2(x1) : x1;
                rs[c & 3] = add2(rs[c & 3], f2(p0, p1));
                pk ^= pack2(p0, p1);
            }
        } else if (MODE == 2) {
            float m0 = s[0], m1 = s[1], m2 = s[2], m3 = s[3];
#pragma unroll
            for (int c = 4; c < 128; c += 4) {
                asm volatile("max.f32 %0, %0, %1;" : "+f"(m0) : "f"(s[c]));
                asm volatile("max.f32 %0, %0, %1;" : "+f"(m1) : "f"(s[c + 1]));
                asm volatile("max.f32 %0, %0, %1;" : "+f"(m2) : "f"(s[c + 2]));
                asm volatile("max.f32 %0, %0, %1;" : "+f"(m3) : "f"(s[c + 3]));
            }
            acc += fmaxf(fmaxf(m0, m1), fmaxf(m2, m3));
            s[0] = acc;
        } else if (MODE == 3) {
            float m0 = s[0], m1 = s[1], m2 = s[2], m3 = s[3];
#pragma unroll
            for (int c = 4; c < 128; c += 8) {
                asm volatile("max.f32 %0, %0, %1, %2;" : "+f"(m0) : "f"(s[c]), "f"(s[c + 1]));
                asm volatile("max.f32 %0, %0, %1, %2;" : "+f"(m1) : "f"(s[c + 2]), "f"(s[c + 3]));
                asm volatile("max.f32 %0, %0, %1, %2;" : "+f"(m2) : "f"(s[c + 4]), "f"(s[(c + 5) & 127]));
                asm volatile("max.f32 %0, %0, %1, %2;" : "+f"(m3) : "f"(s[(c + 6) & 127]), "f"(s[(c + 7) & 127]));
            }
            acc += fmaxf(fmaxf(m0, m1), fmaxf(m2, m3));
            s[0] = acc;
        } else if (MODE == 4) {
            const uint64_t sl2 = f2(seed, seed), nm2 = f2(-seed, -seed);
#pragma unroll
            for (int c = 0; c < 64; ++c) {
                const uint64_t x = fma2(f2(s[2 * c], s[2 * c + 1]), sl2, nm2);
                unf2(x, s[2 * c], s[2 * c + 1]);
            }
        } else if (MODE == 5) {
#pragma unroll
            for (int c = 0; c < 64; ++c) rs[c & 3] = add2(rs[c & 3], f2(s[2 * c], s[2 * c + 1]));
        } else if (MODE == 6) {
#pragma unroll
            for (int c = 0; c < 64; ++c) { uint32_t p = pack2(s[2 * c], s[2 * c + 1]); s[2 * c] = __uint_as_float(p); }
        } else if (MODE == 7) {
#pragma unroll
            for (int i = 0; i < 128; ++i) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(s[i]) : "f"(seed), "f"(-seed));
        }
    }
    long long t1 = clock64();
    float o = acc;
#pragma unroll
    for (int i = 0; i < 128; ++i) o += s[i];
    float a, b;
    unf2(add2(add2(rs[0], rs[1]), add2(rs[2], rs[3])), a, b);
    out[blockIdx.x * blockDim.x + threadIdx.x] = o + a + b + __uint_as_float(pk);
    if (threadIdx.x == 0 && blockIdx.x == 0) *clk = (t1 - t0) / REP;
}

template <int MODE>
void run(const char* name, int n_inst)
{
    float* out;
    long long* clk;
    cudaMalloc(&out, 148 * 256 * 4);
    cudaMalloc(&clk, 8);
    for (int warps : {4, 8}) {
        k<MODE><<<148, warps * 32>>>(out, clk, 0.5f);
        k<MODE><<<148, warps * 32>>>(out, clk, 0.5f);
        long long h;
        cudaMemcpy(&h, clk, 8, cudaMemcpyDeviceToHost);
        printf("%-28s warps/SMSP %d: %6lld clk per rep, %.2f clk per warp-instr (%d instr)\n", name, warps / 4, h, (double)h / n_inst, n_inst);
    }
    cudaError_t e = cudaDeviceSynchronize();
    if (e != cudaSuccess) printf("error %s\n", cudaGetErrorString(e));
    cudaFree(out);
    cudaFree(clk);
}

int main()
{
    run<0>("MUFU.EX2 x128", 128);
    run<1>("mix fma2+2ex2+add2+pack x64", 320);
    run<8>("mix without ex2 x64", 192);
    run<2>("FMNMX x124", 124);
    run<3>("FMNMX3 x62", 62);
    run<4>("FFMA2 x64", 64);
    run<5>("FADD2 x64", 64);
    run<6>("F2FP pack x64", 64);
    run<7>("FFMA x128", 128);
    return 0;
}
