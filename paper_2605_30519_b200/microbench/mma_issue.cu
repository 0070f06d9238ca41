// tcgen05.mma pacing on sm_100a: SS vs TS (A in TMEM), TMEM column placement, issue-queue depth, effect of concurrent tcgen05.ld.
#include <cstdio>
#include <cstdint>
#include <cuda_runtime.h>

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(void* bar, uint32_t count) { asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count)); }
__device__ __forceinline__ bool mbar_try_wait(void* bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}" : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_wait(void* bar, uint32_t parity) { while (!mbar_try_wait(bar, parity)) {} }
__device__ __forceinline__ uint64_t make_desc(uint32_t saddr, uint32_t lbo_bytes, uint32_t sbo_bytes)
{
    return (uint64_t)((saddr & 0x3FFFFu) >> 4) | ((uint64_t)(lbo_bytes >> 4) << 16) | ((uint64_t)(sbo_bytes >> 4) << 32) | ((uint64_t)1 << 46) | ((uint64_t)2 << 61);
}
constexpr uint32_t IDESC_BASE = (1u << 4) | (1u << 7) | (1u << 10) | ((128u >> 3) << 17) | ((128u >> 4) << 24);
__device__ __forceinline__ void mma_ss(uint32_t d, uint64_t a, uint64_t b, uint32_t idesc, uint32_t acc)
{
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\ttcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}" ::"r"(d), "l"(a), "l"(b), "r"(idesc), "r"(acc) : "memory");
}
__device__ __forceinline__ void mma_ts(uint32_t d, uint32_t a, uint64_t b, uint32_t idesc, uint32_t acc)
{
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\ttcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}" ::"r"(d), "r"(a), "l"(b), "r"(idesc), "r"(acc) : "memory");
}
__device__ __forceinline__ void mma_commit(void* bar) { asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory"); }
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, float (&v)[32])
{
    uint32_t* r = reinterpret_cast<uint32_t*>(v);
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
          "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]),
          "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]),
          "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
        : "r"(taddr));
}

__device__ __forceinline__ bool elect_one()
{
    uint32_t pred;
    asm volatile("{\n\t.reg .pred P;\n\telect.sync _|P, 0xffffffff;\n\tselp.u32 %0, 1, 0, P;\n\t}" : "=r"(pred));
    return pred != 0;
}
struct Params {
    int mode;       // 0 SS, 1 TS
    int a_col, d_col, d_col2;  // d alternates between d_col and d_col2 every 8 MMAs
    int n_mma;
    int ld_warps;   // warps 0..3 (x2) doing tcgen05.ld loops concurrently
    int ld_col;
    int same_k;     // 1: every MMA reads the same smem bytes
    int alt1;       // 1: alternate the accumulator every MMA instead of every 8
    int n;          // MMA N
    int tma;        // 1: warp 8 streams 32 KB bulk copies global -> smem meanwhile
};

template <int MODE>
__global__ void __launch_bounds__(320, 1) k(Params p, long long* out, const unsigned char* gsrc)
{
    extern __shared__ unsigned char raw[];
    unsigned char* sm = (unsigned char*)(((uintptr_t)raw + 1023) & ~(uintptr_t)1023);
    unsigned long long* bar = (unsigned long long*)(sm + 4 * 32768);
    uint32_t* tbase = (uint32_t*)(sm + 4 * 32768 + 64);
    volatile int* stop = (volatile int*)(sm + 4 * 32768 + 128);
    const int warp = threadIdx.x >> 5;
    for (int i = threadIdx.x; i < 4 * 32768 / 4; i += blockDim.x) ((uint32_t*)sm)[i] = 0x3c003c00u;
    if (threadIdx.x == 0) { mbar_init(bar, 1); *stop = 0; asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
    if (warp == 9) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tbase)), "r"(512));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem = *tbase;
    if (warp == 9) {
        const uint64_t ad = make_desc(smem_u32(sm), 16, 1024);
        const uint32_t idesc = (1u << 4) | (1u << 7) | (1u << 10) | (((uint32_t)p.n >> 3) << 17) | ((128u >> 4) << 24);
        long long t0 = clock64(), t1 = 0;
        if (MODE >= 5) {
            const uint64_t bd = make_desc(smem_u32(sm + 32768), 16, 1024);
            const uint64_t vd = make_desc(smem_u32(sm + 65536), 16384, 1024);
            const uint32_t idk = idesc, idv = idesc | (1u << 16);
            for (int b = 0; b < p.n_mma / 16; ++b) {
                if (elect_one()) {
#pragma unroll
                    for (int j = 0; j < 8; ++j) {  // first batch of the pair: always SS K-major into S0
                        const uint64_t off = (uint64_t)(((j >> 2) * 16384 + (j & 3) * 32) >> 4);
                        mma_ss(tmem, ad + off, bd + off, idk, j > 0);
                    }
#pragma unroll
                    for (int j = 0; j < 8; ++j) {
                        const uint64_t off = (uint64_t)(((j >> 2) * 16384 + (j & 3) * 32) >> 4);
                        if (MODE == 5) mma_ss(tmem + 128, ad + off, bd + off, idk, j > 0);                                  // SS K-major, other D
                        if (MODE == 6) mma_ts(tmem + 256, tmem + 384 + j * 8, bd + off, idk, j > 0);                        // TS K-major
                        if (MODE == 7) mma_ts(tmem + 256, tmem + 384 + j * 8, vd + (uint64_t)((j * 2048) >> 4), idv, j > 0); // TS MN-major (PV)
                        if (MODE == 8) mma_ss(tmem + 256, ad + off, vd + (uint64_t)((j * 2048) >> 4), idv, j > 0);           // SS MN-major
                    }
                }
                __syncwarp();
            }
        } else
        for (int b = 0; b < p.n_mma / 8; ++b) {
            const int tile = p.same_k ? 0 : b % 3;
            const uint64_t bd0 = make_desc(smem_u32(sm + 32768 * (1 + tile)), 16, 1024);
            const uint32_t d = tmem + ((b & 1) ? p.d_col2 : p.d_col);
            const uint64_t vd0 = make_desc(smem_u32(sm + 32768 * (1 + tile)), 16384, 1024);
            if (elect_one()) {
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    const uint64_t off = (uint64_t)(((j >> 2) * 16384 + (j & 3) * 32) >> 4);
                    const uint32_t dd = p.alt1 ? tmem + ((j & 1) ? p.d_col2 : p.d_col) : d;
                    if (MODE == 0) mma_ss(dd, ad + off, bd0 + off, idesc, j > 1);
                    else if (MODE == 1) mma_ts(dd, tmem + p.a_col + j * 8, bd0 + off, idesc, j > 1);
                    else if (MODE == 4) {
                        if (b & 1) mma_ts(tmem + 256, tmem + 384 + j * 8, vd0 + (uint64_t)((j * 2048) >> 4), idesc | (1u << 16), j > 0);
                        else mma_ss(tmem + ((b & 2) ? 128 : 0), ad + off, bd0 + off, idesc, j > 0);
                    }
                    else if (MODE == 2 || (MODE == 3 && (b & 1))) mma_ts(dd, tmem + 448 + j * 8, vd0 + (uint64_t)((j * 2048) >> 4), idesc | (1u << 16), j > 1);
                    else mma_ts(dd, tmem + p.a_col + j * 8, bd0 + off, idesc, j > 1);
                }
            }
            __syncwarp();
        }
        t1 = clock64();
        if (elect_one()) mma_commit(bar);
        __syncwarp();
        mbar_wait(bar, 0);
        long long t2 = clock64();
        if (blockIdx.x == 0 && threadIdx.x == 9 * 32) { out[0] = t1 - t0; out[1] = t2 - t0; }
        *stop = 1;
    } else if (warp == 8 && p.tma) {
        unsigned long long* tbar = bar + 4;
        long long n = 0;
        if (threadIdx.x == 8 * 32) {
            mbar_init(tbar, 1);
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
            if (p.tma == 2) {
                for (int i = 0; i < 3; ++i) mbar_init(tbar + 1 + i, 1);
                asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
                while (!*stop) {
                    const int st = n % 3;
                    if (n >= 3) mbar_wait(tbar + 1 + st, ((n / 3) - 1) & 1);
                    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(tbar + 1 + st)), "r"(32768) : "memory");
                    for (int c = 0; c < 4; ++c)
                        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                                     ::"r"(smem_u32(sm + 4 * 32768 + 4096 + (st % 2) * 32768 + c * 8192)), "l"(gsrc + ((n * 4 + c) % 128) * 8192), "r"(8192), "r"(smem_u32(tbar + 1 + st)) : "memory");
                    ++n;
                }
            } else
            while (!*stop) {
                asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(tbar)), "r"(32768) : "memory");
                for (int c = 0; c < 2; ++c)
                    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                                 ::"r"(smem_u32(sm + 5 * 32768 + 4096 + c * 16384)), "l"(gsrc + ((n * 2 + c) % 64) * 16384), "r"(16384), "r"(smem_u32(tbar)) : "memory");
                mbar_wait(tbar, n & 1);
                ++n;
            }
            if (blockIdx.x == 0) out[2] = n;
        }
    } else if (warp < p.ld_warps) {
        float v[32];
        float acc = 0.f;
        long long n = 0;
        const uint32_t lane_base = (uint32_t)((warp & 3) * 32) << 16;
        if (p.ld_col < 0) {
            float sacc = 0.f;
            while (!__shfl_sync(0xffffffffu, *stop, 0)) {
                float s[128];
                for (int c = 0; c < 128; c += 32) tmem_ld32(tmem + lane_base + (warp >= 4 ? 128 : 0) + c, *reinterpret_cast<float (*)[32]>(&s[c]));
                asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
                uint32_t pk[32];
#pragma unroll
                for (int c = 0; c < 128; ++c) { float y; asm volatile("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(s[c] * 0.001f - 3.f)); sacc += y; if ((c & 3) == 0) pk[c >> 2] = __float_as_uint(y); }
                if (p.same_k == 2) {
                    asm volatile("tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31,%32};"
                        ::"r"(tmem + lane_base + 384 + (warp >= 4 ? 64 : 0)), "r"(pk[0]), "r"(pk[1]), "r"(pk[2]), "r"(pk[3]), "r"(pk[4]), "r"(pk[5]), "r"(pk[6]), "r"(pk[7]), "r"(pk[8]),
                          "r"(pk[9]), "r"(pk[10]), "r"(pk[11]), "r"(pk[12]), "r"(pk[13]), "r"(pk[14]), "r"(pk[15]), "r"(pk[16]), "r"(pk[17]),
                          "r"(pk[18]), "r"(pk[19]), "r"(pk[20]), "r"(pk[21]), "r"(pk[22]), "r"(pk[23]), "r"(pk[24]), "r"(pk[25]), "r"(pk[26]),
                          "r"(pk[27]), "r"(pk[28]), "r"(pk[29]), "r"(pk[30]), "r"(pk[31]) : "memory");
                    asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
                }
                ++n;
            }
            acc = sacc;
        } else
        while (!__shfl_sync(0xffffffffu, *stop, 0)) {
            for (int c = 0; c < 128; c += 32) {
                tmem_ld32(tmem + lane_base + p.ld_col + c, v);
                asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
                acc += v[0];
            }
            ++n;
        }
        if (blockIdx.x == 0 && (threadIdx.x & 31) == 0) out[2 + warp] = n + (acc == 1234.5f);
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 9) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(512));
}

template <int MODE>
void run(const char* name, Params p)
{
    long long* out;
    cudaMalloc(&out, 16 * 8);
    cudaMemset(out, 0, 16 * 8);
    const int smem = 6 * 32768 + 8192;
    static unsigned char* gsrc = nullptr;
    if (!gsrc) { cudaMalloc(&gsrc, 64 * 16384); cudaMemset(gsrc, 0, 64 * 16384); }
    cudaFuncSetAttribute(k<MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    k<MODE><<<148, 320, smem>>>(p, out, gsrc);
    k<MODE><<<148, 320, smem>>>(p, out, gsrc);
    long long h[16];
    cudaError_t e = cudaMemcpy(h, out, 16 * 8, cudaMemcpyDeviceToHost);
    printf("%-44s n=%4d issue %7lld clk  done %7lld clk  -> %.1f clk/MMA (issue %.1f)  ld/tma iters %lld (%.1f B/clk)\n", name, p.n_mma, h[0], h[1], (double)h[1] / p.n_mma,
           (double)h[0] / p.n_mma, h[2], p.tma ? 32768.0 * h[2] / h[1] : 0.0);
    if (e != cudaSuccess) printf("error %s\n", cudaGetErrorString(e));
    cudaFree(out);
}

int main()
{
    // clean issue loops (no data-dependent control flow between MMAs)
    run<0>("SS K-major", {0, 0, 0, 0, 256, 0, 0, 0, 0, 128, 0});
    run<1>("TS K-major (A in TMEM)", {1, 384, 0, 0, 256, 0, 0, 0, 0, 128, 0});
    run<2>("TS MN-major B (PV-like)", {2, 448, 256, 256, 256, 0, 0, 0, 0, 128, 0});
    run<7>("QK(SS) <-> PV(TS MN-major), 8 + 8 unrolled", {7, 384, 0, 0, 512, 0, 0, 0, 0, 128, 0});
    run<7>("  + TMA stream + 8 softmax-like warps (ld+ex2+st)", {7, 384, 0, 0, 512, 8, -1, 2, 0, 128, 2});
    // the same alternation with one data-dependent branch per batch in the issuing thread
    run<4>("QK(SS) <-> PV(TS), branch per batch", {4, 384, 0, 0, 512, 0, 0, 0, 0, 128, 0});
    run<1>("TS K-major N=256", {1, 448, 0, 0, 256, 0, 0, 1, 0, 256, 0});
    run<0>("SS K-major N=256", {0, 448, 0, 0, 256, 0, 0, 1, 0, 256, 0});
    return 0;
}
