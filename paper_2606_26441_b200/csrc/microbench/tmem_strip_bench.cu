// tmem_strip_bench.cu — microbenchmark behind the tensor-memory strip store of the fp32 batch kernel (score_term.cu):
// TMEM (tcgen05.ld) vs shared memory (LDS.128) as the source of dense strips for an FFMA2 contraction, one CTA of 32 warps
// per SM like the batch kernel, plus a layout check of tcgen05.cp.32x128b.warpx4.  Not part of libgpusparse.so.  Build and run:
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -lineinfo -o tmem_strip_bench tmem_strip_bench.cu && ./tmem_strip_bench
// Results on B200: profiles/r02_tmem_microbench.md.
#include <cstdio>
#include <cstdint>
#include <cstdlib>
#include <vector>
#include <cuda_runtime.h>

#define CK(x) do { cudaError_t e = (x); if (e != cudaSuccess) { printf("CUDA error %s at %d\n", cudaGetErrorString(e), __LINE__); exit(1); } } while (0)

__device__ __forceinline__ unsigned long long fma2(unsigned long long a, unsigned long long b, unsigned long long c) {
    unsigned long long d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__device__ __forceinline__ unsigned long long pk(uint32_t lo, uint32_t hi) {
    unsigned long long d;
    asm("mov.b64 %0, {%1, %2};" : "=l"(d) : "r"(lo), "r"(hi));
    return d;
}
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t (&v)[16]) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                 : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
                   "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
                 : "r"(taddr));
}
__device__ __forceinline__ void tmem_st16(uint32_t taddr, const uint32_t (&v)[16]) {
    asm volatile("tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};"
                 :: "r"(taddr), "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]),
                    "r"(v[8]), "r"(v[9]), "r"(v[10]), "r"(v[11]), "r"(v[12]), "r"(v[13]), "r"(v[14]), "r"(v[15]) : "memory");
}
__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

constexpr int kWarps = 32;
constexpr int kStrips = 32;     // hot strips: 32 x 512 docs x 4 B = 64 KB (a quarter of TMEM, replicated per lane quarter)

// MODE 0: LDS only; 1: TMEM only; 2: alternate 1:1; 3: 3 TMEM : 1 LDS; 4: TMEM with the next load issued before the FMAs; 5: FMA only
template <int MODE>
__global__ void __launch_bounds__(kWarps * 32, 1) k_bench(int iters, float* out, long long* cycles) {
    extern __shared__ __align__(16) unsigned char smem[];
    __shared__ uint32_t s_taddr;
    float* strips = reinterpret_cast<float*>(smem);                 // [kStrips][512]
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int i = threadIdx.x; i < kStrips * 512; i += blockDim.x) strips[i] = 1.0f + (float)(i & 1023) * 1e-3f;
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"((uint32_t)__cvta_generic_to_shared(&s_taddr)), "n"(512));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;");
    const uint32_t tbase = s_taddr + ((uint32_t)(32 * (warp & 3)) << 16);
    // fill the warp's lane quarter (the 8 warps of a quarter write the same values: benign)
    for (int s = 0; s < kStrips; ++s) {
        uint32_t v[16];
#pragma unroll
        for (int r = 0; r < 4; ++r)
#pragma unroll
            for (int u = 0; u < 4; ++u) v[4 * r + u] = __float_as_uint(strips[s * 512 + 4 * (lane + 32 * r) + u]);
        tmem_st16(tbase + s * 16, v);
    }
    tmem_wait_st();
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;");
    unsigned long long acc[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) acc[i] = 0ull;
    const float qf = 1.0f + 1e-6f * lane;
    const unsigned long long q2 = pk(__float_as_uint(qf), __float_as_uint(qf));
    const long long t0 = clock64();
    uint32_t nx[16];
    if (MODE == 4) tmem_ld16(tbase, nx);
#pragma unroll 4
    for (int it = 0; it < iters; ++it) {
        const int s = (it * 7 + warp) & (kStrips - 1);
        bool use_tmem = MODE == 1 || MODE == 4 || (MODE == 2 && (it & 1)) || (MODE == 3 && (it & 3));
        if (MODE == 5) {
#pragma unroll
            for (int i = 0; i < 8; ++i) acc[i] = fma2(acc[i], q2, q2);
        } else if (use_tmem) {
            uint32_t v[16];
            if (MODE == 4) {
                tmem_wait_ld();
#pragma unroll
                for (int i = 0; i < 16; ++i) v[i] = nx[i];
                tmem_ld16(tbase + ((s + 1) & (kStrips - 1)) * 16, nx);
            } else {
                tmem_ld16(tbase + s * 16, v);
                tmem_wait_ld();
            }
#pragma unroll
            for (int i = 0; i < 8; ++i) acc[i] = fma2(pk(v[2 * i], v[2 * i + 1]), q2, acc[i]);
        } else {
            const ulonglong2* src = reinterpret_cast<const ulonglong2*>(strips + s * 512 + 4 * lane);
            ulonglong2 v[4];
#pragma unroll
            for (int r = 0; r < 4; ++r) v[r] = src[32 * r];
#pragma unroll
            for (int r = 0; r < 4; ++r) { acc[2 * r] = fma2(v[r].x, q2, acc[2 * r]); acc[2 * r + 1] = fma2(v[r].y, q2, acc[2 * r + 1]); }
        }
    }
    if (MODE == 4) tmem_wait_ld();
    const long long t1 = clock64();
    float sum = 0.f;
#pragma unroll
    for (int i = 0; i < 8; ++i) { sum += __uint_as_float((uint32_t)acc[i]) + __uint_as_float((uint32_t)(acc[i] >> 32)); }
    if (MODE == 4) sum += __uint_as_float(nx[0]);
    out[blockIdx.x * blockDim.x + threadIdx.x] = sum;
    if (lane == 0) atomicMax((unsigned long long*)&cycles[blockIdx.x], (unsigned long long)(t1 - t0));
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(s_taddr), "n"(512));
}

// Layout check: strips in natural layout in shared memory -> tcgen05.cp 32x128b.warpx4 -> every lane quarter must hold
// TMEM[32k + i][s*16 + 4r + u] = strip[s][4*(i + 32r) + u]
__global__ void __launch_bounds__(kWarps * 32, 1) k_cp_check(uint32_t* dump, int use_cp) {
    extern __shared__ __align__(128) unsigned char smem[];
    __shared__ uint32_t s_taddr;
    __shared__ __align__(8) unsigned long long s_bar;
    uint32_t* strips = reinterpret_cast<uint32_t*>(smem);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int i = threadIdx.x; i < kStrips * 512; i += blockDim.x) strips[i] = (uint32_t)i;
    const uint32_t bar = (uint32_t)__cvta_generic_to_shared(&s_bar);
    if (threadIdx.x == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar) : "memory");
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"((uint32_t)__cvta_generic_to_shared(&s_taddr)), "n"(512));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");      // generic-proxy smem writes -> async proxy (tcgen05.cp reads)
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;");
    const uint32_t t0 = s_taddr;
    if (use_cp) {
        if (threadIdx.x == 0) {
            const uint32_t sbase = (uint32_t)__cvta_generic_to_shared(strips);
            for (int s = 0; s < kStrips; ++s)
                for (int r = 0; r < 4; ++r) {
                    const uint32_t a = sbase + (uint32_t)(s * 2048 + r * 512);
                    // no swizzle, K-major: core matrix = 8 rows x 16 B contiguous; SBO (next 8 rows) = 128 B; LBO unused (one core matrix wide)
                    const unsigned long long desc = (unsigned long long)((a & 0x3FFFF) >> 4) | ((unsigned long long)(16 >> 4) << 16) |
                                                    ((unsigned long long)(128 >> 4) << 32) | (1ull << 46);
                    asm volatile("tcgen05.cp.cta_group::1.32x128b.warpx4 [%0], %1;" ::"r"(t0 + (uint32_t)(s * 16 + r * 4)), "l"(desc) : "memory");
                }
            asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
        }
        uint32_t ok = 0;
        do {
            asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }" : "=r"(ok) : "r"(bar), "r"(0u) : "memory");
        } while (!ok);
        asm volatile("tcgen05.fence::after_thread_sync;");
    }
    if (warp < 4) {
        const uint32_t tb = t0 + ((uint32_t)(32 * warp) << 16);
        for (int s = 0; s < kStrips; ++s) {
            uint32_t v[16];
            tmem_ld16(tb + s * 16, v);
            tmem_wait_ld();
#pragma unroll
            for (int i = 0; i < 16; ++i) dump[((size_t)(32 * warp + lane)) * 512 + s * 16 + i] = v[i];
        }
    }
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(s_taddr), "n"(512));
}

template <int MODE>
void run(const char* name, int iters, float* d_out, long long* d_cyc, int sms) {
    CK(cudaFuncSetAttribute(k_bench<MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, kStrips * 2048));
    CK(cudaMemset(d_cyc, 0, sizeof(long long) * sms));
    cudaEvent_t a, b;
    CK(cudaEventCreate(&a)); CK(cudaEventCreate(&b));
    k_bench<MODE><<<sms, kWarps * 32, kStrips * 2048>>>(iters / 8, d_out, d_cyc);
    CK(cudaMemset(d_cyc, 0, sizeof(long long) * sms));
    CK(cudaEventRecord(a));
    k_bench<MODE><<<sms, kWarps * 32, kStrips * 2048>>>(iters, d_out, d_cyc);
    CK(cudaEventRecord(b));
    CK(cudaDeviceSynchronize());
    float ms = 0;
    CK(cudaEventElapsedTime(&ms, a, b));
    std::vector<long long> h(sms);
    CK(cudaMemcpy(h.data(), d_cyc, sizeof(long long) * sms, cudaMemcpyDeviceToHost));
    long long mx = 0; double avg = 0;
    for (long long c : h) { mx = c > mx ? c : mx; avg += (double)c / sms; }
    printf("%-28s iters %d: %.3f ms, SM cycles per strip-row (one warp, 512 docs x 1 strip): avg %.2f max %.2f  (=> %.1f B/clk/SM)\n", name, iters, ms,
           avg / ((double)iters * kWarps), (double)mx / ((double)iters * kWarps), 2048.0 / (avg / ((double)iters * kWarps)));
}

int main() {
    int dev = 0, sms = 0;
    CK(cudaGetDevice(&dev));
    CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    printf("SMs %d\n", sms);
    float* d_out; long long* d_cyc; uint32_t* d_dump;
    CK(cudaMalloc(&d_out, sizeof(float) * sms * kWarps * 32));
    CK(cudaMalloc(&d_cyc, sizeof(long long) * sms));
    CK(cudaMalloc(&d_dump, sizeof(uint32_t) * 128 * 512));
    // layout check with tcgen05.st (inside k_bench fill) is implicit; explicit check with tcgen05.cp:
    for (int use_cp = 1; use_cp <= 1; ++use_cp) {
        CK(cudaFuncSetAttribute(k_cp_check, cudaFuncAttributeMaxDynamicSharedMemorySize, kStrips * 2048));
        CK(cudaMemset(d_dump, 0xFF, sizeof(uint32_t) * 128 * 512));
        k_cp_check<<<1, kWarps * 32, kStrips * 2048>>>(d_dump, use_cp);
        cudaError_t e = cudaDeviceSynchronize();
        if (e != cudaSuccess) { printf("k_cp_check failed: %s\n", cudaGetErrorString(e)); return 1; }
        std::vector<uint32_t> h(128 * 512);
        CK(cudaMemcpy(h.data(), d_dump, sizeof(uint32_t) * 128 * 512, cudaMemcpyDeviceToHost));
        long bad = 0;
        for (int l = 0; l < 128; ++l)
            for (int c = 0; c < 512; ++c) {
                const int i = l & 31, s = c >> 4, r = (c >> 2) & 3, u = c & 3;
                const uint32_t want = (uint32_t)(s * 512 + 4 * (i + 32 * r) + u);
                if (h[l * 512 + c] != want) { if (bad < 8) printf("  mismatch lane %d col %d: got %u want %u\n", l, c, h[l * 512 + c], want); ++bad; }
            }
        printf("tcgen05.cp 32x128b.warpx4 layout check: %ld mismatches of %d\n", bad, 128 * 512);
    }
    const int iters = 1 << 15;
    run<5>("FFMA2 only", iters, d_out, d_cyc, sms);
    run<0>("LDS.128 x4 + 8 FFMA2", iters, d_out, d_cyc, sms);
    run<1>("tcgen05.ld x16 + 8 FFMA2", iters, d_out, d_cyc, sms);
    run<4>("tcgen05.ld x16 pipelined", iters, d_out, d_cyc, sms);
    run<2>("1 TMEM : 1 LDS", iters, d_out, d_cyc, sms);
    run<3>("3 TMEM : 1 LDS", iters, d_out, d_cyc, sms);
    return 0;
}
