// Machine-model microbenchmarks for the harmonic-sum kernels: what one B200 SM can
// take from an L2-resident spectrum under the access shapes of the gathers, and what shared memory delivers.
//   (1) random line-aligned warp loads with a lane stride of 1..32 words (order h of the greedy gather has
//       lane stride h): requests, 128-byte lines and 32-byte sectors per clock and SM;
//   (2) 1-D bulk async copies (TMA engine) L2 -> shared memory, by chunk size and CTAs per SM;
//   (3) conflict-free LDS.32 / LDS.64 / LDS.128 rates.
// Build and run (one GPU):  nvcc -O3 -std=c++17 -gencode arch=compute_100a,code=sm_100a -o machine_model machine_model.cu
// The numbers measured on this pool's B200 are in profiles/r01b_machine_model.md.
#include <cuda_runtime.h>
#include <cstdio>
#include <cstdlib>
#define CK(x) do { cudaError_t e = (x); if (e != cudaSuccess) { printf("CUDA error %s at %d\n", cudaGetErrorString(e), __LINE__); exit(1); } } while (0)

template <int U, bool CG, bool DEP>
__global__ void k_g(const float* __restrict__ p, unsigned nlines_mask, int stride, int iters, float* out) {
    const unsigned gw = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const unsigned lane = threadIdx.x & 31;
    unsigned state = gw * 2654435761u + 12345u;
    float acc = 0.f;
    for (int it = 0; it < iters; ++it) {
        float v[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            state = state * 1664525u + 1013904223u;
            unsigned line = (state >> 7) & nlines_mask;
            if (DEP) line = (line + (__float_as_uint(acc) & 1u)) & nlines_mask;   // acc is always 0: serialises iterations
            const float* q = p + (size_t)line * 32 + lane * stride;
            v[u] = CG ? __ldcg(q) : __ldg(q);
        }
#pragma unroll
        for (int u = 0; u < U; ++u) acc += v[u];
    }
    if (acc == 123.456f) out[0] = acc;
}

// (3) bulk async copy (TMA 1-D) L2 -> smem streaming: each CTA copies chunks of CH bytes, double buffered
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
template <int CH, int NBUF>
__global__ void k_bulk(const float* __restrict__ p, long long nbytes, int rep, float* out) {
    extern __shared__ float4 sm4[];
    char* sm = (char*)sm4;
    __shared__ unsigned long long bar[NBUF];
    if (threadIdx.x == 0) {
        for (int b = 0; b < NBUF; ++b) asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;\n" :: "r"(smem_u32(&bar[b])));
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    }
    __syncthreads();
    const long long nch = nbytes / CH;
    float acc = 0.f;
    if (threadIdx.x == 0) {
        long long total = 0;
        for (int r = 0; r < rep; ++r) for (long long c = blockIdx.x; c < nch; c += gridDim.x) ++total;
        long long issued = 0, waited = 0;
        int r_i = 0; long long c_i = blockIdx.x;
        unsigned phase[NBUF]; for (int b = 0; b < NBUF; ++b) phase[b] = 0;
        while (waited < total) {
            while (issued < total && issued - waited < NBUF) {
                int b = issued % NBUF;
                asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" :: "r"(smem_u32(&bar[b])), "r"((unsigned)CH) : "memory");
                asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n"
                             :: "r"(smem_u32(sm + (size_t)b * CH)), "l"((const char*)p + c_i * (long long)CH), "r"((unsigned)CH), "r"(smem_u32(&bar[b])) : "memory");
                ++issued; c_i += gridDim.x; if (c_i >= nch) { c_i = blockIdx.x; ++r_i; }
            }
            int b = waited % NBUF;
            unsigned done = 0;
            while (!done) asm volatile("{\n .reg .pred q;\n mbarrier.try_wait.parity.shared::cta.b64 q, [%1], %2;\n selp.u32 %0, 1, 0, q;\n}\n" : "=r"(done) : "r"(smem_u32(&bar[b])), "r"(phase[b]) : "memory");
            phase[b] ^= 1; ++waited;
            acc += ((float*)sm)[b * (CH / 4)];
        }
    }
    if (acc == 123.456f) out[0] = acc;
}

template <int VEC>
__global__ void k_lds(int iters, float* out) {
    __shared__ float4 s4[2048];   // 32 KB
    float* s = (float*)s4;
    for (int i = threadIdx.x; i < 8192; i += blockDim.x) s[i] = 0.f;
    __syncthreads();
    float acc0 = 0.f, acc1 = 0.f, acc2 = 0.f, acc3 = 0.f;
    const float* base = s + (threadIdx.x & 255) * VEC;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            if (VEC == 1) { acc0 += base[u * 1024]; acc1 += base[u * 1024 + 256]; acc2 += base[u * 1024 + 512]; acc3 += base[u * 1024 + 768]; }
            else if (VEC == 2) {
                float2 a = *(const float2*)(base + u * 1024), b = *(const float2*)(base + u * 1024 + 512);
                acc0 += a.x; acc1 += a.y; acc2 += b.x; acc3 += b.y;
            } else {
                float4 a = *(const float4*)(base + u * 1024);
                acc0 += a.x; acc1 += a.y; acc2 += a.z; acc3 += a.w;
            }
        }
        base = (const float*)((unsigned long long)base ^ ((__float_as_int(acc0) & 1) << 4));  // keep the loop alive (acc0 = 0)
    }
    float acc = acc0 + acc1 + acc2 + acc3;
    if (acc == 123.456f) out[0] = acc;
}


template <typename F>
float timeit(F f, int n = 3) {
    cudaEvent_t a, b; cudaEventCreate(&a); cudaEventCreate(&b);
    f(); CK(cudaDeviceSynchronize());
    float best = 1e30f;
    for (int i = 0; i < n; ++i) {
        cudaEventRecord(a); f(); cudaEventRecord(b); CK(cudaEventSynchronize(b));
        float ms; cudaEventElapsedTime(&ms, a, b); if (ms < best) best = ms;
    }
    return best;
}
template <int U, bool CG, bool DEP>
void run(const float* buf, unsigned mask, int stride, float* out, int SM, int wps) {
    int iters = 2000 / U;
    float ms = timeit([&] { k_g<U, CG, DEP><<<SM * wps / 8, 256>>>(buf, mask, stride, iters, out); });
    double wl = (double)SM * wps * iters * U;
    double lines = stride >= 32 ? 32 : stride;             // lines per warp-load
    double sect = stride >= 8 ? 32 : stride * 4;            // sectors per warp-load
    printf("U%d %s %s warps/SM %2d stride %2d: %6.1f Gwarp-loads/s (%5.3f /clk/SM)  lines %6.1f G/s (%5.3f /clk/SM)  sectors %6.2f TB/s\n", U, CG ? "cg" : "nc",
           DEP ? "dep" : "ind", wps, stride, wl / ms / 1e6, wl / ms / 1e6 / SM / 1.965, wl * lines / ms / 1e6, wl * lines / ms / 1e6 / SM / 1.965, wl * sect * 32 / ms / 1e9);
}

int main() {
    float* buf; float* out;
    const size_t bytes = 64u << 20;                       // L2-resident, larger than the L1s
    CK(cudaMalloc(&buf, bytes + (1 << 20))); CK(cudaMalloc(&out, 64));
    CK(cudaMemset(buf, 0, bytes + (1 << 20)));
    cudaDeviceProp pr; cudaGetDeviceProperties(&pr, 0);
    const int SM = pr.multiProcessorCount;
    printf("%s: %d SMs, L2 %d MB, clock %d kHz\n", pr.name, SM, pr.l2CacheSize >> 20, pr.clockRate);
    const unsigned mask = (unsigned)(bytes / 128) - 1;
    for (int stride : {1, 2, 4, 8, 16, 32}) {
        run<4, true, false>(buf, mask, stride, out, SM, 64);
        run<4, false, false>(buf, mask, stride, out, SM, 64);
        run<2, false, true>(buf, mask, stride, out, SM, 64);
        run<4, false, false>(buf, mask, stride, out, SM, 32);
    }
    {
        const long long nbytes = 16 << 20;
        const int rep = 128;
        CK(cudaFuncSetAttribute(k_bulk<16384, 4>, cudaFuncAttributeMaxDynamicSharedMemorySize, 65536));
        for (int cps : {1, 2, 3}) {
            float ms = timeit([&] { k_bulk<16384, 4><<<SM * cps, 32, 65536>>>(buf, nbytes, rep, out); });
            printf("bulk copy 16 KiB x 4 in flight, CTAs/SM %d: %8.1f GB/s\n", cps, (double)nbytes * rep / ms / 1e6);
        }
        CK(cudaFuncSetAttribute(k_bulk<4096, 8>, cudaFuncAttributeMaxDynamicSharedMemorySize, 32768));
        for (int cps : {2, 4, 6}) {
            float ms = timeit([&] { k_bulk<4096, 8><<<SM * cps, 32, 32768>>>(buf, nbytes, rep, out); });
            printf("bulk copy 4 KiB x 8 in flight, CTAs/SM %d: %8.1f GB/s\n", cps, (double)nbytes * rep / ms / 1e6);
        }
    }
    {
        const int iters = 4000, bs = 256;
        double warp_lds = (double)SM * (2048 / 32) * iters * 32;
        float ms = timeit([&] { k_lds<1><<<SM * (2048 / bs), bs>>>(iters, out); });
        printf("LDS.32 : %6.1f Gwarp-LDS/s = %5.2f /clk/SM  %6.1f TB/s\n", warp_lds / ms / 1e6, warp_lds / ms / 1e6 / SM / (pr.clockRate / 1e6), warp_lds * 128 / ms / 1e9);
        warp_lds /= 2;
        ms = timeit([&] { k_lds<2><<<SM * (2048 / bs), bs>>>(iters, out); });
        printf("LDS.64 : %6.1f Gwarp-LDS/s = %5.2f /clk/SM  %6.1f TB/s\n", warp_lds / ms / 1e6, warp_lds / ms / 1e6 / SM / (pr.clockRate / 1e6), warp_lds * 256 / ms / 1e9);
        warp_lds /= 2;
        ms = timeit([&] { k_lds<4><<<SM * (2048 / bs), bs>>>(iters, out); });
        printf("LDS.128: %6.1f Gwarp-LDS/s = %5.2f /clk/SM  %6.1f TB/s\n", warp_lds / ms / 1e6, warp_lds / ms / 1e6 / SM / (pr.clockRate / 1e6), warp_lds * 512 / ms / 1e9);
    }
    return 0;
}
