// PRESTO-like harmonic sum (Alg. 1; eq. 4), shared-memory staged.
//
// With Hq = 2^L the largest power of two <= H, every index Alg. 1 visits for any H' <= Hq is
//     Round(h n / H') = (k n + Hq/2) >> L,   k = h Hq / H'  in  K = {Hq} U {Hq/2^l, (6,10,..,2^l-2) Hq/2^l : l = 1..L}
// (17 fractions k/32 at H = 32; the harmonic sets are nested, see hs_presto.cuh).  A CTA owns T
// consecutive top bins [n0, n0+T), n0 a multiple of T (T a multiple of 128 >= 4 Hq).  For fraction k
// its outputs read the CONTIGUOUS span x[k n0/Hq .. k (n0+T)/Hq]  (the compressing gather of
// SURVEY.md 8(a) a3), k T/Hq + 1 floats, 16-byte aligned.  All spans (8.5 T floats at H = 32) are
// staged once into shared memory -- by 1-D bulk async copies (TMA engine, cp.async.bulk -> UBLKCP)
// on interior tiles, by guarded float4 loads on the tile that touches the end of the row -- and
// every term is then a conflict-free LDS:  lane i of a warp working on outputs n0 + 32 q + i reads
//     span_k[ k (32/Hq) q + ((k i + Hq/2) >> L) ],
// consecutive lanes hit the same or the next word, the per-lane part is a register, the k q part an
// immediate.  L2 -> SM traffic is 4 * sum(k)/Hq = 34 B per bin at H = 32 (each staged float is used
// by 32/k outputs) instead of one 32-byte sector per term and warp-quarter.
#pragma once
#include "hs_common.cuh"

// floats of shared memory used by the spans of one tile (each span padded to a float4 multiple)
template <int L>
__host__ __device__ constexpr int hs_presto_span_floats(int T) {
    constexpr int Hq = 1 << L;
    int tot = 4 * ((T / 4) + 1);                      // k = Hq
    for (int l = 1; l <= L; ++l) {
        const int sc = Hq >> l;                       // k = h * sc
        tot += 4 * (((1 * sc * T) >> L) / 4 + 1);
        for (int h = 6; h < (1 << l); h += 4) tot += 4 * (((h * sc * T) >> L) / 4 + 1);
    }
    return tot;
}

__device__ __forceinline__ unsigned hs_smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }

// stage span k of the tile into sm[off ..]: guarded path (any tile)
template <int BLOCK>
__device__ __forceinline__ void hs_stage_guarded(float* __restrict__ sm, int off, const float* __restrict__ x,
                                                 int g, int len4, int N) {
    float4* dst = reinterpret_cast<float4*>(sm + off);
#pragma unroll 1
    for (int i = threadIdx.x; i < len4; i += BLOCK) {
        const int e = g + 4 * i;
        float4 v;
        if (e + 3 < N) {
            v = __ldg(reinterpret_cast<const float4*>(x + e));
        } else {
            v.x = (e < N) ? __ldg(x + e) : 0.f;
            v.y = (e + 1 < N) ? __ldg(x + e + 1) : 0.f;
            v.z = (e + 2 < N) ? __ldg(x + e + 2) : 0.f;
            v.w = (e + 3 < N) ? __ldg(x + e + 3) : 0.f;
        }
        dst[i] = v;
    }
}

// one 1-D bulk async copy global -> shared, completion counted in bytes on an mbarrier
__device__ __forceinline__ void hs_bulk_g2s(float* dst, const float* src, unsigned bytes, unsigned long long* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n"
                 :: "r"(hs_smem_u32(dst)), "l"(src), "r"(bytes), "r"(hs_smem_u32(bar)) : "memory");
}

template <int T, int L, int BLOCK, bool BULK>
__global__ void __launch_bounds__(BLOCK)
hs_presto_smem_kernel(const __grid_constant__ HsShape sh, const __grid_constant__ HsStats st, HsIO io) {
    constexpr int Hq = 1 << L;
    constexpr int HALF = Hq >> 1;
    constexpr int NW = BLOCK / 32;                    // warps
    constexpr int NQ = T / 32;                        // 32-output groups per tile
    constexpr int Q = 32 >> L;                        // index of output 32 q + i, fraction k: k Q q + ((k i + Hq/2) >> L)
    static_assert(T % 128 == 0 && NQ % NW == 0, "tile shape");
    extern __shared__ float4 hs_smem4[];
    float* sm = reinterpret_cast<float*>(hs_smem4);
    __shared__ unsigned long long bar;

    const int s = blockIdx.y;
    const int N = (int)sh.n_bins;
    const int n_fund = (int)sh.n_fund;
    const int n0 = blockIdx.x * T;
    const int q0 = n0 >> L;                           // n0 / Hq (n0 is a multiple of Hq)
    const float* __restrict__ x = io.x + (long long)s * sh.in_stride;

    // ---- stage the spans ----
    // the tile is interior when every padded span ends inside the row: the largest is k = Hq, [n0, n0+T+4)
    const bool interior = BULK && (n0 + T + 4 <= N);
    if (interior) {
        if (threadIdx.x == 0) {
            asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;\n" :: "r"(hs_smem_u32(&bar)) : "memory");
            asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
            constexpr unsigned total = 4u * (unsigned)hs_presto_span_floats<L>(T);
            asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" :: "r"(hs_smem_u32(&bar)), "r"(total) : "memory");
            int off = 0;
            {
                constexpr int len4 = T / 4 + 1;
                hs_bulk_g2s(sm + off, x + n0, 16u * len4, &bar);
                off += 4 * len4;
            }
#pragma unroll
            for (int l = 1; l <= L; ++l) {
                const int sc = Hq >> l;
                {
                    const int len4 = ((sc * T) >> L) / 4 + 1;
                    hs_bulk_g2s(sm + off, x + sc * q0, 16u * len4, &bar);
                    off += 4 * len4;
                }
#pragma unroll
                for (int h = 6; h < (1 << l); h += 4) {
                    const int k = h * sc;
                    const int len4 = ((k * T) >> L) / 4 + 1;
                    hs_bulk_g2s(sm + off, x + k * q0, 16u * len4, &bar);
                    off += 4 * len4;
                }
            }
        }
    } else {
        int off = 0;
        {
            constexpr int len4 = T / 4 + 1;
            hs_stage_guarded<BLOCK>(sm, off, x, n0, len4, N);
            off += 4 * len4;
        }
#pragma unroll
        for (int l = 1; l <= L; ++l) {
            const int sc = Hq >> l;
            {
                const int len4 = ((sc * T) >> L) / 4 + 1;
                hs_stage_guarded<BLOCK>(sm, off, x, sc * q0, len4, N);
                off += 4 * len4;
            }
#pragma unroll
            for (int h = 6; h < (1 << l); h += 4) {
                const int k = h * sc;
                const int len4 = ((k * T) >> L) / 4 + 1;
                hs_stage_guarded<BLOCK>(sm, off, x, k * q0, len4, N);
                off += 4 * len4;
            }
        }
    }

    // ---- per-lane span addresses (floats): off_k + ((k lane + Hq/2) >> L) + k w ----
    const int lane = threadIdx.x & 31;
    const int w = threadIdx.x >> 5;
    constexpr int NR_MAX = 17;
    int a[NR_MAX];
    {
        int off = 0, r = 0;
        a[r++] = off + lane + 32 * w;                                   // k = Hq: the index is j itself
        off += 4 * (T / 4 + 1);
#pragma unroll
        for (int l = 1; l <= L; ++l) {
            const int sc = Hq >> l;
            a[r++] = off + ((sc * lane + HALF) >> L) + sc * Q * w;
            off += 4 * (((sc * T) >> L) / 4 + 1);
#pragma unroll
            for (int h = 6; h < (1 << l); h += 4) {
                const int k = h * sc;
                a[r++] = off + ((k * lane + HALF) >> L) + k * Q * w;
                off += 4 * (((k * T) >> L) / 4 + 1);
            }
        }
    }

    if (interior) {
        // wait for the bulk copies (phase 0); the barrier init by thread 0 is ordered before by __syncthreads
        __syncthreads();
        unsigned done = 0;
        while (!done) {
            asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], 0;\n selp.u32 %0, 1, 0, p;\n}\n"
                         : "=r"(done) : "r"(hs_smem_u32(&bar)) : "memory");
        }
    } else {
        __syncthreads();
    }

    // ---- accumulate, normalise, max/argmax, store ----
    const long long orow = (long long)s * sh.out_stride;
#pragma unroll
    for (int i = 0; i < NQ / NW; ++i) {
        const int qs = NW * i;                         // q = w + qs; the k*qs part is an immediate
        int r = 0;
        float S = sm[a[r++] + 32 * qs];               // H' = 1: x[n]
        float best = hs_snr(S, st.nmis[0], st.inv_sigma[0]);
        int bh = 1;
#pragma unroll
        for (int l = 1; l <= L; ++l) {
            const int sc = Hq >> l;
            const int Hp = 1 << l;
            float add = sm[a[r++] + sc * Q * qs];         // new fundamental term h = 1
#pragma unroll
            for (int h = 6; h < Hp; h += 4) add = __fadd_rn(add, sm[a[r++] + h * sc * Q * qs]);   // h = 2 mod 4
            S = __fadd_rn(S, add);
            const float snr = hs_snr(S, st.nmis[Hp - 1], st.inv_sigma[Hp - 1]);
            if (snr > best) { best = snr; bh = Hp; }
        }
        const int n = n0 + 32 * (w + qs) + lane;
        if (n < n_fund) {
            st_cs(io.snr + orow + n, best);
            st_cs(io.best_h + orow + n, bh);
        }
    }
}
