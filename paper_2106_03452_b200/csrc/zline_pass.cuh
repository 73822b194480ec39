// zline_pass.cuh -- z (+ y) passes: real lines <-> half spectrum (F1+F2 / F4 and B2+B3 / B5 of SURVEY 8(a)),
// persistent version.  A tile is NL consecutive z-lines of one x-plane: the whole plane for N <= 128 (then the
// y transform is done in the same shared-memory trip), 32 lines for N >= 256.  On the spectrum side a tile is ONE
// contiguous chunk of HBM (NL x H complex) plus NL Nyquist values, on the real side one contiguous chunk of NL x N
// floats, so a tile is fetched with two cp.async.bulk copies that complete on an mbarrier.
//
// The tile sits DENSE in shared memory, [line][H] complex followed by the NL Nyquist values, and every stage
// works in place.  Bank conflicts are avoided not by padding (a bulk copy cannot pad) but by the column swizzle
// of the spectrum layout itself (kz_swz: slot pz of line y lives in column pz ^ (y & 15)): 16 consecutive lines
// hit 16 different 8-byte bank pairs at any fixed slot, so z-stages run "lanes over lines" and y-stages "lanes
// over slots" conflict-free in the same buffer.
//
// A CTA owns a ring of NBUF tile buffers and NG consumer groups of NTC threads; groups take alternate tiles (one
// computes while the other waits at a stage barrier or for its tile) and the thread that sees a buffer released
// refills it at once with the tile NBUF items ahead, so loads are in flight during all of the arithmetic.
//   k_zl_inv       spectrum -> real lines (F4 / B5)
//   k_zl_fwd<GBAR> G (bulk-loaded) + re-rasterised W -> Gbar' -> spectrum (B2+B3)
//   k_zl_fwd<SPLAT> points rasterised in shared memory -> spectrum (F1+F2); no loads, one buffer per group
#pragma once
#include "fft_core.cuh"
#include "zy_pass.cuh"
#include "ring_pass.cuh"

namespace sap {

template <int N> struct ZlCfg {
    static constexpr bool FUSED = (N <= 128);           // tile = whole plane, y transform fused
    static constexpr int NL = FUSED ? N : 32;
    static constexpr int NTC = (N == 512) ? 512 : 256;  // threads per consumer group
    static constexpr int NG = (N == 128 || N == 256) ? 2 : 1;
    // ring buffers (inverse and GBAR); SPLAT uses NG of them
    static constexpr int NBUF = (N == 128) ? 3 : (N == 256) ? 6 : (N == 512) ? 3 : 2;
    static constexpr int MINB = (N == 64) ? 3 : (N == 32) ? 4 : 1;
};
template <int N> constexpr int zl_threads() { return ZlCfg<N>::NTC * ZlCfg<N>::NG; }
template <int N> constexpr int zl_buf_elems() { return ZlCfg<N>::NL * (N / 2) + ZlCfg<N>::NL; }  // float2 per buffer
template <int N> constexpr size_t zl_smem_bytes() {
    return (size_t)ZlCfg<N>::NBUF * zl_buf_elems<N>() * sizeof(float2) + (size_t)N * sizeof(float2) +
           2 * ZlCfg<N>::NBUF * sizeof(uint64_t) + 128;
}

struct ZlInvParams {
    const float2* S;    // [planes][N][N][H] main spectrum (stored order, column swizzle)
    const float2* Q;    // [planes][N][N]   Nyquist plane [x][y]
    float* out;         // [planes][N^3]
    const float2* tw;   // exp(-2 pi i t / N), t < N
    int planes;
};

// plain bulk copy global -> shared, completion on an mbarrier (bytes: multiple of 16, both addresses 16-aligned)
__device__ __forceinline__ void bulk_load(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

// index of (line l, z slot pz) in a tile buffer; the Nyquist value of line l sits at NL*H + l
template <int H> __device__ __forceinline__ int zi(int l, int pz) { return l * H + (pz ^ (l & 15)); }

// ---- z stages, lanes over lines, in place ---------------------------------------------------------------
// Stage S (>= 1) of the H-point plan on NL lines: task = (line, butterfly).
template <int N, int NL, int S, bool INV, int NTC>
__device__ __forceinline__ void zl_stage_lines(float2* s, const float2* tw, int tid) {
    constexpr int H = N / 2;
    constexpr int R = StageInfo<H, S>::R, ST = StageInfo<H, S>::ST;
    constexpr int Q = H / R;
    constexpr int TWMUL = N / (R * ST);
    for (int t = tid; t < NL * Q; t += NTC) {
        const int q = t / NL, l = t - q * NL;
        const int blk = q / ST, j = q - blk * ST;
        const int e0 = blk * (R * ST) + j;
        float2 v[R];
#pragma unroll
        for (int r = 0; r < R; ++r) v[r] = s[zi<H>(l, e0 + r * ST)];
        if (!INV) {
            dft_fwd<R>(v);
            if (ST > 1) {
#pragma unroll
                for (int r = 1; r < R; ++r) v[r] = cmul(v[r], tw[r * j * TWMUL]);
            }
        } else {
            if (ST > 1) {
#pragma unroll
                for (int r = 1; r < R; ++r) v[r] = cmulc(v[r], tw[r * j * TWMUL]);
            }
            dft_inv<R>(v);
        }
#pragma unroll
        for (int r = 0; r < R; ++r) s[zi<H>(l, e0 + r * ST)] = v[r];
    }
}

// Hermitian split of NL lines in place (N >= 256 tiles; the fused planes do it inside the first y stage).
// FWD: slot pos(k) holds Z[k] -> X[k], Nyquist value X[H] written to the tile's Nyquist array.  INV: the reverse.
template <int N, int NL, bool INV, int NTC>
__device__ __forceinline__ void zl_split(float2* s, const float2* tw, int tid) {
    constexpr int H = N / 2;
    for (int t = tid; t < NL * (H / 2 + 1); t += NTC) {
        const int k = t / NL, l = t - k * NL;
        if (k == 0) {
            float2* p0 = s + zi<H>(l, 0);
            float2* pn = s + NL * H + l;
            if (!INV) {
                const float2 z = *p0;
                *p0 = make_float2(z.x + z.y, 0.f);
                *pn = make_float2(z.x - z.y, 0.f);
            } else {
                const float x0 = p0->x, xh = pn->x;
                *p0 = make_float2(0.5f * (x0 + xh), 0.5f * (x0 - xh));
            }
        } else if (k == H / 2) {
            float2* pa = s + zi<H>(l, freq2pos<H>(k));
            const float2 z = *pa;
            *pa = make_float2(z.x, -z.y);
        } else {
            float2* pa = s + zi<H>(l, freq2pos<H>(k));
            float2* pb = s + zi<H>(l, freq2pos<H>(H - k));
            float2 a = *pa, b = *pb;
            if (!INV) r2c_pair(a, b, tw[k]); else c2r_pair(a, b, tw[k]);
            *pa = a;
            *pb = b;
        }
    }
}

}  // namespace sap

namespace sap {

// ring bookkeeping shared by the inverse and the GBAR kernels: item `it` of this CTA is tile blockIdx.x + it * gridDim.x
// and lives in buffer it % NBUF (same protocol as k_ring, one item per tile)
template <int N>
struct ZlRing {
    using C = ZlCfg<N>;
    static constexpr int H = N / 2, NL = C::NL, NBUF = C::NBUF, NTC = C::NTC, BUF = zl_buf_elems<N>();
    float2* bufs;
    uint64_t* full;
    uint64_t* empty;
    long long total;
    const float2* srcS;  // tile g: NL*H complex at srcS + g*NL*H
    const float2* srcQ;  // tile g: NL complex at srcQ + g*NL
    __device__ __forceinline__ void init() const {
        if (threadIdx.x == 0) {
            for (int s = 0; s < NBUF; ++s) { mbar_init(full + s, 1); mbar_init(empty + s, NTC / 32); }
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        }
    }
    __device__ __forceinline__ void issue_load(int it) const {
        const long long g = (long long)blockIdx.x + (long long)it * gridDim.x;
        if (g >= total) return;
        const int s = it % NBUF;
        float2* b = bufs + (size_t)s * BUF;
        mbar_expect_tx(full + s, (uint32_t)(BUF * sizeof(float2)));
        bulk_load(b, srcS + (size_t)g * NL * H, NL * H * sizeof(float2), full + s);
        bulk_load(b + NL * H, srcQ + (size_t)g * NL, NL * sizeof(float2), full + s);
    }
    __device__ __forceinline__ float2* acquire(int it) const {
        const int s = it % NBUF;
        mbar_wait(full + s, (it / NBUF) & 1);
        return bufs + (size_t)s * BUF;
    }
    // tid = thread index inside the consumer group
    __device__ __forceinline__ void release(int it, int tid) const {
        const int s = it % NBUF;
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncwarp();
        if ((tid & 31) == 0) mbar_arrive(empty + s);
        if (tid == 0) {
            mbar_wait(empty + s, (it / NBUF) & 1);
            issue_load(it + NBUF);
        }
    }
};

// ---- inverse: spectrum tile -> real lines ---------------------------------------------------------------------
template <int N>
__global__ void __launch_bounds__(zl_threads<N>(), ZlCfg<N>::MINB) k_zl_inv(const ZlInvParams p) {
    using C = ZlCfg<N>;
    constexpr int H = N / 2, NL = C::NL, NTC = C::NTC, NG = C::NG, NBUF = C::NBUF, BUF = zl_buf_elems<N>();
    constexpr bool FUSED = C::FUSED;
    constexpr int R0 = StageInfo<H, 0>::R, ST0 = StageInfo<H, 0>::ST;
    static_assert(Plan<H>::NS <= 2 && ST0 <= 16, "z plans have at most two stages");
    extern __shared__ __align__(1024) unsigned char zl_smem[];
    ZlRing<N> ring;
    ring.bufs = reinterpret_cast<float2*>(zl_smem);
    float2* tw = ring.bufs + (size_t)NBUF * BUF;
    ring.full = reinterpret_cast<uint64_t*>(tw + N);
    ring.empty = ring.full + NBUF;
    ring.total = (long long)p.planes * (N * N / NL);
    ring.srcS = p.S;
    ring.srcQ = p.Q;
    const int group = threadIdx.x / NTC, tid = threadIdx.x - group * NTC;
    for (int i = threadIdx.x; i < N; i += zl_threads<N>()) tw[i] = p.tw[i];
    ring.init();
    __syncthreads();
    pdl_wait();
    if (threadIdx.x == 0) {
#pragma unroll 1
        for (int it = 0; it < NBUF; ++it) ring.issue_load(it);
    }
    for (long long j = group, g = blockIdx.x + (long long)group * gridDim.x; g < ring.total; j += NG, g += (long long)NG * gridDim.x) {
        float2* s = ring.acquire((int)j);
        if constexpr (FUSED) {
            static_assert(!FUSED || Plan<N>::NS == 2, "fused planes use two-stage y plans");
            // D': inverse of the last y stage, lanes over z slots
            constexpr int R1 = StageInfo<N, 1>::R;
            for (int t = tid; t < H * (N / R1); t += NTC) {
                const int blk = t / H, pz = t - blk * H;
                float2 v[R1];
#pragma unroll
                for (int r = 0; r < R1; ++r) v[r] = s[zi<H>(blk * R1 + r, pz)];
                dft_inv<R1>(v);
#pragma unroll
                for (int r = 0; r < R1; ++r) s[zi<H>(blk * R1 + r, pz)] = v[r];
            }
            for (int blk = tid; blk < N / R1; blk += NTC) {
                float2 v[R1];
#pragma unroll
                for (int r = 0; r < R1; ++r) v[r] = s[NL * H + blk * R1 + r];
                dft_inv<R1>(v);
#pragma unroll
                for (int r = 0; r < R1; ++r) s[NL * H + blk * R1 + r] = v[r];
            }
            consumer_sync<NTC>(group);
            // C': inverse y stage 0 on the slot pair (k, H-k), then the c2r split, in registers
            constexpr int RY = StageInfo<N, 0>::R, STY = StageInfo<N, 0>::ST;
            for (int t = tid; t < (H / 2 + 1) * STY; t += NTC) {
                const int k = t / STY, q = t - k * STY;
                float2 a[RY], b[RY];
                const int ra = (k == 0) ? 0 : freq2pos<H>(k);
                const int rb = (k == 0) ? H : freq2pos<H>(H - k);
#pragma unroll
                for (int r = 0; r < RY; ++r) a[r] = s[zi<H>(q + STY * r, ra)];
                bfly_inv<N, 0, N>(a, q, tw);
                if (rb != ra) {
#pragma unroll
                    for (int r = 0; r < RY; ++r) b[r] = (k == 0) ? s[NL * H + q + STY * r] : s[zi<H>(q + STY * r, rb)];
                    bfly_inv<N, 0, N>(b, q, tw);
                }
                if (k == 0) {
#pragma unroll
                    for (int r = 0; r < RY; ++r)
                        s[zi<H>(q + STY * r, 0)] = make_float2(0.5f * (a[r].x + b[r].x), 0.5f * (a[r].x - b[r].x));
                } else if (k == H / 2) {
#pragma unroll
                    for (int r = 0; r < RY; ++r) s[zi<H>(q + STY * r, ra)] = make_float2(a[r].x, -a[r].y);
                } else {
                    const float2 w = tw[k];
#pragma unroll
                    for (int r = 0; r < RY; ++r) {
                        c2r_pair(a[r], b[r], w);
                        s[zi<H>(q + STY * r, ra)] = a[r];
                        s[zi<H>(q + STY * r, rb)] = b[r];
                    }
                }
            }
            consumer_sync<NTC>(group);
        } else {
            zl_split<N, NL, true, NTC>(s, tw, tid);
            consumer_sync<NTC>(group);
        }
        if constexpr (Plan<H>::NS == 2) {
            zl_stage_lines<N, NL, 1, true, NTC>(s, tw, tid);
            consumer_sync<NTC>(group);
        }
        // A': inverse z stage 0, smem -> registers -> HBM (ST0 consecutive complex = 2 ST0 reals per line and lane group)
        float2* out2 = reinterpret_cast<float2*>(p.out) + (size_t)g * NL * H;
        for (int t = tid; t < NL * ST0; t += NTC) {
            int l, q;
            zline_task<ST0>(t, l, q);
            float2 v[R0];
#pragma unroll
            for (int r = 0; r < R0; ++r) v[r] = s[zi<H>(l, q + ST0 * r)];
            bfly_inv<H, 0, N>(v, q, tw);
#pragma unroll
            for (int r = 0; r < R0; ++r) out2[l * H + q + ST0 * r] = v[r];
        }
        ring.release((int)j, tid);
    }
}

}  // namespace sap
