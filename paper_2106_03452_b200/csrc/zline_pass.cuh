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
//   k_zl_inv   spectrum -> real lines (F4 / B5), every N
//   k_zl_gbar  G (bulk-loaded) + re-rasterised W -> Gbar' -> spectrum (B2+B3), fused planes (N <= 128)
// The splat pass (F1+F2) and the N >= 256 Gbar' pass stay one-tile-per-CTA kernels (zy_pass.cuh): they have little
// or nothing to prefetch and measured faster with 3-4 small CTAs per SM than as a persistent ring.
#pragma once
#include "fft_core.cuh"
#include "zy_pass.cuh"
#include "ring_pass.cuh"

namespace sap {

// INV: the inverse kernel (its tile size is free); the forward kernels tile the lines like the point bins (NL = 32)
template <int N, bool INV> struct ZlCfg {
    static constexpr bool FUSED = (N <= 128);           // tile = whole plane, y transform fused
    static constexpr int NL = FUSED ? N : (N == 512 && INV) ? 16 : 32;
    static constexpr int NTC = (N == 512 && !INV) ? 512 : 256;  // threads per consumer group
    static constexpr int NG = (N == 128 || N == 256 || (N == 512 && INV)) ? 2 : 1;
    static constexpr int NBUF = (N == 128) ? 3 : (N == 256) ? 6 : (N == 512) ? (INV ? 6 : 3) : 2;  // ring buffers
    static constexpr int MINB = (N == 64) ? 3 : (N == 32) ? 4 : 1;
};
template <int N, bool INV> constexpr int zl_threads() { return ZlCfg<N, INV>::NTC * ZlCfg<N, INV>::NG; }
template <int N, bool INV> constexpr int zl_buf_elems() { return ZlCfg<N, INV>::NL * (N / 2) + ZlCfg<N, INV>::NL; }  // float2 per buffer
template <int N, bool INV> constexpr size_t zl_smem_bytes() {
    return (size_t)ZlCfg<N, INV>::NBUF * zl_buf_elems<N, INV>() * sizeof(float2) + (size_t)N * sizeof(float2) +
           3 * ZlCfg<N, INV>::NBUF * sizeof(uint64_t) + (size_t)(N + N / 2 + 4) * sizeof(float) + 128 +
           (INV ? (size_t)zl_threads<N, INV>() * sizeof(int) : 0);   // tile ids of this CTA (listed mode of k_zl_inv)
}

static_assert(zl_smem_bytes<128, true>() <= SMEM_PER_CTA_MAX && zl_smem_bytes<256, true>() <= SMEM_PER_CTA_MAX &&
              zl_smem_bytes<512, true>() <= SMEM_PER_CTA_MAX && zl_smem_bytes<128, false>() <= SMEM_PER_CTA_MAX,
              "tile ring must fit the shared memory of an SM");

struct ZlInvParams {
    const float2* S;    // [planes][N][N][H] main spectrum (stored order, column swizzle)
    const float2* Q;    // [planes][N][N]   Nyquist plane [x][y]
    float* out;         // [planes][N^3]
    const float2* tw;   // exp(-2 pi i t / N), t < N
    int planes;
    // adjoint mode of the fused planes (N <= 128): per item the spectra are (x channel, B, -) and the three output
    // planes are IFFT(plane 0), IFFT(h_y B), IFFT(h_z B): plane 2 is made from plane 1 (fetched again: an L2 hit)
    int adj3;
    const float4* ftab; // per-slot frequency table (spectral.cuh), used in adjoint mode
    // listed mode (the three vbar planes of the backward; see ActLists in sap_dpsr.cu), nullptr = every tile: only the tiles
    // a point can touch are transformed -- the gather (B6) reads nothing else
    const int* zlist;   // ids item * nbins + bin of the active bin tiles (bin = x * NTY + ty, 32 lines for N >= 256, a plane below)
    const int* nact;    // {|zlist|, -, -, -}
    int nbins, nty;
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

// Inverse Hermitian split fused with the inverse of the last z stage (two-stage plans H = R0 x R1, N >= 256 tiles).
// Stored slot p = k0 R1 + k1 holds frequency k = k0 + R0 k1, and H - k sits in block R0 - k0 at index R1 - 1 - k1
// (block 0: index R1 - k1), so the partner of a whole block is one other block: a task loads the block pair
// (k0, R0 - k0), turns X[k], X[H-k] into Z[k], Z[H-k] in registers (c2r_pair) and runs the two R1-point inverse
// butterflies -- one shared-memory round trip and the per-pair index arithmetic of zl_split less.
template <int N, int NL, int NTC>
__device__ __forceinline__ void zl_inv_split_stage1(float2* s, const float2* tw, int tid) {
    constexpr int H = N / 2;
    constexpr int R0 = StageInfo<H, 0>::R, R1 = StageInfo<H, 1>::R;
    static_assert(Plan<H>::NS == 2 && StageInfo<H, 1>::ST == 1 && R0 % 2 == 0 && R1 % 2 == 0, "two-stage z plan");
    constexpr int NTYPE = R0 / 2 + 1;  // block 0, block R0/2, and the pairs (k0, R0 - k0), 1 <= k0 < R0/2
    for (int t = tid; t < NL * NTYPE; t += NTC) {
        const int u = t / NL, l = t - u * NL;
        float2 a[R1];
        if (u == 0) {
            // block 0: k = R0 k1.  k1 = 0 pairs with the Nyquist value, k1 = R1/2 (k = H/2) with itself
#pragma unroll
            for (int i = 0; i < R1; ++i) a[i] = s[zi<H>(l, i)];
            const float xh = s[NL * H + l].x;
            a[0] = make_float2(0.5f * (a[0].x + xh), 0.5f * (a[0].x - xh));
            a[R1 / 2] = make_float2(a[R1 / 2].x, -a[R1 / 2].y);
#pragma unroll
            for (int i = 1; i < R1 / 2; ++i) c2r_pair(a[i], a[R1 - i], tw[R0 * i]);
            dft_inv<R1>(a);
#pragma unroll
            for (int i = 0; i < R1; ++i) s[zi<H>(l, i)] = a[i];
        } else if (u == 1) {
            // block R0/2: k = R0/2 + R0 k1 pairs with index R1 - 1 - k1 of the same block
            constexpr int B0 = (R0 / 2) * R1;
#pragma unroll
            for (int i = 0; i < R1; ++i) a[i] = s[zi<H>(l, B0 + i)];
#pragma unroll
            for (int i = 0; i < R1 / 2; ++i) c2r_pair(a[i], a[R1 - 1 - i], tw[R0 / 2 + R0 * i]);
            dft_inv<R1>(a);
#pragma unroll
            for (int i = 0; i < R1; ++i) s[zi<H>(l, B0 + i)] = a[i];
        } else {
            const int k0 = u - 1;  // 1 .. R0/2 - 1
            const int ba = k0 * R1, bb = (R0 - k0) * R1;
            float2 b[R1];
#pragma unroll
            for (int i = 0; i < R1; ++i) { a[i] = s[zi<H>(l, ba + i)]; b[i] = s[zi<H>(l, bb + i)]; }
#pragma unroll
            for (int i = 0; i < R1; ++i) c2r_pair(a[i], b[R1 - 1 - i], tw[k0 + R0 * i]);
            dft_inv<R1>(a);
            dft_inv<R1>(b);
#pragma unroll
            for (int i = 0; i < R1; ++i) { s[zi<H>(l, ba + i)] = a[i]; s[zi<H>(l, bb + i)] = b[i]; }
        }
    }
}

}  // namespace sap

namespace sap {

// ring bookkeeping shared by the inverse and the GBAR kernels: item `it` of this CTA is tile blockIdx.x + it * gridDim.x
// and lives in buffer it % NBUF (same protocol as k_ring, one item per tile)
template <int N, bool INV>
struct ZlRing {
    using C = ZlCfg<N, INV>;
    static constexpr int H = N / 2, NL = C::NL, NBUF = C::NBUF, NTC = C::NTC, BUF = zl_buf_elems<N, INV>();
    float2* bufs;
    uint64_t* full;
    uint64_t* empty;
    volatile int* issued;  // fills issued into each buffer so far (see k_ring's acquire)
    long long total;
    const float2* srcS;  // tile g: NL*H complex at srcS + g*NL*H
    const float2* srcQ;  // tile g: NL complex at srcQ + g*NL (nullptr: the tile has no Nyquist part, GBAR input)
    int adj3;            // fused adjoint planes: the tiles of plane 3i+2 are fetched from plane 3i+1
    const int* tcache = nullptr;   // listed mode: tile ids of this CTA (shared memory, TCAP entries), else nullptr
    const int* zlist = nullptr;
    int nbins = 0, nty = 1;
    static constexpr int TCAP = ZlCfg<N, INV>::NTC * ZlCfg<N, INV>::NG;
    // listed mode: virtual tile v -> (active bin tile v / (3 SUB), channel, sub-tile) -> dense tile id
    __device__ __forceinline__ long long expand(long long v) const {
        constexpr int SUB = (N <= 128) ? 1 : 32 / NL, TPP = 2 * H * 2 * H / NL;
        const long long e = v / (3 * SUB);
        const int r = (int)(v - e * (3 * SUB)), ch = r / SUB, sub = r - ch * SUB;
        const int id = zlist[e], item = id / nbins, bin = id - item * nbins;
        const int x = bin / nty, ty = bin - x * nty;
        const int tile = (N <= 128) ? x : (x * (2 * H) + ty * 32) / NL + sub;
        return ((long long)item * 3 + ch) * TPP + tile;
    }
    // it-th tile of this CTA (dense tile id), -1 past the end
    __device__ __forceinline__ long long tile_at(int it) const {
        long long v = (long long)blockIdx.x + (long long)it * gridDim.x;
        if (v >= total) return -1;
        // N = 256, inverse (at 512^3 a spectrum is four times the L2: measured no gain): the y pass before this kernel wrote the planes in ascending x; walk them in descending x so
        // that the planes still in L2 are read first
        if (INV && N == 256) v = total - 1 - v;
        if (zlist) return it < TCAP ? (long long)tcache[it] : expand(v);   // (v already reversed above)
        return v;
    }
    __device__ __forceinline__ void init() const {
        if (threadIdx.x == 0) {
            for (int s = 0; s < NBUF; ++s) { mbar_init(full + s, 1); mbar_init(empty + s, NTC / 32); issued[s] = 0; }
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        }
    }
    __device__ __forceinline__ void issue_load(int it) const {
        long long g = tile_at(it);
        if (g < 0) return;
        if (adj3) {
            constexpr int TPP = 2 * H * 2 * H / NL;  // tiles per plane
            if ((g / TPP) % 3 == 2) g -= TPP;
        }
        const int s = it % NBUF;
        float2* b = bufs + (size_t)s * BUF;
        mbar_expect_tx(full + s, (uint32_t)((srcQ ? BUF : NL * H) * sizeof(float2)));
        issued[s] = it / NBUF + 1;
        bulk_load(b, srcS + (size_t)g * NL * H, NL * H * sizeof(float2), full + s);
        if (srcQ) bulk_load(b + NL * H, srcQ + (size_t)g * NL, NL * sizeof(float2), full + s);
    }
    __device__ __forceinline__ float2* acquire(int it) const {
        const int s = it % NBUF;
        while (issued[s] <= it / NBUF) {}  // the fill must be under way before its phase parity means anything
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
        __syncwarp();
    }
};

// ---- inverse: spectrum tile -> real lines ---------------------------------------------------------------------
template <int N>
__global__ void __launch_bounds__(zl_threads<N, true>(), ZlCfg<N, true>::MINB) k_zl_inv(const ZlInvParams p) {
    using C = ZlCfg<N, true>;
    constexpr int H = N / 2, NL = C::NL, NTC = C::NTC, NG = C::NG, NBUF = C::NBUF, BUF = zl_buf_elems<N, true>();
    constexpr bool FUSED = C::FUSED;
    constexpr int R0 = StageInfo<H, 0>::R, ST0 = StageInfo<H, 0>::ST;
    static_assert(Plan<H>::NS <= 2 && ST0 <= 16 && (NL % 32 == 0 || ST0 == 16), "z plans have at most two stages; line-group mapping");
    extern __shared__ __align__(1024) unsigned char zl_smem[];
    ZlRing<N, true> ring;
    ring.bufs = reinterpret_cast<float2*>(zl_smem);
    float2* tw = ring.bufs + (size_t)NBUF * BUF;
    ring.full = reinterpret_cast<uint64_t*>(tw + N);
    ring.empty = ring.full + NBUF;
    ring.issued = reinterpret_cast<volatile int*>(ring.empty + NBUF);
    ring.total = (long long)p.planes * (N * N / NL);
    ring.srcS = p.S;
    ring.srcQ = p.Q;
    ring.adj3 = FUSED ? p.adj3 : 0;
    float* fy = reinterpret_cast<float*>(const_cast<int*>(ring.issued + NBUF));  // h_y per y slot, h_z per z slot (+ Nyquist)
    float* fz = fy + N;
    int* tcache = reinterpret_cast<int*>(fz + H + 4);
    const int group = threadIdx.x / NTC, tid = threadIdx.x - group * NTC;
    for (int i = threadIdx.x; i < N; i += zl_threads<N, true>()) tw[i] = p.tw[i];
    if (FUSED && p.adj3) {
        for (int i = threadIdx.x; i < N; i += zl_threads<N, true>()) fy[i] = p.ftab[i].x;
        for (int i = threadIdx.x; i <= H; i += zl_threads<N, true>()) fz[i] = p.ftab[N + i].x;
    }
    ring.init();
    __syncthreads();
    pdl_wait();
    if (p.zlist) {   // listed mode: the tiles of this CTA are entries blockIdx.x + it * gridDim.x of the expanded active list
        constexpr int SUB = (N <= 128) ? 1 : 32 / NL;
        ring.zlist = p.zlist; ring.nbins = p.nbins; ring.nty = p.nty;
        ring.total = (long long)p.nact[0] * 3 * SUB;
        const long long v = (long long)blockIdx.x + (long long)threadIdx.x * gridDim.x;
        tcache[threadIdx.x] = v < ring.total ? (int)ring.expand(N == 256 ? ring.total - 1 - v : v) : -1;
        ring.tcache = tcache;
        __syncthreads();
    }
    if (threadIdx.x == 0) {
#pragma unroll 1
        for (int it = 0; it < NBUF; ++it) ring.issue_load(it);
    }
    for (long long j = group;; j += NG) {
        const long long g = ring.tile_at((int)j);
        if (g < 0) break;
        float2* s = ring.acquire((int)j);
        if constexpr (FUSED) {
            static_assert(!FUSED || Plan<N>::NS == 2, "fused planes use two-stage y plans");
            // D': inverse of the last y stage, lanes over z slots
            constexpr int R1 = StageInfo<N, 1>::R;
            const int ch = p.adj3 ? (int)((g / (N * N / NL)) % 3) : 0;  // adjoint mode: 1 = h_y on the way in, 2 = h_z
            for (int t = tid; t < H * (N / R1); t += NTC) {
                const int blk = t / H, pz = t - blk * H;
                float2 v[R1];
#pragma unroll
                for (int r = 0; r < R1; ++r) v[r] = s[zi<H>(blk * R1 + r, pz)];
                if (ch == 1) {
#pragma unroll
                    for (int r = 0; r < R1; ++r) v[r] = cscale(fy[blk * R1 + r], v[r]);
                } else if (ch == 2) {
                    const float w = fz[pz];
#pragma unroll
                    for (int r = 0; r < R1; ++r) v[r] = cscale(w, v[r]);
                }
                dft_inv<R1>(v);
#pragma unroll
                for (int r = 0; r < R1; ++r) s[zi<H>(blk * R1 + r, pz)] = v[r];
            }
            for (int blk = tid; blk < N / R1; blk += NTC) {
                float2 v[R1];
#pragma unroll
                for (int r = 0; r < R1; ++r) v[r] = s[NL * H + blk * R1 + r];
                if (ch == 1) {
#pragma unroll
                    for (int r = 0; r < R1; ++r) v[r] = cscale(fy[blk * R1 + r], v[r]);
                } else if (ch == 2) {
#pragma unroll
                    for (int r = 0; r < R1; ++r) v[r] = cscale(fz[H], v[r]);  // h_z = 0 on the Nyquist plane (R3)
                }
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
        }
        if constexpr (!FUSED) {
            zl_inv_split_stage1<N, NL, NTC>(s, tw, tid);  // c2r split + inverse of the last z stage in one pass
            consumer_sync<NTC>(group);
        } else if constexpr (Plan<H>::NS == 2) {
            zl_stage_lines<N, NL, 1, true, NTC>(s, tw, tid);
            consumer_sync<NTC>(group);
        }
        // A': inverse z stage 0, smem -> registers -> HBM (ST0 consecutive complex = 2 ST0 reals per line and lane group)
        float2* out2 = reinterpret_cast<float2*>(p.out) + (size_t)g * NL * H;
        for (int t = tid; t < NL * ST0; t += NTC) {
            int l, q;
            if constexpr (ST0 == 16) { l = t >> 4; q = t & 15; }  // 16 consecutive complex of a line per half-warp
            else zline_task<ST0>(t, l, q);
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

namespace sap {

// ---- forward: real lines -> spectrum tile ----------------------------------------------------------------------
// B2+B3: G is bulk-loaded into the tile, W = sum_i w is rasterised on top of it from the binned points (same
// weights as the splat, Eq.10-11) scaled by (beta/P)/s, and the first stage multiplies by s:
//   Gbar' = s (G + ((beta/P)/s) W) - (S1/a) delta_0.
struct ZlFwdParams {
    ZyFwdParams z;   // points, bins, G, bw, S, Q (N <= 128: [x][y]; N >= 256: transposed [y][x]), tw, nch
    int planes;      // batch * nch
};

template <int N>
__global__ void __launch_bounds__(zl_threads<N, false>(), ZlCfg<N, false>::MINB) k_zl_gbar(const ZlFwdParams pp) {
    using C = ZlCfg<N, false>;
    constexpr int H = N / 2, NL = C::NL, NTC = C::NTC, NG = C::NG, BUF = zl_buf_elems<N, false>();
    constexpr int NBUF = C::NBUF;
    constexpr bool FUSED = C::FUSED;
    constexpr int R0 = StageInfo<H, 0>::R, ST0 = StageInfo<H, 0>::ST;
    constexpr int TPP = N * N / NL;  // tiles per plane
    constexpr int NTY = N / NL, NBINS = N * NTY, M = N - 1;
    static_assert(Plan<H>::NS <= 2 && ST0 <= 16 && (NL * ST0) % 32 == 0, "z plan / line-group mapping");
    const ZyFwdParams& p = pp.z;
    extern __shared__ __align__(1024) unsigned char zl_smem[];
    ZlRing<N, false> ring;
    ring.bufs = reinterpret_cast<float2*>(zl_smem);
    float2* tw = ring.bufs + (size_t)C::NBUF * BUF;
    ring.full = reinterpret_cast<uint64_t*>(tw + N);
    ring.empty = ring.full + C::NBUF;
    ring.issued = reinterpret_cast<volatile int*>(ring.empty + C::NBUF);
    ring.total = (long long)pp.planes * TPP;
    ring.srcS = reinterpret_cast<const float2*>(p.G);  // GBAR: tile g = NL*N floats = NL*H float2 at G + g*NL*N
    ring.srcQ = nullptr;
    ring.adj3 = 0;
    const int group = threadIdx.x / NTC, tid = threadIdx.x - group * NTC;
    for (int i = threadIdx.x; i < N; i += zl_threads<N, false>()) tw[i] = p.tw[i];
    ring.init();
    __syncthreads();
    pdl_wait();
    if (threadIdx.x == 0) {
#pragma unroll 1
        for (int it = 0; it < NBUF; ++it) ring.issue_load(it);
    }
    for (long long j = group, g = blockIdx.x + (long long)group * gridDim.x; g < ring.total; j += NG, g += (long long)NG * gridDim.x) {
        const int by = (int)(g / TPP), bx = (int)(g - (long long)by * TPP);
        const int item = by / p.nch;
        const int line0 = bx * NL, x = line0 / N, y0 = line0 - x * N, ty = y0 / NL;
        float2* So = p.S + (size_t)g * NL * H;
        // A0: bins that can touch lines [line0, line0 + NL): x-slabs {x, x-1} x y-tiles {ty, ty-1}
        const int* bs = p.bin_start + (size_t)item * (NBINS + 1);
        int b_lo[4], b_n[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const int xb = (k & 1) ? ((x - 1) & M) : x;
            const int tb = (k & 2) ? ((ty + NTY - 1) % NTY) : ty;
            const bool use = (NTY > 1) || !(k & 2);
            const int bin = xb * NTY + tb;
            b_lo[k] = use ? bs[bin] : 0;
            b_n[k] = use ? bs[bin + 1] - b_lo[k] : 0;
        }
        float2* s = ring.acquire((int)j);
        // A1: rasterise the points of the bins into the tile, natural order: float (l, z) at l*N + z
        const float gs = p.bw[item * 4 + 0], wscale = p.bw[item * 4 + 1] / gs, gc0 = p.bw[item * 4 + 2];
        {
            float* sf = reinterpret_cast<float*>(s);
            const float4* sp = p.spts + (size_t)item * p.P;
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                for (int i = b_lo[k] + tid; i < b_lo[k] + b_n[k]; i += NTC) {
                    const float4 c = sp[i];
                    const float val = wscale;
                    const float tx = c.x * (float)N, tyf = c.y * (float)N, tz = c.z * (float)N;
                    const float fx0 = floorf(tx), fy0 = floorf(tyf), fz0 = floorf(tz);
                    const int jx = (int)fx0, jy = (int)fy0, jz = (int)fz0;
                    const float fx = tx - fx0, fy = tyf - fy0, fz = tz - fz0;
#pragma unroll
                    for (int dx = 0; dx < 2; ++dx) {
                        if (((jx + dx) & M) != x) continue;
                        const float wx = (dx ? fx : 1.f - fx) * val;
#pragma unroll
                        for (int dy = 0; dy < 2; ++dy) {
                            const int ly = ((jy + dy) & M) - y0;
                            if ((unsigned)ly >= (unsigned)NL) continue;
                            const float wxy = wx * (dy ? fy : 1.f - fy);
#pragma unroll
                            for (int dz = 0; dz < 2; ++dz)
                                atomicAdd(sf + ly * N + ((jz + dz) & M), wxy * (dz ? fz : 1.f - fz));
                        }
                    }
                }
            }
        }
        consumer_sync<NTC>(group);
        // A2: z stage 0.  Reads the natural-order line, writes the swizzled slots: the ST0 butterflies of a line sit
        // in one warp (zline_task), so a __syncwarp between its loads and its stores is all the ordering needed.
        for (int t = tid; t < NL * ST0; t += NTC) {
            int l, q;
            zline_task<ST0>(t, l, q);
            float2 v[R0];
#pragma unroll
            for (int r = 0; r < R0; ++r) {
                float2 xv = cscale(gs, s[l * H + q + ST0 * r]);
                if (line0 == 0 && l == 0 && q == 0 && r == 0) xv.x -= gc0;
                v[r] = xv;
            }
            __syncwarp();
            bfly_fwd<H, 0, N>(v, q, tw);
#pragma unroll
            for (int r = 0; r < R0; ++r) s[zi<H>(l, q + ST0 * r)] = v[r];
        }
        consumer_sync<NTC>(group);
        if constexpr (Plan<H>::NS == 2) {
            zl_stage_lines<N, NL, 1, false, NTC>(s, tw, tid);
            consumer_sync<NTC>(group);
        }
        if constexpr (!FUSED) {
            // C: Hermitian split in place, then the tile IS the HBM chunk: straight 16-byte copy out
            zl_split<N, NL, false, NTC>(s, tw, tid);
            consumer_sync<NTC>(group);
            const float4* s4 = reinterpret_cast<const float4*>(s);
            float4* So4 = reinterpret_cast<float4*>(So);
            for (int i = tid; i < NL * H / 2; i += NTC) So4[i] = s4[i];
            float2* Qt = p.Q + (size_t)by * ((size_t)N * N);  // transposed Nyquist plane [y][x]
            for (int l = tid; l < NL; l += NTC) Qt[(size_t)(y0 + l) * N + x] = s[NL * H + l];
        } else {
            static_assert(!FUSED || Plan<N>::NS == 2, "fused planes use two-stage y plans");
            // C: r2c split fused into y stage 0.  One task owns the slot pair (k, H-k) for RY y-values.
            constexpr int RY = StageInfo<N, 0>::R, STY = StageInfo<N, 0>::ST;
            for (int t = tid; t < (H / 2 + 1) * STY; t += NTC) {
                const int k = t / STY, q = t - k * STY;
                float2 a[RY], b[RY];
                int ra, rb;
                if (k == 0) {
                    ra = 0; rb = H;
#pragma unroll
                    for (int r = 0; r < RY; ++r) {
                        const float2 z = s[zi<H>(q + STY * r, 0)];
                        a[r] = make_float2(z.x + z.y, 0.f);
                        b[r] = make_float2(z.x - z.y, 0.f);
                    }
                } else if (k == H / 2) {
                    ra = rb = freq2pos<H>(k);
#pragma unroll
                    for (int r = 0; r < RY; ++r) {
                        const float2 z = s[zi<H>(q + STY * r, ra)];
                        a[r] = make_float2(z.x, -z.y);
                        b[r] = a[r];
                    }
                } else {
                    ra = freq2pos<H>(k); rb = freq2pos<H>(H - k);
                    const float2 w = tw[k];
#pragma unroll
                    for (int r = 0; r < RY; ++r) {
                        a[r] = s[zi<H>(q + STY * r, ra)];
                        b[r] = s[zi<H>(q + STY * r, rb)];
                        r2c_pair(a[r], b[r], w);
                    }
                }
                bfly_fwd<N, 0, N>(a, q, tw);
#pragma unroll
                for (int r = 0; r < RY; ++r) s[zi<H>(q + STY * r, ra)] = a[r];
                if (rb != ra) {
                    bfly_fwd<N, 0, N>(b, q, tw);
#pragma unroll
                    for (int r = 0; r < RY; ++r) {
                        if (k == 0) s[NL * H + q + STY * r] = b[r];
                        else s[zi<H>(q + STY * r, rb)] = b[r];
                    }
                }
            }
            consumer_sync<NTC>(group);
            // D: last y stage smem -> registers -> HBM; lanes over z slots (the stored column of slot pz in row y is
            // exactly its shared-memory column)
            constexpr int R1 = StageInfo<N, 1>::R;
            static_assert(StageInfo<N, 1>::ST == 1, "last stage");
            for (int t = tid; t < H * (N / R1); t += NTC) {
                const int blk = t / H, pz = t - blk * H;
                float2 v[R1];
#pragma unroll
                for (int r = 0; r < R1; ++r) v[r] = s[zi<H>(blk * R1 + r, pz)];
                dft_fwd<R1>(v);
#pragma unroll
                for (int r = 0; r < R1; ++r) So[zi<H>(blk * R1 + r, pz)] = v[r];
            }
            float2* Qo = p.Q + (size_t)by * ((size_t)N * N) + line0;
            for (int blk = tid; blk < N / R1; blk += NTC) {
                float2 v[R1];
#pragma unroll
                for (int r = 0; r < R1; ++r) v[r] = s[NL * H + blk * R1 + r];
                dft_fwd<R1>(v);
#pragma unroll
                for (int r = 0; r < R1; ++r) Qo[blk * R1 + r] = v[r];
            }
        }
        ring.release((int)j, tid);
    }
}

}  // namespace sap
