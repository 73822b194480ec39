// sap_dpsr.cu -- the C-ABI library of the B200-native DPSR layer (include/sap_dpsr.h).
// Kernels: splat (F1), z/y/x FFT passes with the fused spectral solve (F2-F4, B3-B5), normalisation
// (F5), grid reductions (B1), Gbar' assembly fused into the first backward pass (B2), gather (B6).
// Step names F1..B6: SURVEY.md 8(a).  No cuFFT, no CPU fallback.
#include <cuda_runtime.h>
#include <math.h>
#include <stdio.h>
#include <string.h>
#include <stdlib.h>
#include <new>
#include <string>

#include "../../include/sap_dpsr.h"
#include "dpsr_kernels.cuh"
#include "fused_small.cuh"

namespace sap {

struct DevCtx {
    int tid, nthr;
    __device__ __forceinline__ void sync() const { __syncthreads(); }
    __device__ __forceinline__ void atomic_add(float* p, float v) const { atomicAdd(p, v); }
    __device__ __forceinline__ void atomic_add(int* p, int v) const { atomicAdd(p, v); }
};

// ------------------------------------------------------------------------------------------------
// __global__ wrappers around the block bodies
// ------------------------------------------------------------------------------------------------
// minimum resident CTAs per SM the register allocation must allow (a register cliff halves occupancy)
template <int N> constexpr int zy_min_blocks() { return (N == 128 || N == 512) ? 3 : 4; }
template <int N, int NL, bool DO_Y, int SRC, int NT>
__global__ void __launch_bounds__(NT, zy_min_blocks<N>()) k_zy_fwd(ZyFwdParams p) {
    extern __shared__ __align__(16) float2 smem[];
    DevCtx ctx{(int)threadIdx.x, NT};
    pdl_wait();
    zy_fwd_body<N, NL, DO_Y, SRC>(ctx, p, smem, (int)blockIdx.x, (int)blockIdx.y);
}

// ------------------------------------------------------------------------------------------------
// pointwise / point kernels
// ------------------------------------------------------------------------------------------------
struct Corner {
    int j0[3];
    float f[3];
};
// t = c N, j0 = floor(t), f = t - j0 (Eq.10-11; readings R1/R2).  N is a power
// of two, so t, floor and f are exact in fp32.
__device__ __forceinline__ Corner corner_of(const float* __restrict__ c, int N) {
    Corner k;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const float t = c[a] * (float)N;
        const float fl = floorf(t);
        k.j0[a] = (int)fl;
        k.f[a] = t - fl;
    }
    return k;
}
__device__ __forceinline__ size_t vox(int N, int jx, int jy, int jz) {
    const int M = N - 1;  // periodic wrap (R1)
    return ((size_t)(jx & M) * N + (jy & M)) * N + (jz & M);
}

// ---- F1a: counting sort of the points by bin key j0x * NTY + j0y / NL (NTY = N / NL) -----------------
// The z/y forward kernel rasterises each block's lines from the bins that can touch them, so the
// splatted field never exists in HBM (no zero fill, no global atomics on the grid).
__device__ __forceinline__ int bin_key(const float* __restrict__ c, int N, int NL) {
    const int M = N - 1;
    const int jx = (int)floorf(c[0] * (float)N) & M, jy = (int)floorf(c[1] * (float)N) & M;
    return jx * (N / NL) + jy / NL;
}
constexpr int BIN_CS = 8;    // one bin counter / cursor per 32-byte sector (atomics to one 128-byte line serialise in L2)
__global__ void k_bin_count(const float* __restrict__ pts, int P, int N, int NL, int nbins, int* __restrict__ cnt,
                            int* __restrict__ nact) {
    pdl_wait();
    const int i = blockIdx.x * blockDim.x + threadIdx.x, b = blockIdx.y;
    if (i == 0 && b == 0) { nact[0] = 0; nact[1] = 0; nact[2] = 0; nact[3] = 0; }  // lengths of the active-tile lists (k_bin_scan appends)
    if (i >= P) return;
    atomicAdd(cnt + ((size_t)b * nbins + bin_key(pts + ((size_t)b * P + i) * 3, N, NL)) * BIN_CS, 1);
}
// one block per item: exclusive scan of the counts -> start[nbins+1]; cursor = start; counts reset to 0
// Activity lists ("nobody computes what nobody reads").  A tile (x, ty) = the NL z-lines y in [ty NL, (ty+1) NL) of plane x is
// ACTIVE when a point can touch it: one of the bins (x, ty), (x-1, ty), (x, ty-1), (x-1, ty-1) is non-empty -- the test the
// splat pass uses for its own tile.  A plane is active when one of its tiles is.  The splatted field is identically zero
// on inactive tiles and the gather (B6) never reads vbar there, so
//   - the forward y pass (N >= 256) neither loads nor transforms inactive planes (it writes their zeros),
//   - the inverse y pass of the adjoint skips inactive planes and the inverse z pass of the adjoint inactive tiles.
// zlist: ids item * nbins + bin of the active tiles; ylist: global tile ids of the y-pass tiles of the active planes and of
// all Nyquist-plane tiles; nact = {|zlist|, |ylist|, number of active planes, -} (reset by the binning kernel).  Items append their segments with one atomicAdd each: the order of the items in the lists is arbitrary,
// the results do not depend on it (tiles are independent).
struct ActLists {
    int* plane_act;   // [B][N] 1 = active
    int* zlist;       // [B * nbins]
    int* ylist;       // [B * (N * KT + NYQT)]  (N >= 256)
    int* nact;        // [4]
    unsigned* tile_bits;  // [B][nbins / 32] activity bits of the tiles, bit = bin index
    unsigned* plane_bits; // [B][N / 32] activity bits of the planes
    int N, NTY, KT, NYQT;  // KT = y-pass tiles per plane (0: no y pass), NYQT = Nyquist tiles per item
};
__device__ __forceinline__ int block_excl_scan_1024(int v, int* wsum, int& total) {
    const int tid = threadIdx.x, nt = blockDim.x;
    int incl = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int t = __shfl_up_sync(0xffffffffu, incl, o);
        if ((tid & 31) >= o) incl += t;
    }
    __syncthreads();
    if ((tid & 31) == 31) wsum[tid >> 5] = incl;
    __syncthreads();
    if (tid < 32) {
        int w = (tid < (nt >> 5)) ? wsum[tid] : 0;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, w, o);
            if (tid >= o) w += t;
        }
        wsum[tid] = w;
    }
    __syncthreads();
    total = wsum[31];
    return incl - v + ((tid >> 5) ? wsum[(tid >> 5) - 1] : 0);
}
// Builds the lists of one item from its exclusive bin offsets start_at(0..nbins) (whole block, blockDim.x a multiple of 32
// and >= nbins / 32; wsum = 32 ints of shared memory).  Bins are visited lanes-over-bins (conflict-free reads of the
// offsets), the activity flags are packed with warp ballots and the lists are the set bits in increasing order.
template <class F>
__device__ __forceinline__ void build_act_lists(const ActLists& al, int b, int nbins, int* wsum, F start_at) {
    __shared__ int s_base[2];
    __shared__ int s_planes[512];
    __shared__ unsigned s_bits[256];   // nbins <= 8192
    const int tid = threadIdx.x, nt = blockDim.x;
    const int N = al.N, NTY = al.NTY, lg = 31 - __clz(NTY);   // N and NTY are powers of two
    auto bin_n = [&](int x, int t) { const int i = ((x & (N - 1)) << lg) + (t & (NTY - 1)); return start_at(i + 1) - start_at(i); };
    for (int i = tid; i < nbins; i += nt) {   // nbins and nt are multiples of 32: whole warps
        const int x = i >> lg, t = i & (NTY - 1);
        int n = bin_n(x, t) + bin_n(x - 1, t);
        if (NTY > 1) n += bin_n(x, t - 1) + bin_n(x - 1, t - 1);
        const unsigned word = __ballot_sync(0xffffffffu, n > 0);
        if ((tid & 31) == 0) s_bits[i >> 5] = word;
    }
    __syncthreads();
    // active tiles: word w -> its set bits
    const int nwords = nbins >> 5;
    const unsigned myw = tid < nwords ? s_bits[tid] : 0u;
    if (tid < nwords) al.tile_bits[(size_t)b * nwords + tid] = myw;
    int ztot;
    int zoff = block_excl_scan_1024(__popc(myw), wsum, ztot);
    if (tid == 0) s_base[0] = atomicAdd(al.nact + 0, ztot);
    // active planes: one of the NTY tiles of the plane is active (NTY <= 16 divides 32: the bits sit in one word)
    int ptot = 0;
    for (int x0 = 0; x0 < N; x0 += nt) {   // one round unless the block has fewer threads than planes
        const int x = x0 + tid;
        int pact = 0;
        if (x < N) {
            const int bit0 = x << lg;
            pact = ((s_bits[bit0 >> 5] >> (bit0 & 31)) & ((NTY >= 32) ? 0xffffffffu : ((1u << NTY) - 1u))) ? 1 : 0;
            al.plane_act[(size_t)b * N + x] = pact;
        }
        if (x0 + (tid & ~31) < N) {   // whole warps: N is a multiple of 32
            const unsigned pw = __ballot_sync(0xffffffffu, pact != 0);
            if ((tid & 31) == 0) al.plane_bits[(size_t)b * (N >> 5) + (x >> 5)] = pw;
        }
        int tot;
        const int poff = ptot + block_excl_scan_1024(pact, wsum, tot);
        if (x < N && pact) s_planes[poff] = x;
        ptot += tot;
    }
    if (tid == 0) {
        s_base[1] = al.KT ? atomicAdd(al.nact + 1, ptot * al.KT + al.NYQT) : 0;
        atomicAdd(al.nact + 2, ptot);
    }
    __syncthreads();
    {
        int* zl = al.zlist + s_base[0];
        unsigned w = myw;
        while (w) { const int bit = __ffs(w) - 1; w &= w - 1; zl[zoff++] = b * nbins + (tid << 5) + bit; }
    }
    if (al.KT) {
        const int tpu = N * al.KT + al.NYQT;   // y-pass tiles per item (dense numbering)
        const int lk = 31 - __clz(al.KT);      // KT is a power of two
        int* yl = al.ylist + s_base[1];
        for (int e = tid; e < ptot * al.KT; e += nt) yl[e] = b * tpu + (s_planes[e >> lk] << lk) + (e & (al.KT - 1));
        for (int e = tid; e < al.NYQT; e += nt) yl[ptot * al.KT + e] = b * tpu + N * al.KT + e;
    }
}
__global__ void k_bin_scan(int* __restrict__ cnt, int nbins, int P, int* __restrict__ start, int* __restrict__ cursor,
                           unsigned* __restrict__ nmax) {
    pdl_wait();
    if (threadIdx.x == 0) nmax[blockIdx.x] = 0u;   // k_bin_scatter (the next launch) takes the max of |n| into it
    __shared__ int wsum[32];
    const int b = blockIdx.x, tid = threadIdx.x, nt = blockDim.x;
    int* c = cnt + (size_t)b * nbins * BIN_CS;
    int* st = start + (size_t)b * (nbins + 1);
    int* cu = cursor + (size_t)b * nbins * BIN_CS;
    extern __shared__ int s_cnt[];   // [nbins] the counts, fetched with independent loads (one sector each) and cleared
    for (int i = tid; i < nbins; i += nt) { s_cnt[i] = c[i * BIN_CS]; c[i * BIN_CS] = 0; }
    __syncthreads();
    const int per = (nbins + nt - 1) / nt;
    const int lo = tid * per, hi = min(lo + per, nbins);
    int local = 0;
    for (int i = lo; i < hi; ++i) local += s_cnt[i];
    int incl = local;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int t = __shfl_up_sync(0xffffffffu, incl, o);
        if ((tid & 31) >= o) incl += t;
    }
    if ((tid & 31) == 31) wsum[tid >> 5] = incl;
    __syncthreads();
    if (tid < 32) {
        int w = (tid < (nt >> 5)) ? wsum[tid] : 0;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, w, o);
            if (tid >= o) w += t;
        }
        wsum[tid] = w;  // inclusive over warps
    }
    __syncthreads();
    int run = incl - local + ((tid >> 5) ? wsum[(tid >> 5) - 1] : 0);
    for (int i = lo; i < hi; ++i) {
        const int n = s_cnt[i];
        st[i] = run;
        cu[i * BIN_CS] = run;
        run += n;
    }
    if (tid == 0) st[nbins] = P;
}
// ---- F1a in ONE launch (the default): count + rank | per-item barrier | offsets (every block, in shared memory) + scatter ----
// Phase 1 takes each point's rank inside its bin from the return value of the counting atomicAdd; after the barrier every
// block of the item scans the item's counts itself (nbins <= 8192: 32 per thread) and places its points at
// start[bin] + rank -- no second round of atomics, no second barrier, and the launch and drain latencies of two kernels
// less (the three-kernel version below stays as the fall-back for batches too large to be co-resident).  The splat pass that
// follows clears the counts and re-arms the barrier, so a forward leaves the state it found (replayable in a CUDA graph).
struct BinSortParams {
    const float* pts; const float* nrm;
    int P, N, NL, nbins;
    int* cnt;        // [B][nbins][BIN_CS] (entry 0 of each group of BIN_CS) zero on entry; cleared by the splat pass
    int* start;      // [B][nbins + 1]
    float4* spts; float4* snrm;
    unsigned* nmax;  // [B]
    unsigned* bsync; // [3] arrivals, -, time-out flag
    ActLists al;
};
constexpr int BIN_PPT = 8;   // points per thread of k_bin_sort; bin and rank stay in registers across the barrier
__global__ void __launch_bounds__(256, 6) k_bin_sort(const BinSortParams p) {
    extern __shared__ int s_start[];   // [nbins + 1]
    __shared__ int wsum[32];
    pdl_wait();
    // blocks 0 .. gx-1 of an item own its points (point i of block x, thread t, round k: i = (k gx + x) 256 + t); block gx
    // owns none: it publishes the offsets and builds the activity lists while the others scatter
    const int b = blockIdx.y, gx = gridDim.x - 1, tid = threadIdx.x, B = gridDim.y;
    const bool publisher = (int)blockIdx.x == gx;
    const unsigned nblk = gridDim.x * gridDim.y;
    const int nbins = p.nbins, P = p.P;
    int* cnt = p.cnt + (size_t)b * nbins * BIN_CS;
    const float* pts = p.pts + (size_t)b * P * 3;
    const float* nrm = p.nrm + (size_t)b * P * 3;
    int key[BIN_PPT], rank[BIN_PPT];
    if (publisher) {
        if (tid == 0) {
            p.nmax[b] = 0u;
            if (b == 0 && p.al.nact) { p.al.nact[0] = 0; p.al.nact[1] = 0; p.al.nact[2] = 0; p.al.nact[3] = 0; }
        }
    } else {
        // phase 1: count; the value the atomic returns is the point's rank in its bin.  All loads first, then all atomics;
        // the normals (read in phase 3) are pulled into L2 meanwhile.
#pragma unroll
        for (int k = 0; k < BIN_PPT; ++k) {
            const int i = (k * gx + blockIdx.x) * 256 + tid;
            key[k] = 0;
            if (i < P) {
                key[k] = bin_key(pts + (size_t)i * 3, p.N, p.NL);
                asm volatile("prefetch.global.L2 [%0];" ::"l"(nrm + (size_t)i * 3));
            }
        }
#pragma unroll
        for (int k = 0; k < BIN_PPT; ++k) {
            const int i = (k * gx + blockIdx.x) * 256 + tid;
            rank[k] = 0;
            if (i < P) rank[k] = atomicAdd(cnt + key[k] * BIN_CS, 1);
        }
    }
    // barrier over all blocks of the launch (co-resident: cooperative launch); bounded spin, sticky time-out flag
    __syncthreads();
    if (tid == 0) {
        asm volatile("fence.acq_rel.gpu;" ::: "memory");
        atomicAdd(p.bsync, 1u);
        unsigned seen, spins = 0;
        unsigned long long t0 = 0;
        do {
            asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(seen) : "l"(p.bsync) : "memory");
            if (seen < nblk && (++spins & 1023u) == 0) {
                unsigned long long t;
                asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t));
                if (t0 == 0) t0 = t;
                else if (t - t0 > 2000000000ull) { atomicExch(p.bsync + 2, 1u); break; }
            }
        } while (seen < nblk);
        asm volatile("fence.acq_rel.gpu;" ::: "memory");
    }
    __syncthreads();
    // phase 2: exclusive scan of the item's counts into shared memory (every block)
    for (int i = tid; i < nbins; i += 256) s_start[i] = __ldcg(cnt + i * BIN_CS);   // independent loads (L2: written by atomics)
    __syncthreads();
    const int per = (nbins + 255) / 256;
    const int lo = min(tid * per, nbins), hi = min(lo + per, nbins);
    int local = 0;
    for (int i = lo; i < hi; ++i) local += s_start[i];
    int tot;
    int run = block_excl_scan_1024(local, wsum, tot);
    for (int i = lo; i < hi; ++i) { const int n = s_start[i]; s_start[i] = run; run += n; }
    if (tid == 0) s_start[nbins] = P;
    __syncthreads();
    if (publisher) {
        int* st = p.start + (size_t)b * (nbins + 1);
        for (int i = tid; i <= nbins; i += 256) st[i] = s_start[i];
        if (p.al.zlist) build_act_lists(p.al, b, nbins, wsum, [&](int i) { return s_start[i]; });
    } else {
        // phase 3: scatter
        unsigned amax = 0u;
#pragma unroll
        for (int k = 0; k < BIN_PPT; ++k) {
            const int i = (k * gx + blockIdx.x) * 256 + tid;
            if (i < P) {
                const float* c = pts + (size_t)i * 3;
                const float* n = nrm + (size_t)i * 3;
                const float n0 = __ldg(n), n1 = __ldg(n + 1), n2 = __ldg(n + 2);
                const int pos = s_start[key[k]] + rank[k];
                p.spts[(size_t)b * P + pos] = make_float4(__ldg(c), __ldg(c + 1), __ldg(c + 2), __int_as_float(i));  // .w: index in the caller's order
                p.snrm[(size_t)b * P + pos] = make_float4(n0, n1, n2, 0.f);
                amax = max(amax, __float_as_uint(fmaxf(fmaxf(fabsf(n0), fabsf(n1)), fabsf(n2))));
            }
        }
        amax = __reduce_max_sync(0xffffffffu, amax);
        if ((tid & 31) == 0 && amax) atomicMax(p.nmax + b, amax);
    }
    // The counts and the barrier word are cleared by the NEXT kernel of the forward (the splat pass, which starts when
    // every block of this one is done): no exit round trip here, and a call still leaves the state it found.
    (void)B;
}
// (the last block of each item owns no points: it builds the activity lists from the offsets meanwhile)
__global__ void k_bin_scatter(const float* __restrict__ pts, const float* __restrict__ nrm, int P, int N, int NL,
                              int nbins, int* __restrict__ cursor, float4* __restrict__ spts,
                              float4* __restrict__ snrm, unsigned* __restrict__ nmax, const int* __restrict__ start, ActLists al) {
    pdl_wait();
    const int i = blockIdx.x * blockDim.x + threadIdx.x, b = blockIdx.y;
    if (blockIdx.x == gridDim.x - 1) {
        if (!al.zlist) return;
        extern __shared__ int s_st[];   // [nbins + 1] copy of the offsets
        __shared__ int wsum[32];
        const int tid = threadIdx.x, nt = blockDim.x;
        const int* st = start + (size_t)b * (nbins + 1);
        for (int k = tid; k <= nbins; k += nt) s_st[k] = st[k];
        __syncthreads();
        build_act_lists(al, b, nbins, wsum, [&](int k) { return s_st[k]; });
        return;
    }
    unsigned amax = 0u;   // bit pattern of max_c |n_c| (non-negative floats order like their bits): scale of the fixed-point splat
    if (i < P) {
        const float* c = pts + ((size_t)b * P + i) * 3;
        const float* n = nrm + ((size_t)b * P + i) * 3;
        const int pos = atomicAdd(cursor + ((size_t)b * nbins + bin_key(c, N, NL)) * BIN_CS, 1);
        spts[(size_t)b * P + pos] = make_float4(c[0], c[1], c[2], __int_as_float(i));  // .w: index in the caller's order
        snrm[(size_t)b * P + pos] = make_float4(n[0], n[1], n[2], 0.f);
        amax = __float_as_uint(fmaxf(fmaxf(fabsf(n[0]), fabsf(n[1])), fabsf(n[2])));
    }
    amax = __reduce_max_sync(0xffffffffu, amax);
    if ((threadIdx.x & 31) == 0 && amax) atomicMax(nmax + b, amax);
}

__device__ __forceinline__ float warp_sum(float x) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
    return x;
}
// block sum of one float per thread; result valid in thread 0
__device__ __forceinline__ float block_sum(float x, float* sh) {
    x = warp_sum(x);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    __syncthreads();
    if (lane == 0) sh[wid] = x;
    __syncthreads();
    float r = 0.f;
    if (wid == 0) {
        r = (lane < (int)(blockDim.x >> 5)) ? sh[lane] : 0.f;
        r = warp_sum(r);
    }
    return r;
}

// F5a: mu = mean_i interp(chi', c_i); a = chi'[0,0,0] - mu; s = 0.5/|a| (Eq.4; R5, R11).
// Partial sums go to a double accumulator; the last block of an item finalises stats = {mu, a, s, 0}.
// Walks the points in bin order (neighbours in memory are neighbours in space: the 8 gathers hit L1/L2).
__global__ void k_sample_mean(const float4* __restrict__ spts, int P, int N, const float* __restrict__ chi_p,
                              double* __restrict__ acc, unsigned* __restrict__ ticket,
                              float* __restrict__ stats) {
    pdl_wait();
    __shared__ float sh[32];
    const int b = blockIdx.y;
    const size_t V = (size_t)N * N * N;
    const float* g = chi_p + (size_t)b * V;
    float sum = 0.f;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < P; i += gridDim.x * blockDim.x) {
        const float4 c4 = __ldg(spts + (size_t)b * P + i);
        const float cc[3] = {c4.x, c4.y, c4.z};
        const Corner k = corner_of(cc, N);
        float s = 0.f;
#pragma unroll
        for (int d = 0; d < 8; ++d) {
            const int dx = d >> 2, dy = (d >> 1) & 1, dz = d & 1;
            const float w = (dx ? k.f[0] : 1.f - k.f[0]) * (dy ? k.f[1] : 1.f - k.f[1]) * (dz ? k.f[2] : 1.f - k.f[2]);
            s += w * __ldg(g + vox(N, k.j0[0] + dx, k.j0[1] + dy, k.j0[2] + dz));
        }
        sum += s;
    }
    const float bs = block_sum(sum, sh);
    if (threadIdx.x == 0) {
        atomicAdd(acc + b, (double)bs);
        __threadfence();
        const unsigned t = atomicAdd(ticket + b, 1u);
        if (t == gridDim.x - 1) {
            const double tot = atomicAdd(acc + b, 0.0);
            const double mu = tot / (double)P;
            const double a = (double)g[0] - mu;
            const double s = 0.5 / fabs(a);  // m = 0.5
            stats[b * 4 + 0] = (float)mu;
            stats[b * 4 + 1] = (float)a;
            stats[b * 4 + 2] = (float)s;
            stats[b * 4 + 3] = 0.f;
            acc[b] = 0.0;
            ticket[b] = 0u;
        }
    }
}

// F5b: chi = s (chi' - mu), in place
__global__ void k_scale_shift(float4* __restrict__ chi, size_t n4_per_item, const float* __restrict__ stats) {
    pdl_wait();
    const int b = blockIdx.y;
    const float mu = stats[b * 4 + 0], s = stats[b * 4 + 2];
    float4* p = chi + (size_t)b * n4_per_item;
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n4_per_item; i += stride) {
        float4 v = p[i];
        v.x = s * (v.x - mu); v.y = s * (v.y - mu); v.z = s * (v.z - mu); v.w = s * (v.w - mu);
        p[i] = v;
    }
}

// F5b fused with the loss of the learning-based setting (Eq.9): L = || chi - chi_gt ||^2.  The same
// pass writes chi = s (chi' - mu), the upstream gradient G = dL/dchi = 2 (chi - chi_gt) and accumulates L together
// with the reductions S0 = sum G, S1 = sum G chi of the backward (B1), so G never makes a round trip through the
// caller and k_reduce_g is not needed.  The last block writes loss[b] and bw = {s, beta/P, S1/a, beta/(P s)}.
__global__ void k_scale_shift_mse(float4* __restrict__ chi, const float4* __restrict__ chi_gt, float4* __restrict__ G,
                                  size_t n4_per_item, int P, const float* __restrict__ stats, double* __restrict__ acc,
                                  unsigned* __restrict__ ticket, float* __restrict__ bw, float* __restrict__ loss) {
    pdl_wait();
    __shared__ float sh[32];
    const int b = blockIdx.y;
    const float mu = stats[b * 4 + 0], s = stats[b * 4 + 2];
    float4* c = chi + (size_t)b * n4_per_item;
    const float4* t = chi_gt + (size_t)b * n4_per_item;
    float4* g = G + (size_t)b * n4_per_item;
    float s0 = 0.f, s1 = 0.f, l = 0.f;
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n4_per_item; i += stride) {
        float4 v = c[i];
        const float4 w = t[i];
        v.x = s * (v.x - mu); v.y = s * (v.y - mu); v.z = s * (v.z - mu); v.w = s * (v.w - mu);
        const float4 d = make_float4(v.x - w.x, v.y - w.y, v.z - w.z, v.w - w.w);
        const float4 gg = make_float4(2.f * d.x, 2.f * d.y, 2.f * d.z, 2.f * d.w);
        c[i] = v;
        g[i] = gg;
        l += (d.x * d.x + d.y * d.y) + (d.z * d.z + d.w * d.w);
        s0 += (gg.x + gg.y) + (gg.z + gg.w);
        s1 += (gg.x * v.x + gg.y * v.y) + (gg.z * v.z + gg.w * v.w);
    }
    const float b0 = block_sum(s0, sh);
    const float b1 = block_sum(s1, sh);
    const float b2 = block_sum(l, sh);
    if (threadIdx.x == 0) {
        atomicAdd(acc + 3 * b, (double)b0);
        atomicAdd(acc + 3 * b + 1, (double)b1);
        atomicAdd(acc + 3 * b + 2, (double)b2);
        __threadfence();
        const unsigned tk = atomicAdd(ticket + b, 1u);
        if (tk == gridDim.x - 1) {
            const double S0 = atomicAdd(acc + 3 * b, 0.0), S1 = atomicAdd(acc + 3 * b + 1, 0.0), L = atomicAdd(acc + 3 * b + 2, 0.0);
            const double a = stats[b * 4 + 1], sd = stats[b * 4 + 2];
            const double beta = S1 / a - sd * S0;
            bw[b * 4 + 0] = (float)sd;
            bw[b * 4 + 1] = (float)(beta / (double)P);
            bw[b * 4 + 2] = (float)(S1 / a);
            bw[b * 4 + 3] = (float)(beta / ((double)P * sd));
            loss[b] = (float)L;
            acc[3 * b] = 0.0; acc[3 * b + 1] = 0.0; acc[3 * b + 2] = 0.0;
            ticket[b] = 0u;
        }
    }
}

// B1: S0 = sum G, S1 = sum G chi; the last block writes bw = {s, beta/P, S1/a, beta/(P s)},
// beta = S1/a - s S0.
__global__ void k_reduce_g(const float4* __restrict__ G, const float4* __restrict__ chi, size_t n4_per_item,
                           int P, const float* __restrict__ stats, double* __restrict__ acc,
                           unsigned* __restrict__ ticket, float* __restrict__ bw) {
    pdl_wait();
    __shared__ float sh[32];
    const int b = blockIdx.y;
    const float4* g = G + (size_t)b * n4_per_item;
    const float4* c = chi + (size_t)b * n4_per_item;
    float s0 = 0.f, s1 = 0.f;
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    // (walks the grids from the END: chi was written front to back by the normalisation pass, its tail is still in L2)
    const size_t last = n4_per_item - 1;
    for (; i + 3 * stride < n4_per_item; i += 4 * stride) {  // 8 independent 16-byte loads in flight per thread
        float4 a[4], x[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) { a[u] = __ldcs(g + (last - (i + u * stride))); x[u] = __ldcs(c + (last - (i + u * stride))); }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            s0 += (a[u].x + a[u].y) + (a[u].z + a[u].w);
            s1 += (a[u].x * x[u].x + a[u].y * x[u].y) + (a[u].z * x[u].z + a[u].w * x[u].w);
        }
    }
    for (; i < n4_per_item; i += stride) {
        const float4 a = g[last - i], x = c[last - i];
        s0 += (a.x + a.y) + (a.z + a.w);
        s1 += (a.x * x.x + a.y * x.y) + (a.z * x.z + a.w * x.w);
    }
    const float b0 = block_sum(s0, sh);
    const float b1 = block_sum(s1, sh);
    if (threadIdx.x == 0) {
        atomicAdd(acc + 2 * b, (double)b0);
        atomicAdd(acc + 2 * b + 1, (double)b1);
        __threadfence();
        const unsigned t = atomicAdd(ticket + b, 1u);
        if (t == gridDim.x - 1) {
            const double S0 = atomicAdd(acc + 2 * b, 0.0), S1 = atomicAdd(acc + 2 * b + 1, 0.0);
            const double a = stats[b * 4 + 1], s = stats[b * 4 + 2];
            const double beta = S1 / a - s * S0;
            bw[b * 4 + 0] = (float)s;
            bw[b * 4 + 1] = (float)(beta / (double)P);
            bw[b * 4 + 2] = (float)(S1 / a);
            bw[b * 4 + 3] = (float)(beta / ((double)P * s));
            acc[2 * b] = 0.0;
            acc[2 * b + 1] = 0.0;
            ticket[b] = 0u;
        }
    }
}

// B6: dL/dn_i = sum_corners w vbar[corner];
//     dL/dc_i[a] = sum_corners (dw/dc_a) (n_i . vbar[corner] + (beta/(P s)) chi[corner]),
//     dw/dc_a = N (d_a ? +1 : -1) prod_{b != a} w_b   (adjoint of F1 and F5; the mu part of chi' = chi/s + mu
//     cancels because sum_corners dw/dc_a = 0).
//     Walks the points in bin order (spatial locality of the 32 gathers) and scatters the two gradients back to
//     the caller's order through the index kept in spts.w.
__global__ void k_gather_grads(const float4* __restrict__ spts, const float4* __restrict__ snrm, int P, int N,
                               const float* __restrict__ vbar, const float* __restrict__ chi,
                               const float* __restrict__ bw, float* __restrict__ gp, float* __restrict__ gn) {
    pdl_wait();
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int b = blockIdx.y;
    if (i >= P) return;
    const size_t V = (size_t)N * N * N;
    const float4 c4 = __ldg(spts + (size_t)b * P + i), n4 = __ldg(snrm + (size_t)b * P + i);
    const size_t o = ((size_t)b * P + __float_as_int(c4.w)) * 3;
    const float cc[3] = {c4.x, c4.y, c4.z};
    const Corner k = corner_of(cc, N);
    const float n0 = n4.x, n1 = n4.y, n2 = n4.z;
    const float cchi = bw[b * 4 + 3];
    const float* vb = vbar + (size_t)b * 3 * V;
    const float* cb = chi + (size_t)b * V;
    float g0 = 0.f, g1 = 0.f, g2 = 0.f, c0 = 0.f, c1 = 0.f, c2 = 0.f;
#pragma unroll
    for (int d = 0; d < 8; ++d) {
        const int dx = d >> 2, dy = (d >> 1) & 1, dz = d & 1;
        const float wx = dx ? k.f[0] : 1.f - k.f[0];
        const float wy = dy ? k.f[1] : 1.f - k.f[1];
        const float wz = dz ? k.f[2] : 1.f - k.f[2];
        const size_t j = vox(N, k.j0[0] + dx, k.j0[1] + dy, k.j0[2] + dz);
        const float a0 = __ldg(vb + j), a1 = __ldg(vb + V + j), a2 = __ldg(vb + 2 * V + j);
        const float x = __ldg(cb + j);
        const float w = wx * wy * wz;
        g0 += w * a0; g1 += w * a1; g2 += w * a2;
        const float val = n0 * a0 + n1 * a1 + n2 * a2 + cchi * x;
        c0 += (dx ? val : -val) * (wy * wz);
        c1 += (dy ? val : -val) * (wx * wz);
        c2 += (dz ? val : -val) * (wx * wy);
    }
    const float fN = (float)N;
    gn[o] = g0; gn[o + 1] = g1; gn[o + 2] = g2;
    gp[o] = fN * c0; gp[o + 1] = fN * c1; gp[o + 2] = fN * c2;
}

}  // namespace sap

// ================================================================================================
// handle, launch plumbing
// ================================================================================================
struct sap_dpsr {
    int N = 0, batch = 0, max_points = 0, device = 0, num_sms = 148;
    float sigma = 0.f;
    // workspace (device)
    float* v = nullptr;        // [B][3][N^3]  splatted field / vbar
    float4* spts = nullptr;    // [B][max_points] points sorted by bin
    float4* snrm = nullptr;    // [B][max_points] normals, same order
    int* bin_cnt = nullptr;    // [B][nbins]   (zero between calls)
    int* bin_cursor = nullptr; // [B][nbins]
    int* bin_start = nullptr;  // [B][nbins+1]
    unsigned* bsync = nullptr; // [3] barrier of k_bin_sort: arrivals, exits, time-out flag
    int bin_gx_max = 0;        // co-resident blocks of k_bin_sort per batch item (0: three-kernel fall-back)
    int coop_pdl = 1;          // cooperative launches also take the programmatic-serialization attribute (probed on first use)
    int nbins = 0;
    float2* S3 = nullptr;      // [B*3][N*N*H] 3-channel spectra
    float2* Q3 = nullptr;      // [B*3][N*N]
    float2* S1 = nullptr;      // [B][N*N*H]   1-channel spectrum
    float2* Q1 = nullptr;      // [B][N*N]
    float2* tw = nullptr;      // [N]
    float4* ftab = nullptr;    // [N + N/2 + 1] per-slot frequency table of the spectral multiplier
    // TMA descriptors of the spectra (ring_pass.cuh): main arrays with the x-pass / y-pass tile box, Nyquist planes
    CUtensorMap mS3x, mS3y, mS1x, mS1y, mQ3, mQ1, mQT3, mQT1;
    float2* QT3 = nullptr;     // [B*3][N*N] transposed Nyquist planes (N >= 256: staging between the z/x passes and the y pass)
    float2* QT1 = nullptr;     // [B][N*N]
    double* acc = nullptr;     // [B][3] reduction accumulators (mean | S0,S1)
    unsigned* ticket = nullptr;  // [B][2]
    float* stats = nullptr;    // [B][4] {mu, a, s, -}
    float* bw = nullptr;       // [B][4] {s, beta/P, S1/a, beta/(P s)}
    unsigned* nmax = nullptr;  // [B] bit pattern of the largest |normal component| of the item (fixed-point scale of the splat)
    // activity lists (ActLists, written by k_bin_scan): which planes / tiles a point can touch
    int* plane_act = nullptr;  // [B][N]
    int* zlist = nullptr;      // [B * nbins]
    int* ylist = nullptr;      // [B * (N * KT + NYQT)] (N >= 256)
    int* nact = nullptr;       // [4]
    unsigned* tile_bits = nullptr;  // [B][nbins / 32]
    unsigned* plane_bits = nullptr; // [B][N / 32]
    bool mask_solve = false;   // fused planes in the throughput regime: the splat pass writes no zeros for inactive planes, the solve masks them
    bool sparse = true;        // use the lists (SAP_DENSE=1 in the environment of sap_dpsr_create: every tile is processed)
    bool lists_valid = false;  // the lists belong to the bins in the workspace (the latency path does not write them)
    // staging for the *_host entry points (allocated on first use)
    float *h_pts = nullptr, *h_nrm = nullptr, *h_chi = nullptr, *h_gchi = nullptr, *h_gp = nullptr, *h_gn = nullptr;
    int host_P = 0;
    int binned_P = 0;          // num_points of the forward whose bins are in the workspace
    // which forward the workspace state (bins, stats, bw, gmse) belongs to: bumped by EVERY forward variant, so that a
    // backward can tell whether another forward has run on the handle since the one it differentiates
    unsigned long long epoch = 0;
    enum FwdKind { FWD_NONE = 0, FWD_DEVICE = 1, FWD_MSE = 2, FWD_HOST = 3 };
    int fwd_kind = FWD_NONE;
    // fused-loss path (sap_dpsr_forward_mse / backward_mse), allocated on first use
    float* gmse = nullptr;     // [B][N^3] G = 2 (chi - chi_gt)
    double* acc_mse = nullptr; // [B][3]   S0, S1, L accumulators
    bool mse_valid = false;    // bw and gmse belong to the last forward
    // latency path (fused_small.cuh): one cooperative kernel per direction when all x-planes fit one wave of CTAs
    bool fused_ok = false;     // N <= 128 and batch * N <= #SMs
    int path = SAP_PATH_AUTO;
    int fused_pdl = 1;         // the cooperative launch also takes the programmatic-serialization attribute (probed on first use)
    int* fhist = nullptr;      // [B][#SMs][N]
    double* facc = nullptr;    // [B][2]
    unsigned* fsync = nullptr; // [4] barrier arrivals, exits, time-out flag
    long long* fstamps = nullptr;  // [64] clock64 of CTA 0 at the marks of the phase bodies
    size_t ws_bytes = 0;
    int launches = 0;
    // optional per-kernel timing (sap_dpsr_set_profiling): one event before the first launch, one after each
    bool prof = false;
    static constexpr int MAX_EV = 24;
    cudaEvent_t ev[MAX_EV] = {};
    const char* ev_name[MAX_EV] = {};
    int nev = 0;
    std::string err;
};

namespace sap {

static thread_local std::string g_create_err;

static bool cuda_ok(sap_dpsr* h, cudaError_t e, const char* what) {
    if (e == cudaSuccess) return true;
    char buf[512];
    snprintf(buf, sizeof buf, "%s: %s", what, cudaGetErrorString(e));
    if (h) h->err = buf; else g_create_err = buf;
    return false;
}

template <class T> static cudaError_t dev_alloc(sap_dpsr* h, T** p, size_t count) {
    cudaError_t e = cudaMalloc((void**)p, count * sizeof(T));
    if (e == cudaSuccess) h->ws_bytes += count * sizeof(T);
    return e;
}

#define SAP_LAUNCH_CHECK(h, name)                                          \
    do {                                                                   \
        ++(h)->launches;                                                   \
        if (!cuda_ok((h), cudaGetLastError(), name)) return SAP_ERR_CUDA;  \
        prof_mark((h), name, st);                                          \
    } while (0)

static void prof_mark(sap_dpsr* h, const char* name, cudaStream_t st) {
    if (!h->prof || h->nev >= sap_dpsr::MAX_EV) return;
    h->ev_name[h->nev] = name;
    cudaEventRecord(h->ev[h->nev], st);
    ++h->nev;
}
static void prof_begin(sap_dpsr* h, cudaStream_t st) {
    h->nev = 0;
    prof_mark(h, "begin", st);
}

// Every kernel of the path is launched with programmatic dependent launch (see pdl_wait in fft_core.cuh): the
// launch latency of kernel n+1 hides behind kernel n.
template <class... KArgs, class... Args>
static void launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args&&... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}

// cooperative launch (all blocks co-resident: the kernel has a grid barrier), with programmatic dependent launch on top
// where the driver combines the two attributes
template <class P>
static cudaError_t launch_coop(sap_dpsr* h, void (*kernel)(P), dim3 grid, dim3 block, size_t smem, cudaStream_t st, const P& p) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute at[2];
    at[0].id = cudaLaunchAttributeCooperative; at[0].val.cooperative = 1;
    at[1].id = cudaLaunchAttributeProgrammaticStreamSerialization; at[1].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = h->coop_pdl ? 2 : 1;
    static const bool plain = getenv("SAP_BIN_COOP") && getenv("SAP_BIN_COOP")[0] == '0';   // experiment
    if (plain) { at[0] = at[1]; cfg.numAttrs = 1; }
    cudaError_t e = cudaLaunchKernelEx(&cfg, kernel, p);
    if (e != cudaSuccess && h->coop_pdl) {
        cudaGetLastError();
        h->coop_pdl = 0;
        cfg.numAttrs = 1;
        e = cudaLaunchKernelEx(&cfg, kernel, p);
    }
    return e;
}

template <class K> static cudaError_t set_smem(K kernel, size_t bytes) {
    return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
}

// ---- TMA descriptors -------------------------------------------------------------------------------
// cuTensorMapEncodeTiled is reached through the runtime's driver entry point (no link against libcuda).
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static EncodeTiledFn encode_tiled_fn(sap_dpsr* h) {
    static EncodeTiledFn fn = nullptr;
    if (fn) return fn;
    void* ptr = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (!cuda_ok(h, cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &ptr, cudaEnableDefault, &q), "cudaGetDriverEntryPoint")) return nullptr;
    if (q != cudaDriverEntryPointSuccess || !ptr) { h->err = "cuTensorMapEncodeTiled not available in this driver"; return nullptr; }
    fn = (EncodeTiledFn)ptr;
    return fn;
}
// float view of a complex array: dims[0] counts floats (2 per complex), strides in bytes for dims 1..rank-1
static bool make_map(sap_dpsr* h, CUtensorMap* m, void* base, int rank, const cuuint64_t* dims, const cuuint64_t* strides,
                     const cuuint32_t* box) {
    EncodeTiledFn fn = encode_tiled_fn(h);
    if (!fn) return false;
    const cuuint32_t es[4] = {1, 1, 1, 1};
    const CUresult r = fn(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, (cuuint32_t)rank, base, dims, strides, box, es,
                          CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                          CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        char buf[128];
        snprintf(buf, sizeof buf, "cuTensorMapEncodeTiled failed (CUresult %d)", (int)r);
        h->err = buf;
        return false;
    }
    return true;
}

// threads per block of the FFT kernels
template <int N> struct Cfg {
    static constexpr bool FUSED_ZY = (N <= 128);  // a whole (y,z) plane fits one CTA's shared memory
    static constexpr int NL = FUSED_ZY ? N : 32;
    static constexpr int NT_ZY = 256;
};

template <int N> struct Runner {
    static constexpr int H = N / 2;
    using C = Cfg<N>;

    static sap_status_t prepare(sap_dpsr* h) {
        cudaError_t e = cudaSuccess;
        {   // frequency table of the multiplier, in stored-slot order
            float4 tab[N + H + 1];
            const float cg = 2.f * h->sigma * h->sigma / ((float)N * (float)N);
            for (int i = 0; i < N; ++i) tab[i] = freq_entry_n<N>(i, cg);
            for (int i = 0; i <= H; ++i) tab[N + i] = freq_entry_z<N>(i, cg);
            e = cudaMemcpy(h->ftab, tab, sizeof(tab), cudaMemcpyHostToDevice);
        }
        auto upd = [&](cudaError_t x) { if (e == cudaSuccess) e = x; };
        upd(set_smem(k_zl_inv<N>, zl_smem_bytes<N, true>()));
        if constexpr (C::FUSED_ZY) {
            upd(set_smem(k_zy_fwd<N, C::NL, C::FUSED_ZY, SRC_SPLAT, C::NT_ZY>, zy_smem_bytes<N, C::NL>()));
            upd(set_smem(k_zl_gbar<N>, zl_smem_bytes<N, false>()));
        } else {
            upd(set_smem(k_zw_fwd<N, SRC_SPLAT>, ZwCfg<N>::SMEM));
            upd(set_smem(k_zw_fwd<N, SRC_GBAR>, ZwCfg<N>::SMEM));
            upd(set_smem(k_zw_inv<N>, ZwCfg<N>::SMEM));
        }
        upd(set_smem(k_ring<N, MODE_SOLVE>, ring_smem_bytes<N, MODE_SOLVE>()));
        upd(set_smem(k_ring<N, MODE_ADJ>, ring_smem_bytes<N, MODE_ADJ>()));
        if constexpr (!C::FUSED_ZY) {
            upd(set_smem(k_ring<N, MODE_FWD>, ring_smem_bytes<N, MODE_FWD>()));
            upd(set_smem(k_ring<N, MODE_FWD3>, ring_smem_bytes<N, MODE_FWD3>()));
            upd(set_smem(k_ring<N, MODE_INV3>, ring_smem_bytes<N, MODE_INV3>()));
            upd(set_smem(k_ring<N, MODE_INV>, ring_smem_bytes<N, MODE_INV>()));
        }
        if constexpr (N <= 128) {
            upd(set_smem(k_fused_fwd<N>, FusedCfg<N>::BYTES));
            upd(set_smem(k_fused_bwd<N>, FusedCfg<N>::BYTES));
        }
        if (!cuda_ok(h, e, "cudaFuncSetAttribute")) return SAP_ERR_CUDA;
        // TMA descriptors: tile = NB points along the pass axis x W contiguous kz (or y, Nyquist plane) slots
        constexpr cuuint32_t W2 = 2 * RingCfg<N>::W, NB = ring_box_rows<N>();
        const cuuint64_t B3 = (cuuint64_t)h->batch * 3, B1 = (cuuint64_t)h->batch;
        const cuuint64_t sS[3] = {(cuuint64_t)H * 8, (cuuint64_t)N * H * 8, (cuuint64_t)N * N * H * 8};
        const cuuint64_t sQ[2] = {(cuuint64_t)N * 8, (cuuint64_t)N * N * 8};
        const cuuint64_t dS3[4] = {(cuuint64_t)2 * H, N, N, B3}, dS1[4] = {(cuuint64_t)2 * H, N, N, B1};
        const cuuint64_t dQ3[3] = {(cuuint64_t)2 * N, N, B3}, dQ1[3] = {(cuuint64_t)2 * N, N, B1};
        const cuuint32_t bx[4] = {W2, 1, NB, 1}, by[4] = {W2, NB, 1, 1}, bq[3] = {W2, NB, 1};
        const bool ok = make_map(h, &h->mS3x, h->S3, 4, dS3, sS, bx) && make_map(h, &h->mS3y, h->S3, 4, dS3, sS, by) &&
                        make_map(h, &h->mS1x, h->S1, 4, dS1, sS, bx) && make_map(h, &h->mS1y, h->S1, 4, dS1, sS, by) &&
                        make_map(h, &h->mQ3, h->Q3, 3, dQ3, sQ, bq) && make_map(h, &h->mQ1, h->Q1, 3, dQ1, sQ, bq) &&
                        (C::FUSED_ZY || (make_map(h, &h->mQT3, h->QT3, 3, dQ3, sQ, bq) && make_map(h, &h->mQT1, h->QT1, 3, dQ1, sQ, bq)));
        return ok ? SAP_OK : SAP_ERR_CUDA;
    }

    // persistent ring pass (ring_pass.cuh).  axis 0: x pass, axis 1: y pass (N >= 256).  Nyquist plane: the z
    // pass leaves it transposed ([y][x]) for the y pass, which writes it back as [x][y] for the x pass (and the
    // other way round on the inverse side), so every tile of every pass is a TMA box with contiguous rows.
    template <int MODE>
    static void launch_ring(sap_dpsr* h, cudaStream_t st, int units, const CUtensorMap& mS, const CUtensorMap& mQ,
                            float2* outS, float2* outQ, int axis) {
        using RC = RingCfgM<N, MODE>;
        RingParams p;
        p.mapS = mS; p.mapQ = mQ; p.outS = outS; p.outQ = outQ; p.tw = h->tw; p.ftab = h->ftab;
        (void)axis;
        p.units = units; p.nyq_out_t = C::FUSED_ZY ? 0 : 1;
        const bool listed = (MODE == MODE_FWD3 || MODE == MODE_INV3) && h->sparse && h->lists_valid;
        p.ylist = listed ? h->ylist : nullptr; p.nact = h->nact;
        p.tile_bits = h->tile_bits;
        p.plane_bits = (MODE == MODE_SOLVE && h->sparse && h->mask_solve) ? h->plane_bits : nullptr;
        p.cs = (float)((2.0 / ((double)N * N * N)) / (-2.0 * 3.14159265358979323846));
        const long long total = (long long)units * (N * (H / RC::W) + N / RC::W);
        long long grid = (long long)RC::MINB * h->num_sms;
        if (grid > total) grid = total;
        launch_pdl(k_ring<N, MODE>, dim3((unsigned)grid), dim3(ring_threads<N, MODE>()), ring_smem_bytes<N, MODE>(), st, p);
    }

    static void launch_zl_gbar(sap_dpsr* h, cudaStream_t st, const ZyFwdParams& z, int planes) {
        using ZC = ZlCfg<N, false>;
        ZlFwdParams p{z, planes};
        const long long total = (long long)planes * (N * N / ZC::NL);
        long long grid = (long long)ZC::MINB * h->num_sms;
        if (grid > total) grid = total;
        launch_pdl(k_zl_gbar<N>, dim3((unsigned)grid), dim3(zl_threads<N, false>()), zl_smem_bytes<N, false>(), st, p);
    }
    static void launch_zl_inv(sap_dpsr* h, cudaStream_t st, const float2* S, const float2* Q, float* out, int planes, int adj3 = 0,
                              bool listed = false) {
        using ZC = ZlCfg<N, true>;
        ZlInvParams p{S, Q, out, h->tw, planes, adj3, h->ftab, nullptr, h->nact, h->nbins, C::FUSED_ZY ? 1 : N / 32};
        if (listed && h->sparse && h->lists_valid) p.zlist = h->zlist;
        if constexpr (!C::FUSED_ZY) {
            static const bool ring = getenv("SAP_ZL_RING") && getenv("SAP_ZL_RING")[0] == '1';   // experiment: the ring kernel
            if (!ring) {
                const long long total = (long long)planes * (N * N / ZwCfg<N>::NL);
                long long grid = (long long)ZwCfg<N>::MINB * h->num_sms;
                if (grid > total) grid = total;
                launch_pdl(k_zw_inv<N>, dim3((unsigned)grid), dim3(ZwCfg<N>::NT), ZwCfg<N>::SMEM, st, p);
                return;
            }
        }
        const long long total = (long long)planes * (N * N / ZC::NL);
        long long grid = (long long)ZC::MINB * h->num_sms;
        if (grid > total) grid = total;
        launch_pdl(k_zl_inv<N>, dim3((unsigned)grid), dim3(zl_threads<N, true>()), zl_smem_bytes<N, true>(), st, p);
    }

    // ---- latency path: the whole forward / backward as one cooperative kernel (fused_small.cuh) ----
    static FusedParams fused_params(sap_dpsr* h, const float* pts, const float* nrm, int P, float* chi, const float* G, float* gp, float* gn) {
        FusedParams p;
        p.pts = pts; p.nrm = nrm; p.chi = chi; p.G = G; p.gp = gp; p.gn = gn; p.P = P; p.B = h->batch;
        p.spts = h->spts; p.snrm = h->snrm; p.bin_start = h->bin_start; p.hist = h->fhist;
        p.S3 = h->S3; p.Q3 = h->Q3; p.S1 = h->S1; p.Q1 = h->Q1; p.tw = h->tw; p.ftab = h->ftab;
        p.acc = h->facc; p.stats = h->stats; p.bw = h->bw; p.sync = h->fsync; p.stamps = h->fstamps;
        p.cs = (float)((2.0 / ((double)N * N * N)) / (-2.0 * 3.14159265358979323846));
        return p;
    }
    template <class K> static cudaError_t launch_fused(sap_dpsr* h, K kernel, cudaStream_t st, const FusedParams& p) {
        if constexpr (N <= 128) {
            cudaLaunchConfig_t cfg = {};
            cfg.gridDim = dim3((unsigned)h->num_sms); cfg.blockDim = dim3(FusedCfg<N>::NT);
            cfg.dynamicSmemBytes = FusedCfg<N>::BYTES; cfg.stream = st;
            cudaLaunchAttribute at[2];
            at[0].id = cudaLaunchAttributeCooperative; at[0].val.cooperative = 1;
            at[1].id = cudaLaunchAttributeProgrammaticStreamSerialization; at[1].val.programmaticStreamSerializationAllowed = 1;
            static const bool coop = !(getenv("SAP_FUSED_COOP") && getenv("SAP_FUSED_COOP")[0] == '0');
            if (!coop) at[0] = at[1];   // experiment: plain launch (148 CTAs of one per SM are co-resident in practice)
            cfg.attrs = at; cfg.numAttrs = (coop && h->fused_pdl) ? 2 : 1;
            cudaError_t e = cudaLaunchKernelEx(&cfg, kernel, p);
            if (e != cudaSuccess && h->fused_pdl) {  // this driver does not combine the two attributes: cooperative only
                cudaGetLastError();
                h->fused_pdl = 0;
                cfg.numAttrs = 1;
                e = cudaLaunchKernelEx(&cfg, kernel, p);
            }
            return e;
        } else {
            return cudaErrorInvalidValue;
        }
    }
    // SAP_PATH_AUTO: the latency path where it measured at least as fast as the 13-launch chain with a flushed L2 and
    // clearly faster back to back / from the host (2 launches instead of 13): N <= 64.  At 128^3 the chain of
    // programmatic dependent launches hides its launch latencies and wins (DESIGN.md 8a has the phase table).
    static bool use_fused(const sap_dpsr* h) {
        if (!h->fused_ok || h->path == SAP_PATH_THROUGHPUT) return false;
        return h->path == SAP_PATH_LATENCY || N <= 64;
    }

    static sap_status_t forward(sap_dpsr* h, const float* pts, const float* nrm, int P, float* chi, cudaStream_t st,
                                const float* chi_gt = nullptr, float* loss = nullptr) {
        const int B = h->batch;
        const size_t V = (size_t)N * N * N;
        prof_begin(h, st);
        if constexpr (N <= 128) {
            if (use_fused(h) && !chi_gt) {
                const FusedParams p = fused_params(h, pts, nrm, P, chi, nullptr, nullptr, nullptr);
                if (!cuda_ok(h, launch_fused(h, k_fused_fwd<N>, st, p), "k_fused_fwd")) return SAP_ERR_CUDA;
                SAP_LAUNCH_CHECK(h, "k_fused_fwd");
                h->binned_P = P;
                h->mse_valid = false;
                h->lists_valid = false;   // the latency path bins the points itself and writes no activity lists
                return SAP_OK;
            }
        }
        // F1a: bin the points (counting sort); the rasterisation itself happens inside k_zy_fwd
        bool sorted_in_one = false;
        {
            const dim3 gp((P + 255) / 256, B);
            constexpr int KT = C::FUSED_ZY ? 0 : H / RingCfg<N>::W, NYQT = C::FUSED_ZY ? 0 : N / RingCfg<N>::W;
            static_assert(C::FUSED_ZY || RingCfg<N>::W == 16, "ylist is sized for 16-column y-pass tiles");
            const ActLists al{h->plane_act, h->sparse ? h->zlist : nullptr, h->ylist, h->nact, h->tile_bits, h->plane_bits, N, N / C::NL, KT, NYQT};
            // one launch when every point fits the registers of a co-resident grid (BIN_PPT per thread), else three
            int gx = (int)gp.x < h->bin_gx_max ? (int)gp.x : h->bin_gx_max;
            if (P >= 65536) {   // large clouds: four points per thread -- every block scans all the bin counts (64 KB of sectors at
                                // 256^3) and arrives at the grid barrier, so fewer, fatter blocks (256^3, 100,000 points: 19.4 -> 17.7 us)
                int want = (P + 1023) / 1024;
                const int floor_ = (h->num_sms + B - 1) / B;
                if (want < floor_) want = floor_;
                if (want < gx) gx = want;
            }
            // (measured with one counter per 32-byte sector: 480,000 points 31 us against 48 us for the three kernels, 10^6 points
            // 131 us against 98 us -- every counting atomic returns a value and they all arrive at once)
            constexpr long long bin1_max = 524288;
            sorted_in_one = h->bin_gx_max >= 1 && (long long)gx * 256 * BIN_PPT >= P && (long long)B * P <= bin1_max;
            if (sorted_in_one) {
                const BinSortParams bp{pts, nrm, P, N, C::NL, h->nbins, h->bin_cnt, h->bin_start, h->spts, h->snrm, h->nmax, h->bsync, al};
                if (!cuda_ok(h, launch_coop(h, k_bin_sort, dim3(gx + 1, B), dim3(256), (size_t)(h->nbins + 1) * sizeof(int), st, bp), "k_bin_sort")) return SAP_ERR_CUDA;
                SAP_LAUNCH_CHECK(h, "k_bin_sort");
            } else {
                launch_pdl(k_bin_count, dim3(gp), dim3(256), 0, st, pts, P, N, C::NL, h->nbins, h->bin_cnt, h->nact);
                SAP_LAUNCH_CHECK(h, "k_bin_count");
                launch_pdl(k_bin_scan, dim3(B), dim3(1024), (size_t)h->nbins * sizeof(int), st, h->bin_cnt, h->nbins, P, h->bin_start, h->bin_cursor, h->nmax);
                SAP_LAUNCH_CHECK(h, "k_bin_scan");
                launch_pdl(k_bin_scatter, dim3(gp.x + 1, B), dim3(256), (size_t)(h->nbins + 1) * sizeof(int), st, pts, nrm, P, N, C::NL, h->nbins, h->bin_cursor,
                           h->spts, h->snrm, h->nmax, (const int*)h->bin_start, al);
                SAP_LAUNCH_CHECK(h, "k_bin_scatter");
            }
            h->lists_valid = h->sparse;
            h->binned_P = P;
        }
        // F2 z (+y) forward, 3 channels
        {
            ZyFwdParams p{h->spts, h->snrm, h->bin_start, P, nullptr, nullptr, h->S3, C::FUSED_ZY ? h->Q3 : h->QT3, h->tw, 3, h->nmax,
                          (h->sparse && (!C::FUSED_ZY || h->mask_solve)) ? h->plane_act : nullptr, sorted_in_one ? h->bin_cnt : nullptr, B * h->nbins * BIN_CS, h->bsync};
            if constexpr (C::FUSED_ZY)
                launch_pdl(k_zy_fwd<N, C::NL, C::FUSED_ZY, SRC_SPLAT, C::NT_ZY>, dim3(N * N / C::NL, B * 3), dim3(C::NT_ZY), zy_smem_bytes<N, C::NL>(), st, p);
            else
                launch_pdl(k_zw_fwd<N, SRC_SPLAT>, dim3(N * N / ZwCfg<N>::NL, B), dim3(ZwCfg<N>::NT), ZwCfg<N>::SMEM, st, p);
            SAP_LAUNCH_CHECK(h, C::FUSED_ZY ? "k_zy_fwd" : "k_zw_fwd<SPLAT>");
        }
        if constexpr (!C::FUSED_ZY) {
            launch_ring<MODE_FWD3>(h, st, B, h->mS3y, h->mQT3, h->S3, h->Q3, 1);  // planes (x, u, -) out of (x, y, z)
            SAP_LAUNCH_CHECK(h, "k_ring<FWD,y>");
        }
        // F2x + F3 + F4x: x forward, spectral solve, x inverse (3 -> 1)
        launch_ring<MODE_SOLVE>(h, st, B, h->mS3x, h->mQ3, h->S1, C::FUSED_ZY ? h->Q1 : h->QT1, 0);
        SAP_LAUNCH_CHECK(h, "k_ring<SOLVE>");
        if constexpr (!C::FUSED_ZY) {
            launch_ring<MODE_INV>(h, st, B, h->mS1y, h->mQT1, h->S1, h->Q1, 1);
            SAP_LAUNCH_CHECK(h, "k_ring<INV,y>");
        }
        // F4 (y +) z inverse -> chi'
        {
            launch_zl_inv(h, st, h->S1, h->Q1, chi, B);
            SAP_LAUNCH_CHECK(h, C::FUSED_ZY ? "k_zl_inv" : "k_zw_inv");
        }
        // F5 normalise
        {
            int nb = (P + 255) / 256; if (nb > 2 * h->num_sms) nb = 2 * h->num_sms;
            launch_pdl(k_sample_mean, dim3(dim3(nb, B)), dim3(256), 0, st, (const float4*)h->spts, P, N, (const float*)chi, h->acc, h->ticket, h->stats);
            SAP_LAUNCH_CHECK(h, "k_sample_mean");
            const size_t n4 = V / 4;
            int gb = (int)((n4 + 255) / 256); const int cap = (h->num_sms * 8 + B - 1) / B; if (gb > cap) gb = cap; if (gb < 1) gb = 1;
            if (chi_gt) {
                launch_pdl(k_scale_shift_mse, dim3(gb, B), dim3(256), 0, st, reinterpret_cast<float4*>(chi), reinterpret_cast<const float4*>(chi_gt),
                           reinterpret_cast<float4*>(h->gmse), n4, P, (const float*)h->stats, h->acc_mse, h->ticket + B, h->bw, loss);
            } else {
                launch_pdl(k_scale_shift, dim3(gb, B), dim3(256), 0, st, reinterpret_cast<float4*>(chi), n4, (const float*)h->stats);
            }
            h->mse_valid = chi_gt != nullptr;
            SAP_LAUNCH_CHECK(h, chi_gt ? "k_scale_shift_mse" : "k_scale_shift");
        }
        return SAP_OK;
    }

    static sap_status_t backward(sap_dpsr* h, const float* pts, const float* nrm, int P, const float* chi,
                                 const float* gchi, float* gp, float* gn, cudaStream_t st, bool have_bw = false) {
        const int B = h->batch;
        const size_t V = (size_t)N * N * N;
        prof_begin(h, st);
        if constexpr (N <= 128) {
            if (use_fused(h) && !have_bw) {
                const FusedParams p = fused_params(h, pts, nrm, P, const_cast<float*>(chi), gchi, gp, gn);
                if (!cuda_ok(h, launch_fused(h, k_fused_bwd<N>, st, p), "k_fused_bwd")) return SAP_ERR_CUDA;
                SAP_LAUNCH_CHECK(h, "k_fused_bwd");
                return SAP_OK;
            }
        }
        // B1 reductions (already done by the fused loss pass of sap_dpsr_forward_mse)
        if (!have_bw) {
            const size_t n4 = V / 4;
            int gb = (int)((n4 + 255) / 256); const int cap = (h->num_sms * 4 + B - 1) / B; if (gb > cap) gb = cap; if (gb < 1) gb = 1;
            launch_pdl(k_reduce_g, dim3(dim3(gb, B)), dim3(256), 0, st, reinterpret_cast<const float4*>(gchi), reinterpret_cast<const float4*>(chi),
                                                   n4, P, h->stats, h->acc + B, h->ticket + B, h->bw);
            SAP_LAUNCH_CHECK(h, "k_reduce_g");
        }
        // B2 + B3: Gbar' assembled on load, z (+y) forward
        {
            ZyFwdParams p{h->spts, h->snrm, h->bin_start, P, gchi, h->bw, h->S1, C::FUSED_ZY ? h->Q1 : h->QT1, h->tw, 1, h->nmax, nullptr, nullptr, 0, nullptr};
            if constexpr (C::FUSED_ZY) launch_zl_gbar(h, st, p, B);
            else launch_pdl(k_zw_fwd<N, SRC_GBAR>, dim3(N * N / ZwCfg<N>::NL, B), dim3(ZwCfg<N>::NT), ZwCfg<N>::SMEM, st, p);
            SAP_LAUNCH_CHECK(h, C::FUSED_ZY ? "k_zl_gbar" : "k_zw_fwd<GBAR>");
        }
        if constexpr (!C::FUSED_ZY) {
            launch_ring<MODE_FWD>(h, st, B, h->mS1y, h->mQT1, h->S1, h->Q1, 1);
            SAP_LAUNCH_CHECK(h, "k_ring<FWD,y>");
        }
        // B3x + B4 + B5x: x forward, transposed multiplier, 3 x inverse
        launch_ring<MODE_ADJ>(h, st, B, h->mS1x, h->mQ1, h->S3, C::FUSED_ZY ? h->Q3 : h->QT3, 0);
        SAP_LAUNCH_CHECK(h, "k_ring<ADJ>");
        if constexpr (!C::FUSED_ZY) {
            launch_ring<MODE_INV3>(h, st, B, h->mS3y, h->mQT3, h->S3, h->Q3, 1);  // planes (x, y, z) out of (x, B, -)
            SAP_LAUNCH_CHECK(h, "k_ring<INV,y>");
        }
        // B5 (y +) z inverse -> vbar (into the v workspace)
        {
            launch_zl_inv(h, st, h->S3, h->Q3, h->v, B * 3, C::FUSED_ZY ? 1 : 0, true);  // fused: planes (x, B, -) -> (x, y, z)
            SAP_LAUNCH_CHECK(h, C::FUSED_ZY ? "k_zl_inv" : "k_zw_inv");
        }
        // B6 gather
        launch_pdl(k_gather_grads, dim3(dim3((P + 127) / 128, B)), dim3(128), 0, st, (const float4*)h->spts, (const float4*)h->snrm, P, N, (const float*)h->v, chi, (const float*)h->bw, gp, gn);
        SAP_LAUNCH_CHECK(h, "k_gather_grads");
        return SAP_OK;
    }
};

template <class F> static sap_status_t dispatch(int N, F&& f) {
    switch (N) {
        case 32: return f(Runner<32>{});
        case 64: return f(Runner<64>{});
        case 128: return f(Runner<128>{});
        case 256: return f(Runner<256>{});
        case 512: return f(Runner<512>{});
        default: return SAP_ERR_UNSUPPORTED;
    }
}

}  // namespace sap

// ================================================================================================
// C ABI (include/sap_dpsr.h)
// ================================================================================================
using namespace sap;

static bool supported_N(int N) { return N == 32 || N == 64 || N == 128 || N == 256 || N == 512; }

static void free_all(sap_dpsr* h) {
    for (int i = 0; i < sap_dpsr::MAX_EV; ++i) if (h->ev[i]) cudaEventDestroy(h->ev[i]);
    cudaFree(h->v); cudaFree(h->spts); cudaFree(h->snrm); cudaFree(h->bin_cnt); cudaFree(h->bin_cursor); cudaFree(h->bin_start); cudaFree(h->S3); cudaFree(h->Q3); cudaFree(h->S1); cudaFree(h->Q1); cudaFree(h->QT3); cudaFree(h->QT1); cudaFree(h->tw); cudaFree(h->ftab);
    cudaFree(h->fhist); cudaFree(h->facc); cudaFree(h->fsync); cudaFree(h->fstamps);
    cudaFree(h->bsync);
    cudaFree(h->tile_bits); cudaFree(h->plane_bits); cudaFree(h->plane_act); cudaFree(h->zlist); cudaFree(h->ylist); cudaFree(h->nact);
    cudaFree(h->gmse); cudaFree(h->acc_mse); cudaFree(h->acc); cudaFree(h->ticket); cudaFree(h->stats); cudaFree(h->bw); cudaFree(h->nmax);
    cudaFree(h->h_pts); cudaFree(h->h_nrm); cudaFree(h->h_chi); cudaFree(h->h_gchi); cudaFree(h->h_gp); cudaFree(h->h_gn);
}

extern "C" sap_status_t sap_dpsr_create(int N, float sigma, int batch, int max_points, sap_dpsr_t** out) {
    g_create_err.clear();
    if (!out) { g_create_err = "out is NULL"; return SAP_ERR_INVALID_ARG; }
    if (N <= 0 || batch <= 0 || max_points <= 0) { g_create_err = "N, batch and max_points must be positive"; return SAP_ERR_INVALID_ARG; }
    if (!(sigma >= 0.f) || !isfinite(sigma)) { g_create_err = "sigma must be finite and >= 0"; return SAP_ERR_INVALID_ARG; }
    if (!supported_N(N)) { g_create_err = "N must be one of 32, 64, 128, 256, 512"; return SAP_ERR_UNSUPPORTED; }
    if ((long long)batch * 3 > 65535) { g_create_err = "batch too large (batch*3 must fit gridDim.y)"; return SAP_ERR_UNSUPPORTED; }
    int dev = 0;
    if (!cuda_ok(nullptr, cudaGetDevice(&dev), "cudaGetDevice")) return SAP_ERR_CUDA;
    cudaDeviceProp prop;
    if (!cuda_ok(nullptr, cudaGetDeviceProperties(&prop, dev), "cudaGetDeviceProperties")) return SAP_ERR_CUDA;
    if (prop.major != 10) { g_create_err = "device is not sm_100 (Blackwell B200); this library has no other code path"; return SAP_ERR_UNSUPPORTED; }

    sap_dpsr* h = new (std::nothrow) sap_dpsr;
    if (!h) { g_create_err = "host allocation failed"; return SAP_ERR_OOM; }
    h->num_sms = prop.multiProcessorCount; h->N = N; h->sigma = sigma; h->batch = batch; h->max_points = max_points; h->device = dev;
    const size_t V = (size_t)N * N * N, SP = (size_t)N * N * (N / 2), QP = (size_t)N * N, B = (size_t)batch;
    cudaError_t e = cudaSuccess;
    auto upd = [&](cudaError_t x) { if (e == cudaSuccess) e = x; };
    h->nbins = N * (N <= 128 ? 1 : N / 32);
    upd(dev_alloc(h, &h->v, B * 3 * V));
    upd(dev_alloc(h, &h->spts, B * (size_t)max_points));
    upd(dev_alloc(h, &h->snrm, B * (size_t)max_points));
    upd(dev_alloc(h, &h->bin_cnt, B * (size_t)h->nbins * BIN_CS));
    upd(dev_alloc(h, &h->bin_cursor, B * (size_t)h->nbins * BIN_CS));
    upd(dev_alloc(h, &h->bin_start, B * (size_t)(h->nbins + 1)));
    upd(dev_alloc(h, &h->bsync, (size_t)4));
    upd(dev_alloc(h, &h->S3, B * 3 * SP));
    upd(dev_alloc(h, &h->Q3, B * 3 * QP));
    upd(dev_alloc(h, &h->S1, B * SP));
    upd(dev_alloc(h, &h->Q1, B * QP));
    if (N >= 256) { upd(dev_alloc(h, &h->QT3, B * 3 * QP)); upd(dev_alloc(h, &h->QT1, B * QP)); }
    upd(dev_alloc(h, &h->tw, (size_t)N));
    upd(dev_alloc(h, &h->ftab, (size_t)(N + N / 2 + 1)));
    upd(dev_alloc(h, &h->acc, B * 3));
    upd(dev_alloc(h, &h->ticket, B * 2));
    upd(dev_alloc(h, &h->stats, B * 4));
    upd(dev_alloc(h, &h->bw, B * 4));
    upd(dev_alloc(h, &h->nmax, B));
    {
        const char* dense = getenv("SAP_DENSE");
        h->sparse = !(dense && dense[0] == '1');
        upd(dev_alloc(h, &h->plane_act, B * (size_t)N));
        upd(dev_alloc(h, &h->zlist, B * (size_t)h->nbins));
        if (N >= 256) upd(dev_alloc(h, &h->ylist, B * ((size_t)N * (N / 2 / 16) + N / 16)));
        upd(dev_alloc(h, &h->nact, (size_t)4));
        upd(dev_alloc(h, &h->tile_bits, B * (size_t)(h->nbins / 32)));
        upd(dev_alloc(h, &h->plane_bits, B * (size_t)(N / 32)));
        // Measured: at 128^3 x 32 the splat pass drops from 224 to 192 us when it need not write the zeros of the inactive planes and
        // the (memory-bound) solve is not slower for masking them; with one grid in flight the masks cost the solve 1.7 us and
        // buy nothing, and for N >= 256 they cost the instruction-bound solve more than the z pass gains
        h->mask_solve = N <= 128 && (long long)batch * N >= 4LL * h->num_sms;
    }
    h->fused_ok = (N <= 128) && ((long long)batch * N <= h->num_sms) && batch <= (N == 32 ? 4 : N == 64 ? 2 : 1);
    if (h->fused_ok) {
        upd(dev_alloc(h, &h->fhist, B * (size_t)h->num_sms * N));
        upd(dev_alloc(h, &h->facc, B * 2));
        upd(dev_alloc(h, &h->fsync, (size_t)4));
        upd(dev_alloc(h, &h->fstamps, (size_t)64));
    }
    if (e != cudaSuccess) {
        cuda_ok(nullptr, e, "cudaMalloc(workspace)");
        const bool oom = (e == cudaErrorMemoryAllocation);
        free_all(h); delete h; cudaGetLastError();
        return oom ? SAP_ERR_OOM : SAP_ERR_CUDA;
    }
    // twiddle table exp(-2 pi i t / N) computed in double
    float2* tw = new (std::nothrow) float2[N];
    if (!tw) { free_all(h); delete h; g_create_err = "host allocation failed"; return SAP_ERR_OOM; }
    for (int t = 0; t < N; ++t) {
        const double a = -2.0 * 3.14159265358979323846 * (double)t / (double)N;
        tw[t] = make_float2((float)cos(a), (float)sin(a));
    }
    upd(cudaMemcpy(h->tw, tw, sizeof(float2) * N, cudaMemcpyHostToDevice));
    delete[] tw;
    upd(cudaMemset(h->bin_cnt, 0, sizeof(int) * B * h->nbins * BIN_CS));
    upd(cudaMemset(h->acc, 0, sizeof(double) * B * 3));
    upd(cudaMemset(h->ticket, 0, sizeof(unsigned) * B * 2));
    upd(cudaMemset(h->stats, 0, sizeof(float) * B * 4));
    upd(cudaMemset(h->bw, 0, sizeof(float) * B * 4));
    upd(cudaMemset(h->nmax, 0, sizeof(unsigned) * B));
    upd(cudaMemset(h->nact, 0, sizeof(int) * 4));
    upd(cudaMemset(h->bsync, 0, sizeof(unsigned) * 4));
    {   // single-launch binning: all its blocks must be co-resident (grid barrier)
        int occ = 0;
        const size_t sm = (size_t)(h->nbins + 1) * sizeof(int);
        upd(cudaFuncSetAttribute(k_bin_sort, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm));
        upd(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_bin_sort, 256, sm));
        const char* b3 = getenv("SAP_BIN3");
        h->bin_gx_max = (b3 && b3[0] == '1') ? 0 : (int)(((long long)occ * h->num_sms) / batch) - 1;   // + 1 publisher block per item
    }
    if (h->fused_ok) {
        upd(cudaMemset(h->facc, 0, sizeof(double) * B * 2));
        upd(cudaMemset(h->fsync, 0, sizeof(unsigned) * 4));
        upd(cudaMemset(h->fstamps, 0, sizeof(long long) * 64));
    }
    sap_status_t st = SAP_OK;
    if (e != cudaSuccess) { cuda_ok(nullptr, e, "workspace init"); st = SAP_ERR_CUDA; }
    if (st == SAP_OK) {
        st = dispatch(N, [&](auto r) { return decltype(r)::prepare(h); });
        if (st != SAP_OK) g_create_err = h->err;
    }
    if (st != SAP_OK) { free_all(h); delete h; return st; }
    *out = h;
    return SAP_OK;
}

// the workspace, the TMA descriptors and every buffer the caller passes live on the device the handle was created on
static sap_status_t check_device(sap_dpsr* h) {
    int dev = -1;
    if (!cuda_ok(h, cudaGetDevice(&dev), "cudaGetDevice")) return SAP_ERR_CUDA;
    if (dev != h->device) {
        char buf[160];
        snprintf(buf, sizeof buf, "current CUDA device is %d but the handle was created on device %d (call cudaSetDevice first)", dev, h->device);
        h->err = buf;
        return SAP_ERR_INVALID_ARG;
    }
    return SAP_OK;
}
static void mark_forward(sap_dpsr* h, int kind) { ++h->epoch; h->fwd_kind = kind; }

static sap_status_t check_common(sap_dpsr* h, int num_points) {
    if (!h) return SAP_ERR_INVALID_ARG;
    h->err.clear();
    h->launches = 0;
    if (num_points < 1 || num_points > h->max_points) { h->err = "num_points out of range [1, max_points]"; return SAP_ERR_INVALID_ARG; }
    return check_device(h);
}

extern "C" sap_status_t sap_dpsr_forward(sap_dpsr_t* h, const float* points, const float* normals, int num_points,
                                         float* chi, void* stream) {
    sap_status_t st = check_common(h, num_points);
    if (st != SAP_OK) return st;
    if (!points || !normals || !chi) { h->err = "null pointer argument"; return SAP_ERR_INVALID_ARG; }
    mark_forward(h, sap_dpsr::FWD_DEVICE);
    return dispatch(h->N, [&](auto r) { return decltype(r)::forward(h, points, normals, num_points, chi, (cudaStream_t)stream); });
}

extern "C" sap_status_t sap_dpsr_backward(sap_dpsr_t* h, const float* points, const float* normals, int num_points,
                                          const float* chi, const float* grad_chi, float* grad_points,
                                          float* grad_normals, void* stream) {
    sap_status_t st = check_common(h, num_points);
    if (st != SAP_OK) return st;
    if (!points || !normals || !chi || !grad_chi || !grad_points || !grad_normals) { h->err = "null pointer argument"; return SAP_ERR_INVALID_ARG; }
    if ((h->fwd_kind != sap_dpsr::FWD_DEVICE && h->fwd_kind != sap_dpsr::FWD_MSE) || num_points != h->binned_P) {
        h->err = "sap_dpsr_backward must follow sap_dpsr_forward (or sap_dpsr_forward_mse) on this handle with the same num_points";
        return SAP_ERR_INVALID_ARG;
    }
    return dispatch(h->N, [&](auto r) {
        return decltype(r)::backward(h, points, normals, num_points, chi, grad_chi, grad_points, grad_normals, (cudaStream_t)stream);
    });
}

static sap_status_t ensure_mse(sap_dpsr* h) {
    if (h->gmse) return SAP_OK;
    const size_t V = (size_t)h->N * h->N * h->N, B = (size_t)h->batch;
    cudaError_t e = dev_alloc(h, &h->gmse, B * V);
    if (e == cudaSuccess) e = dev_alloc(h, &h->acc_mse, B * 3);
    if (e == cudaSuccess) e = cudaMemset(h->acc_mse, 0, sizeof(double) * B * 3);
    if (e != cudaSuccess) {
        cuda_ok(h, e, "cudaMalloc(fused-loss workspace)");
        cudaFree(h->gmse); cudaFree(h->acc_mse);
        h->gmse = nullptr; h->acc_mse = nullptr;
        cudaGetLastError();
        return e == cudaErrorMemoryAllocation ? SAP_ERR_OOM : SAP_ERR_CUDA;
    }
    return SAP_OK;
}

extern "C" sap_status_t sap_dpsr_forward_mse(sap_dpsr_t* h, const float* points, const float* normals, int num_points,
                                             const float* chi_gt, float* chi, float* loss, void* stream) {
    sap_status_t st = check_common(h, num_points);
    if (st != SAP_OK) return st;
    if (!points || !normals || !chi_gt || !chi || !loss) { h->err = "null pointer argument"; return SAP_ERR_INVALID_ARG; }
    if ((st = ensure_mse(h)) != SAP_OK) return st;
    mark_forward(h, sap_dpsr::FWD_MSE);
    return dispatch(h->N, [&](auto r) {
        return decltype(r)::forward(h, points, normals, num_points, chi, (cudaStream_t)stream, chi_gt, loss);
    });
}

extern "C" sap_status_t sap_dpsr_backward_mse(sap_dpsr_t* h, const float* points, const float* normals, int num_points,
                                              const float* chi, float* grad_points, float* grad_normals, void* stream) {
    sap_status_t st = check_common(h, num_points);
    if (st != SAP_OK) return st;
    if (!points || !normals || !chi || !grad_points || !grad_normals) { h->err = "null pointer argument"; return SAP_ERR_INVALID_ARG; }
    if (h->fwd_kind != sap_dpsr::FWD_MSE || !h->mse_valid || num_points != h->binned_P) {
        h->err = "sap_dpsr_backward_mse must follow sap_dpsr_forward_mse on this handle with the same num_points";
        return SAP_ERR_INVALID_ARG;
    }
    return dispatch(h->N, [&](auto r) {
        return decltype(r)::backward(h, points, normals, num_points, chi, h->gmse, grad_points, grad_normals, (cudaStream_t)stream, true);
    });
}

static sap_status_t ensure_staging(sap_dpsr* h) {
    if (h->h_pts) return SAP_OK;
    const size_t V = (size_t)h->N * h->N * h->N, B = (size_t)h->batch, PP = B * (size_t)h->max_points * 3;
    cudaError_t e = cudaSuccess;
    auto upd = [&](cudaError_t x) { if (e == cudaSuccess) e = x; };
    upd(dev_alloc(h, &h->h_pts, PP)); upd(dev_alloc(h, &h->h_nrm, PP));
    upd(dev_alloc(h, &h->h_gp, PP)); upd(dev_alloc(h, &h->h_gn, PP));
    upd(dev_alloc(h, &h->h_chi, B * V)); upd(dev_alloc(h, &h->h_gchi, B * V));
    if (e != cudaSuccess) {
        cuda_ok(h, e, "cudaMalloc(staging)");
        cudaFree(h->h_pts); cudaFree(h->h_nrm); cudaFree(h->h_gp); cudaFree(h->h_gn); cudaFree(h->h_chi); cudaFree(h->h_gchi);
        h->h_pts = h->h_nrm = h->h_gp = h->h_gn = h->h_chi = h->h_gchi = nullptr;
        cudaGetLastError();
        return e == cudaErrorMemoryAllocation ? SAP_ERR_OOM : SAP_ERR_CUDA;
    }
    return SAP_OK;
}

extern "C" sap_status_t sap_dpsr_forward_host(sap_dpsr_t* h, const float* points_host, const float* normals_host,
                                              int num_points, float* chi_host, void* stream) {
    sap_status_t st = check_common(h, num_points);
    if (st != SAP_OK) return st;
    if (!points_host || !normals_host) { h->err = "null pointer argument"; return SAP_ERR_INVALID_ARG; }
    if ((st = ensure_staging(h)) != SAP_OK) return st;
    mark_forward(h, sap_dpsr::FWD_HOST);
    cudaStream_t s = (cudaStream_t)stream;
    const size_t pb = (size_t)h->batch * num_points * 3 * sizeof(float);
    const size_t vb = (size_t)h->batch * h->N * h->N * h->N * sizeof(float);
    if (!cuda_ok(h, cudaMemcpyAsync(h->h_pts, points_host, pb, cudaMemcpyHostToDevice, s), "H2D points")) return SAP_ERR_CUDA;
    if (!cuda_ok(h, cudaMemcpyAsync(h->h_nrm, normals_host, pb, cudaMemcpyHostToDevice, s), "H2D normals")) return SAP_ERR_CUDA;
    st = dispatch(h->N, [&](auto r) { return decltype(r)::forward(h, h->h_pts, h->h_nrm, num_points, h->h_chi, s); });
    if (st != SAP_OK) return st;
    h->host_P = num_points;
    if (chi_host && !cuda_ok(h, cudaMemcpyAsync(chi_host, h->h_chi, vb, cudaMemcpyDeviceToHost, s), "D2H chi")) return SAP_ERR_CUDA;
    if (!cuda_ok(h, cudaStreamSynchronize(s), "cudaStreamSynchronize")) return SAP_ERR_CUDA;
    return SAP_OK;
}

extern "C" sap_status_t sap_dpsr_backward_host(sap_dpsr_t* h, const float* grad_chi_host, float* grad_points_host,
                                               float* grad_normals_host, void* stream) {
    if (!h) return SAP_ERR_INVALID_ARG;
    h->err.clear();
    const int keep = h->launches;
    if (check_device(h) != SAP_OK) return SAP_ERR_INVALID_ARG;
    if (!h->h_pts || h->host_P < 1 || h->fwd_kind != sap_dpsr::FWD_HOST) {
        h->err = "sap_dpsr_backward_host must follow sap_dpsr_forward_host (no other forward on this handle in between)";
        return SAP_ERR_INVALID_ARG;
    }
    if (!grad_chi_host || !grad_points_host || !grad_normals_host) { h->err = "null pointer argument"; return SAP_ERR_INVALID_ARG; }
    (void)keep;
    h->launches = 0;
    cudaStream_t s = (cudaStream_t)stream;
    const int P = h->host_P;
    const size_t pb = (size_t)h->batch * P * 3 * sizeof(float);
    const size_t vb = (size_t)h->batch * h->N * h->N * h->N * sizeof(float);
    if (!cuda_ok(h, cudaMemcpyAsync(h->h_gchi, grad_chi_host, vb, cudaMemcpyHostToDevice, s), "H2D grad_chi")) return SAP_ERR_CUDA;
    sap_status_t st = dispatch(h->N, [&](auto r) {
        return decltype(r)::backward(h, h->h_pts, h->h_nrm, P, h->h_chi, h->h_gchi, h->h_gp, h->h_gn, s);
    });
    if (st != SAP_OK) return st;
    if (!cuda_ok(h, cudaMemcpyAsync(grad_points_host, h->h_gp, pb, cudaMemcpyDeviceToHost, s), "D2H grad_points")) return SAP_ERR_CUDA;
    if (!cuda_ok(h, cudaMemcpyAsync(grad_normals_host, h->h_gn, pb, cudaMemcpyDeviceToHost, s), "D2H grad_normals")) return SAP_ERR_CUDA;
    if (!cuda_ok(h, cudaStreamSynchronize(s), "cudaStreamSynchronize")) return SAP_ERR_CUDA;
    return SAP_OK;
}

extern "C" sap_status_t sap_dpsr_get_stats(sap_dpsr_t* h, float* stats_host, void* stream) {
    if (!h) return SAP_ERR_INVALID_ARG;
    h->err.clear();
    if (!stats_host) { h->err = "null pointer argument"; return SAP_ERR_INVALID_ARG; }
    cudaStream_t s = (cudaStream_t)stream;
    float* tmp = new (std::nothrow) float[(size_t)h->batch * 4];
    if (!tmp) { h->err = "host allocation failed"; return SAP_ERR_OOM; }
    unsigned flag = 0, bflag = 0;
    bool ok = cuda_ok(h, cudaMemcpyAsync(tmp, h->stats, sizeof(float) * 4 * h->batch, cudaMemcpyDeviceToHost, s), "D2H stats") &&
              (!h->fsync || cuda_ok(h, cudaMemcpyAsync(&flag, h->fsync + 2, sizeof(unsigned), cudaMemcpyDeviceToHost, s), "D2H flag")) &&
              cuda_ok(h, cudaMemcpyAsync(&bflag, h->bsync + 2, sizeof(unsigned), cudaMemcpyDeviceToHost, s), "D2H flag") &&
              cuda_ok(h, cudaStreamSynchronize(s), "cudaStreamSynchronize");
    if (ok && bflag) {  // the barrier of k_bin_sort gave up waiting
        h->err = "k_bin_sort: grid barrier timed out; results of that call are invalid";
        cudaMemsetAsync(h->bsync, 0, sizeof(unsigned) * 4, s);
        cudaMemsetAsync(h->bin_cnt, 0, sizeof(int) * (size_t)h->batch * h->nbins * BIN_CS, s);
        cudaStreamSynchronize(s);
        delete[] tmp;
        return SAP_ERR_CUDA;
    }
    if (ok && flag) {  // a grid barrier of the fused path gave up waiting (the CTAs of the launch were not co-resident)
        h->err = "fused path: grid barrier timed out; results of that call are invalid";
        cudaMemsetAsync(h->fsync, 0, sizeof(unsigned) * 4, s);
        cudaMemsetAsync(h->facc, 0, sizeof(double) * 2 * h->batch, s);
        cudaStreamSynchronize(s);
        delete[] tmp;
        return SAP_ERR_CUDA;
    }
    if (ok) for (int b = 0; b < h->batch; ++b) for (int k = 0; k < 3; ++k) stats_host[b * 3 + k] = tmp[b * 4 + k];
    delete[] tmp;
    return ok ? SAP_OK : SAP_ERR_CUDA;
}

extern "C" sap_status_t sap_dpsr_set_sparse(sap_dpsr_t* h, int on) {
    if (!h) return SAP_ERR_INVALID_ARG;
    h->err.clear();
    h->sparse = on != 0;
    h->lists_valid = false;   // the next forward rebuilds (or drops) the lists
    return SAP_OK;
}
extern "C" sap_status_t sap_dpsr_get_activity(sap_dpsr_t* h, int* out_host, void* stream) {
    if (!h) return SAP_ERR_INVALID_ARG;
    h->err.clear();
    if (!out_host) { h->err = "null pointer argument"; return SAP_ERR_INVALID_ARG; }
    if (!h->sparse || !h->lists_valid) { h->err = "no activity lists (switched off, or the last forward took the latency path)"; return SAP_ERR_INVALID_ARG; }
    int n[4] = {0, 0, 0, 0};
    cudaStream_t s = (cudaStream_t)stream;
    if (!cuda_ok(h, cudaMemcpyAsync(n, h->nact, sizeof n, cudaMemcpyDeviceToHost, s), "D2H activity") ||
        !cuda_ok(h, cudaStreamSynchronize(s), "cudaStreamSynchronize")) return SAP_ERR_CUDA;
    out_host[0] = n[0]; out_host[1] = h->batch * h->nbins; out_host[2] = n[2]; out_host[3] = h->batch * h->N;
    return SAP_OK;
}

extern "C" void sap_dpsr_destroy(sap_dpsr_t* h) {
    if (!h) return;
    free_all(h);
    delete h;
}

extern "C" unsigned long long sap_dpsr_epoch(const sap_dpsr_t* h) { return h ? h->epoch : 0ull; }
extern "C" sap_status_t sap_dpsr_check_epoch(sap_dpsr_t* h, unsigned long long epoch) {
    if (!h) return SAP_ERR_INVALID_ARG;
    h->err.clear();
    if (epoch != h->epoch) {
        h->err = "stale forward: another forward has run on this handle since the one being differentiated "
                 "(bins and normalisation statistics now belong to the later call)";
        return SAP_ERR_INVALID_ARG;
    }
    return SAP_OK;
}

extern "C" sap_status_t sap_dpsr_reserve(sap_dpsr_t* h, int what) {
    if (!h) return SAP_ERR_INVALID_ARG;
    h->err.clear();
    sap_status_t st = check_device(h);
    if (st != SAP_OK) return st;
    if ((what & ~(SAP_RESERVE_MSE | SAP_RESERVE_HOST)) != 0) { h->err = "unknown reserve flag"; return SAP_ERR_INVALID_ARG; }
    if ((what & SAP_RESERVE_MSE) && (st = ensure_mse(h)) != SAP_OK) return st;
    if ((what & SAP_RESERVE_HOST) && (st = ensure_staging(h)) != SAP_OK) return st;
    return SAP_OK;
}

extern "C" const char* sap_dpsr_last_error(const sap_dpsr_t* h) { return h ? h->err.c_str() : g_create_err.c_str(); }
extern "C" size_t sap_dpsr_workspace_bytes(const sap_dpsr_t* h) { return h ? h->ws_bytes : 0; }
extern "C" int sap_dpsr_last_launch_count(const sap_dpsr_t* h) { return h ? h->launches : 0; }

extern "C" sap_status_t sap_dpsr_set_path(sap_dpsr_t* h, int path) {
    if (!h) return SAP_ERR_INVALID_ARG;
    h->err.clear();
    if (path != SAP_PATH_AUTO && path != SAP_PATH_THROUGHPUT && path != SAP_PATH_LATENCY) { h->err = "unknown path"; return SAP_ERR_INVALID_ARG; }
    if (path == SAP_PATH_LATENCY && !h->fused_ok) {
        h->err = "the latency path needs N <= 128 and batch * N <= number of SMs";
        return SAP_ERR_UNSUPPORTED;
    }
    h->path = path;
    return SAP_OK;
}
extern "C" int sap_dpsr_get_path(const sap_dpsr_t* h) {
    if (!h) return -1;
    if (!h->fused_ok || h->path == SAP_PATH_THROUGHPUT) return SAP_PATH_THROUGHPUT;
    return (h->path == SAP_PATH_LATENCY || h->N <= 64) ? SAP_PATH_LATENCY : SAP_PATH_THROUGHPUT;
}
// marks of the last fused forward (ids 0..28) and backward (32..52), stamped by CTA 0 with clock64
extern "C" int sap_dpsr_get_fused_phases(sap_dpsr_t* h, float* us, const char** names, int cap) {
    if (!h || !h->fstamps) return 0;
    long long t[64];
    if (cudaMemcpy(t, h->fstamps, sizeof t, cudaMemcpyDeviceToHost) != cudaSuccess) { cudaGetLastError(); return 0; }
    int khz = 1965000;
    cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, h->device);   // cycles -> microseconds at the nominal SM clock
    static const char* nm[64] = {};
    if (!nm[1]) {
        nm[1] = "F:hist"; nm[2] = "F:barrier1"; nm[3] = "F:offsets+scatter"; nm[4] = "F:barrier2"; nm[5] = "F:zero planes";
        nm[6] = "F:rasterise"; nm[7] = "F:z stage0"; nm[8] = "F:z stage1"; nm[9] = "F:split+y stage0"; nm[10] = "F:y last->HBM";
        nm[12] = "F:barrier3"; nm[13] = "F:x load+stage0"; nm[14] = "F:x last+solve"; nm[15] = "F:x inverse->HBM";
        nm[16] = "F:barrier4"; nm[17] = "F:load plane"; nm[22] = "F:inv y last"; nm[23] = "F:inv y stage0+split"; nm[24] = "F:inv z stage1";
        nm[25] = "F:inv z stage0"; nm[26] = "F:sample mean"; nm[27] = "F:barrier5"; nm[28] = "F:scale+store";
        nm[33] = "B:load+reduce+zero"; nm[34] = "B:barrier1"; nm[36] = "B:chi term+raster W"; nm[37] = "B:z stage0"; nm[38] = "B:z stage1";
        nm[39] = "B:split+y stage0"; nm[40] = "B:y last->HBM"; nm[42] = "B:barrier2"; nm[43] = "B:x load+stage0"; nm[44] = "B:x last+adjoint";
        nm[45] = "B:x inverse x2->HBM"; nm[46] = "B:barrier3"; nm[47] = "B:load planes"; nm[48] = "B:inv y last x3"; nm[49] = "B:inv y stage0+split x3"; nm[50] = "B:inv z stage1 x3";
        nm[51] = "B:inv z stage0 x3"; nm[52] = "B:gather";
    }
    int n = 0, prev = -1;
    for (int i = 0; i < 64 && n < cap; ++i) {
        if (i == 32) prev = -1;   // the backward is another launch (maybe another SM): its clock has another origin
        if (t[i] == 0) continue;
        if (prev >= 0 && nm[i] && t[i] >= t[prev]) {
            if (us) us[n] = (float)((double)(t[i] - t[prev]) / ((double)khz * 1e-3));
            if (names) names[n] = nm[i];
            ++n;
        }
        prev = i;
    }
    return n;
}

extern "C" sap_status_t sap_dpsr_set_profiling(sap_dpsr_t* h, int on) {
    if (!h) return SAP_ERR_INVALID_ARG;
    h->err.clear();
    if (on && !h->ev[0]) {
        for (int i = 0; i < sap_dpsr::MAX_EV; ++i)
            if (!cuda_ok(h, cudaEventCreate(&h->ev[i]), "cudaEventCreate")) return SAP_ERR_CUDA;
    }
    h->prof = on != 0;
    h->nev = 0;
    return SAP_OK;
}

extern "C" int sap_dpsr_get_profile(sap_dpsr_t* h, float* ms, const char** names, int cap) {
    if (!h || h->nev < 2) return 0;
    if (cudaEventSynchronize(h->ev[h->nev - 1]) != cudaSuccess) return 0;
    int n = 0;
    for (int i = 1; i < h->nev && n < cap; ++i, ++n) {
        float t = 0.f;
        cudaEventElapsedTime(&t, h->ev[i - 1], h->ev[i]);
        if (ms) ms[n] = t;
        if (names) names[n] = h->ev_name[i];
    }
    return n;
}
