// ring_pass.cuh -- persistent, TMA-fed strided-axis passes (x pass with the fused spectral solve; y pass for
// N >= 256).  A CTA owns a ring of NSTAGE shared-memory buffers, each one tile of N points x W contiguous columns
// (W*8-byte rows) fetched by ONE cp.async.bulk.tensor whose completion lands on an mbarrier.  NG consumer groups
// take alternate tiles: a group transforms its tile IN PLACE in the buffer, writes the result to HBM straight
// from registers and releases the buffer; the thread that sees the last warp of the group release it refills it
// at once with the tile NSTAGE items ahead.  Loads are therefore in flight during all of the arithmetic whatever
// the register count (the earlier one-tile-per-CTA kernel depended on occupancy for that overlap), and there is
// no producer warp.
//   MODE_FWD / MODE_INV : forward / inverse transform along y
//   MODE_SOLVE (F2x+F3+F4x): chi~ = i sum_c m_c v~_c; the y and z channels are combined before the x transform (their
//                            factors do not depend on x): 2 forward x transforms, the multiplier, 1 inverse, 1 channel out
//   MODE_ADJ   (B3x+B4+B5x): forward x on 1 channel, vbar~_c = -i m_c Gbar'~; the y and z channels are one inverse x
//                            transform scaled per column: 2 inverse x transforms, 3 channels out
// Equations: Eq.3 / Eq.12-17; multiplier and readings as in spectral.cuh.
#pragma once
#include <cuda.h>
#include <stdint.h>
#include "fft_core.cuh"
#include "spectral.cuh"

namespace sap {

template <int N> struct RingCfg;
// W columns per tile, NG consumer groups of NTC threads each (a group owns a tile from load to store; groups take
// alternate tiles so that one computes while the other waits at a stage barrier), NSTAGE ring buffers, MINB
// resident CTAs per SM
template <> struct RingCfg<32>  { static constexpr int W = 16, NTC = 128, NG = 1, NSTAGE = 4, MINB = 4; };
template <> struct RingCfg<64>  { static constexpr int W = 32, NTC = 256, NG = 1, NSTAGE = 4, MINB = 3; };
template <> struct RingCfg<128> { static constexpr int W = 16, NTC = 128, NG = 4, NSTAGE = 12, MINB = 1; };
template <> struct RingCfg<256> { static constexpr int W = 16, NTC = 256, NG = 2, NSTAGE = 6, MINB = 1; };
template <> struct RingCfg<512> { static constexpr int W = 16, NTC = 512, NG = 1, NSTAGE = 3, MINB = 1; };  // 64-byte rows (W = 8) measured 25% slower
// per-mode overrides (same W: the TMA boxes are shared); none at present.  Measured and rejected at N = 128: the
// solve with 3 groups and 13 buffers (4 spare for prefetch) was 7% slower than 4 groups and 12 buffers; at N = 512 the
// solve with 2 groups of 256 threads (64 accumulator registers per thread, spills) 18% slower than 1 group of 512.
template <int N, int MODE> struct RingCfgM : RingCfg<N> {};
template <int N, int MODE> constexpr int ring_threads() { return RingCfgM<N, MODE>::NTC * RingCfgM<N, MODE>::NG; }

// twiddle tables in shared memory: per stage with a stride > 1, ST x R entries [j][r] of float4 (see cmul4), one
// table for the forward direction and one (conjugated) for the inverse
template <int N> constexpr int ring_tw_entries() {
    return N + (Plan<N>::NS == 3 ? StageInfo<N, 1>::ST * StageInfo<N, 1>::R : 0);
}
template <int N, int MODE> constexpr size_t ring_smem_bytes() {
    using C = RingCfgM<N, MODE>;
    return (size_t)C::NSTAGE * N * C::W * sizeof(float2) + 2 * (size_t)ring_tw_entries<N>() * sizeof(float4) +
           (size_t)N * sizeof(float4) + 3 * C::NSTAGE * sizeof(uint64_t) + 128 +
           (size_t)ring_threads<N, MODE>() * sizeof(int) +  // tile ids of this CTA (listed mode)
           (N >= 256 && (MODE == MODE_FWD3 || MODE == MODE_INV3) ? 256 * sizeof(unsigned) : 0);   // activity bits of the z-pass tiles
}
constexpr size_t SMEM_PER_CTA_MAX = 227 * 1024;  // sm_100a opt-in limit per CTA
static_assert(ring_smem_bytes<32, MODE_SOLVE>() * 4 <= SMEM_PER_CTA_MAX + 4096 && ring_smem_bytes<64, MODE_SOLVE>() * 3 <= SMEM_PER_CTA_MAX &&
              ring_smem_bytes<128, MODE_SOLVE>() <= SMEM_PER_CTA_MAX && ring_smem_bytes<256, MODE_SOLVE>() <= SMEM_PER_CTA_MAX &&
              ring_smem_bytes<512, MODE_SOLVE>() <= SMEM_PER_CTA_MAX, "ring buffers + tables must fit the shared memory of an SM");
template <int N> constexpr int ring_box_rows() { return N < 256 ? N : 256; }  // TMA box dimension limit

struct RingParams {
    CUtensorMap mapS;    // main spectrum of the input array, box = one tile (or half a tile at N = 512)
    CUtensorMap mapQ;    // Nyquist plane of the input: [x][y] for the x pass, the transposed copy [y][x] for the y pass
    float2* outS;
    float2* outQ;
    const float2* tw;
    const float4* ftab;
    int units;           // planes (FWD / INV) or batch items (SOLVE / ADJ)
    int nyq_out_t;       // x pass: Nyquist-plane output is written transposed ([y][x]); the y pass always reads [y][x], writes [x][y]
    float cs;
    // listed mode of the 3-channel y passes (MODE_FWD3 / MODE_INV3; see ActLists in sap_dpsr.cu), nullptr = every tile:
    const int* ylist;    // global tile ids (unit * tiles_per_unit + T) of the tiles of the active planes + all Nyquist tiles.
                         // MODE_FWD3 runs in place: the rows of an inactive plane in the output planes 0 and 1 are the zeros
                         // the splat pass wrote there; MODE_INV3's output there is never read
    const int* nact;     // {-, |ylist|, -, -}
    // ... and inside an active plane the rows of the INACTIVE z-pass tiles (32 lines each) are neither written by the splat pass
    // (MODE_FWD3 fetches whatever is there with the tile and its stage 0 reads those rows as zeros; fetching only the active
    // rows with one 32-row box each was measured slower: 4 KB boxes, 8-16 per tile) nor stored by MODE_INV3 (the inverse z pass
    // does not read them)
    const unsigned* tile_bits;   // [units][N * (N / 32) / 32] activity bits of the z-pass tiles, bit x * (N / 32) + ty
    // MODE_SOLVE of the fused planes (N <= 128) in the throughput regime (sap_dpsr.cu decides), else nullptr: the splat pass
    // has not written the zeros of the inactive planes, the solve reads those rows as zeros (xrow_masks)
    const unsigned* plane_bits;  // [units][N / 32] activity bits of the x-planes
};

// ---- PTX wrappers ---------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* b, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* b, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(b)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* b) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(b)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* b, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "LAB_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
        "@P1 bra DONE;\n"
        "bra LAB_WAIT;\n"
        "DONE:\n"
        "}\n" ::"r"(smem_u32(b)), "r"(parity) : "memory");
}
__device__ __forceinline__ void tma_load_4d(uint32_t dst, const CUtensorMap* map, int c0, int c1, int c2, int c3, uint64_t* bar) {
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];"
        ::"r"(dst), "l"(reinterpret_cast<uint64_t>(map)), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tma_load_3d(uint32_t dst, const CUtensorMap* map, int c0, int c1, int c2, uint64_t* bar) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
        ::"r"(dst), "l"(reinterpret_cast<uint64_t>(map)), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(bar)) : "memory");
}
template <int NTC> __device__ __forceinline__ void consumer_sync(int group) { asm volatile("bar.sync %0, %1;" ::"r"(group + 1), "n"(NTC) : "memory"); }
// a * w with the table entry t = {w.x, w.y, -w.y, w.x} (forward) or {w.x, -w.y, w.y, w.x} (a * conj w): two
// packed instructions, no operand fix-ups
__device__ __forceinline__ float2 cmul4(float2 a, float4 t) {
    return __ffma2_rn(make_float2(a.y, a.y), make_float2(t.z, t.w), __fmul2_rn(make_float2(a.x, a.x), make_float2(t.x, t.y)));
}

}  // namespace sap

namespace sap {

// ---- in-place stages on a dense [N][W] tile; lanes run over the W columns -------------------------------
// Stage S (S = 0 or the middle stage of a 3-stage plan).  tab = this stage's twiddle table for this direction.
// swz = 15 for a y-pass tile of the main spectrum (row n holds z slot c in column c ^ (n & 15), see kz_swz), else 0.
// 32-row group of tile row q + r ST (q < ST): rowmask bit of the z-pass tile (32 lines) the row belongs to
template <int ST> __device__ __forceinline__ int ring_row_group(int q, int r) { return ((r * ST) >> 5) + (ST >= 32 ? (q >> 5) : 0); }
// rowmask (y-pass tiles, listed mode): bit g set = rows [32 g, 32 g + 32) of the tile belong to an active z-pass tile; the
// rows of the other groups are zeros that nobody wrote: stage 0 reads them as 0 whatever the buffer holds
// x-pass tiles of the solve (rows = x-planes) with the plane masks on: bit r of xm[i] says whether row q + r ST of the thread's
// i-th stage-0 task lies in an ACTIVE plane.  The rows of inactive planes are zeros that the splat pass did not write: stage 0
// reads them as 0 whatever the tile holds.  pw = the unit's N/32 plane-activity words.
template <int N, int W, int NTC>
__device__ __forceinline__ void xrow_masks(const unsigned* __restrict__ pw, int tid, unsigned (&xm)[2]) {
    constexpr int R = StageInfo<N, 0>::R, ST = StageInfo<N, 0>::ST, NT = ST * W;
    static_assert((NT + NTC - 1) / NTC <= 2, "at most two stage-0 tasks per thread");
#pragma unroll
    for (int i = 0; i < (NT + NTC - 1) / NTC; ++i) {
        const int q = (tid + i * NTC) / W;
        unsigned m = 0u;
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int x = (q + r * ST) & (N - 1);
            m |= ((__ldg(pw + (x >> 5)) >> (x & 31)) & 1u) << r;
        }
        xm[i] = m;
    }
}
template <int N, int S, int W, int NTC, bool INV>
__device__ __forceinline__ void ring_stage(float2* s, const float4* tab, int tid, int swz = 0, unsigned rowmask = 0xffffffffu,
                                           const unsigned* xm = nullptr) {
    constexpr int R = StageInfo<N, S>::R, ST = StageInfo<N, S>::ST;
    constexpr int NT = (N / R) * W;  // butterflies of the tile
#pragma unroll
    for (int i = 0; i < (NT + NTC - 1) / NTC; ++i) {
        const int t = tid + i * NTC;
        if (NT % NTC != 0 && t >= NT) break;
        const int q = t / W, c = t - q * W;
        const int blk = q / ST, j = q - blk * ST;
        const int row0 = blk * (R * ST) + j;
        const float4* tr = tab + j * R;
        float2 v[R];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            v[r] = s[(row0 + r * ST) * W + (c ^ ((row0 + r * ST) & swz))];
            if (S == 0 && !INV && !((rowmask >> ring_row_group<ST>(j, r)) & 1u)) v[r] = make_float2(0.f, 0.f);
            if (S == 0 && !INV && xm && !((xm[i] >> r) & 1u)) v[r] = make_float2(0.f, 0.f);
        }
        if (!INV) {
            dft_fwd<R>(v);
            if constexpr (ST > 1) {
#pragma unroll
                for (int r = 1; r < R; ++r) v[r] = cmul4(v[r], tr[r]);
            }
        } else {
            if constexpr (ST > 1) {
#pragma unroll
                for (int r = 1; r < R; ++r) v[r] = cmul4(v[r], tr[r]);
            }
            dft_inv<R>(v);
        }
#pragma unroll
        for (int r = 0; r < R; ++r) s[(row0 + r * ST) * W + (c ^ ((row0 + r * ST) & swz))] = v[r];
    }
}
// inverse stage 0: smem -> registers -> HBM.  out + off(row n, column c) = out[n * sn + c * sc]
template <int N, int W, int NTC>
__device__ __forceinline__ void ring_stage0_inv_store(const float2* s, const float4* tab, int tid, float2* out, unsigned sn, unsigned sc, int swz = 0,
                                                      unsigned rowmask = 0xffffffffu) {
    constexpr int R = StageInfo<N, 0>::R, ST = StageInfo<N, 0>::ST;
    constexpr int NT = ST * W;
#pragma unroll
    for (int i = 0; i < (NT + NTC - 1) / NTC; ++i) {
        const int t = tid + i * NTC;
        if (NT % NTC != 0 && t >= NT) break;
        const int q = t / W, c = t - q * W;
        const float4* tr = tab + q * R;
        float2 v[R];
#pragma unroll
        for (int r = 0; r < R; ++r) v[r] = s[(q + r * ST) * W + (c ^ ((q + r * ST) & swz))];
#pragma unroll
        for (int r = 1; r < R; ++r) v[r] = cmul4(v[r], tr[r]);
        dft_inv<R>(v);
#pragma unroll
        for (int r = 0; r < R; ++r)
            if ((rowmask >> ring_row_group<ST>(q, r)) & 1u) out[(unsigned)(q + r * ST) * sn + (unsigned)(c ^ ((q + r * ST) & swz)) * sc] = v[r];
    }
}

}  // namespace sap

namespace sap {

// Forward stage 0 of the x pass on the combination wy * s1 + wz * s2 of two channels, result in s1.  The y and z
// factors of the divergence (and of the adjoint) do not depend on x, so they commute with the transform along x:
// sum_c h_c v~_c needs two forward x transforms, not three (and the adjoint two inverse ones).
template <int N, int W, int NTC>
__device__ __forceinline__ void ring_stage0_fwd2(float2* s1, const float2* s2, const float4* tab, int tid, float wy, float wz,
                                                 const unsigned* xm = nullptr) {
    constexpr int R = StageInfo<N, 0>::R, ST = StageInfo<N, 0>::ST;
    constexpr int NT = ST * W;
#pragma unroll
    for (int i = 0; i < (NT + NTC - 1) / NTC; ++i) {
        const int t = tid + i * NTC;
        if (NT % NTC != 0 && t >= NT) break;
        const int q = t / W, c = t - q * W;
        const float4* tr = tab + q * R;
        float2 v[R];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            v[r] = caxpy(wz, s2[(q + r * ST) * W + c], cscale(wy, s1[(q + r * ST) * W + c]));
            if (xm && !((xm[i] >> r) & 1u)) v[r] = make_float2(0.f, 0.f);
        }
        dft_fwd<R>(v);
#pragma unroll
        for (int r = 1; r < R; ++r) v[r] = cmul4(v[r], tr[r]);
#pragma unroll
        for (int r = 0; r < R; ++r) s1[(q + r * ST) * W + c] = v[r];
    }
}
// inverse stage 0 of a y-pass tile with a per-column output factor scale(c), c = z slot inside the tile
template <int N, int W, int NTC, class F>
__device__ __forceinline__ void ring_stage0_inv_store_scaled(const float2* s, const float4* tab, int tid, float2* out, unsigned sn,
                                                             unsigned sc, int swz, F scale, unsigned rowmask = 0xffffffffu) {
    constexpr int R = StageInfo<N, 0>::R, ST = StageInfo<N, 0>::ST;
    constexpr int NT = ST * W;
#pragma unroll
    for (int i = 0; i < (NT + NTC - 1) / NTC; ++i) {
        const int t = tid + i * NTC;
        if (NT % NTC != 0 && t >= NT) break;
        const int q = t / W, c = t - q * W;
        const float4* tr = tab + q * R;
        const float w = scale(c);
        float2 v[R];
#pragma unroll
        for (int r = 0; r < R; ++r) v[r] = s[(q + r * ST) * W + (c ^ ((q + r * ST) & swz))];
#pragma unroll
        for (int r = 1; r < R; ++r) v[r] = cmul4(v[r], tr[r]);
        dft_inv<R>(v);
#pragma unroll
        for (int r = 0; r < R; ++r)
            if ((rowmask >> ring_row_group<ST>(q, r)) & 1u) out[(unsigned)(q + r * ST) * sn + (unsigned)(c ^ ((q + r * ST) & swz)) * sc] = cscale(w, v[r]);
    }
}
// forward stage 0 of a y-pass tile with a per-column input factor scale(c)
template <int N, int W, int NTC, class F>
__device__ __forceinline__ void ring_stage0_fwd_scaled(float2* s, const float4* tab, int tid, int swz, F scale, unsigned rowmask = 0xffffffffu) {
    constexpr int R = StageInfo<N, 0>::R, ST = StageInfo<N, 0>::ST;
    constexpr int NT = ST * W;
#pragma unroll
    for (int i = 0; i < (NT + NTC - 1) / NTC; ++i) {
        const int t = tid + i * NTC;
        if (NT % NTC != 0 && t >= NT) break;
        const int q = t / W, c = t - q * W;
        const float4* tr = tab + q * R;
        const float w = scale(c);
        float2 v[R];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            v[r] = cscale(w, s[(q + r * ST) * W + (c ^ ((q + r * ST) & swz))]);
            if (!((rowmask >> ring_row_group<ST>(q, r)) & 1u)) v[r] = make_float2(0.f, 0.f);
        }
        dft_fwd<R>(v);
#pragma unroll
        for (int r = 1; r < R; ++r) v[r] = cmul4(v[r], tr[r]);
#pragma unroll
        for (int r = 0; r < R; ++r) s[(q + r * ST) * W + (c ^ ((q + r * ST) & swz))] = v[r];
    }
}
template <int N, int MODE>
__global__ void __launch_bounds__(ring_threads<N, MODE>(), RingCfgM<N, MODE>::MINB) k_ring(const __grid_constant__ RingParams p) {
    using C = RingCfgM<N, MODE>;
    constexpr int W = C::W, NTC = C::NTC, NG = C::NG, NSTAGE = C::NSTAGE, H = N / 2;
    constexpr int AXIS = (MODE == MODE_FWD || MODE == MODE_INV || MODE == MODE_FWD3 || MODE == MODE_INV3) ? 1 : 0;  // y : x pass
    constexpr bool TWO_SPECTRA = (N >= 256);  // the y and z channels reach / leave the x pass as one spectrum
    constexpr int NS = Plan<N>::NS, LS = NS - 1, RL = StageInfo<N, LS>::R;
    static_assert(StageInfo<N, LS>::ST == 1 && NS >= 2, "plan");
    constexpr int R0 = StageInfo<N, 0>::R, R1 = StageInfo<N, 1>::R;
    constexpr int TWE = ring_tw_entries<N>();
    constexpr int TILE_ELEMS = N * W;
    constexpr uint32_t TILE_BYTES = TILE_ELEMS * sizeof(float2);
    constexpr int NB = ring_box_rows<N>();
    constexpr int NTASK = (N / RL) * W, TPT = NTASK / NTC;
    static_assert(NTASK % NTC == 0, "last-stage tasks divide evenly over the consumers");
    constexpr int KT = H / W, TILES_MAIN = N * KT, TILES_NYQ = N / W;
    // input items per tile, and the plane strides of the 3-channel arrays on either side
    constexpr int IN_CH = (MODE == MODE_SOLVE) ? (TWO_SPECTRA ? 2 : 3) : (MODE == MODE_FWD3 || MODE == MODE_INV3) ? 3 : 1;
    constexpr int IN_STRIDE = (MODE == MODE_SOLVE || MODE == MODE_FWD3 || MODE == MODE_INV3) ? 3 : 1;
    constexpr int OUT_CH = (MODE == MODE_ADJ || MODE == MODE_FWD3 || MODE == MODE_INV3) ? 3 : 1;
    constexpr size_t SPLANE = (size_t)N * N * H, QPLANE = (size_t)N * N;
    constexpr int tiles_per_unit = TILES_MAIN + TILES_NYQ;
    constexpr int IT_PER_TILE = IN_CH;

    extern __shared__ __align__(1024) unsigned char ring_smem[];
    float2* bufs = reinterpret_cast<float2*>(ring_smem);
    float4* tabF = reinterpret_cast<float4*>(bufs + (size_t)NSTAGE * TILE_ELEMS);
    float4* tabI = tabF + TWE;
    float4* fx = tabI + TWE;
    uint64_t* full = reinterpret_cast<uint64_t*>(fx + N);
    uint64_t* empty = full + NSTAGE;
    volatile int* issued = reinterpret_cast<volatile int*>(empty + NSTAGE);  // fills issued into each buffer so far
    int* tcache = const_cast<int*>(reinterpret_cast<volatile int*>(issued + NSTAGE + (NSTAGE & 1)));  // listed mode: this CTA's tile ids
    constexpr int TCAP = ring_threads<N, MODE>();
    constexpr bool CAN_LIST = (MODE == MODE_FWD3 || MODE == MODE_INV3);
    // The forward y passes read what the z pass before them wrote plane by plane in ascending x: they walk the planes in
    // DESCENDING x, so that the planes written last -- still in the 126 MB L2 -- are read first.
    constexpr bool REVERSED = (MODE == MODE_FWD3 || MODE == MODE_FWD);
    const int group = threadIdx.x / NTC, tid = threadIdx.x - group * NTC;

    for (int i = threadIdx.x; i < TWE; i += ring_threads<N, MODE>()) {
        int e;  // the entry is w_N^e
        if (i < N) { const int j = i / R0, r = i - j * R0; e = r * j; }
        else { const int k = i - N, j = k / R1, r = k - j * R1; e = r * j * R0; }
        const float2 w = p.tw[e];
        tabF[i] = make_float4(w.x, w.y, -w.y, w.x);
        tabI[i] = make_float4(w.x, -w.y, w.y, w.x);
    }
    for (int i = threadIdx.x; i < N; i += ring_threads<N, MODE>()) fx[i] = p.ftab[i];
    if (threadIdx.x == 0) {
        for (int s = 0; s < NSTAGE; ++s) { mbar_init(full + s, 1); mbar_init(empty + s, NTC / 32); issued[s] = 0; }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    pdl_wait();  // the tables above are constants of the handle; the spectra below are the predecessor's output
    const bool listed = CAN_LIST && p.ylist != nullptr;
    const long long total = listed ? (long long)p.nact[1] : (long long)p.units * tiles_per_unit;
    // activity bits of the z-pass tiles (listed mode, N >= 256): cached when they fit, else read from global memory
    constexpr int BITW = N * (N / 32) / 32;   // words per unit
    unsigned* bits_s = reinterpret_cast<unsigned*>(tcache + TCAP);
    const bool bits_cached = CAN_LIST && listed && (long long)p.units * BITW <= 256;
    if (bits_cached)
        for (int i = threadIdx.x; i < p.units * BITW; i += TCAP) bits_s[i] = p.tile_bits[i];
    // rowmask of the y-pass tile of plane o: bit ty = z-pass tile (o, ty) is active
    auto rowmask_of = [&](int unit, int o) -> unsigned {
        constexpr int NTY = N / 32;
        const int bit0 = o * NTY, w = unit * BITW + (bit0 >> 5);
        const unsigned word = bits_cached ? bits_s[w] : p.tile_bits[w];
        return (word >> (bit0 & 31)) & ((NTY >= 32) ? 0xffffffffu : ((1u << NTY) - 1u));
    };
    if (CAN_LIST && listed) {
        const long long idx = (long long)blockIdx.x + (long long)threadIdx.x * gridDim.x;
        tcache[threadIdx.x] = idx < total ? p.ylist[REVERSED ? total - 1 - idx : idx] : -1;
        __syncthreads();
    }
    // j-th tile of this CTA (global tile id), -1 past the end
    auto tile_at = [&](int j) -> long long {
        long long idx = (long long)blockIdx.x + (long long)j * gridDim.x;
        if (idx >= total) return -1;
        if (REVERSED) idx = total - 1 - idx;
        if (CAN_LIST && listed) return j < TCAP ? (long long)tcache[j] : (long long)p.ylist[idx];
        return idx;
    };

    // One item = one (tile, input channel) = one ring buffer fill.  Item `it` of this CTA lives in buffer it % NSTAGE;
    // the thread that sees the last consumer warp release item `it` immediately refills the buffer with item
    // it + NSTAGE, so there is no producer warp (a 17th warp would cost every thread 1/5 of its registers).
    auto issue_load = [&](int it) {
        const int j = it / IT_PER_TILE, ch = it - j * IT_PER_TILE;
        const long long g = tile_at(j);
        if (g < 0) return;
        const int unit = (int)(g / tiles_per_unit), T = (int)(g - (long long)unit * tiles_per_unit);
        const int s = it % NSTAGE;
        const int plane = unit * IN_STRIDE + ((MODE == MODE_INV3 && ch == 2) ? 1 : ch);  // INV3 fetches plane 1 twice
        const uint32_t dst = smem_u32(bufs + (size_t)s * TILE_ELEMS);
        mbar_expect_tx(full + s, TILE_BYTES);
        issued[s] = it / NSTAGE + 1;
        if (T < TILES_MAIN) {
            const int o = T / KT, kt = T - o * KT;
#pragma unroll
            for (int n0 = 0; n0 < N; n0 += NB) {
                if (AXIS == 0) tma_load_4d(dst + n0 * W * 8, &p.mapS, 2 * kt * W, o, n0, plane, full + s);
                else tma_load_4d(dst + n0 * W * 8, &p.mapS, 2 * kt * W, n0, o, plane, full + s);
            }
        } else {
            const int t = T - TILES_MAIN;
#pragma unroll
            for (int n0 = 0; n0 < N; n0 += NB) tma_load_3d(dst + n0 * W * 8, &p.mapQ, 2 * t * W, n0, plane, full + s);
        }
    };
    // consumers hand item `it` back; thread 0 of the group waits for the group's last warp and refills the buffer
    auto release = [&](int it) {
        const int s = it % NSTAGE;
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncwarp();
        if ((tid & 31) == 0) mbar_arrive(empty + s);
        if (tid == 0) {
            mbar_wait(empty + s, (it / NSTAGE) & 1);
            issue_load(it + NSTAGE);
        }
        __syncwarp();  // warp 0 is converged again before the next aligned group barrier
    };
    // A parity wait is only meaningful once the barrier has reached the phase waited for: a group may get here
    // before the fill it wants has even been issued (the previous fill of the buffer belongs to another group), and a
    // wait one phase early would return at once.  `issued` says the fill is under way, i.e. the phase is current.
    auto acquire = [&](int it) -> float2* {
        const int s = it % NSTAGE;
        while (issued[s] <= it / NSTAGE) {}
        mbar_wait(full + s, (it / NSTAGE) & 1);
        return bufs + (size_t)s * TILE_ELEMS;
    };
    if (threadIdx.x == 0) {
#pragma unroll 1
        for (int it = 0; it < NSTAGE; ++it) issue_load(it);
    }
    // ---------------- per-tile work of a consumer group ----------------
    for (int j = group;; j += NG) {
        const long long gl = tile_at(j);
        if (gl < 0) break;
        const int g = (int)gl;
        const int it = j * IT_PER_TILE;  // ring position of this tile's first item
        const int unit = g / tiles_per_unit, T = g - unit * tiles_per_unit;
        TileDesc d = tile_desc<N, W>(AXIS, T);
        if (AXIS == 0 && d.nyq && p.nyq_out_t) { d.base = (size_t)(T - TILES_MAIN) * W * N; d.sn = 1; d.sc = N; }
        const unsigned sn = (unsigned)d.sn, sc = (unsigned)d.sc;
        const int swz = (AXIS == 1 && !d.nyq) ? 15 : 0;  // y-pass tiles of the main spectrum: column swizzle per row
        const int xswz = (AXIS == 0 && !d.nyq) ? (d.other & 15) : 0;  // x-pass tile at y = d.other: one XOR for the tile
        // listed 3-channel y passes: which 32-row groups of this tile exist (d.other = the plane x of a main tile)
        const unsigned rowmask = (CAN_LIST && N >= 256 && listed && !d.nyq) ? rowmask_of(unit, d.other) : 0xffffffffu;
        unsigned xmv[2] = {0xffffffffu, 0xffffffffu};
        const bool xmasked = MODE == MODE_SOLVE && N <= 128 && p.plane_bits != nullptr && !d.nyq;
        if (MODE == MODE_SOLVE && N <= 128 && xmasked) xrow_masks<N, W, NTC>(p.plane_bits + (size_t)unit * (N / 32), tid, xmv);
        const unsigned* xm = xmasked ? xmv : nullptr;
        auto out_tile = [&](int c) {  // first element of this tile in output channel c
            const size_t plane = (size_t)unit * OUT_CH + c;
            return (d.nyq ? p.outQ + plane * QPLANE : p.outS + plane * SPLANE) + d.base;
        };
        auto col_freq = [&](int c, float4& ey, float4& ez) {
            ey = __ldg(p.ftab + (d.nyq ? d.other + c : d.other));
            ez = __ldg(p.ftab + N + (d.nyq ? H : d.pz0 + (c ^ xswz)));
        };

        if constexpr (MODE == MODE_FWD) {
            float2* buf = acquire(it);
            ring_stage<N, 0, W, NTC, false>(buf, tabF, tid, swz);
            consumer_sync<NTC>(group);
            if constexpr (NS == 3) {
                ring_stage<N, 1, W, NTC, false>(buf, tabF + N, tid, swz);
                consumer_sync<NTC>(group);
            }
            float2* out = out_tile(0);
#pragma unroll
            for (int i = 0; i < TPT; ++i) {
                const int t = tid + i * NTC, blk = t / W, c = t - blk * W;
                float2 v[RL];
#pragma unroll
                for (int r = 0; r < RL; ++r) v[r] = buf[(blk * RL + r) * W + (c ^ ((blk * RL + r) & swz))];
                dft_fwd<RL>(v);
#pragma unroll
                for (int r = 0; r < RL; ++r)
                    out[(unsigned)(blk * RL + r) * sn + (unsigned)(c ^ ((blk * RL + r) & swz)) * sc] = v[r];
            }
            release(it);
        } else if constexpr (MODE == MODE_INV) {
            float2* buf = acquire(it);
            ring_stage<N, LS, W, NTC, true>(buf, nullptr, tid, swz);
            consumer_sync<NTC>(group);
            if constexpr (NS == 3) {
                ring_stage<N, 1, W, NTC, true>(buf, tabI + N, tid, swz);
                consumer_sync<NTC>(group);
            }
            ring_stage0_inv_store<N, W, NTC>(buf, tabI, tid, out_tile(0), sn, sc, swz);
            release(it);
        } else if constexpr (MODE == MODE_FWD3) {
            // y pass of the three splat channels: plane 0 = FFT_y(v_x); plane 1 = u = h_y FFT_y(v_y) + FFT_y(h_z v_z)
            // (h_z is constant along y: applied on the way into the transform; h_y on the way out)
            auto hz_of = [&](int c) { return __ldg(p.ftab + N + (d.nyq ? H : d.pz0 + c)).x; };  // a thread follows the z SLOT c across rows
            float2 acc[TPT][RL];
#pragma unroll
            for (int ch = 0; ch < 3; ++ch) {
                float2* buf = acquire(it + ch);
                if (ch == 2) ring_stage0_fwd_scaled<N, W, NTC>(buf, tabF, tid, swz, hz_of, rowmask);
                else ring_stage<N, 0, W, NTC, false>(buf, tabF, tid, swz, rowmask);
                consumer_sync<NTC>(group);
                if constexpr (NS == 3) {
                    ring_stage<N, 1, W, NTC, false>(buf, tabF + N, tid, swz);
                    consumer_sync<NTC>(group);
                }
                float2* out = out_tile(ch == 0 ? 0 : 1);
#pragma unroll
                for (int i = 0; i < TPT; ++i) {
                    const int t = tid + i * NTC, blk = t / W, c = t - blk * W;
                    float2 v[RL];
#pragma unroll
                    for (int r = 0; r < RL; ++r) v[r] = buf[(blk * RL + r) * W + (c ^ ((blk * RL + r) & swz))];
                    dft_fwd<RL>(v);
                    if (ch == 1) {
#pragma unroll
                        for (int r = 0; r < RL; ++r) acc[i][r] = cscale(fx[blk * RL + r].x, v[r]);
                    } else {
#pragma unroll
                        for (int r = 0; r < RL; ++r)
                            out[(unsigned)(blk * RL + r) * sn + (unsigned)(c ^ ((blk * RL + r) & swz)) * sc] =
                                (ch == 0) ? v[r] : cadd(v[r], acc[i][r]);
                    }
                }
                release(it + ch);
            }
        } else if constexpr (MODE == MODE_INV3) {
            // inverse y pass of the adjoint: plane 0 = IFFT_y(plane 0); from B (plane 1, fetched twice -- the second fetch
            // is an L2 hit): plane 1 = IFFT_y(h_y B), plane 2 = h_z IFFT_y(B)
            auto hz_of = [&](int c) { return __ldg(p.ftab + N + (d.nyq ? H : d.pz0 + c)).x; };  // a thread follows the z SLOT c across rows
#pragma unroll
            for (int ch = 0; ch < 3; ++ch) {
                float2* buf = acquire(it + ch);
                if (ch == 1) {  // inverse of the last plan stage with h_y on the way in
#pragma unroll
                    for (int i = 0; i < TPT; ++i) {
                        const int t = tid + i * NTC, blk = t / W, c = t - blk * W;
                        float2 v[RL];
#pragma unroll
                        for (int r = 0; r < RL; ++r)
                            v[r] = cscale(fx[blk * RL + r].x, buf[(blk * RL + r) * W + (c ^ ((blk * RL + r) & swz))]);
                        dft_inv<RL>(v);
#pragma unroll
                        for (int r = 0; r < RL; ++r) buf[(blk * RL + r) * W + (c ^ ((blk * RL + r) & swz))] = v[r];
                    }
                } else {
                    ring_stage<N, LS, W, NTC, true>(buf, nullptr, tid, swz);
                }
                consumer_sync<NTC>(group);
                if constexpr (NS == 3) {
                    ring_stage<N, 1, W, NTC, true>(buf, tabI + N, tid, swz);
                    consumer_sync<NTC>(group);
                }
                // The pass runs in place and plane 1 is fetched twice (items ch = 1 and ch = 2): the second fetch must have
                // LANDED before plane 1 of this tile is overwritten (an issued bulk load is not ordered against later
                // generic stores), so wait for the ch = 2 buffer's full barrier first.  It is a separate buffer: no cost.
                if (ch == 1) acquire(it + 2);
                if (ch < 2) ring_stage0_inv_store<N, W, NTC>(buf, tabI, tid, out_tile(ch), sn, sc, swz, rowmask);
                else ring_stage0_inv_store_scaled<N, W, NTC>(buf, tabI, tid, out_tile(2), sn, sc, swz, hz_of, rowmask);
                release(it + ch);
            }
        } else if constexpr (MODE == MODE_SOLVE) {
            // chi~ = i f (h_x v~_x + h_y v~_y + h_z v~_z).  h_y and h_z are constant along x, so the y and z channels
            // are combined BEFORE the x transform: two forward x transforms per tile, not three.  The multiplier and the
            // first inverse stage happen on the registers of the last forward stage (same slots, no barrier).
            float4 ey, ez;
            col_freq(tid % W, ey, ez);  // NTC % W == 0: every task of this thread is in column tid % W
            const MultCol mc = mult_col(ey, ez, p.cs);
            float2 acc[TPT][RL];
            (void)acc;
            constexpr bool SIDE = NSTAGE >= 2 * 3;  // the ring can hold whole tiles and still prefetch
            float2* b0 = acquire(it);
            ring_stage<N, 0, W, NTC, false>(b0, tabF, tid, 0, 0xffffffffu, xm);
            if constexpr (!SIDE) {  // N = 512: finish the x channel and hand its buffer back first
                consumer_sync<NTC>(group);
                if constexpr (NS == 3) {
                    ring_stage<N, 1, W, NTC, false>(b0, tabF + N, tid);
                    consumer_sync<NTC>(group);
                }
#pragma unroll
                for (int i = 0; i < TPT; ++i) {
                    const int t = tid + i * NTC, blk = t / W, c = t - blk * W;
                    float2 v[RL];
#pragma unroll
                    for (int r = 0; r < RL; ++r) v[r] = b0[(blk * RL + r) * W + c];
                    dft_fwd<RL>(v);
#pragma unroll
                    for (int r = 0; r < RL; ++r) acc[i][r] = cscale(fx[blk * RL + r].x, v[r]);
                }
                release(it);
            }
            float2* b1 = acquire(it + 1);
            if constexpr (TWO_SPECTRA) {  // the y pass has already formed u = h_y v~_y + h_z v~_z
                ring_stage<N, 0, W, NTC, false>(b1, tabF, tid);
                consumer_sync<NTC>(group);
            } else {
                float2* b2 = acquire(it + 2);
                ring_stage0_fwd2<N, W, NTC>(b1, b2, tabF, tid, ey.x, ez.x, xm);
                consumer_sync<NTC>(group);
                release(it + 2);  // the z channel has been folded into b1
            }
            if constexpr (NS == 3) {
                if constexpr (SIDE) ring_stage<N, 1, W, NTC, false>(b0, tabF + N, tid);
                ring_stage<N, 1, W, NTC, false>(b1, tabF + N, tid);
                consumer_sync<NTC>(group);
            }
#pragma unroll
            for (int i = 0; i < TPT; ++i) {
                const int t = tid + i * NTC, blk = t / W, c = t - blk * W;
                const int e0 = blk * RL * W + c;
                float2 v[RL], a[RL];
                if constexpr (SIDE) {
#pragma unroll
                    for (int r = 0; r < RL; ++r) v[r] = b0[e0 + r * W];
                    dft_fwd<RL>(v);
#pragma unroll
                    for (int r = 0; r < RL; ++r) a[r] = cscale(fx[blk * RL + r].x, v[r]);
                } else {
#pragma unroll
                    for (int r = 0; r < RL; ++r) a[r] = acc[i][r];
                }
#pragma unroll
                for (int r = 0; r < RL; ++r) v[r] = b1[e0 + r * W];
                dft_fwd<RL>(v);
#pragma unroll
                for (int r = 0; r < RL; ++r) {
                    const float f = mult_fc(fx[blk * RL + r], mc);
                    const float2 dv = cscale(f, cadd(a[r], v[r]));
                    a[r] = make_float2(-dv.y, dv.x);  // chi~ = i (div)
                }
                dft_inv<RL>(a);
#pragma unroll
                for (int r = 0; r < RL; ++r) b1[e0 + r * W] = a[r];
            }
            if constexpr (SIDE) release(it);
            consumer_sync<NTC>(group);
            if constexpr (NS == 3) {
                ring_stage<N, 1, W, NTC, true>(b1, tabI + N, tid);
                consumer_sync<NTC>(group);
            }
            ring_stage0_inv_store<N, W, NTC>(b1, tabI, tid, out_tile(0), sn, sc);
            release(it + 1);
        } else {  // MODE_ADJ
            // vbar~_c = h_c A, A = -i f Gbar'~.  h_y and h_z are constant along x: the y and z channels are the SAME inverse
            // x transform B of A, so a tile needs two inverse x transforms, not three, and writes two spectra.
            float4 ey, ez;
            col_freq(tid % W, ey, ez);
            const MultCol mc = mult_col(ey, ez, p.cs);
            float2* buf = acquire(it);
            ring_stage<N, 0, W, NTC, false>(buf, tabF, tid);
            consumer_sync<NTC>(group);
            if constexpr (NS == 3) {
                ring_stage<N, 1, W, NTC, false>(buf, tabF + N, tid);
                consumer_sync<NTC>(group);
            }
            float2 acc[TPT][RL];  // A on the slots of this thread's last-stage butterflies
#pragma unroll
            for (int i = 0; i < TPT; ++i) {
                const int t = tid + i * NTC, blk = t / W, c = t - blk * W;
                float2 v[RL];
#pragma unroll
                for (int r = 0; r < RL; ++r) v[r] = buf[(blk * RL + r) * W + c];
                dft_fwd<RL>(v);
#pragma unroll
                for (int r = 0; r < RL; ++r) {
                    const float f = mult_fc(fx[blk * RL + r], mc);
                    acc[i][r] = cscale(f, mul_mi(v[r]));   // -i f v: one packed multiply (half swap + negate are operand modifiers)
                }
            }
#pragma unroll
            for (int pass = 0; pass < 2; ++pass) {  // 0: x channel (h_x varies along x), 1: y and z channels
                if (pass > 0) consumer_sync<NTC>(group);  // stage-0 reads of the previous pass are done
#pragma unroll
                for (int i = 0; i < TPT; ++i) {
                    const int t = tid + i * NTC, blk = t / W, c = t - blk * W;
                    float2 v[RL];
#pragma unroll
                    for (int r = 0; r < RL; ++r) v[r] = (pass == 0) ? cscale(fx[blk * RL + r].x, acc[i][r]) : acc[i][r];
                    dft_inv<RL>(v);
#pragma unroll
                    for (int r = 0; r < RL; ++r) buf[(blk * RL + r) * W + c] = v[r];
                }
                consumer_sync<NTC>(group);
                if constexpr (NS == 3) {
                    ring_stage<N, 1, W, NTC, true>(buf, tabI + N, tid);
                    consumer_sync<NTC>(group);
                }
                // pass 1 stores B unscaled as plane 1: the next pass (k_ring<INV3> or the fused k_zl_inv) makes the y and
                // z channels from it with h_y and h_z on the way into ITS first stage
                ring_stage0_inv_store<N, W, NTC>(buf, tabI, tid, out_tile(pass), sn, sc);
            }
            release(it);
        }
    }
}

}  // namespace sap
