// ring_pass.cuh -- persistent, TMA-fed version of the strided-axis passes (x pass with the fused spectral
// solve, y pass for N >= 256).  One CTA = NTC consumer threads + one producer warp.  The producer streams
// tiles of N points x W contiguous columns (W*8-byte rows) from HBM into a ring of NSTAGE shared-memory
// buffers with cp.async.bulk.tensor (one instruction per tile, completion on an mbarrier); the consumers
// transform a tile IN PLACE in its buffer, write the result to HBM straight from registers and hand the
// buffer back.  Loads of the next tiles are therefore in flight during all of the arithmetic, whatever the
// register count -- the earlier one-tile-per-CTA version depended on occupancy for that overlap.
//   MODE_FWD / MODE_INV : forward / inverse transform along `axis`
//   MODE_SOLVE (F2x+F3+F4x): forward x on 3 channels, chi~ = i sum_c m_c v~_c, inverse x, 1 channel out
//   MODE_ADJ   (B3x+B4+B5x): forward x on 1 channel, vbar~_c = -i m_c Gbar'~, 3 inverse x
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
template <> struct RingCfg<128> { static constexpr int W = 32, NTC = 256, NG = 2, NSTAGE = 6, MINB = 1; };
template <> struct RingCfg<256> { static constexpr int W = 16, NTC = 256, NG = 2, NSTAGE = 6, MINB = 1; };
template <> struct RingCfg<512> { static constexpr int W = 16, NTC = 512, NG = 1, NSTAGE = 3, MINB = 1; };
template <int N> constexpr int ring_threads() { return RingCfg<N>::NTC * RingCfg<N>::NG; }

template <int N> constexpr size_t ring_smem_bytes() {
    using C = RingCfg<N>;
    return (size_t)C::NSTAGE * N * C::W * sizeof(float2) + (size_t)N * sizeof(float2) + (size_t)N * sizeof(float4) +
           2 * C::NSTAGE * sizeof(uint64_t) + 128;
}
template <int N> constexpr int ring_box_rows() { return N < 256 ? N : 256; }  // TMA box dimension limit

struct RingParams {
    CUtensorMap mapS;    // main spectrum of the input array, box = one tile (or half a tile at N = 512)
    CUtensorMap mapQ;    // Nyquist plane of the input: [x][y] for the x pass, the transposed copy [y][x] for the y pass
    float2* outS;
    float2* outQ;
    const float2* tw;
    const float4* ftab;
    int axis;            // 0: x pass, 1: y pass (main spectrum only)
    int units;           // planes (FWD / INV) or batch items (SOLVE / ADJ)
    int nyq_out_t;       // Nyquist-plane output is written transposed ([y][x] <-> [x][y]); always so for axis 1
    float cs;
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
// consumers hand a ring buffer back: order their generic-proxy accesses before the producer's next TMA write
__device__ __forceinline__ void ring_release(uint64_t* empty_bar) {
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    __syncwarp();
    if ((threadIdx.x & 31) == 0) mbar_arrive(empty_bar);
}

}  // namespace sap

namespace sap {

// stage 0 of the length-N plan, in place in a dense [N][W] tile; lanes over columns
template <int N, int W, int NTC, bool INV>
__device__ __forceinline__ void ring_stage0(float2* s, const float2* tw, int tid) {
    constexpr int R = StageInfo<N, 0>::R, ST = StageInfo<N, 0>::ST;
    for (int t = tid; t < ST * W; t += NTC) {
        const int q = t / W, c = t - q * W;
        float2 v[R];
#pragma unroll
        for (int r = 0; r < R; ++r) v[r] = s[(q + ST * r) * W + c];
        if (INV) bfly_inv<N, 0, N>(v, q, tw); else bfly_fwd<N, 0, N>(v, q, tw);
#pragma unroll
        for (int r = 0; r < R; ++r) s[(q + ST * r) * W + c] = v[r];
    }
}

template <int N, int MODE>
__global__ void __launch_bounds__(ring_threads<N>(), RingCfg<N>::MINB) k_ring(const __grid_constant__ RingParams p) {
    using C = RingCfg<N>;
    constexpr int W = C::W, NTC = C::NTC, NG = C::NG, NSTAGE = C::NSTAGE, H = N / 2;
    constexpr int NS = Plan<N>::NS, LS = NS - 1, RL = StageInfo<N, LS>::R;
    static_assert(StageInfo<N, LS>::ST == 1 && NS >= 2, "plan");
    constexpr int R0 = StageInfo<N, 0>::R, ST0 = StageInfo<N, 0>::ST;
    constexpr int TILE_ELEMS = N * W;
    constexpr uint32_t TILE_BYTES = TILE_ELEMS * sizeof(float2);
    constexpr int NB = ring_box_rows<N>();
    constexpr int NTASK = (N / RL) * W, TPT = (NTASK + NTC - 1) / NTC;
    static_assert(NTASK % NTC == 0, "last-stage tasks divide evenly over the consumers");
    constexpr int KT = H / W, TILES_MAIN = N * KT, TILES_NYQ = N / W;
    constexpr int IN_CH = (MODE == MODE_SOLVE) ? 3 : 1, OUT_CH = (MODE == MODE_ADJ) ? 3 : 1;
    constexpr size_t SPLANE = (size_t)N * N * H, QPLANE = (size_t)N * N;

    extern __shared__ __align__(1024) unsigned char ring_smem[];
    float2* bufs = reinterpret_cast<float2*>(ring_smem);
    float2* tw = bufs + (size_t)NSTAGE * TILE_ELEMS;
    float4* fx = reinterpret_cast<float4*>(tw + N);
    uint64_t* full = reinterpret_cast<uint64_t*>(fx + N);
    uint64_t* empty = full + NSTAGE;
    const int group = threadIdx.x / NTC, tid = threadIdx.x - group * NTC;

    for (int i = threadIdx.x; i < N; i += ring_threads<N>()) { tw[i] = p.tw[i]; fx[i] = p.ftab[i]; }
    if (threadIdx.x == 0) {
        for (int s = 0; s < NSTAGE; ++s) { mbar_init(full + s, 1); mbar_init(empty + s, NTC / 32); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    constexpr int tiles_per_unit = TILES_MAIN + TILES_NYQ;
    constexpr int IT_PER_TILE = IN_CH;
    const long long total = (long long)p.units * tiles_per_unit;

    // One item = one (tile, input channel) = one ring buffer fill.  Item `it` of this CTA lives in buffer it % NSTAGE;
    // the thread that sees the last consumer warp release item `it` immediately refills the buffer with item
    // it + NSTAGE, so there is no producer warp (a 17th warp would cost every thread 1/5 of its registers).
    auto issue_load = [&](int it) {
        const int j = it / IT_PER_TILE, ch = it - j * IT_PER_TILE;
        const long long g = (long long)blockIdx.x + (long long)j * gridDim.x;
        if (g >= total) return;
        const int unit = (int)(g / tiles_per_unit), T = (int)(g - (long long)unit * tiles_per_unit);
        const int s = it % NSTAGE;
        mbar_expect_tx(full + s, TILE_BYTES);
        const int plane = unit * IN_CH + ch;
        const uint32_t dst = smem_u32(bufs + (size_t)s * TILE_ELEMS);
        if (T < TILES_MAIN) {
            const int o = T / KT, kt = T - o * KT;
#pragma unroll
            for (int n0 = 0; n0 < N; n0 += NB) {
                if (p.axis == 0) tma_load_4d(dst + n0 * W * 8, &p.mapS, 2 * kt * W, o, n0, plane, full + s);
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
    };
    if (threadIdx.x == 0) {
#pragma unroll 1
        for (int it = 0; it < NSTAGE; ++it) issue_load(it);
    }

    // ---------------- consumers ----------------
    float2 acc[TPT][RL];  // SOLVE: divergence accumulators; ADJ: -i f Gbar'~
    (void)acc;
    for (int j = group, g = blockIdx.x + group * gridDim.x; g < total; j += NG, g += NG * gridDim.x) {
        int it = j * IT_PER_TILE;  // ring position of this tile's first buffer (same order as the producer)
        const int unit = g / tiles_per_unit, T = g - unit * tiles_per_unit;
        TileDesc d = tile_desc<N, W>(p.axis, T);
        if (d.nyq && p.nyq_out_t) { d.base = (size_t)(T - TILES_MAIN) * W * N; d.sn = 1; d.sc = N; }
        auto out_plane = [&](int c) {
            const size_t plane = (size_t)unit * OUT_CH + c;
            return d.nyq ? p.outQ + plane * QPLANE : p.outS + plane * SPLANE;
        };
        auto col_freq = [&](int c, float4& ey, float4& ez) {
            ey = __ldg(p.ftab + (d.nyq ? d.other + c : d.other));
            ez = __ldg(p.ftab + N + (d.nyq ? H : d.pz0 + c));
        };
        float2* buf = nullptr;
        int s = 0;
        // ---- forward half
        if constexpr (MODE != MODE_INV) {
#pragma unroll
            for (int ch = 0; ch < IN_CH; ++ch, ++it) {
                s = it % NSTAGE;
                buf = bufs + (size_t)s * TILE_ELEMS;
                mbar_wait(full + s, (it / NSTAGE) & 1);
                ring_stage0<N, W, NTC, false>(buf, tw, tid);
                consumer_sync<NTC>(group);
                if constexpr (NS == 3) {
                    fft_stage<N, 1, false, N, true>(buf, W, 1, W, tw, tid, NTC);
                    consumer_sync<NTC>(group);
                }
#pragma unroll
                for (int i = 0; i < TPT; ++i) {
                    const int t = tid + i * NTC;
                    const int blk = t / W, c = t - blk * W;
                    float2 v[RL];
#pragma unroll
                    for (int r = 0; r < RL; ++r) v[r] = buf[(blk * RL + r) * W + c];
                    dft_fwd<RL>(v);
                    if constexpr (MODE == MODE_FWD) {
                        float2* gout = out_plane(0);
#pragma unroll
                        for (int r = 0; r < RL; ++r)
                            gout[d.base + (size_t)(blk * RL + r) * d.sn + (size_t)c * d.sc] = v[r];
                    } else {
                        float4 ey, ez;
                        col_freq(c, ey, ez);
                        if (MODE == MODE_ADJ || ch == 2) {
#pragma unroll
                            for (int r = 0; r < RL; ++r) {
                                const float f = mult_f(fx[blk * RL + r], ey, ez, p.cs);
                                if constexpr (MODE == MODE_SOLVE) {
                                    const float2 dv = cscale(f, caxpy(ez.x, v[r], acc[i][r]));
                                    acc[i][r] = make_float2(-dv.y, dv.x);  // chi~ = i (div)
                                } else {
                                    acc[i][r] = make_float2(f * v[r].y, -f * v[r].x);  // -i f Gbar'~
                                }
                            }
                        } else if (ch == 0) {
#pragma unroll
                            for (int r = 0; r < RL; ++r) acc[i][r] = cscale(fx[blk * RL + r].x, v[r]);
                        } else {
#pragma unroll
                            for (int r = 0; r < RL; ++r) acc[i][r] = caxpy(ey.x, v[r], acc[i][r]);
                        }
                    }
                }
                if (MODE == MODE_FWD || (MODE == MODE_SOLVE && ch < 2)) release(it);
            }
        } else {
            s = it % NSTAGE;
            buf = bufs + (size_t)s * TILE_ELEMS;
            mbar_wait(full + s, (it / NSTAGE) & 1);
            ++it;
        }
        // ---- inverse half, in the buffer of the last input channel
        if constexpr (MODE != MODE_FWD) {
#pragma unroll
            for (int ch = 0; ch < OUT_CH; ++ch) {
                if (ch > 0) consumer_sync<NTC>(group);  // stage-0 reads of the previous channel are done
#pragma unroll
                for (int i = 0; i < TPT; ++i) {
                    const int t = tid + i * NTC;
                    const int blk = t / W, c = t - blk * W;
                    float2 v[RL];
                    if constexpr (MODE == MODE_INV) {
#pragma unroll
                        for (int r = 0; r < RL; ++r) v[r] = buf[(blk * RL + r) * W + c];
                    } else if constexpr (MODE == MODE_SOLVE) {
#pragma unroll
                        for (int r = 0; r < RL; ++r) v[r] = acc[i][r];
                    } else {
                        float4 ey, ez;
                        col_freq(c, ey, ez);
#pragma unroll
                        for (int r = 0; r < RL; ++r) {
                            const float h = (ch == 0) ? fx[blk * RL + r].x : (ch == 1) ? ey.x : ez.x;
                            v[r] = cscale(h, acc[i][r]);
                        }
                    }
                    dft_inv<RL>(v);
#pragma unroll
                    for (int r = 0; r < RL; ++r) buf[(blk * RL + r) * W + c] = v[r];
                }
                consumer_sync<NTC>(group);
                if constexpr (NS == 3) {
                    fft_stage<N, 1, true, N, true>(buf, W, 1, W, tw, tid, NTC);
                    consumer_sync<NTC>(group);
                }
                float2* gout = out_plane(ch);
                for (int t = tid; t < ST0 * W; t += NTC) {
                    const int q = t / W, c = t - q * W;
                    float2 v[R0];
#pragma unroll
                    for (int r = 0; r < R0; ++r) v[r] = buf[(q + ST0 * r) * W + c];
                    bfly_inv<N, 0, N>(v, q, tw);
#pragma unroll
                    for (int r = 0; r < R0; ++r) gout[d.base + (size_t)(q + ST0 * r) * d.sn + (size_t)c * d.sc] = v[r];
                }
            }
            release(it - 1);
        }
    }
}

}  // namespace sap
