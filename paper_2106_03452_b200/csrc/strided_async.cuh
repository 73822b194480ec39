// strided_async.cuh -- persistent, software-pipelined version of the strided-axis pass.
//
// Each CTA loops over tiles (N points x W contiguous columns).  The raw rows of the next slabs (a slab
// = one channel of one tile, N rows of W*8 bytes) are fetched by the copy engine with
// cp.async.bulk (global -> shared, completion on an mbarrier) into a ring of NB buffers while the
// current slab is transformed, so HBM reads stay in flight through the compute and store phases even
// with one CTA per SM.  The transform is the same as strided_pass.cuh: stage 0 in place in the slab,
// (middle stage for three-stage plans), then the stride-1 stage in registers with the spectral
// multiplier applied between its forward and inverse halves; outputs go registers -> global.
//
// The memory-pipeline primitives come from the context (device: PTX mbarrier / cp.async.bulk; the
// host debugging harness: a synchronous copy), everything else is shared with strided_pass.cuh.
#pragma once
#include "strided_pass.cuh"

namespace sap {

template <int N, int MODE, int W, int NB> constexpr size_t strided_async_smem_bytes() {
    // NB raw slabs (pitch W, 16-byte aligned rows) + an output staging tile (pitch W+1) for SOLVE/ADJ
    // + twiddles + NB mbarriers
    return ((size_t)NB * N * W + ((MODE == MODE_SOLVE || MODE == MODE_ADJ) ? (size_t)N * (W + 1) : 0) + N) * sizeof(float2) +
           16 * sizeof(unsigned long long);
}

// stage 0 forward, in place in a raw slab (pitch W)
template <int N, int W, int NT, class Ctx>
SAP_HD void slab_stage0_fwd(Ctx& ctx, float2* s, const float2* tw) {
    constexpr int R = StageInfo<N, 0>::R, ST = StageInfo<N, 0>::ST;
    for (int t = ctx.tid; t < ST * W; t += NT) {
        const int q = t / W, c = t - q * W;
        float2 v[R];
#pragma unroll
        for (int r = 0; r < R; ++r) v[r] = s[(q + ST * r) * W + c];
        bfly_fwd<N, 0, N>(v, q, tw);
#pragma unroll
        for (int r = 0; r < R; ++r) s[(q + ST * r) * W + c] = v[r];
    }
}
// stage 0 inverse: smem (pitch P) -> registers -> global
template <int N, int W, int P, int NT, class Ctx>
SAP_HD void slab_stage0_inv(Ctx& ctx, float2* g, const TileDesc& d, const float2* s, const float2* tw) {
    constexpr int R = StageInfo<N, 0>::R, ST = StageInfo<N, 0>::ST;
    for (int t = ctx.tid; t < ST * W; t += NT) {
        const int q = t / W, c = t - q * W;
        float2 v[R];
#pragma unroll
        for (int r = 0; r < R; ++r) v[r] = s[(q + ST * r) * P + c];
        bfly_inv<N, 0, N>(v, q, tw);
#pragma unroll
        for (int r = 0; r < R; ++r) g[d.base + (size_t)(q + ST * r) * d.sn + (size_t)c * d.sc] = v[r];
    }
}

// bx: CTA index, nbx: number of CTAs (persistent loop stride); nby: planes (FWD/INV: item*nch + ch) or batch
// items (SOLVE/ADJ).  Work item w = bx + k*nbx covers tile w % NTILES of plane w / NTILES.
template <int N, int MODE, int NT, int W, int NB, class Ctx>
SAP_HD void strided_async_body(Ctx& ctx, const StridedParams& p, float2* smem, int bx, int nbx, int nby) {
    constexpr int H = N / 2;
    constexpr int NS = Plan<N>::NS;
    constexpr int RL = StageInfo<N, NS - 1>::R;
    static_assert(StageInfo<N, NS - 1>::ST == 1 && NS >= 2, "plan");
    constexpr int NTASK = (N / RL) * W;
    constexpr int TPT = (NTASK + NT - 1) / NT;
    constexpr int SLAB = N * W;
    constexpr int OP = W + 1;  // pitch of the output staging tile
    constexpr size_t SPLANE = (size_t)N * N * H;
    constexpr size_t QPLANE = (size_t)N * N;
    constexpr int IN_CH = (MODE == MODE_SOLVE) ? 3 : 1;
    constexpr int OUT_CH = (MODE == MODE_ADJ) ? 3 : 1;
    constexpr bool HAS_OUT = (MODE == MODE_SOLVE || MODE == MODE_ADJ);
    constexpr int NTILES = strided_tiles<N, W>();

    float2* slabs = smem;
    float2* obuf = smem + NB * SLAB;
    float2* tw = obuf + (HAS_OUT ? N * OP : 0);
    unsigned long long* bars = reinterpret_cast<unsigned long long*>(tw + N);

    for (int i = ctx.tid; i < N; i += NT) tw[i] = p.tw[i];
    if (ctx.tid == 0)
        for (int b = 0; b < NB; ++b) ctx.bar_init(bars + b);
    ctx.fence_init();
    ctx.sync();

    const int total = NTILES * nby;
    const int my_tiles = (bx < total) ? (total - 1 - bx) / nbx + 1 : 0;
    const int my_slabs = my_tiles * IN_CH;
    auto in_plane = [&](const TileDesc& d, int by, int c) {
        const size_t plane = (size_t)by * IN_CH + c;
        return d.nyq ? p.inQ + plane * QPLANE : p.inS + plane * SPLANE;
    };
    auto out_plane = [&](const TileDesc& d, int by, int c) {
        const size_t plane = (size_t)by * OUT_CH + c;
        return d.nyq ? p.outQ + plane * QPLANE : p.outS + plane * SPLANE;
    };
    // enqueue the copy of slab j (tile j / IN_CH, channel j % IN_CH) into ring slot j % NB
    auto issue = [&](int j) {
        if (j >= my_slabs) return;
        const int w = bx + (j / IN_CH) * nbx;
        const TileDesc d = tile_desc<N, W>(p.axis, w % NTILES);
        if (d.sc != 1) return;  // rows not contiguous (Nyquist plane along y): loaded synchronously at use
        const float2* g = in_plane(d, w / NTILES, j % IN_CH) + d.base;
        float2* dst = slabs + (j % NB) * SLAB;
        unsigned long long* bar = bars + (j % NB);
        if (ctx.tid == 0) ctx.bar_expect(bar, (unsigned)(SLAB * sizeof(float2)));
        for (int n = ctx.tid; n < N; n += NT) ctx.bulk_row(dst + n * W, g + (size_t)n * d.sn, (unsigned)(W * sizeof(float2)), bar);
    };
    unsigned phase_bits = 0;  // per ring slot: parity of the next completion to wait for
    for (int j = 0; j < NB; ++j) issue(j);

    float2 acc[TPT][RL];
    (void)acc;
    int j = 0;
    for (int k = 0; k < my_tiles; ++k) {
        const int by = (bx + k * nbx) / NTILES;
        const TileDesc d = tile_desc<N, W>(p.axis, (bx + k * nbx) % NTILES);
        auto col_freq = [&](int c, int& uy, int& uz, float& hy, float& hz) {
            const int ky = pos2freq<N>(d.nyq ? d.other + c : d.other);
            const int kz = d.nyq ? H : pos2freq<H>(d.pz0 + c);
            uy = signed_freq<N>(ky); uz = signed_freq<N>(kz);
            hy = (ky == H) ? 0.f : (float)uy; hz = (kz == H) ? 0.f : (float)uz;
        };
#pragma unroll
        for (int ch = 0; ch < IN_CH; ++ch, ++j) {
            const int slot = j % NB;
            float2* s = slabs + slot * SLAB;
            if (d.sc == 1) {
                ctx.bar_wait(bars + slot, (phase_bits >> slot) & 1u);
                phase_bits ^= 1u << slot;
            } else {
                const float2* g = in_plane(d, by, ch);
                for (int i = ctx.tid; i < N * W; i += NT) {
                    const int c = i / N, n = i - c * N;
                    s[n * W + c] = g[d.base + (size_t)c * d.sc + n];
                }
                ctx.sync();
            }
            if constexpr (MODE != MODE_INV) {
                slab_stage0_fwd<N, W, NT>(ctx, s, tw);
                ctx.sync();
                if constexpr (NS == 3) {
                    fft_stage<N, 1, false, N, true>(s, W, 1, W, tw, ctx.tid, NT);
                    ctx.sync();
                }
            }
            // stride-1 stage
#pragma unroll
            for (int i = 0; i < TPT; ++i) {
                const int t = ctx.tid + i * NT;
                if (NTASK % NT == 0 || t < NTASK) {
                    const int blk = t / W, c = t - blk * W;
                    const int e0 = blk * RL * W + c;
                    float2 v[RL];
#pragma unroll
                    for (int r = 0; r < RL; ++r) v[r] = s[e0 + r * W];
                    if constexpr (MODE == MODE_INV) {
                        dft_inv<RL>(v);
#pragma unroll
                        for (int r = 0; r < RL; ++r) s[e0 + r * W] = v[r];
                    } else {
                        dft_fwd<RL>(v);
                        if constexpr (MODE == MODE_FWD) {
                            float2* g = out_plane(d, by, 0);
#pragma unroll
                            for (int r = 0; r < RL; ++r)
                                g[d.base + (size_t)(blk * RL + r) * d.sn + (size_t)c * d.sc] = v[r];
                        } else {
                            int uy, uz; float hy, hz;
                            col_freq(c, uy, uz, hy, hz);
                            if (MODE == MODE_ADJ || ch == 2) {
#pragma unroll
                                for (int r = 0; r < RL; ++r) {
                                    const int ux = signed_freq<N>(pos2freq<N>(blk * RL + r));
                                    const float f = mult_f<N>(ux, uy, uz, p.cg, p.cs);
                                    if constexpr (MODE == MODE_SOLVE) {
                                        const float dr = f * (acc[i][r].x + hz * v[r].x), di = f * (acc[i][r].y + hz * v[r].y);
                                        acc[i][r] = make_float2(-di, dr);
                                    } else {
                                        acc[i][r] = make_float2(f * v[r].y, -f * v[r].x);
                                    }
                                }
                            } else if (ch == 0) {
#pragma unroll
                                for (int r = 0; r < RL; ++r) {
                                    const int kx = pos2freq<N>(blk * RL + r);
                                    const float hx = (kx == H) ? 0.f : (float)signed_freq<N>(kx);
                                    acc[i][r] = make_float2(hx * v[r].x, hx * v[r].y);
                                }
                            } else {
#pragma unroll
                                for (int r = 0; r < RL; ++r) { acc[i][r].x += hy * v[r].x; acc[i][r].y += hy * v[r].y; }
                            }
                        }
                    }
                }
            }
            ctx.sync();
            if constexpr (MODE == MODE_INV) {
                if constexpr (NS == 3) {
                    fft_stage<N, 1, true, N, true>(s, W, 1, W, tw, ctx.tid, NT);
                    ctx.sync();
                }
                slab_stage0_inv<N, W, W, NT>(ctx, out_plane(d, by, 0), d, s, tw);
                ctx.sync();
            }
            // the slot is free: refill it with the slab NB ahead
            ctx.fence_async();
            issue(j + NB);
        }
        if constexpr (HAS_OUT) {
#pragma unroll
            for (int ch = 0; ch < OUT_CH; ++ch) {
#pragma unroll
                for (int i = 0; i < TPT; ++i) {
                    const int t = ctx.tid + i * NT;
                    if (NTASK % NT == 0 || t < NTASK) {
                        const int blk = t / W, c = t - blk * W;
                        float2 v[RL];
                        if constexpr (MODE == MODE_SOLVE) {
#pragma unroll
                            for (int r = 0; r < RL; ++r) v[r] = acc[i][r];
                        } else {
                            int uy, uz; float hy, hz;
                            col_freq(c, uy, uz, hy, hz);
#pragma unroll
                            for (int r = 0; r < RL; ++r) {
                                float h;
                                if (ch == 0) {
                                    const int kx = pos2freq<N>(blk * RL + r);
                                    h = (kx == H) ? 0.f : (float)signed_freq<N>(kx);
                                } else h = (ch == 1) ? hy : hz;
                                v[r] = make_float2(h * acc[i][r].x, h * acc[i][r].y);
                            }
                        }
                        dft_inv<RL>(v);
#pragma unroll
                        for (int r = 0; r < RL; ++r) obuf[(blk * RL + r) * OP + c] = v[r];
                    }
                }
                ctx.sync();
                if constexpr (NS == 3) {
                    fft_stage<N, 1, true, N, true>(obuf, OP, 1, W, tw, ctx.tid, NT);
                    ctx.sync();
                }
                slab_stage0_inv<N, W, OP, NT>(ctx, out_plane(d, by, ch), d, obuf, tw);
                ctx.sync();
            }
        }
    }
}

}  // namespace sap
