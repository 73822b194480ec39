// strided_pass.cuh -- transforms along a strided axis over tiles of N points x 16 contiguous columns
// (128-byte rows), with the spectral solve fused between the last forward and the first inverse stage.
//   MODE_FWD / MODE_INV : plain forward / inverse transform along `axis` (the y pass when N >= 256)
//   MODE_SOLVE (F2x+F3+F4x): forward x on 3 channels, chi~ = i sum_c m_c v~_c, inverse x, 1 channel out
//   MODE_ADJ   (B3x+B4+B5x): forward x on 1 channel, vbar~_c = conj(M_c) Gbar'~ = -i m_c Gbar'~, 3 inverse x
// Shared-memory traffic: the first stage runs global -> registers -> smem and the last one smem ->
// registers -> global; the multiplier is applied on the registers of the middle stage, which is at
// once the last forward (DIF) and the first inverse (DIT) stage -- both act on the same R slots.
// Tiles cover the main spectrum and then the Nyquist plane (different strides, same code).
#pragma once
#include "fft_core.cuh"

namespace sap {

// Columns per tile: 32 contiguous complex values (256-byte rows, one warp per row); 16 when H = 16.
// (W is a template parameter of the kernels: 16 or 32, W <= N/2.)

// Spectral multiplier of Eq.3 / Eq.16 with readings R3 (Nyquist derivative zeroed),
// R4 (DC zero), R6 (integer frequencies, literal Gaussian):
//   M_c(k) = i m_c,  m_c = f uh_c,  f = cs exp(-cg q) / q,  q = |u|^2,  cg = 2 sigma^2 / N^2,
//   cs = (2 / N^3) / (-2 pi): folds the inverse-transform scale (R8) and the factor 2 of the half-length
//   c2r trick into the multiplier.
// Per-slot table (built once in sap_dpsr_create, float4 {uh, u^2, exp(-cg u^2), 0}): entries [0, N) for the
// slots of a length-N axis (x, y), entries [N, N + H] for the z slots (slot H = the Nyquist plane).
template <int N> SAP_HD int signed_freq(int k) { return (k < N / 2) ? k : k - N; }
template <int N> SAP_HD float4 freq_entry_n(int slot, float cg) {
    const int k = pos2freq<N>(slot), u = signed_freq<N>(k);
    return make_float4((k == N / 2) ? 0.f : (float)u, (float)(u * u), expf(-cg * (float)(u * u)), 0.f);
}
template <int N> SAP_HD float4 freq_entry_z(int slot, float cg) {
    constexpr int H = N / 2;
    const int k = (slot == H) ? H : pos2freq<H>(slot);
    return make_float4((k == H) ? 0.f : (float)k, (float)(k * k), expf(-cg * (float)(k * k)), 0.f);
}
SAP_HD float fast_rcp(float x) {
#ifdef __CUDA_ARCH__
    return __frcp_rn(x);
#else
    return 1.f / x;
#endif
}
// f = cs g / q from three table entries (0 at DC)
SAP_HD float mult_f(const float4& ex, const float4& ey, const float4& ez, float cs) {
    const float q = ex.y + ey.y + ez.y;
    return (q == 0.f) ? 0.f : cs * (ex.z * ey.z) * ez.z * fast_rcp(q);
}

enum { MODE_FWD = 0, MODE_INV = 1, MODE_SOLVE = 2, MODE_ADJ = 3 };

struct StridedParams {
    const float2* inS;
    const float2* inQ;
    float2* outS;
    float2* outQ;
    const float2* tw;
    const float4* ftab;  // [N + H + 1] frequency table (see freq_entry_*)
    int axis;     // 0: along x (stride N*H / N), 1: along y (stride H / 1)
    float cg;     // 2 sigma^2 / N^2
    float cs;     // (2 / N^3) / (-2 pi)
};

template <int N, int W> constexpr int strided_tiles() { return N * (N / 2 / W) + N / W; }
// one tile buffer for every mode: SOLVE streams its 3 input channels through it (the divergence is
// accumulated in registers), ADJ streams its 3 output channels
template <int N, int W> constexpr size_t strided_smem_bytes() { return ((size_t)N * (W + 1) + N) * sizeof(float2) + (size_t)N * sizeof(float4); }

struct TileDesc {
    size_t base;   // element offset inside one channel array
    int sn, sc;    // strides (in float2) of the point index n and the column index c
    bool nyq;
    int other;     // x pass: slot py (main) or first py of the tile (nyq)
    int pz0;       // x pass main: first z slot of the tile
};

template <int N, int W> SAP_HD TileDesc tile_desc(int axis, int T) {
    constexpr int H = N / 2;
    constexpr int TILE_W = W;
    constexpr int KT = H / TILE_W;
    TileDesc d;
    if (T < N * KT) {
        const int o = T / KT, kt = T - o * KT;
        d.nyq = false;
        d.other = o;
        d.pz0 = kt * TILE_W;
        d.sc = 1;
        if (axis == 0) { d.base = (size_t)o * H + kt * TILE_W; d.sn = N * H; }
        else { d.base = (size_t)o * N * H + kt * TILE_W; d.sn = H; }
    } else {
        const int t = T - N * KT;
        d.nyq = true;
        d.other = t * TILE_W;
        d.pz0 = 0;
        if (axis == 0) { d.base = (size_t)t * TILE_W; d.sn = N; d.sc = 1; }
        else { d.base = (size_t)t * TILE_W * N; d.sn = 1; d.sc = N; }
    }
    return d;
}

// stage 0, forward: global -> registers -> smem.  Task = (column c, butterfly q); lanes over columns.
template <int N, int W, class Ctx>
SAP_HD void st_first_fwd(Ctx& ctx, const float2* g, const TileDesc& d, float2* s, const float2* tw) {
    constexpr int R = StageInfo<N, 0>::R, ST = StageInfo<N, 0>::ST;
    constexpr int TILE_W = W, TILE_PITCH = W + 1;
    for (int t = ctx.tid; t < ST * TILE_W; t += ctx.nthr) {
        const int q = t / TILE_W, c = t - q * TILE_W;
        float2 v[R];
#pragma unroll
        for (int r = 0; r < R; ++r) v[r] = g[d.base + (size_t)(q + ST * r) * d.sn + (size_t)c * d.sc];
        bfly_fwd<N, 0, N>(v, q, tw);
#pragma unroll
        for (int r = 0; r < R; ++r) s[(q + ST * r) * TILE_PITCH + c] = v[r];
    }
}
// stage 0, inverse: smem -> registers -> global
template <int N, int W, class Ctx>
SAP_HD void st_first_inv(Ctx& ctx, float2* g, const TileDesc& d, const float2* s, const float2* tw) {
    constexpr int R = StageInfo<N, 0>::R, ST = StageInfo<N, 0>::ST;
    constexpr int TILE_W = W, TILE_PITCH = W + 1;
    for (int t = ctx.tid; t < ST * TILE_W; t += ctx.nthr) {
        const int q = t / TILE_W, c = t - q * TILE_W;
        float2 v[R];
#pragma unroll
        for (int r = 0; r < R; ++r) v[r] = s[(q + ST * r) * TILE_PITCH + c];
        bfly_inv<N, 0, N>(v, q, tw);
#pragma unroll
        for (int r = 0; r < R; ++r) g[d.base + (size_t)(q + ST * r) * d.sn + (size_t)c * d.sc] = v[r];
    }
}

// bx: tile index; by: plane index for FWD/INV (item*nch + ch), batch item for SOLVE/ADJ.
// NT = threads per block (compile time: the stride-1 stage keeps per-task accumulators in registers
// across the channel loop, so the task -> thread assignment must be static).
template <int N, int MODE, int NT, int W, class Ctx>
SAP_HD void strided_body(Ctx& ctx, const StridedParams& p, float2* smem, int bx, int by) {
    constexpr int H = N / 2;
    constexpr int NS = Plan<N>::NS;
    constexpr int LS = NS - 1;                      // last plan stage: stride 1
    constexpr int RL = StageInfo<N, LS>::R;
    static_assert(StageInfo<N, LS>::ST == 1 && NS >= 2, "plan");
    constexpr int TILE_W = W, TILE_PITCH = W + 1;
    constexpr int NTASK = (N / RL) * TILE_W;        // butterflies of the stride-1 stage
    constexpr int TPT = (NTASK + NT - 1) / NT;      // per thread
    constexpr size_t SPLANE = (size_t)N * N * H;
    constexpr size_t QPLANE = (size_t)N * N;
    constexpr int IN_CH = (MODE == MODE_SOLVE) ? 3 : 1;
    constexpr int OUT_CH = (MODE == MODE_ADJ) ? 3 : 1;
    float2* s = smem;
    float2* tw = smem + N * TILE_PITCH;
    float4* fx = reinterpret_cast<float4*>(tw + N);  // x-axis frequency entries (SOLVE / ADJ)
    for (int i = ctx.tid; i < N; i += NT) tw[i] = p.tw[i];
    if constexpr (MODE == MODE_SOLVE || MODE == MODE_ADJ)
        for (int i = ctx.tid; i < N; i += NT) fx[i] = p.ftab[i];
    ctx.sync();
    const TileDesc d = tile_desc<N, W>(p.axis, bx);
    auto in_plane = [&](int c) {
        const size_t plane = (size_t)by * IN_CH + c;
        return d.nyq ? p.inQ + plane * QPLANE : p.inS + plane * SPLANE;
    };
    auto out_plane = [&](int c) {
        const size_t plane = (size_t)by * OUT_CH + c;
        return d.nyq ? p.outQ + plane * QPLANE : p.outS + plane * SPLANE;
    };
    // frequency helpers for the stride-1 stage (SOLVE / ADJ)
    auto col_freq = [&](int c, float4& ey, float4& ez) {
        ey = p.ftab[d.nyq ? d.other + c : d.other];
        ez = p.ftab[N + (d.nyq ? H : d.pz0 + c)];
    };

    float2 acc[TPT][RL];  // SOLVE: divergence accumulators; ADJ: -i f Gbar'~ ; FWD/INV: unused
    (void)acc;

    // ---- forward half, channel by channel through the single tile buffer
    if constexpr (MODE != MODE_INV) {
#pragma unroll
        for (int ch = 0; ch < IN_CH; ++ch) {
            if (ch > 0) ctx.sync();  // previous channel's stride-1 reads are done
            st_first_fwd<N, W>(ctx, in_plane(ch), d, s, tw);
            ctx.sync();
            if constexpr (NS == 3) {
                fft_stage<N, 1, false, N, true>(s, TILE_PITCH, 1, TILE_W, tw, ctx.tid, NT);
                ctx.sync();
            }
#pragma unroll
            for (int i = 0; i < TPT; ++i) {
                const int t = ctx.tid + i * NT;
                if (NTASK % NT == 0 || t < NTASK) {
                    const int blk = t / TILE_W, c = t - blk * TILE_W;
                    const int e0 = blk * RL * TILE_PITCH + c;
                    float2 v[RL];
#pragma unroll
                    for (int r = 0; r < RL; ++r) v[r] = s[e0 + r * TILE_PITCH];
                    dft_fwd<RL>(v);
                    if constexpr (MODE == MODE_FWD) {
                        float2* g = out_plane(0);
#pragma unroll
                        for (int r = 0; r < RL; ++r)
                            g[d.base + (size_t)(blk * RL + r) * d.sn + (size_t)c * d.sc] = v[r];
                    } else {
                        float4 ey, ez;
                        col_freq(c, ey, ez);
                        const float hy = ey.x, hz = ez.x;
                        if (MODE == MODE_ADJ || ch == 2) {
                            // finish: multiply by f = cs g / q (and by i or -i)
#pragma unroll
                            for (int r = 0; r < RL; ++r) {
                                const float f = mult_f(fx[blk * RL + r], ey, ez, p.cs);
                                if constexpr (MODE == MODE_SOLVE) {
                                    const float dr = f * (acc[i][r].x + hz * v[r].x), di = f * (acc[i][r].y + hz * v[r].y);
                                    acc[i][r] = make_float2(-di, dr);  // chi~ = i (dr + i di)
                                } else {
                                    acc[i][r] = make_float2(f * v[r].y, -f * v[r].x);  // -i f Gbar'~
                                }
                            }
                        } else if (ch == 0) {
#pragma unroll
                            for (int r = 0; r < RL; ++r) {
                                const float hx = fx[blk * RL + r].x;
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
    }
    // ---- inverse half
    if constexpr (MODE != MODE_FWD) {
#pragma unroll
        for (int ch = 0; ch < OUT_CH; ++ch) {
            if (MODE != MODE_INV || ch > 0) ctx.sync();  // buffer free: stride-1 reads / previous stores done
#pragma unroll
            for (int i = 0; i < TPT; ++i) {
                const int t = ctx.tid + i * NT;
                if (NTASK % NT == 0 || t < NTASK) {
                    const int blk = t / TILE_W, c = t - blk * TILE_W;
                    const int e0 = blk * RL * TILE_PITCH + c;
                    float2 v[RL];
                    if constexpr (MODE == MODE_INV) {
                        const float2* g = in_plane(0);
#pragma unroll
                        for (int r = 0; r < RL; ++r)
                            v[r] = g[d.base + (size_t)(blk * RL + r) * d.sn + (size_t)c * d.sc];
                    } else if constexpr (MODE == MODE_SOLVE) {
#pragma unroll
                        for (int r = 0; r < RL; ++r) v[r] = acc[i][r];
                    } else {
                        float4 ey, ez;
                        col_freq(c, ey, ez);
#pragma unroll
                        for (int r = 0; r < RL; ++r) {
                            const float h = (ch == 0) ? fx[blk * RL + r].x : (ch == 1) ? ey.x : ez.x;
                            v[r] = make_float2(h * acc[i][r].x, h * acc[i][r].y);
                        }
                    }
                    dft_inv<RL>(v);
#pragma unroll
                    for (int r = 0; r < RL; ++r) s[e0 + r * TILE_PITCH] = v[r];
                }
            }
            ctx.sync();
            if constexpr (NS == 3) {
                fft_stage<N, 1, true, N, true>(s, TILE_PITCH, 1, TILE_W, tw, ctx.tid, NT);
                ctx.sync();
            }
            st_first_inv<N, W>(ctx, out_plane(ch), d, s, tw);
        }
    }
}

}  // namespace sap
