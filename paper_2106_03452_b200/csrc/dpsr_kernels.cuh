// dpsr_kernels.cuh -- block bodies of the FFT / spectral-solve kernels of the DPSR path.
//
// Data layout in HBM (per batch item, per channel), H = N/2:
//   real grids      float  [N][N][N]            x slowest, z fastest (the C-ABI layout)
//   main spectrum   float2 [N][N][H]            slots (px, py, pz) in *stored order* on every axis
//   Nyquist plane   float2 [N][N]               the kz = N/2 column of every z-line, slots (px, py)
// "Stored order": slot p of an axis holds frequency pos2freq<len>(p) (fft_core.cuh); x and y are
// length-N complex transforms, z is a real transform done as an H-point complex FFT + split.
//
// Bodies are templates over a context (thread id, thread count, barrier) so the same source can be
// stepped on the host by a debugging harness; the library only instantiates them with DevCtx.
#pragma once
#include "fft_core.cuh"

namespace sap {

constexpr int TILE_W = 16;             // columns (contiguous complex values) per strided tile: 128 B rows
constexpr int TILE_PITCH = TILE_W + 1; // odd pitch: conflict-free for both lane mappings

// ------------------------------------------------------------------------------------------------
// Spectral multiplier of Eq.3 / Eq.16 with readings R3 (Nyquist derivative
// zeroed), R4 (DC zero), R6 (integer frequencies, literal Gaussian):
//   M_c(k) = i m_c,  m_c = g uh_c / (-2 pi q),  g = exp(-2 sigma^2 q / N^2),  q = |u|^2.
// `cg` = 2 sigma^2 / N^2;  `cs` = (2 / N^3) / (-2 pi) folds the inverse-transform scale (R8) and the
// factor 2 of the half-length c2r trick into the multiplier.
// ------------------------------------------------------------------------------------------------
template <int N> SAP_HD void spectral_multiplier(int kx, int ky, int kz, float cg, float cs, float (&m)[3]) {
    constexpr int H = N / 2;
    const int ux = (kx < H) ? kx : kx - N;
    const int uy = (ky < H) ? ky : ky - N;
    const int uz = (kz < H) ? kz : kz - N;
    const int qi = ux * ux + uy * uy + uz * uz;
    if (qi == 0) { m[0] = m[1] = m[2] = 0.f; return; }
    const float q = (float)qi;
    const float f = cs * expf(-cg * q) / q;
    m[0] = (kx == H) ? 0.f : f * (float)ux;
    m[1] = (ky == H) ? 0.f : f * (float)uy;
    m[2] = (kz == H) ? 0.f : f * (float)uz;
}

// ------------------------------------------------------------------------------------------------
// z (+ y) forward: real lines -> half spectrum.  One block owns NL z-lines (consecutive in memory);
// with DO_Y, NL == N and the block owns one whole x-plane and also transforms along y, so the plane
// makes one trip through shared memory for two axes (F2 of SURVEY 8(a); B3 with GBAR).
// GBAR (backward, B2): the input is assembled on the fly, Gbar' = s G + (beta/P) W - (S1/a) delta_0.
// ------------------------------------------------------------------------------------------------
struct ZyFwdParams {
    const float* in;    // [planes][N^3] real input (v, or G in GBAR mode)
    const float* W;     // GBAR: [batch][N^3] point density
    const float* bw;    // GBAR: [batch][4] = {s, beta/P, S1/a, -}
    float2* S;          // [planes][N*N*H]
    float2* Q;          // [planes][N*N]
    const float2* tw;   // exp(-2 pi i t / N), t < N
    int nch;            // planes per batch item
};

template <int N, int NL, bool DO_Y, bool GBAR>
constexpr size_t zy_smem_bytes() { return ((size_t)(N / 2 + 1) * (NL + 1) + N) * sizeof(float2); }

template <int N, int NL, bool DO_Y, bool GBAR, class Ctx>
SAP_HD void zy_fwd_body(Ctx& ctx, const ZyFwdParams& p, float2* smem, int bx, int by) {
    constexpr int H = N / 2;
    constexpr int PITCH = NL + 1;
    static_assert(!DO_Y || NL == N, "plane mode owns N lines");
    float2* s = smem;
    float2* tw = smem + (H + 1) * PITCH;
    const size_t V = (size_t)N * N * N;
    const size_t line0 = (size_t)bx * NL;  // global line index = x*N + y
    for (int i = ctx.tid; i < N; i += ctx.nthr) tw[i] = p.tw[i];

    const float2* in2 = reinterpret_cast<const float2*>(p.in + (size_t)by * V) + line0 * H;
    if (!GBAR) {
        for (int i = ctx.tid; i < NL * H; i += ctx.nthr) {
            const int l = i / H, m = i - l * H;
            s[m * PITCH + l] = in2[i];
        }
    } else {
        const int item = by / p.nch;
        const float2* w2 = reinterpret_cast<const float2*>(p.W + (size_t)item * V) + line0 * H;
        const float cs_ = p.bw[item * 4 + 0], cw = p.bw[item * 4 + 1], c0 = p.bw[item * 4 + 2];
        for (int i = ctx.tid; i < NL * H; i += ctx.nthr) {
            const int l = i / H, m = i - l * H;
            float2 g = in2[i], w = w2[i];
            float2 v = make_float2(cs_ * g.x + cw * w.x, cs_ * g.y + cw * w.y);
            if (line0 == 0 && i == 0) v.x -= c0;
            s[m * PITCH + l] = v;
        }
    }
    ctx.sync();
    // z: H-point complex FFT of the packed (even, odd) samples, one line per lane
    fft_lines<H, false, N, true>(ctx, s, PITCH, 1, NL, tw);
    r2c_split<N, N>(ctx, s, PITCH, 1, NL, tw);
    ctx.sync();
    if constexpr (DO_Y) {
        // y: N-point complex FFT along the fast smem index, lines = the H+1 kz rows
        constexpr int NS = Plan<N>::NS;
        fft_stage<N, 0, false, N, true>(s, 1, PITCH, H, tw, ctx.tid, ctx.nthr);
        fft_stage<N, 0, false, N, false>(s + H * PITCH, 1, PITCH, 1, tw, ctx.tid, ctx.nthr);
        ctx.sync();
        if constexpr (NS > 1) {
            fft_stage<N, 1, false, N, true>(s, 1, PITCH, H, tw, ctx.tid, ctx.nthr);
            fft_stage<N, 1, false, N, false>(s + H * PITCH, 1, PITCH, 1, tw, ctx.tid, ctx.nthr);
            ctx.sync();
        }
        if constexpr (NS > 2) {
            fft_stage<N, 2, false, N, true>(s, 1, PITCH, H, tw, ctx.tid, ctx.nthr);
            fft_stage<N, 2, false, N, false>(s + H * PITCH, 1, PITCH, 1, tw, ctx.tid, ctx.nthr);
            ctx.sync();
        }
    }
    float2* So = p.S + (size_t)by * ((size_t)N * N * H) + line0 * H;
    for (int i = ctx.tid; i < NL * H; i += ctx.nthr) {
        const int l = i / H, pz = i - l * H;
        So[i] = s[pz * PITCH + l];
    }
    float2* Qo = p.Q + (size_t)by * ((size_t)N * N) + line0;
    for (int l = ctx.tid; l < NL; l += ctx.nthr) Qo[l] = s[H * PITCH + l];
}

// ------------------------------------------------------------------------------------------------
// (y +) z inverse: half spectrum -> real lines (F4 / B5).  Mirror image of zy_fwd_body.
// ------------------------------------------------------------------------------------------------
struct ZyInvParams {
    const float2* S;   // [planes][N*N*H]
    const float2* Q;   // [planes][N*N]
    float* out;        // [planes][N^3]
    const float2* tw;
};

template <int N, int NL, bool DO_Y, class Ctx>
SAP_HD void zy_inv_body(Ctx& ctx, const ZyInvParams& p, float2* smem, int bx, int by) {
    constexpr int H = N / 2;
    constexpr int PITCH = NL + 1;
    float2* s = smem;
    float2* tw = smem + (H + 1) * PITCH;
    const size_t V = (size_t)N * N * N;
    const size_t line0 = (size_t)bx * NL;
    for (int i = ctx.tid; i < N; i += ctx.nthr) tw[i] = p.tw[i];
    const float2* Si = p.S + (size_t)by * ((size_t)N * N * H) + line0 * H;
    for (int i = ctx.tid; i < NL * H; i += ctx.nthr) {
        const int l = i / H, pz = i - l * H;
        s[pz * PITCH + l] = Si[i];
    }
    const float2* Qi = p.Q + (size_t)by * ((size_t)N * N) + line0;
    for (int l = ctx.tid; l < NL; l += ctx.nthr) s[H * PITCH + l] = Qi[l];
    ctx.sync();
    if constexpr (DO_Y) {
        constexpr int NS = Plan<N>::NS;
        if constexpr (NS > 2) {
            fft_stage<N, 2, true, N, true>(s, 1, PITCH, H, tw, ctx.tid, ctx.nthr);
            fft_stage<N, 2, true, N, false>(s + H * PITCH, 1, PITCH, 1, tw, ctx.tid, ctx.nthr);
            ctx.sync();
        }
        if constexpr (NS > 1) {
            fft_stage<N, 1, true, N, true>(s, 1, PITCH, H, tw, ctx.tid, ctx.nthr);
            fft_stage<N, 1, true, N, false>(s + H * PITCH, 1, PITCH, 1, tw, ctx.tid, ctx.nthr);
            ctx.sync();
        }
        fft_stage<N, 0, true, N, true>(s, 1, PITCH, H, tw, ctx.tid, ctx.nthr);
        fft_stage<N, 0, true, N, false>(s + H * PITCH, 1, PITCH, 1, tw, ctx.tid, ctx.nthr);
        ctx.sync();
    }
    c2r_split<N, N>(ctx, s, PITCH, 1, NL, tw);
    ctx.sync();
    fft_lines<H, true, N, true>(ctx, s, PITCH, 1, NL, tw);
    float2* out2 = reinterpret_cast<float2*>(p.out + (size_t)by * V) + line0 * H;
    for (int i = ctx.tid; i < NL * H; i += ctx.nthr) {
        const int l = i / H, m = i - l * H;
        out2[i] = s[m * PITCH + l];
    }
}

// ------------------------------------------------------------------------------------------------
// Strided-axis pass over tiles of N points x 16 contiguous columns.
//   MODE_FWD / MODE_INV : plain forward / inverse transform along `axis` (the y pass when N >= 256)
//   MODE_SOLVE (F2x+F3+F4x): forward x on 3 channels, chi~ = i sum_c m_c v~_c, inverse x, 1 channel out
//   MODE_ADJ   (B3x+B4+B5x): forward x on 1 channel, vbar~_c = conj(M_c) Gbar'~ = -i m_c Gbar'~, 3 inverse x
// Tiles cover the main spectrum and then the Nyquist plane (different strides, same code).
// ------------------------------------------------------------------------------------------------
enum { MODE_FWD = 0, MODE_INV = 1, MODE_SOLVE = 2, MODE_ADJ = 3 };

struct StridedParams {
    const float2* inS;
    const float2* inQ;
    float2* outS;
    float2* outQ;
    const float2* tw;
    int axis;     // 0: along x (stride N*H / N), 1: along y (stride H / 1)
    float cg;     // 2 sigma^2 / N^2
    float cs;     // (2 / N^3) / (-2 pi)
};

template <int N> constexpr int strided_tiles() { return N * (N / 2 / TILE_W) + N / TILE_W; }
template <int N, int MODE> constexpr int strided_channels() { return (MODE == MODE_SOLVE || MODE == MODE_ADJ) ? 3 : 1; }
template <int N, int MODE>
constexpr size_t strided_smem_bytes() {
    return ((size_t)strided_channels<N, MODE>() * N * TILE_PITCH + N) * sizeof(float2);
}

struct TileDesc {
    size_t base;   // element offset inside one channel array
    int sn, sc;    // strides (in float2) of the point index n and the column index c
    bool nyq;
    int other;     // x pass: slot py (main) or first py of the tile (nyq); y pass: unused
    int pz0;       // x pass main: first z slot of the tile
};

template <int N> SAP_HD TileDesc tile_desc(int axis, int T) {
    constexpr int H = N / 2;
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

template <int N, class Ctx>
SAP_HD void tile_load(Ctx& ctx, const float2* g, const TileDesc& d, float2* s) {
    if (d.sc == 1) {
        for (int i = ctx.tid; i < N * TILE_W; i += ctx.nthr) {
            const int n = i / TILE_W, c = i - n * TILE_W;
            s[n * TILE_PITCH + c] = g[d.base + (size_t)n * d.sn + c];
        }
    } else {
        for (int i = ctx.tid; i < N * TILE_W; i += ctx.nthr) {
            const int c = i / N, n = i - c * N;
            s[n * TILE_PITCH + c] = g[d.base + (size_t)c * d.sc + n];
        }
    }
}
template <int N, class Ctx>
SAP_HD void tile_store(Ctx& ctx, float2* g, const TileDesc& d, const float2* s) {
    if (d.sc == 1) {
        for (int i = ctx.tid; i < N * TILE_W; i += ctx.nthr) {
            const int n = i / TILE_W, c = i - n * TILE_W;
            g[d.base + (size_t)n * d.sn + c] = s[n * TILE_PITCH + c];
        }
    } else {
        for (int i = ctx.tid; i < N * TILE_W; i += ctx.nthr) {
            const int c = i / N, n = i - c * N;
            g[d.base + (size_t)c * d.sc + n] = s[n * TILE_PITCH + c];
        }
    }
}

// bx: tile index; by: plane index of the INPUT side for FWD/INV (item*nch + ch), batch item for SOLVE/ADJ
template <int N, int MODE, class Ctx>
SAP_HD void strided_body(Ctx& ctx, const StridedParams& p, float2* smem, int bx, int by) {
    constexpr int H = N / 2;
    constexpr int CH = strided_channels<N, MODE>();
    constexpr int BUF = N * TILE_PITCH;
    constexpr size_t SPLANE = (size_t)N * N * H;
    constexpr size_t QPLANE = (size_t)N * N;
    float2* s = smem;
    float2* tw = smem + CH * BUF;
    for (int i = ctx.tid; i < N; i += ctx.nthr) tw[i] = p.tw[i];
    const TileDesc d = tile_desc<N>(p.axis, bx);
    constexpr int IN_CH = (MODE == MODE_SOLVE) ? 3 : 1;
    constexpr int OUT_CH = (MODE == MODE_ADJ) ? 3 : 1;
    for (int c = 0; c < IN_CH; ++c) {
        const size_t plane = (size_t)by * IN_CH + c;
        const float2* g = d.nyq ? p.inQ + plane * QPLANE : p.inS + plane * SPLANE;
        tile_load<N>(ctx, g, d, s + c * BUF);
    }
    ctx.sync();
    if constexpr (MODE != MODE_INV) {
        for (int c = 0; c < IN_CH; ++c) {
            // stages of different channels are independent: barrier once per stage, not per channel
            fft_stage<N, 0, false, N, true>(s + c * BUF, TILE_PITCH, 1, TILE_W, tw, ctx.tid, ctx.nthr);
        }
        ctx.sync();
        if constexpr (Plan<N>::NS > 1) {
            for (int c = 0; c < IN_CH; ++c)
                fft_stage<N, 1, false, N, true>(s + c * BUF, TILE_PITCH, 1, TILE_W, tw, ctx.tid, ctx.nthr);
            ctx.sync();
        }
        if constexpr (Plan<N>::NS > 2) {
            for (int c = 0; c < IN_CH; ++c)
                fft_stage<N, 2, false, N, true>(s + c * BUF, TILE_PITCH, 1, TILE_W, tw, ctx.tid, ctx.nthr);
            ctx.sync();
        }
    }
    if constexpr (MODE == MODE_SOLVE || MODE == MODE_ADJ) {
        for (int i = ctx.tid; i < N * TILE_W; i += ctx.nthr) {
            const int n = i / TILE_W, c = i - n * TILE_W;
            const int kx = pos2freq<N>(n);
            const int ky = pos2freq<N>(d.nyq ? d.other + c : d.other);
            const int kz = d.nyq ? H : pos2freq<H>(d.pz0 + c);
            float m[3];
            spectral_multiplier<N>(kx, ky, kz, p.cg, p.cs, m);
            const int e = n * TILE_PITCH + c;
            if constexpr (MODE == MODE_SOLVE) {
                const float2 a = s[e], b = s[BUF + e], cc = s[2 * BUF + e];
                const float dr = m[0] * a.x + m[1] * b.x + m[2] * cc.x;
                const float di = m[0] * a.y + m[1] * b.y + m[2] * cc.y;
                s[e] = make_float2(-di, dr);  // i * (dr + i di)
            } else {
                const float2 g = s[e];
                s[e] = make_float2(m[0] * g.y, -m[0] * g.x);  // -i m (gr + i gi)
                s[BUF + e] = make_float2(m[1] * g.y, -m[1] * g.x);
                s[2 * BUF + e] = make_float2(m[2] * g.y, -m[2] * g.x);
            }
        }
        ctx.sync();
    }
    if constexpr (MODE != MODE_FWD) {
        if constexpr (Plan<N>::NS > 2) {
            for (int c = 0; c < OUT_CH; ++c)
                fft_stage<N, 2, true, N, true>(s + c * BUF, TILE_PITCH, 1, TILE_W, tw, ctx.tid, ctx.nthr);
            ctx.sync();
        }
        if constexpr (Plan<N>::NS > 1) {
            for (int c = 0; c < OUT_CH; ++c)
                fft_stage<N, 1, true, N, true>(s + c * BUF, TILE_PITCH, 1, TILE_W, tw, ctx.tid, ctx.nthr);
            ctx.sync();
        }
        for (int c = 0; c < OUT_CH; ++c)
            fft_stage<N, 0, true, N, true>(s + c * BUF, TILE_PITCH, 1, TILE_W, tw, ctx.tid, ctx.nthr);
        ctx.sync();
    }
    for (int c = 0; c < OUT_CH; ++c) {
        const size_t plane = (size_t)by * OUT_CH + c;
        float2* g = d.nyq ? p.outQ + plane * QPLANE : p.outS + plane * SPLANE;
        tile_store<N>(ctx, g, d, s + c * BUF);
    }
}

}  // namespace sap
