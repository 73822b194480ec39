// fused_small.cuh -- the latency path: the WHOLE forward (F1-F5) and the WHOLE backward (B1-B6) of SURVEY 8(a) as
// ONE cooperative kernel each, for grids whose x-planes all fit one wave of CTAs (N <= 128 and batch * N <= #CTAs:
// the coarse-to-fine levels 32^3 / 64^3 / 128^3 of PAPER.md:L121 / L396 and the 128^3 headline config at batch 1).
//
// Why: at these sizes the 13-launch chain of the throughput path is latency-bound (every launch is one wave of
// CTAs whose critical path is a chain of dependent loads and block barriers; 0.09-0.10 ms per forward+backward at
// 32^3 / 64^3 against a microsecond of HBM time).  Here the phases of the path are separated by grid barriers
// (one atomic arrive + an acquire spin, ~1 us) instead of kernel boundaries, data that a CTA produces and consumes
// itself stays in its shared memory ACROSS the barrier, and several HBM round trips disappear altogether:
//   forward  : [bin count] | [bin offsets + scatter] | [splat + z + y forward, 3 channels of an x-plane per CTA]
//              | [x forward + spectral solve + x inverse, 4 column-tile groups per CTA]
//              | [y + z inverse of an x-plane; partial sum of chi' at the points]  | [chi = s (chi' - mu), written once]
//              (chi' never exists in HBM: the plane waits in shared memory for mu)
//   backward : [S0, S1 partial sums; chi and G planes stay in shared memory] | [chi term of dL/dc; Gbar' assembled on
//              top of G; z + y forward] | [x forward + transposed multiplier + 2 x inverses] | [y + z inverse of the 3
//              channels of an x-plane; owner-computes gather of dL/dn and dL/dc from shared memory]
//              (vbar never exists in HBM; the gradients are accumulated with float atomics: each point receives the
//              contributions of its two x-planes)
// Equations: Eq.10-11 (splat), Eq.12-17 (FFTs, solve), Eq.4/18 (normalisation); backward: DESIGN.md 3.
//
// Every phase body is a __host__ __device__ template on a small context (thread index, barrier, atomics), so the
// whole path also runs on the CPU, CTA after CTA, phase after phase (tests/host/fused_emulate.cpp): index logic is
// checked against the oracle without a GPU.  The spectra use the same stored order / column swizzle as the
// throughput path (dpsr_kernels.cuh), so the two paths can be mixed phase by phase.
#pragma once
#include <math.h>
#include "fft_core.cuh"
#include "spectral.cuh"
#include "zy_pass.cuh"

namespace sap {

struct FusedParams {
    // caller's buffers
    const float* pts;   // [B][P][3]
    const float* nrm;   // [B][P][3]
    float* chi;         // [B][N^3]  forward: written; backward: read
    const float* G;     // [B][N^3]  backward: dL/dchi
    float* gp;          // [B][P][3] backward: dL/dpoints
    float* gn;          // [B][P][3] backward: dL/dnormals
    int P, B;
    // workspace of the handle
    float4* spts;       // [B][P] points sorted by x-slab {cx, cy, cz, original index}
    float4* snrm;       // [B][P]
    int* bin_start;     // [B][N + 1]
    int* hist;          // [B][#CTAs][N] per-CTA histograms of the counting sort
    float2* S3;         // [B*3][N*N*H] + Q3 [B*3][N*N]: 3-channel spectrum (stored order, swizzled columns)
    float2* Q3;
    float2* S1;         // [B][N*N*H] + Q1 [B][N*N]
    float2* Q1;
    const float2* tw;   // exp(-2 pi i t / N)
    const float4* ftab; // per-slot frequency table (spectral.cuh)
    double* acc;        // [B][2] reduction accumulators, zero between launches
    float* stats;       // [B][4] {mu, a, s, chi'[0,0,0]}
    float* bw;          // [B][4] {s, beta/P, S1/a, beta/(P s)}
    unsigned* sync;     // [0] barrier arrivals, [1] exits (both zero between launches), [2] sticky time-out flag
    long long* stamps;  // [64] clock64 of CTA 0 at the marks of the phase bodies (profiling; may be null)
    float cs;           // (2 / N^3) / (-2 pi): inverse-transform scale and the c2r factor folded into the multiplier
};

// ---- shared-memory carve-up ---------------------------------------------------------------------------------------
template <int N> struct FusedCfg {
    static constexpr int H = N / 2, PITCH = N + 1;
    static constexpr int NT = 512;                       // threads per CTA
    static constexpr int XW = 16, XNTC = 128, XNG = NT / XNTC;  // x pass: 4 groups of 128 threads, tiles of N x 16 columns
    static constexpr int MAXB = (N == 32) ? 4 : (N == 64) ? 2 : 1;
    static constexpr size_t PAD = (size_t)(H + 1) * PITCH;   // float2 per padded plane (forward z/y layout)
    static constexpr size_t DENSE = (size_t)N * H + N;       // float2 per dense plane + its Nyquist values
    static constexpr size_t XBUF = (size_t)N * XW;           // float2 per x-pass buffer
    static constexpr size_t cmax(size_t a, size_t b) { return a > b ? a : b; }
    static constexpr size_t PADA = (PAD + 1) / 2 * 2;              // 16-byte aligned start of what follows a padded plane
    static constexpr size_t BIG = cmax(cmax(3 * PAD + 1, 3 * DENSE), cmax((size_t)XNG * 2 * XBUF, PADA + (size_t)N * H + PAD));
    // byte offsets
    static constexpr size_t o_tw = 0;                                   // float2[N]
    static constexpr size_t o_tabF = o_tw + (size_t)N * 8;              // float4[N]
    static constexpr size_t o_tabI = o_tabF + (size_t)N * 16;           // float4[N]
    static constexpr size_t o_fx = o_tabI + (size_t)N * 16;             // float4[N]
    static constexpr size_t o_fz = o_fx + (size_t)N * 16;               // float[H + 1] (+ pad)
    static constexpr size_t o_bins = o_fz + (size_t)(H + 4) * 4;        // int[MAXB][N + 1]
    static constexpr size_t o_scr = (o_bins + (size_t)MAXB * (N + 1) * 4 + 15) / 16 * 16;  // int[8 * NT + 2 * N + 64]
    static constexpr size_t o_big = (o_scr + (size_t)(8 * NT + 2 * N + 64) * 4 + 127) / 128 * 128;
    static constexpr size_t BYTES = o_big + BIG * 8;
};
static_assert(FusedCfg<128>::BYTES <= 227 * 1024, "fused kernels must fit the shared memory of an SM");

template <int N> struct FusedSmem {
    using C = FusedCfg<N>;
    float2* tw; float4* tabF; float4* tabI; float4* fx; float* fz; int* bins; int* scr; float2* big;
    SAP_HD explicit FusedSmem(unsigned char* base)
        : tw(reinterpret_cast<float2*>(base + C::o_tw)), tabF(reinterpret_cast<float4*>(base + C::o_tabF)),
          tabI(reinterpret_cast<float4*>(base + C::o_tabI)), fx(reinterpret_cast<float4*>(base + C::o_fx)),
          fz(reinterpret_cast<float*>(base + C::o_fz)), bins(reinterpret_cast<int*>(base + C::o_bins)),
          scr(reinterpret_cast<int*>(base + C::o_scr)), big(reinterpret_cast<float2*>(base + C::o_big)) {}
};

// ---- small helpers ---------------------------------------------------------------------------------------------------
// loads of data another CTA wrote in an earlier phase: L2 only (no stale or polluted L1 lines)
SAP_HD float2 ld2(const float2* p) {
#ifdef __CUDA_ARCH__
    return __ldcg(p);
#else
    return *p;
#endif
}
SAP_HD int4 ldi4(const int4* p) {
#ifdef __CUDA_ARCH__
    return __ldcg(p);
#else
    return *p;
#endif
}
SAP_HD float4 ld4(const float4* p) {
#ifdef __CUDA_ARCH__
    return __ldcg(p);
#else
    return *p;
#endif
}
// a * w with the table entry t = {w.x, w.y, -w.y, w.x} (forward) or {w.x, -w.y, w.y, w.x} (a * conj w)
SAP_HD float2 fcmul4(float2 a, float4 t) {
#ifdef __CUDA_ARCH__
    return __ffma2_rn(make_float2(a.y, a.y), make_float2(t.z, t.w), __fmul2_rn(make_float2(a.x, a.x), make_float2(t.x, t.y)));
#else
    return make_float2(a.x * t.x + a.y * t.z, a.x * t.y + a.y * t.w);
#endif
}
SAP_HD float bits_i2f(int i) {
#ifdef __CUDA_ARCH__
    return __int_as_float(i);
#else
    union { int i; float f; } u; u.i = i; return u.f;
#endif
}
SAP_HD int bits_f2i(float f) {
#ifdef __CUDA_ARCH__
    return __float_as_int(f);
#else
    union { int i; float f; } u; u.f = f; return u.i;
#endif
}
// index of (line l, z slot pz) in a dense plane (column swizzle of the HBM layout, see kz_swz)
template <int H> SAP_HD int dzi(int l, int pz) { return l * H + (pz ^ (l & 15)); }

// trilinear footprint of a point restricted to ONE x-plane: the plane takes the (1 - fx) share of the points of its own
// slab (k = 0) and the fx share of the points of the slab before it (k = 1)  (Eq.10-11; R1, R2)
struct Foot {
    int jy, jz;
    float wx, fy, fz;
    float sx;   // sign of dw/dcx on this plane: -1 (k = 0), +1 (k = 1)
};
template <int N> SAP_HD Foot foot_of(float4 c, int k) {
    const float tx = c.x * (float)N, ty = c.y * (float)N, tz = c.z * (float)N;
    const float fx0 = floorf(tx), fy0 = floorf(ty), fz0 = floorf(tz);
    const float fx = tx - fx0;
    Foot f;
    f.jy = (int)fy0; f.jz = (int)fz0;
    f.fy = ty - fy0; f.fz = tz - fz0;
    f.wx = k ? fx : 1.f - fx;
    f.sx = k ? 1.f : -1.f;
    return f;
}
template <int N> SAP_HD int slab_of(const float* c) { return (int)floorf(c[0] * (float)N) & (N - 1); }

// ---- tables (constants of the handle; built before the dependency wait) -------------------------------------------
template <int N, class Ctx> SAP_HD void fused_tables(Ctx& ctx, const FusedParams& p, FusedSmem<N>& sm) {
    constexpr int H = N / 2, R0 = StageInfo<N, 0>::R;
    static_assert(Plan<N>::NS == 2, "x and y plans of the fused path have two stages");
    for (int i = ctx.tid; i < N; i += ctx.nthr) {
        sm.tw[i] = p.tw[i];
        const int j = i / R0, r = i - j * R0;
        const float2 w = p.tw[r * j];   // stage-0 twiddle w_N^{r j}
        sm.tabF[i] = make_float4(w.x, w.y, -w.y, w.x);
        sm.tabI[i] = make_float4(w.x, -w.y, w.y, w.x);
        sm.fx[i] = p.ftab[i];
    }
    for (int i = ctx.tid; i <= H; i += ctx.nthr) sm.fz[i] = p.ftab[N + i].x;
}

// =====================================================================================================================
// forward z + y transform of NCH real x-planes held in shared memory in the padded layout of zy_pass.cuh:
// value (line l = y, z = 2m + par) of channel ch at s[ch*PAD + m*PITCH + l].{x,y}.  Result: S[ch] (main spectrum of
// this x-plane, N*H complex, swizzled columns) and Q[ch] (Nyquist values of its N lines).  The first stage applies
// v <- gs * v (- c0 at voxel (y,z) = (0,0) when `origin`): Gbar' = s (G + W (beta/P)/s) - (S1/a) delta_0 in the backward.
// =====================================================================================================================
// Input of the first stage:
//   FIX  the planes hold 32-bit fixed-point sums (rasterised field): v = int * gs           (gs = 1 / S)
//   GBAR plane 0 holds G (float), `wpl` the fixed-point density W: v = gs * G + cw * W      (cw = (beta/P) / S_w)
enum { PSRC_FIX = 0, PSRC_GBAR = 1 };
template <int N, int NCH, int PSRC, class Ctx>
SAP_HD void plane_fwd_zy(Ctx& ctx, float2* s, const int2* wpl, const float2* tw, float gs, float cw, float c0, bool origin,
                         float2* So, size_t strideS, float2* Qo, size_t strideQ, int sid) {
    constexpr int H = N / 2, PITCH = N + 1;
    constexpr size_t PAD = FusedCfg<N>::PAD;
    constexpr int R0 = StageInfo<H, 0>::R, ST0 = StageInfo<H, 0>::ST;
    static_assert(Plan<H>::NS <= 2 && ST0 <= 16, "z plans have at most two stages");
    // z stage 0
    for (int t = ctx.tid; t < NCH * N * ST0; t += ctx.nthr) {
        const int ch = t / (N * ST0), tt = t - ch * (N * ST0);
        int l, q;
        zline_task<ST0>(tt, l, q);
        float2* sc = s + ch * PAD;
        float2 v[R0];
#pragma unroll
        for (int r = 0; r < R0; ++r) {
            const int e = (q + ST0 * r) * PITCH + l;
            if (PSRC == PSRC_FIX) {
                const int2 iv = reinterpret_cast<const int2*>(sc)[e];
                v[r] = make_float2(gs * (float)iv.x, gs * (float)iv.y);
            } else {
                const float2 g = sc[e];
                const int2 iw = wpl[e];
                v[r] = make_float2(gs * g.x + cw * (float)iw.x, gs * g.y + cw * (float)iw.y);
            }
        }
        if (origin && l == 0 && q == 0) v[0].x -= c0;
        bfly_fwd<H, 0, N>(v, q, tw);
#pragma unroll
        for (int r = 0; r < R0; ++r) sc[(q + ST0 * r) * PITCH + l] = v[r];
    }
    ctx.sync();
    ctx.stamp(sid);
    if constexpr (Plan<H>::NS > 1) {
        for (int ch = 0; ch < NCH; ++ch) fft_stage<H, 1, false, N, true>(s + ch * PAD, PITCH, 1, N, tw, ctx.tid, ctx.nthr);
        ctx.sync();
    }
    ctx.stamp(sid + 1);
    // r2c split fused into y stage 0: one task owns the row pair (k, H-k) for RY y-values
    constexpr int RY = StageInfo<N, 0>::R, STY = StageInfo<N, 0>::ST;
    constexpr int TC = (H / 2 + 1) * STY;
    for (int t = ctx.tid; t < NCH * TC; t += ctx.nthr) {
        const int ch = t / TC, tt = t - ch * TC;
        const int k = tt / STY, q = tt - k * STY;
        float2* sc = s + ch * PAD;
        float2 a[RY], b[RY];
        int ra, rb;
        if (k == 0) {
            ra = 0; rb = H;
#pragma unroll
            for (int r = 0; r < RY; ++r) {
                const float2 z = sc[q + STY * r];
                a[r] = make_float2(z.x + z.y, 0.f);
                b[r] = make_float2(z.x - z.y, 0.f);
            }
        } else if (k == H / 2) {
            ra = rb = freq2pos<H>(k);
#pragma unroll
            for (int r = 0; r < RY; ++r) {
                const float2 z = sc[ra * PITCH + q + STY * r];
                a[r] = make_float2(z.x, -z.y);
                b[r] = a[r];
            }
        } else {
            ra = freq2pos<H>(k); rb = freq2pos<H>(H - k);
            const float2 w = tw[k];
#pragma unroll
            for (int r = 0; r < RY; ++r) {
                a[r] = sc[ra * PITCH + q + STY * r];
                b[r] = sc[rb * PITCH + q + STY * r];
                r2c_pair(a[r], b[r], w);
            }
        }
        bfly_fwd<N, 0, N>(a, q, tw);
#pragma unroll
        for (int r = 0; r < RY; ++r) sc[ra * PITCH + q + STY * r] = a[r];
        if (rb != ra) {
            bfly_fwd<N, 0, N>(b, q, tw);
#pragma unroll
            for (int r = 0; r < RY; ++r) sc[rb * PITCH + q + STY * r] = b[r];
        }
    }
    ctx.sync();
    ctx.stamp(sid + 2);
    // last y stage: smem -> registers -> HBM, lanes over z slots (contiguous in HBM)
    constexpr int R1 = StageInfo<N, 1>::R;
    static_assert(StageInfo<N, 1>::ST == 1, "last stage");
    constexpr int TD = H * (N / R1);
    for (int t = ctx.tid; t < NCH * TD; t += ctx.nthr) {
        const int ch = t / TD, tt = t - ch * TD;
        const int blk = tt / H, pz = tt - blk * H;
        const float2* sc = s + ch * PAD;
        float2* out = So + ch * strideS;
        float2 v[R1];
#pragma unroll
        for (int r = 0; r < R1; ++r) v[r] = sc[pz * PITCH + blk * R1 + r];
        dft_fwd<R1>(v);
#pragma unroll
        for (int r = 0; r < R1; ++r) out[(size_t)(blk * R1 + r) * H + kz_swz(pz, blk * R1 + r)] = v[r];
    }
    for (int t = ctx.tid; t < NCH * (N / R1); t += ctx.nthr) {  // Nyquist row
        const int ch = t / (N / R1), blk = t - ch * (N / R1);
        const float2* sc = s + ch * PAD;
        float2* out = Qo + ch * strideQ;
        float2 v[R1];
#pragma unroll
        for (int r = 0; r < R1; ++r) v[r] = sc[H * PITCH + blk * R1 + r];
        dft_fwd<R1>(v);
#pragma unroll
        for (int r = 0; r < R1; ++r) out[blk * R1 + r] = v[r];
    }
    ctx.stamp(sid + 3);
}

// =====================================================================================================================
// inverse y + z transform, in place, of NCH spectrum planes held DENSE in shared memory (plane ch at s + ch*DENSE:
// N*H complex in the HBM layout of an x-plane followed by its N Nyquist values).  On return the real value (line l, z)
// of channel ch sits at component z & 1 of s[ch*DENSE + dzi<H>(l, z >> 1)].
// ADJ: channels 1 and 2 are both the spectrum B of the adjoint; h_y (per y slot) / h_z (per z slot) are applied on the
// way into the first stage: vbar_y = IFFT(h_y B), vbar_z = IFFT(h_z B).
// =====================================================================================================================
template <int N, int NCH, bool ADJ, class Ctx>
SAP_HD void plane_inv_yz(Ctx& ctx, float2* s, const float2* tw, const float4* fy, const float* fz, int sid) {
    constexpr int H = N / 2;
    constexpr size_t DENSE = FusedCfg<N>::DENSE;
    constexpr int R1 = StageInfo<N, 1>::R;
    // inverse of the last y stage, lanes over z slots
    constexpr int TD = H * (N / R1);
    for (int t = ctx.tid; t < NCH * TD; t += ctx.nthr) {
        const int ch = t / TD, tt = t - ch * TD;
        const int blk = tt / H, pz = tt - blk * H;
        float2* sc = s + ch * DENSE;
        float2 v[R1];
#pragma unroll
        for (int r = 0; r < R1; ++r) v[r] = sc[dzi<H>(blk * R1 + r, pz)];
        if (ADJ && ch == 1) {
#pragma unroll
            for (int r = 0; r < R1; ++r) v[r] = cscale(fy[blk * R1 + r].x, v[r]);
        } else if (ADJ && ch == 2) {
            const float w = fz[pz];
#pragma unroll
            for (int r = 0; r < R1; ++r) v[r] = cscale(w, v[r]);
        }
        dft_inv<R1>(v);
#pragma unroll
        for (int r = 0; r < R1; ++r) sc[dzi<H>(blk * R1 + r, pz)] = v[r];
    }
    for (int t = ctx.tid; t < NCH * (N / R1); t += ctx.nthr) {
        const int ch = t / (N / R1), blk = t - ch * (N / R1);
        float2* sc = s + ch * DENSE + (size_t)N * H;
        float2 v[R1];
#pragma unroll
        for (int r = 0; r < R1; ++r) v[r] = sc[blk * R1 + r];
        if (ADJ && ch == 1) {
#pragma unroll
            for (int r = 0; r < R1; ++r) v[r] = cscale(fy[blk * R1 + r].x, v[r]);
        } else if (ADJ && ch == 2) {
#pragma unroll
            for (int r = 0; r < R1; ++r) v[r] = cscale(fz[H], v[r]);  // h_z = 0 on the Nyquist plane (R3)
        }
        dft_inv<R1>(v);
#pragma unroll
        for (int r = 0; r < R1; ++r) sc[blk * R1 + r] = v[r];
    }
    ctx.sync();
    ctx.stamp(sid);
    // inverse y stage 0 on the slot pair (k, H-k), then the c2r split, in registers
    constexpr int RY = StageInfo<N, 0>::R, STY = StageInfo<N, 0>::ST;
    constexpr int TC = (H / 2 + 1) * STY;
    for (int t = ctx.tid; t < NCH * TC; t += ctx.nthr) {
        const int ch = t / TC, tt = t - ch * TC;
        const int k = tt / STY, q = tt - k * STY;
        float2* sc = s + ch * DENSE;
        float2 a[RY], b[RY];
        const int ra = (k == 0) ? 0 : freq2pos<H>(k);
        const int rb = (k == 0) ? H : freq2pos<H>(H - k);
#pragma unroll
        for (int r = 0; r < RY; ++r) a[r] = sc[dzi<H>(q + STY * r, ra)];
        bfly_inv<N, 0, N>(a, q, tw);
        if (rb != ra) {
#pragma unroll
            for (int r = 0; r < RY; ++r) b[r] = (k == 0) ? sc[N * H + q + STY * r] : sc[dzi<H>(q + STY * r, rb)];
            bfly_inv<N, 0, N>(b, q, tw);
        }
        if (k == 0) {
#pragma unroll
            for (int r = 0; r < RY; ++r)
                sc[dzi<H>(q + STY * r, 0)] = make_float2(0.5f * (a[r].x + b[r].x), 0.5f * (a[r].x - b[r].x));
        } else if (k == H / 2) {
#pragma unroll
            for (int r = 0; r < RY; ++r) sc[dzi<H>(q + STY * r, ra)] = make_float2(a[r].x, -a[r].y);
        } else {
            const float2 w = tw[k];
#pragma unroll
            for (int r = 0; r < RY; ++r) {
                c2r_pair(a[r], b[r], w);
                sc[dzi<H>(q + STY * r, ra)] = a[r];
                sc[dzi<H>(q + STY * r, rb)] = b[r];
            }
        }
    }
    ctx.sync();
    ctx.stamp(sid + 1);
    // inverse z stages, lanes over lines
    if constexpr (Plan<H>::NS == 2) {
        constexpr int R = StageInfo<H, 1>::R, Q = H / R;
        static_assert(StageInfo<H, 1>::ST == 1, "last z stage");
        for (int t = ctx.tid; t < NCH * N * Q; t += ctx.nthr) {
            const int ch = t / (N * Q), tt = t - ch * (N * Q);
            const int q = tt / N, l = tt - q * N;
            float2* sc = s + ch * DENSE;
            float2 v[R];
#pragma unroll
            for (int r = 0; r < R; ++r) v[r] = sc[dzi<H>(l, q * R + r)];
            dft_inv<R>(v);
#pragma unroll
            for (int r = 0; r < R; ++r) sc[dzi<H>(l, q * R + r)] = v[r];
        }
        ctx.sync();
    }
    ctx.stamp(sid + 2);
    constexpr int R0 = StageInfo<H, 0>::R, ST0 = StageInfo<H, 0>::ST;
    for (int t = ctx.tid; t < NCH * N * ST0; t += ctx.nthr) {
        const int ch = t / (N * ST0), tt = t - ch * (N * ST0);
        int l, q;
        zline_task<ST0>(tt, l, q);
        float2* sc = s + ch * DENSE;
        float2 v[R0];
#pragma unroll
        for (int r = 0; r < R0; ++r) v[r] = sc[dzi<H>(l, q + ST0 * r)];
        bfly_inv<H, 0, N>(v, q, tw);
#pragma unroll
        for (int r = 0; r < R0; ++r) sc[dzi<H>(l, q + ST0 * r)] = v[r];
    }
    ctx.sync();
}
// real value (line l, z) of a dense plane after plane_inv_yz
template <int N> SAP_HD float dense_at(const float2* sc, int l, int z) {
    const float2 v = sc[dzi<N / 2>(l, z >> 1)];
    return (z & 1) ? v.y : v.x;
}

// =====================================================================================================================
// forward phases
// =====================================================================================================================
// F1a: histogram of this CTA's chunk of the points over the N x-slabs
template <int N, class Ctx>
SAP_HD void fwd_hist(Ctx& ctx, const FusedParams& p, FusedSmem<N>& sm, int cta, int ncta) {
    const int chunk = (p.P + ncta - 1) / ncta;
    const int i0 = cta * chunk, i1 = (i0 + chunk < p.P) ? i0 + chunk : p.P;
    int* h = sm.scr;
    for (int item = 0; item < p.B; ++item) {
        for (int b = ctx.tid; b < N; b += ctx.nthr) h[b] = 0;
        ctx.sync();
        for (int i = i0 + ctx.tid; i < i1; i += ctx.nthr) ctx.atomic_inc(h + slab_of<N>(p.pts + ((size_t)item * p.P + i) * 3));
        ctx.sync();
        int* gh = p.hist + ((size_t)item * ncta + cta) * N;
        for (int b = ctx.tid; b < N; b += ctx.nthr) gh[b] = h[b];
        ctx.sync();
    }
}
// F1b: slab offsets (every CTA keeps the whole table in its shared memory; CTA 0 also writes it to the handle for
// the backward) and scatter of this CTA's chunk into the sorted arrays
template <int N, class Ctx>
SAP_HD void fwd_scatter(Ctx& ctx, const FusedParams& p, FusedSmem<N>& sm, int cta, int ncta) {
    constexpr int NSL = FusedCfg<N>::NT / N;
    const int chunk = (p.P + ncta - 1) / ncta;
    const int i0 = cta * chunk, i1 = (i0 + chunk < p.P) ? i0 + chunk : p.P;
    int* part_tot = sm.scr;                         // [4 NSL][N]
    int* part_off = sm.scr + 4 * FusedCfg<N>::NT;   // [4 NSL][N]
    int* cursor = sm.scr + 8 * FusedCfg<N>::NT;     // [N]
    for (int item = 0; item < p.B; ++item) {
        const int4* gh4 = reinterpret_cast<const int4*>(p.hist + (size_t)item * ncta * N);
        int* bs = sm.bins + item * (N + 1);
        // thread (slice sl, 4 slabs b4): sums the histograms of the CTAs of its slice, 4 independent 16-byte loads in flight
        constexpr int N4 = N / 4, NSL4 = FusedCfg<N>::NT / N4;
        const int per = (ncta + NSL4 - 1) / NSL4;
        int4* ptot4 = reinterpret_cast<int4*>(part_tot);   // [NSL4][N4]: slice sl of slab b at part_tot[sl * N + b]
        int4* poff4 = reinterpret_cast<int4*>(part_off);
        static_assert(NSL4 * N4 * 4 <= 4 * FusedCfg<N>::NT && NSL4 == 4 * NSL, "partial sums fit the scratch arrays");
        for (int t = ctx.tid; t < NSL4 * N4; t += ctx.nthr) {
            const int sl = t / N4, b4 = t - sl * N4;
            int4 tot = make_int4(0, 0, 0, 0), off = make_int4(0, 0, 0, 0);
            const int c1 = ((sl + 1) * per < ncta) ? (sl + 1) * per : ncta;
#pragma unroll 4
            for (int c = sl * per; c < c1; ++c) {
                const int4 v = ldi4(gh4 + (size_t)c * N4 + b4);
                tot.x += v.x; tot.y += v.y; tot.z += v.z; tot.w += v.w;
                if (c < cta) { off.x += v.x; off.y += v.y; off.z += v.z; off.w += v.w; }
            }
            ptot4[t] = tot;
            poff4[t] = off;
        }
        ctx.sync();
        for (int b = ctx.tid; b < N; b += ctx.nthr) {
            int tot = 0, off = 0;
            for (int sl = 0; sl < 4 * NSL; ++sl) { tot += part_tot[sl * N + b]; off += part_off[sl * N + b]; }
            part_tot[b] = tot;   // slice 0 of the array: only read by this thread above
            cursor[b] = off;
        }
        ctx.sync();
        {   // exclusive scan of the N slab totals: log2(N) ping-pong steps (a serial loop in one thread cost 2-3 us)
            int* a = part_tot;             // inclusive sums so far: slice 0 of part_tot ...
            int* b2 = part_tot + N;        // ... and slice 1 (both free now)
            for (int d = 1; d < N; d <<= 1) {
                for (int b = ctx.tid; b < N; b += ctx.nthr) b2[b] = a[b] + (b >= d ? a[b - d] : 0);
                ctx.sync();
                int* t = a; a = b2; b2 = t;
            }
            for (int b = ctx.tid; b < N; b += ctx.nthr) bs[b + 1] = a[b];
            if (ctx.tid == 0) bs[0] = 0;
        }
        ctx.sync();
        for (int b = ctx.tid; b < N; b += ctx.nthr) cursor[b] += bs[b];
        if (cta == 0) {
            int* gbs = p.bin_start + (size_t)item * (N + 1);
            for (int b = ctx.tid; b <= N; b += ctx.nthr) gbs[b] = bs[b];
        }
        ctx.sync();
        for (int i = i0 + ctx.tid; i < i1; i += ctx.nthr) {
            const float* c = p.pts + ((size_t)item * p.P + i) * 3;
            const float* n = p.nrm + ((size_t)item * p.P + i) * 3;
            const int pos = ctx.atomic_inc(cursor + slab_of<N>(c));
            p.spts[(size_t)item * p.P + pos] = make_float4(c[0], c[1], c[2], bits_i2f(i));
            p.snrm[(size_t)item * p.P + pos] = make_float4(n[0], n[1], n[2], 0.f);
        }
        ctx.sync();
    }
}

// F1 + F2zy: rasterise the three channels of x-plane `tile` (owner computes) and transform along z and y
template <int N, class Ctx>
SAP_HD void fwd_splat_zy(Ctx& ctx, const FusedParams& p, FusedSmem<N>& sm, int tile) {
    constexpr int H = N / 2, PITCH = N + 1, M = N - 1;
    constexpr size_t PAD = FusedCfg<N>::PAD;
    const int item = tile / N, x = tile - item * N;
    float2* s = sm.big;
    {
        float4* s4 = reinterpret_cast<float4*>(s);
        for (int i = ctx.tid; i < (int)((3 * PAD + 1) / 2); i += ctx.nthr) s4[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
    ctx.sync();
    ctx.stamp(5);
    const int* bs = sm.bins + item * (N + 1);
    const float4* sp = p.spts + (size_t)item * p.P;
    const float4* sn = p.snrm + (size_t)item * p.P;
    // fixed-point scale of this plane: bound = sum_i max_c |n_ic| over the points that touch it
    float bound = 0.f;
    for (int k = 0; k < 2; ++k) {
        const int bin = (x - k) & M;
        for (int i = bs[bin] + ctx.tid; i < bs[bin + 1]; i += ctx.nthr) {
            const float4 n = ld4(sn + i);
            bound += fmaxf(fmaxf(fabsf(n.x), fabsf(n.y)), fabsf(n.z));
        }
    }
    const FixScale fs = fix_scale(ctx.block_sum_all(bound, reinterpret_cast<float*>(sm.scr)));
    int* si = reinterpret_cast<int*>(s);
    for (int k = 0; k < 2; ++k) {
        const int bin = (x - k) & M;
        for (int i = bs[bin] + ctx.tid; i < bs[bin + 1]; i += ctx.nthr) {
            const float4 c = ld4(sp + i), n = ld4(sn + i);
            const Foot f = foot_of<N>(c, k);
            const float nx = n.x * fs.S, ny = n.y * fs.S, nz = n.z * fs.S;
#pragma unroll
            for (int dy = 0; dy < 2; ++dy) {
                const int ly = (f.jy + dy) & M;
                const float wxy = f.wx * (dy ? f.fy : 1.f - f.fy);
#pragma unroll
                for (int dz = 0; dz < 2; ++dz) {
                    const int z = (f.jz + dz) & M;
                    const float w = wxy * (dz ? f.fz : 1.f - f.fz);
                    int* cell = si + ((size_t)(z >> 1) * PITCH + ly) * 2 + (z & 1);
                    ctx.atomic_add(cell, fix_round(w * nx));
                    ctx.atomic_add(cell + 2 * PAD, fix_round(w * ny));
                    ctx.atomic_add(cell + 4 * PAD, fix_round(w * nz));
                }
            }
        }
    }
    ctx.sync();
    ctx.stamp(6);
    const size_t SPLANE = (size_t)N * N * H, QPLANE = (size_t)N * N;
    plane_fwd_zy<N, 3, PSRC_FIX>(ctx, s, nullptr, sm.tw, fs.invS, 0.f, 0.f, false, p.S3 + (size_t)item * 3 * SPLANE + (size_t)x * N * H,
                                 SPLANE, p.Q3 + (size_t)item * 3 * QPLANE + (size_t)x * N, QPLANE, 7);
}

// tile geometry of the x pass: which y slot / z slots the XW columns of tile T hold
template <int N> struct XTile {
    TileDesc d;
    int xswz;
    SAP_HD explicit XTile(int T) : d(tile_desc<N, FusedCfg<N>::XW>(0, T)), xswz(0) { xswz = d.nyq ? 0 : (d.other & 15); }
    SAP_HD void col_freq(const float4* ftab, int c, float4& ey, float4& ez) const {
        ey = ftab[d.nyq ? d.other + c : d.other];
        ez = ftab[N + (d.nyq ? N / 2 : d.pz0 + (c ^ xswz))];
    }
};
template <int N> constexpr int x_tiles() { return N * ((N / 2) / FusedCfg<N>::XW) + N / FusedCfg<N>::XW; }

// F2x + F3 + F4x: x forward of (v~_x, h_y v~_y + h_z v~_z), spectral multiplier, x inverse (3 spectra -> 1).
// chi~ = i f (h_x v~_x + h_y v~_y + h_z v~_z), f = cs g / |u|^2 (Eq.3 / Eq.16; R3, R4, R6).
template <int N, class Ctx>
SAP_HD void fwd_x_solve(Ctx& ctx, const FusedParams& p, const FusedSmem<N>& sm, float2* b0, float2* b1, int item, int T) {
    constexpr int H = N / 2, W = FusedCfg<N>::XW;
    constexpr int R0 = StageInfo<N, 0>::R, ST = StageInfo<N, 0>::ST, RL = StageInfo<N, 1>::R;
    const size_t SPLANE = (size_t)N * N * H, QPLANE = (size_t)N * N;
    const XTile<N> xt(T);
    const unsigned sn = (unsigned)xt.d.sn, sc = (unsigned)xt.d.sc;
    const float2* src0 = (xt.d.nyq ? p.Q3 + (size_t)item * 3 * QPLANE : p.S3 + (size_t)item * 3 * SPLANE) + xt.d.base;
    const size_t cstride = xt.d.nyq ? QPLANE : SPLANE;
    float2* out = (xt.d.nyq ? p.Q1 + (size_t)item * QPLANE : p.S1 + (size_t)item * SPLANE) + xt.d.base;
    for (int t = ctx.tid; t < ST * W; t += ctx.nthr) {  // forward stage 0: HBM -> registers -> smem
        const int q = t / W, c = t - q * W;
        float4 ey, ez;
        xt.col_freq(p.ftab, c, ey, ez);
        const float4* tr = sm.tabF + q * R0;
        float2 v[R0], u[R0];
#pragma unroll
        for (int r = 0; r < R0; ++r) {
            const size_t off = (size_t)((unsigned)(q + r * ST) * sn + (unsigned)c * sc);
            v[r] = ld2(src0 + off);
            u[r] = caxpy(ez.x, ld2(src0 + 2 * cstride + off), cscale(ey.x, ld2(src0 + cstride + off)));
        }
        dft_fwd<R0>(v);
        dft_fwd<R0>(u);
#pragma unroll
        for (int r = 1; r < R0; ++r) { v[r] = fcmul4(v[r], tr[r]); u[r] = fcmul4(u[r], tr[r]); }
#pragma unroll
        for (int r = 0; r < R0; ++r) { b0[(q + r * ST) * W + c] = v[r]; b1[(q + r * ST) * W + c] = u[r]; }
    }
    ctx.sync();
    ctx.stamp(13);
    for (int t = ctx.tid; t < (N / RL) * W; t += ctx.nthr) {  // last forward stage, multiplier, first inverse stage
        const int blk = t / W, c = t - blk * W, e0 = blk * RL * W + c;
        float4 ey, ez;
        xt.col_freq(p.ftab, c, ey, ez);
        const MultCol mc = mult_col(ey, ez, p.cs);
        float2 v[RL], a[RL];
#pragma unroll
        for (int r = 0; r < RL; ++r) v[r] = b0[e0 + r * W];
        dft_fwd<RL>(v);
#pragma unroll
        for (int r = 0; r < RL; ++r) a[r] = cscale(sm.fx[blk * RL + r].x, v[r]);
#pragma unroll
        for (int r = 0; r < RL; ++r) v[r] = b1[e0 + r * W];
        dft_fwd<RL>(v);
#pragma unroll
        for (int r = 0; r < RL; ++r) {
            const float f = mult_fc(sm.fx[blk * RL + r], mc);
            const float2 dv = cscale(f, cadd(a[r], v[r]));
            a[r] = make_float2(-dv.y, dv.x);  // chi~ = i (div)
        }
        dft_inv<RL>(a);
#pragma unroll
        for (int r = 0; r < RL; ++r) b1[e0 + r * W] = a[r];
    }
    ctx.sync();
    ctx.stamp(14);
    for (int t = ctx.tid; t < ST * W; t += ctx.nthr) {  // inverse stage 0: smem -> registers -> HBM
        const int q = t / W, c = t - q * W;
        const float4* tr = sm.tabI + q * R0;
        float2 v[R0];
#pragma unroll
        for (int r = 0; r < R0; ++r) v[r] = b1[(q + r * ST) * W + c];
#pragma unroll
        for (int r = 1; r < R0; ++r) v[r] = fcmul4(v[r], tr[r]);
        dft_inv<R0>(v);
#pragma unroll
        for (int r = 0; r < R0; ++r) out[(size_t)((unsigned)(q + r * ST) * sn + (unsigned)c * sc)] = v[r];
    }
    ctx.sync();
}

// F4yz + F5a: inverse y/z of x-plane `tile` into shared memory; partial sum of chi' at the points (Eq.4, R11)
template <int N, class Ctx>
SAP_HD void fwd_inv_mean(Ctx& ctx, const FusedParams& p, FusedSmem<N>& sm, int tile) {
    constexpr int H = N / 2, M = N - 1;
    const int item = tile / N, x = tile - item * N;
    float2* s = sm.big;
    {
        const float4* g4 = reinterpret_cast<const float4*>(p.S1 + (size_t)tile * N * H);
        float4* s4 = reinterpret_cast<float4*>(s);
#pragma unroll 8
        for (int i = ctx.tid; i < N * H / 2; i += ctx.nthr) s4[i] = ld4(g4 + i);
        const float2* q2 = p.Q1 + (size_t)tile * N;
        for (int i = ctx.tid; i < N; i += ctx.nthr) s[N * H + i] = ld2(q2 + i);
    }
    ctx.sync();
    ctx.stamp(17);
    plane_inv_yz<N, 1, false>(ctx, s, sm.tw, sm.fx, sm.fz, 22);
    ctx.stamp(25);
    const int* bs = sm.bins + item * (N + 1);
    const float4* sp = p.spts + (size_t)item * p.P;
    float sum = 0.f;
    for (int k = 0; k < 2; ++k) {
        const int bin = (x - k) & M;
        for (int i = bs[bin] + ctx.tid; i < bs[bin + 1]; i += ctx.nthr) {
            const Foot f = foot_of<N>(ld4(sp + i), k);
            float a = 0.f;
#pragma unroll
            for (int dy = 0; dy < 2; ++dy) {
                const int ly = (f.jy + dy) & M;
                const float wy = dy ? f.fy : 1.f - f.fy;
#pragma unroll
                for (int dz = 0; dz < 2; ++dz) a += wy * (dz ? f.fz : 1.f - f.fz) * dense_at<N>(s, ly, (f.jz + dz) & M);
            }
            sum += f.wx * a;
        }
    }
    const float tot = ctx.block_sum(sum, reinterpret_cast<float*>(sm.scr));
    if (ctx.tid == 0) {
        ctx.gatomic_add(p.acc + 2 * item, (double)tot);
        if (x == 0) p.stats[item * 4 + 3] = s[0].x;  // chi'[0,0,0]
    }
}
// F5b (after the grid barrier): mu, a, s; chi = s (chi' - mu) written from shared memory
template <int N, class Ctx>
SAP_HD void fwd_scale_store(Ctx& ctx, const FusedParams& p, FusedSmem<N>& sm, int tile) {
    constexpr int H = N / 2;
    const int item = tile / N, x = tile - item * N;
    const double mu_d = ctx.gload(p.acc + 2 * item) / (double)p.P;
    const double a_d = (double)ctx.gload(p.stats + item * 4 + 3) - mu_d;
    const double s_d = 0.5 / fabs(a_d);  // m = 0.5; reading R5
    const float mu = (float)mu_d, sc = (float)s_d;
    const float2* s = sm.big;
    float2* out = reinterpret_cast<float2*>(p.chi) + (size_t)tile * N * H;
    {
        // 16-byte stores: the complex pair (m, m+1), m even, of line l sits in the 16-byte word (m ^ k) >> 1, k = l & 15,
        // with its halves swapped when k is odd
        const float4* s4 = reinterpret_cast<const float4*>(s);
        float4* out4 = reinterpret_cast<float4*>(out);
#pragma unroll 4
        for (int t = ctx.tid; t < N * H / 2; t += ctx.nthr) {
            const int l = t / (H / 2), m2 = t - l * (H / 2), k = l & 15;
            const float4 v = s4[l * (H / 2) + (m2 ^ (k >> 1))];
            const float4 w = (k & 1) ? make_float4(v.z, v.w, v.x, v.y) : v;
            out4[t] = make_float4(sc * (w.x - mu), sc * (w.y - mu), sc * (w.z - mu), sc * (w.w - mu));
        }
    }
    if (x == 0 && ctx.tid == 0) {
        p.stats[item * 4 + 0] = mu;
        p.stats[item * 4 + 1] = (float)a_d;
        p.stats[item * 4 + 2] = sc;
    }
}

// =====================================================================================================================
// backward phases
// =====================================================================================================================
// B1a: chi and G planes of x-plane `tile` into shared memory (chi natural, G in the padded layout of the forward
// transform); partial sums S0 = sum G, S1 = sum G chi
template <int N, class Ctx>
SAP_HD void bwd_load_reduce(Ctx& ctx, const FusedParams& p, FusedSmem<N>& sm, int tile) {
    constexpr int H = N / 2, PITCH = N + 1;
    constexpr size_t PAD = FusedCfg<N>::PAD;
    const int item = tile / N;
    float2* gpl = sm.big;
    float2* cpl = sm.big + FusedCfg<N>::PADA;
    int2* wpl = reinterpret_cast<int2*>(sm.big + FusedCfg<N>::PADA + (size_t)N * H);   // fixed-point density W, padded layout
    for (int i = ctx.tid; i < (int)PAD; i += ctx.nthr) wpl[i] = make_int2(0, 0);
    const float2* g2 = reinterpret_cast<const float2*>(p.G) + (size_t)tile * N * H;
    const float2* c2 = reinterpret_cast<const float2*>(p.chi) + (size_t)tile * N * H;
    float s0 = 0.f, s1 = 0.f;
    {
        const float4* g4 = reinterpret_cast<const float4*>(g2);
        const float4* c4 = reinterpret_cast<const float4*>(c2);
        float4* cpl4 = reinterpret_cast<float4*>(cpl);
#pragma unroll 8
        for (int t = ctx.tid; t < N * H / 2; t += ctx.nthr) {
            const int l = t / (H / 2), m = 2 * (t - l * (H / 2));
            const float4 g = ld4(g4 + t), c = ld4(c4 + t);
            s0 += (g.x + g.y) + (g.z + g.w);
            s1 += (g.x * c.x + g.y * c.y) + (g.z * c.z + g.w * c.w);
            gpl[m * PITCH + l] = make_float2(g.x, g.y);
            gpl[(m + 1) * PITCH + l] = make_float2(g.z, g.w);
            cpl4[t] = c;
        }
    }
    const float t0 = ctx.block_sum(s0, reinterpret_cast<float*>(sm.scr));
    const float t1 = ctx.block_sum(s1, reinterpret_cast<float*>(sm.scr));
    if (ctx.tid == 0) {
        ctx.gatomic_add(p.acc + 2 * item, (double)t0);
        ctx.gatomic_add(p.acc + 2 * item + 1, (double)t1);
    }
}
// the gradients are accumulated with atomics: clear them first (all CTAs, before the first barrier)
template <class Ctx> SAP_HD void bwd_zero_grads(Ctx& ctx, const FusedParams& p, int cta, int ncta) {
    const size_t n = (size_t)p.B * p.P * 3;
    for (size_t i = (size_t)cta * ctx.nthr + ctx.tid; i < n; i += (size_t)ncta * ctx.nthr) { p.gp[i] = 0.f; p.gn[i] = 0.f; }
}
// B1b + B2 + B3zy (after the barrier): beta; chi term of dL/dc; Gbar' assembled on the G plane; z + y forward
template <int N, class Ctx>
SAP_HD void bwd_gbar_zy(Ctx& ctx, const FusedParams& p, FusedSmem<N>& sm, int tile) {
    constexpr int H = N / 2, PITCH = N + 1, M = N - 1;
    constexpr size_t PAD = FusedCfg<N>::PAD;
    const int item = tile / N, x = tile - item * N;
    const double S0 = ctx.gload(p.acc + 2 * item), S1 = ctx.gload(p.acc + 2 * item + 1);
    const double a = (double)ctx.gload(p.stats + item * 4 + 1), sd = (double)ctx.gload(p.stats + item * 4 + 2);
    const double beta = S1 / a - sd * S0;
    const float gs = (float)sd, cw = (float)(beta / (double)p.P), c0 = (float)(S1 / a), cchi = (float)(beta / ((double)p.P * sd));
    if (x == 0 && ctx.tid == 0) {
        p.bw[item * 4 + 0] = gs; p.bw[item * 4 + 1] = cw; p.bw[item * 4 + 2] = c0; p.bw[item * 4 + 3] = cchi;
    }
    float2* gpl = sm.big;
    const float* cpl = reinterpret_cast<const float*>(sm.big + FusedCfg<N>::PADA);
    int2* wpl = reinterpret_cast<int2*>(sm.big + FusedCfg<N>::PADA + (size_t)N * H);
    int* wi = reinterpret_cast<int*>(wpl);
    const int* bs = p.bin_start + (size_t)item * (N + 1);
    const float4* sp = p.spts + (size_t)item * p.P;
    const int n_x = (bs[x + 1] - bs[x]) + (bs[((x - 1) & M) + 1] - bs[(x - 1) & M]);
    const FixScale fs = fix_scale((float)n_x);   // every weight is <= 1: no cell of W can exceed the number of points
    for (int k = 0; k < 2; ++k) {
        const int bin = (x - k) & M;
        const int lo = bs[bin], hi = bs[bin + 1];
        for (int i = lo + ctx.tid; i < hi; i += ctx.nthr) {
            const float4 c = sp[i];
            const Foot f = foot_of<N>(c, k);
            float g0 = 0.f, g1 = 0.f, g2 = 0.f;
#pragma unroll
            for (int dy = 0; dy < 2; ++dy) {
                const int ly = (f.jy + dy) & M;
                const float wy = dy ? f.fy : 1.f - f.fy;
#pragma unroll
                for (int dz = 0; dz < 2; ++dz) {
                    const int z = (f.jz + dz) & M;
                    const float wz = dz ? f.fz : 1.f - f.fz;
                    ctx.atomic_add(wi + ((size_t)(z >> 1) * PITCH + ly) * 2 + (z & 1), fix_round(f.wx * wy * wz * fs.S));
                    const float val = cchi * cpl[ly * N + z];
                    g0 += f.sx * val * (wy * wz);
                    g1 += (dy ? val : -val) * (f.wx * wz);
                    g2 += (dz ? val : -val) * (f.wx * wy);
                }
            }
            float* o = p.gp + ((size_t)item * p.P + bits_f2i(c.w)) * 3;
            ctx.gatomic_add(o, (float)N * g0);
            ctx.gatomic_add(o + 1, (float)N * g1);
            ctx.gatomic_add(o + 2, (float)N * g2);
        }
    }
    ctx.sync();
    ctx.stamp(36);
    plane_fwd_zy<N, 1, PSRC_GBAR>(ctx, gpl, wpl, sm.tw, gs, cw * fs.invS, c0, x == 0, p.S1 + (size_t)tile * N * H, 0,
                                  p.Q1 + (size_t)tile * N, 0, 37);
}

// B3x + B4 + B5x: x forward of Gbar'~, A = -i f Gbar'~, two x inverses: plane 0 = IFFT_x(h_x A), plane 1 = B = IFFT_x(A)
// (vbar_y and vbar_z are made from B by the next phase: h_y and h_z commute with the x transform)
template <int N, class Ctx>
SAP_HD void bwd_x_adj(Ctx& ctx, const FusedParams& p, const FusedSmem<N>& sm, float2* b0, float2* b1, int item, int T) {
    constexpr int H = N / 2, W = FusedCfg<N>::XW;
    constexpr int R0 = StageInfo<N, 0>::R, ST = StageInfo<N, 0>::ST, RL = StageInfo<N, 1>::R;
    const size_t SPLANE = (size_t)N * N * H, QPLANE = (size_t)N * N;
    const XTile<N> xt(T);
    const unsigned sn = (unsigned)xt.d.sn, sc = (unsigned)xt.d.sc;
    const float2* src = (xt.d.nyq ? p.Q1 + (size_t)item * QPLANE : p.S1 + (size_t)item * SPLANE) + xt.d.base;
    float2* out0 = (xt.d.nyq ? p.Q3 + (size_t)item * 3 * QPLANE : p.S3 + (size_t)item * 3 * SPLANE) + xt.d.base;
    float2* out1 = out0 + (xt.d.nyq ? QPLANE : SPLANE);
    for (int t = ctx.tid; t < ST * W; t += ctx.nthr) {
        const int q = t / W, c = t - q * W;
        const float4* tr = sm.tabF + q * R0;
        float2 v[R0];
#pragma unroll
        for (int r = 0; r < R0; ++r) v[r] = ld2(src + (size_t)((unsigned)(q + r * ST) * sn + (unsigned)c * sc));
        dft_fwd<R0>(v);
#pragma unroll
        for (int r = 1; r < R0; ++r) v[r] = fcmul4(v[r], tr[r]);
#pragma unroll
        for (int r = 0; r < R0; ++r) b0[(q + r * ST) * W + c] = v[r];
    }
    ctx.sync();
    ctx.stamp(43);
    for (int t = ctx.tid; t < (N / RL) * W; t += ctx.nthr) {
        const int blk = t / W, c = t - blk * W, e0 = blk * RL * W + c;
        float4 ey, ez;
        xt.col_freq(p.ftab, c, ey, ez);
        const MultCol mc = mult_col(ey, ez, p.cs);
        float2 v[RL], a[RL];
#pragma unroll
        for (int r = 0; r < RL; ++r) v[r] = b0[e0 + r * W];
        dft_fwd<RL>(v);
#pragma unroll
        for (int r = 0; r < RL; ++r) {
            const float f = mult_fc(sm.fx[blk * RL + r], mc);
            a[r] = make_float2(f * v[r].y, -f * v[r].x);          // A = -i f Gbar'~
            v[r] = cscale(sm.fx[blk * RL + r].x, a[r]);            // h_x A
        }
        dft_inv<RL>(v);
        dft_inv<RL>(a);
#pragma unroll
        for (int r = 0; r < RL; ++r) { b0[e0 + r * W] = v[r]; b1[e0 + r * W] = a[r]; }
    }
    ctx.sync();
    ctx.stamp(44);
    for (int t = ctx.tid; t < 2 * ST * W; t += ctx.nthr) {
        const int pl = t / (ST * W), tt = t - pl * (ST * W);
        const int q = tt / W, c = tt - q * W;
        const float4* tr = sm.tabI + q * R0;
        const float2* b = pl ? b1 : b0;
        float2* out = pl ? out1 : out0;
        float2 v[R0];
#pragma unroll
        for (int r = 0; r < R0; ++r) v[r] = b[(q + r * ST) * W + c];
#pragma unroll
        for (int r = 1; r < R0; ++r) v[r] = fcmul4(v[r], tr[r]);
        dft_inv<R0>(v);
#pragma unroll
        for (int r = 0; r < R0; ++r) out[(size_t)((unsigned)(q + r * ST) * sn + (unsigned)c * sc)] = v[r];
    }
    ctx.sync();
}

// B5yz + B6: inverse y/z of the three channels of x-plane `tile` in shared memory, then the owner-computes gather:
//   dL/dn_i += sum_corners w vbar[corner],  dL/dc_i[a] += N sum_corners (dw/dc_a)/N (n_i . vbar[corner])
// restricted to the corners on this plane (the chi term of dL/dc was added by bwd_gbar_zy).
template <int N, class Ctx>
SAP_HD void bwd_inv_gather(Ctx& ctx, const FusedParams& p, FusedSmem<N>& sm, int tile) {
    constexpr int H = N / 2, M = N - 1;
    constexpr size_t DENSE = FusedCfg<N>::DENSE;
    const size_t SPLANE = (size_t)N * N * H, QPLANE = (size_t)N * N;
    const int item = tile / N, x = tile - item * N;
    float2* s = sm.big;
    {
        const float4* g0 = reinterpret_cast<const float4*>(p.S3 + (size_t)item * 3 * SPLANE + (size_t)x * N * H);
        const float4* g1 = g0 + SPLANE / 2;
        float4* d0 = reinterpret_cast<float4*>(s);
        float4* d1 = reinterpret_cast<float4*>(s + DENSE);
        float4* d2 = reinterpret_cast<float4*>(s + 2 * DENSE);
#pragma unroll 8
        for (int i = ctx.tid; i < N * H / 2; i += ctx.nthr) {
            d0[i] = ld4(g0 + i);
            const float4 b = ld4(g1 + i);
            d1[i] = b;
            d2[i] = b;
        }
        const float2* q0 = p.Q3 + (size_t)item * 3 * QPLANE + (size_t)x * N;
        for (int i = ctx.tid; i < N; i += ctx.nthr) {
            s[N * H + i] = ld2(q0 + i);
            const float2 b = ld2(q0 + QPLANE + i);
            s[DENSE + N * H + i] = b;
            s[2 * DENSE + N * H + i] = b;
        }
    }
    ctx.sync();
    ctx.stamp(47);
    plane_inv_yz<N, 3, true>(ctx, s, sm.tw, sm.fx, sm.fz, 48);
    ctx.stamp(51);
    const int* bs = p.bin_start + (size_t)item * (N + 1);
    const float4* sp = p.spts + (size_t)item * p.P;
    const float4* sn = p.snrm + (size_t)item * p.P;
    for (int k = 0; k < 2; ++k) {
        const int bin = (x - k) & M;
        const int lo = bs[bin], hi = bs[bin + 1];
        for (int i = lo + ctx.tid; i < hi; i += ctx.nthr) {
            const float4 c = sp[i], n = sn[i];
            const Foot f = foot_of<N>(c, k);
            float n0 = 0.f, n1 = 0.f, n2 = 0.f, g0 = 0.f, g1 = 0.f, g2 = 0.f;
#pragma unroll
            for (int dy = 0; dy < 2; ++dy) {
                const int ly = (f.jy + dy) & M;
                const float wy = dy ? f.fy : 1.f - f.fy;
#pragma unroll
                for (int dz = 0; dz < 2; ++dz) {
                    const int z = (f.jz + dz) & M;
                    const float wz = dz ? f.fz : 1.f - f.fz;
                    const float a0 = dense_at<N>(s, ly, z), a1 = dense_at<N>(s + DENSE, ly, z), a2 = dense_at<N>(s + 2 * DENSE, ly, z);
                    const float w = f.wx * wy * wz;
                    n0 += w * a0; n1 += w * a1; n2 += w * a2;
                    const float val = n.x * a0 + n.y * a1 + n.z * a2;
                    g0 += f.sx * val * (wy * wz);
                    g1 += (dy ? val : -val) * (f.wx * wz);
                    g2 += (dz ? val : -val) * (f.wx * wy);
                }
            }
            const size_t o = ((size_t)item * p.P + bits_f2i(c.w)) * 3;
            ctx.gatomic_add(p.gn + o, n0);
            ctx.gatomic_add(p.gn + o + 1, n1);
            ctx.gatomic_add(p.gn + o + 2, n2);
            ctx.gatomic_add(p.gp + o, (float)N * g0);
            ctx.gatomic_add(p.gp + o + 1, (float)N * g1);
            ctx.gatomic_add(p.gp + o + 2, (float)N * g2);
        }
    }
}

}  // namespace sap

// =====================================================================================================================
// device side: contexts, grid barrier, the two kernels
// =====================================================================================================================
#ifdef __CUDACC__
namespace sap {

__device__ __forceinline__ float fused_warp_sum(float x) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
    return x;
}
template <int NTHR> struct FusedCtaCtx {
    int tid;
    long long* stamps;   // CTA 0 only: clock64 at the marks of the phase bodies (profiling), else null
    static constexpr int nthr = NTHR;
    __device__ __forceinline__ void stamp(int i) const { if (stamps && tid == 0) stamps[i] = clock64(); }
    __device__ __forceinline__ void sync() const { __syncthreads(); }
    __device__ __forceinline__ void atomic_add(int* p, int v) const { atomicAdd(p, v); }
    __device__ __forceinline__ int atomic_inc(int* p) const { return atomicAdd(p, 1); }
    __device__ __forceinline__ void gatomic_add(float* p, float v) const { atomicAdd(p, v); }
    __device__ __forceinline__ void gatomic_add(double* p, double v) const { atomicAdd(p, v); }
    __device__ __forceinline__ double gload(const double* p) const { return __ldcg(p); }
    __device__ __forceinline__ float gload(const float* p) const { return __ldcg(p); }
    // block sum, valid in thread 0; scratch: 32 floats
    __device__ __forceinline__ float block_sum(float x, float* scratch) const {
        x = fused_warp_sum(x);
        __syncthreads();
        if ((tid & 31) == 0) scratch[tid >> 5] = x;
        __syncthreads();
        float r = 0.f;
        if (tid < 32) {
            r = (tid < NTHR / 32) ? scratch[tid] : 0.f;
            r = fused_warp_sum(r);
        }
        return r;
    }
    // block sum, valid in every thread; scratch: 33 floats
    __device__ __forceinline__ float block_sum_all(float x, float* scratch) const {
        const float r = block_sum(x, scratch);
        if (tid == 0) scratch[32] = r;
        __syncthreads();
        return scratch[32];
    }
};
template <int NTHR> struct FusedGroupCtx {
    int tid, group;
    long long* stamps;
    static constexpr int nthr = NTHR;
    __device__ __forceinline__ void stamp(int i) const { if (stamps && tid == 0) stamps[i] = clock64(); }
    __device__ __forceinline__ void sync() const { asm volatile("bar.sync %0, %1;" ::"r"(group + 1), "n"(NTHR) : "memory"); }
};

// Grid barrier k (k = 1, 2, ...) of a cooperative launch: every CTA arrives once on a monotonic counter and spins until
// k * #CTAs arrivals are visible.  The spin is bounded (2 s): a time-out sets a sticky flag the host reports instead
// of hanging the device.
__device__ __forceinline__ void fused_grid_barrier(const FusedParams& p, unsigned k) {
    __syncthreads();
    if (threadIdx.x == 0) {
        const unsigned target = k * gridDim.x;
        asm volatile("fence.acq_rel.gpu;" ::: "memory");
        atomicAdd(p.sync, 1u);
        unsigned seen;
        unsigned long long t0 = 0;
        int spins = 0;
        do {
            asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(seen) : "l"(p.sync) : "memory");
            if (seen < target && (++spins & 1023) == 0) {   // every ~1000 polls look at the clock: give up after 2 s
                unsigned long long t;
                asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t));
                if (t0 == 0) t0 = t;
                else if (t - t0 > 2000000000ull) { atomicExch(p.sync + 2, 1u); break; }
            }
        } while (seen < target);
        asm volatile("fence.acq_rel.gpu;" ::: "memory");
    }
    __syncthreads();
}
// last CTA out clears the counters and the accumulators for the next launch
__device__ __forceinline__ void fused_finish(const FusedParams& p) {
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        const unsigned t = atomicAdd(p.sync + 1, 1u);
        if (t == gridDim.x - 1) {
            for (int i = 0; i < 2 * p.B; ++i) p.acc[i] = 0.0;
            p.sync[0] = 0u;
            p.sync[1] = 0u;
            __threadfence();
        }
    }
}
__device__ __forceinline__ void fused_stamp(const FusedParams& p, int i) {
    if (p.stamps && blockIdx.x == 0 && threadIdx.x == 0) p.stamps[i] = clock64();
}

template <int N>
__global__ void __launch_bounds__(FusedCfg<N>::NT, 1) k_fused_fwd(const FusedParams p) {
    using C = FusedCfg<N>;
    extern __shared__ __align__(128) unsigned char fused_smem[];
    FusedSmem<N> sm(fused_smem);
    FusedCtaCtx<C::NT> ctx{(int)threadIdx.x, blockIdx.x == 0 ? p.stamps : nullptr};
    const int cta = blockIdx.x, ncta = gridDim.x;
    fused_tables<N>(ctx, p, sm);
    __syncthreads();
    pdl_wait();
    unsigned k = 0;
    fused_stamp(p, 0);
    fwd_hist<N>(ctx, p, sm, cta, ncta);
    fused_stamp(p, 1);
    fused_grid_barrier(p, ++k);
    fused_stamp(p, 2);
    fwd_scatter<N>(ctx, p, sm, cta, ncta);
    fused_stamp(p, 3);
    fused_grid_barrier(p, ++k);
    fused_stamp(p, 4);
    for (int tile = cta; tile < p.B * N; tile += ncta) fwd_splat_zy<N>(ctx, p, sm, tile);
    fused_grid_barrier(p, ++k);
    fused_stamp(p, 12);
    {
        FusedGroupCtx<C::XNTC> g{(int)threadIdx.x % C::XNTC, (int)threadIdx.x / C::XNTC, (blockIdx.x == 0 && threadIdx.x < C::XNTC) ? p.stamps : nullptr};
        float2* b0 = sm.big + (size_t)g.group * 2 * C::XBUF;
        const int per = x_tiles<N>();
        for (int T = cta * C::XNG + g.group; T < p.B * per; T += ncta * C::XNG) fwd_x_solve<N>(g, p, sm, b0, b0 + C::XBUF, T / per, T % per);
    }
    fused_stamp(p, 15);
    fused_grid_barrier(p, ++k);
    fused_stamp(p, 16);
    const bool mine = cta < p.B * N;   // host guarantees B * N <= #CTAs: the plane waits in shared memory for mu
    if (mine) fwd_inv_mean<N>(ctx, p, sm, cta);
    fused_stamp(p, 26);
    fused_grid_barrier(p, ++k);
    fused_stamp(p, 27);
    if (mine) fwd_scale_store<N>(ctx, p, sm, cta);
    fused_stamp(p, 28);
    fused_finish(p);
}

template <int N>
__global__ void __launch_bounds__(FusedCfg<N>::NT, 1) k_fused_bwd(const FusedParams p) {
    using C = FusedCfg<N>;
    extern __shared__ __align__(128) unsigned char fused_smem[];
    FusedSmem<N> sm(fused_smem);
    FusedCtaCtx<C::NT> ctx{(int)threadIdx.x, blockIdx.x == 0 ? p.stamps : nullptr};
    const int cta = blockIdx.x, ncta = gridDim.x;
    fused_tables<N>(ctx, p, sm);
    __syncthreads();
    pdl_wait();
    unsigned k = 0;
    fused_stamp(p, 32);
    const bool mine = cta < p.B * N;
    if (mine) bwd_load_reduce<N>(ctx, p, sm, cta);
    bwd_zero_grads(ctx, p, cta, ncta);
    fused_stamp(p, 33);
    fused_grid_barrier(p, ++k);
    fused_stamp(p, 34);
    if (mine) bwd_gbar_zy<N>(ctx, p, sm, cta);
    fused_grid_barrier(p, ++k);
    fused_stamp(p, 42);
    {
        FusedGroupCtx<C::XNTC> g{(int)threadIdx.x % C::XNTC, (int)threadIdx.x / C::XNTC, (blockIdx.x == 0 && threadIdx.x < C::XNTC) ? p.stamps : nullptr};
        float2* b0 = sm.big + (size_t)g.group * 2 * C::XBUF;
        const int per = x_tiles<N>();
        for (int T = cta * C::XNG + g.group; T < p.B * per; T += ncta * C::XNG) bwd_x_adj<N>(g, p, sm, b0, b0 + C::XBUF, T / per, T % per);
    }
    fused_stamp(p, 45);
    fused_grid_barrier(p, ++k);
    fused_stamp(p, 46);
    for (int tile = cta; tile < p.B * N; tile += ncta) { bwd_inv_gather<N>(ctx, p, sm, tile); __syncthreads(); }
    fused_stamp(p, 52);
    fused_finish(p);
}

}  // namespace sap
#endif
