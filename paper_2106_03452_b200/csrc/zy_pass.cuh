// zy_pass.cuh -- forward z (+ y) pass, one tile per CTA: real lines -> half spectrum (F1+F2, and B2+B3 for N >= 256).
// (The inverse pass and the fused Gbar' pass are the persistent kernels of zline_pass.cuh.)
//
// One block owns NL z-lines (consecutive in memory, NL % 32 == 0).  With DO_Y (N <= 128) NL == N: the
// block owns a whole x-plane and transforms along z and y in ONE trip through shared memory.
// Shared-memory traffic is kept to ~6 passes per plane: the first z stage runs global -> registers ->
// smem, the r2c split is fused into the first y stage, and the last y stage runs smem -> registers ->
// global.
// smem: (H+1) rows (kz slots + Nyquist) x PITCH = NL+1 columns (lines); PITCH == 1 (mod 16).
#pragma once
#include <math.h>
#include "fft_core.cuh"

namespace sap {

// Input of the forward pass.  The real plane is never read from HBM: it is rasterised on the fly
// ("owner computes") from the points of the bins that can touch this block's lines.
//   SRC_SPLAT (F1+F2): v_ch = sum_i w n_i[ch]                      (Eq.10-11)
//   SRC_GBAR  (B2+B3): Gbar' = s G + (beta/P) W - (S1/a) delta_0,  W = sum_i w rasterised the same way
// Points are pre-sorted by bin key j0x * (N/NL) + j0y / NL (k_bin_* kernels); bin_start has NBINS+1 entries.
enum { SRC_SPLAT = 0, SRC_GBAR = 1 };
struct ZyFwdParams {
    const float4* spts;    // [batch][P] sorted points  {cx, cy, cz, index in the caller's order (int bits)}
    const float4* snrm;    // [batch][P] sorted normals {nx, ny, nz, -}
    const int* bin_start;  // [batch][NBINS + 1]
    int P;
    const float* G;        // GBAR: [batch][N^3] upstream gradient
    const float* bw;       // GBAR: [batch][4] = {s, beta/P, S1/a, -}
    float2* S;             // [planes][N*N*H]
    float2* Q;             // [planes][N*N]  ([x][y] when the plane is fused (N <= 128), transposed [y][x] otherwise)
    const float2* tw;      // exp(-2 pi i t / N), t < N
    int nch;               // planes per batch item (3 for SPLAT, 1 for GBAR)
    const unsigned* nmax;  // SPLAT: [batch] bit pattern of max_i max_c |n_ic| (k_bin_scatter), for the fixed-point scale
    const int* plane_act;  // SPLAT, N >= 256: [batch][N] activity of the x-planes (k_bin_scan), or nullptr.  The y pass
                           // neither loads nor transforms an inactive plane: its tiles of channel 2 are not written
    int* clear_cnt;        // SPLAT after k_bin_sort: the bin counts [clear_n] and the barrier word, cleared here for the next
    int clear_n;           // forward (every block of k_bin_sort is done with them when this kernel starts), or nullptr
    unsigned* clear_sync;
};

// Column swizzle of the main spectrum in HBM: the value of z slot pz of line (x, y) is stored in column
// pz ^ (y & 15).  Within a 16-column group the columns of 16 consecutive lines are then all different, so a tile
// of lines that a bulk copy drops DENSE into shared memory can be walked "lanes over lines" without bank
// conflicts.  An involution: the same function maps a stored column back to its slot.
SAP_HD int kz_swz(int pz, int y) { return pz ^ (y & 15); }

// ---- fixed-point rasterisation ---------------------------------------------------------------------------------------
// The trilinear splat accumulates into shared memory with NATIVE 32-bit integer atomics (a float atomicAdd on shared
// memory is a compare-and-swap loop, measured at ~400 cycles per add here: 12 of them per point were the straggler
// of the whole forward).  Each contribution w * n_c is rounded once to a multiple of the quantum 1/S; S is a power of
// two chosen per tile from bound = sum over the tile's points of max_c |n_ic|  >=  |any cell sum|, so that
// bound * S < 2^30: overflow is impossible, whatever the point distribution.  Integer addition is associative, so the
// rasterised field is bit-identical from run to run (the float atomics were not).  Error: <= quantum / 2 per
// contribution, quantum <= bound / 2^29 (for 650 unit normals on a plane: 1.2e-6, about 10 fp32 ulps of 1; the
// tolerance of the path is 1e-4 max|chi|).
SAP_HD float bits_u2f(unsigned u) {
#ifdef __CUDA_ARCH__
    return __uint_as_float(u);
#else
    union { unsigned u; float f; } v; v.u = u; return v.f;
#endif
}
struct FixScale { float S, invS; };
SAP_HD FixScale fix_scale(float bound) {
    FixScale f;
    if (!(bound > 0.f) || !(bound < 3.0e38f)) { f.S = 1.f; f.invS = 1.f; return f; }
    int e;
    (void)frexpf(bound, &e);          // bound = m 2^e, m in [0.5, 1)  =>  bound < 2^e
    int k = 30 - e;                   // S = 2^k: bound S < 2^30
    if (k > 120) k = 120;
    if (k < -120) k = -120;
    f.S = ldexpf(1.f, k);
    f.invS = ldexpf(1.f, -k);
    return f;
}
SAP_HD int fix_round(float v) {
#ifdef __CUDA_ARCH__
    return __float2int_rn(v);
#else
    return (int)lrintf(v);
#endif
}
template <int N, int NL> constexpr size_t zy_smem_bytes() { return ((size_t)(N / 2 + 1) * (NL + 1) + N) * sizeof(float2); }

// task t -> (line, q) for the global<->smem z stage: q (ST0 consecutive complex of one line) fastest,
// the 32/ST0 lines of a warp spaced ST0 apart so that (q + line) is distinct mod 16 per half-warp.
template <int ST0> SAP_HD void zline_task(int t, int& line, int& q) {
    constexpr int s = (ST0 > 16) ? 16 : ST0;  // ST0 <= 16 for every supported plan
    const int g = t >> 5, w = t & 31;
    q = w % s;
    const int i = w / s;
    line = i * s + (g % s) + 32 * (g / s);
}

// ---- forward ---------------------------------------------------------------------------------------
template <int N, int NL, bool DO_Y, int SRC, class Ctx>
SAP_HD void zy_fwd_body(Ctx& ctx, const ZyFwdParams& p, float2* smem, int bx, int by) {
    constexpr int H = N / 2;
    constexpr int PITCH = NL + 1;
    constexpr int R0 = StageInfo<H, 0>::R, ST0 = StageInfo<H, 0>::ST;
    static_assert(NL % 32 == 0 && ST0 <= 16, "line-group mapping");
    static_assert(!DO_Y || NL == N, "plane mode owns N lines");
    float2* s = smem;
    float2* tw = smem + (H + 1) * PITCH;
    const size_t V = (size_t)N * N * N;
    const size_t line0 = (size_t)bx * NL;  // global line index = x*N + y

    if (SRC == SRC_SPLAT && p.clear_cnt && bx == 0 && by == 0) {
        for (int i = ctx.tid; i < p.clear_n; i += ctx.nthr) p.clear_cnt[i] = 0;
        if (ctx.tid == 0) p.clear_sync[0] = 0u;
    }
    float2* So = p.S + (size_t)by * ((size_t)N * N * H) + line0 * H;
    float2* Qo = p.Q + (size_t)by * ((size_t)N * N) + line0;
    // A0: which bins can touch lines [line0, line0 + NL): x-slabs {x, x-1} x y-tiles {ty, ty-1}
    constexpr int NTY = N / NL, NBINS = N * NTY, M = N - 1;
    const int item = by / p.nch, ch = by - item * p.nch;
    const int x = (int)(line0 / N), y0 = (int)(line0 % N), ty = y0 / NL;
    const int* bs = p.bin_start + (size_t)item * (NBINS + 1);
    int b_lo[4], b_n[4], total = 0;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const int xb = (k & 1) ? ((x - 1) & M) : x;
        const int tb = (k & 2) ? ((ty + NTY - 1) % NTY) : ty;
        const bool use = (NTY > 1) || !(k & 2);
        const int bin = xb * NTY + tb;
        b_lo[k] = use ? bs[bin] : 0;
        b_n[k] = use ? bs[bin + 1] - b_lo[k] : 0;
        total += b_n[k];
    }
    if (SRC == SRC_SPLAT && total == 0) {  // nothing lands here: the spectrum of zeros is zeros (before any other work)
        // fused planes with the solve's plane masks on (plane_act set): the solve reads the rows of an inactive plane as zeros
        // whatever the spectrum holds there, nobody has to write them
        const bool skip_main = p.plane_act != nullptr;
        float4* So4 = reinterpret_cast<float4*>(So);
        if (!skip_main)
            for (int i = ctx.tid; i < NL * H / 2; i += ctx.nthr) So4[i] = make_float4(0.f, 0.f, 0.f, 0.f);
        if constexpr (DO_Y) {
            for (int l = ctx.tid; l < NL; l += ctx.nthr) Qo[l] = make_float2(0.f, 0.f);
        } else {
            float2* Qt = p.Q + (size_t)by * ((size_t)N * N);
            for (int l = ctx.tid; l < NL; l += ctx.nthr) Qt[(size_t)(y0 + l) * N + x] = make_float2(0.f, 0.f);
        }
        return;
    }
    // A1: zero the plane, rasterise the points into it, z = 2m + parity.  The plane holds 32-bit FIXED-POINT sums while it
    // is rasterised (native integer shared-memory atomics; a float atomicAdd on shared memory is a compare-and-swap loop):
    // scale 2^k with (number of points that can touch the tile) x (largest normal component of the item) x 2^k < 2^30.
    for (int i = ctx.tid; i < N; i += ctx.nthr) tw[i] = p.tw[i];
    {
        float4* s4 = reinterpret_cast<float4*>(s);
        for (int i = ctx.tid; i < (H * PITCH + 1) / 2; i += ctx.nthr) s4[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
    const float amax = (SRC == SRC_SPLAT) ? bits_u2f(p.nmax[item]) : 1.f;
    const FixScale fs = fix_scale((float)total * amax);
    ctx.sync();
    {
        int* si = reinterpret_cast<int*>(s);
        const float4* sp = p.spts + (size_t)item * p.P;
        const float4* sn = p.snrm + (size_t)item * p.P;
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            for (int i = b_lo[k] + ctx.tid; i < b_lo[k] + b_n[k]; i += ctx.nthr) {
                const float4 c = sp[i];
                float val = fs.S;
                if (SRC == SRC_SPLAT) {
                    const float4 n = sn[i];
                    val *= (ch == 0) ? n.x : (ch == 1) ? n.y : n.z;
                }
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
                        for (int dz = 0; dz < 2; ++dz) {
                            const int z = (jz + dz) & M;
                            ctx.atomic_add(si + ((z >> 1) * PITCH + ly) * 2 + (z & 1), fix_round(wxy * (dz ? fz : 1.f - fz)));
                        }
                    }
                }
            }
        }
    }
    ctx.sync();
    // A2: z stage 0 in place (GBAR: combined with G from HBM on the way)
    {
        const float2* g2 = nullptr;
        float cs_ = 0.f, cw = 0.f, c0 = 0.f;
        if (SRC == SRC_GBAR) {
            g2 = reinterpret_cast<const float2*>(p.G + (size_t)item * V) + line0 * H;
            cs_ = p.bw[item * 4 + 0]; cw = p.bw[item * 4 + 1]; c0 = p.bw[item * 4 + 2];
        }
        for (int t = ctx.tid; t < NL * ST0; t += ctx.nthr) {
            int l, q;
            zline_task<ST0>(t, l, q);
            float2 v[R0];
#pragma unroll
            for (int r = 0; r < R0; ++r) {
                const int2 iv = reinterpret_cast<const int2*>(s)[(q + ST0 * r) * PITCH + l];   // fixed-point sums
                float2 xv = cscale(fs.invS, make_float2((float)iv.x, (float)iv.y));
                if (SRC == SRC_GBAR) {
                    const int e = l * H + q + ST0 * r;
                    const float2 g = g2[e];
                    xv = caxpy(cs_, g, cscale(cw, xv));
                    if (line0 == 0 && e == 0) xv.x -= c0;
                }
                v[r] = xv;
            }
            bfly_fwd<H, 0, N>(v, q, tw);
#pragma unroll
            for (int r = 0; r < R0; ++r) s[(q + ST0 * r) * PITCH + l] = v[r];
        }
        ctx.sync();
    }
    // B: remaining z stages in shared memory, one line per lane
    static_assert(Plan<H>::NS <= 2, "z plans have at most two stages");
    // (the fused variant holds a block pair = 2 R1 complex values per thread: worth it where the kernel has the
    // registers, i.e. at 3 CTAs per SM (N = 512); at N = 256 the kernel runs 4 CTAs per SM on 64 registers)
    constexpr bool FUSE_SPLIT = !DO_Y && N >= 512;   // at 256 it spills at 4 CTAs/SM and is no faster at 3 (r2: 67.6 vs 66.0 us)
    if constexpr (Plan<H>::NS > 1 && !FUSE_SPLIT) {
        fft_stage<H, 1, false, N, true>(s, PITCH, 1, NL, tw, ctx.tid, ctx.nthr);
        ctx.sync();
    }
    if constexpr (!DO_Y && !FUSE_SPLIT) {
        r2c_split<N, N>(ctx, s, PITCH, 1, NL, tw);
        ctx.sync();
    }
    if constexpr (FUSE_SPLIT) {
        // B+C: last z stage fused with the Hermitian split.  Stored slot p = k0 R1 + k1 holds frequency k0 + R0 k1 and
        // H - k sits in block R0 - k0 at index R1 - 1 - k1 (block 0: R1 - k1): a task transforms the block pair
        // (k0, R0 - k0) of one line and applies r2c_pair to the 2 R1 values in registers (mirror of zl_inv_split_stage1).
        static_assert(DO_Y || Plan<H>::NS == 2, "tiles of N >= 256 use two-stage z plans");
        constexpr int ZR0 = StageInfo<H, 0>::R, ZR1 = StageInfo<H, 1>::R, NTYPE = ZR0 / 2 + 1;
        for (int t = ctx.tid; t < NL * NTYPE; t += ctx.nthr) {
            const int u = t / NL, l = t - u * NL;
            float2* col = s + l;
            float2 a[ZR1];
            if (u == 0) {
#pragma unroll
                for (int i = 0; i < ZR1; ++i) a[i] = col[i * PITCH];
                dft_fwd<ZR1>(a);
                const float2 z = a[0];
                a[0] = make_float2(z.x + z.y, 0.f);
                col[H * PITCH] = make_float2(z.x - z.y, 0.f);
                a[ZR1 / 2] = make_float2(a[ZR1 / 2].x, -a[ZR1 / 2].y);
#pragma unroll
                for (int i = 1; i < ZR1 / 2; ++i) r2c_pair(a[i], a[ZR1 - i], tw[ZR0 * i]);
#pragma unroll
                for (int i = 0; i < ZR1; ++i) col[i * PITCH] = a[i];
            } else if (u == 1) {
                float2* blk = col + (ZR0 / 2) * ZR1 * PITCH;
#pragma unroll
                for (int i = 0; i < ZR1; ++i) a[i] = blk[i * PITCH];
                dft_fwd<ZR1>(a);
#pragma unroll
                for (int i = 0; i < ZR1 / 2; ++i) r2c_pair(a[i], a[ZR1 - 1 - i], tw[ZR0 / 2 + ZR0 * i]);
#pragma unroll
                for (int i = 0; i < ZR1; ++i) blk[i * PITCH] = a[i];
            } else {
                const int k0 = u - 1;
                float2* ba = col + k0 * ZR1 * PITCH;
                float2* bb = col + (ZR0 - k0) * ZR1 * PITCH;
                float2 b[ZR1];
#pragma unroll
                for (int i = 0; i < ZR1; ++i) { a[i] = ba[i * PITCH]; b[i] = bb[i * PITCH]; }
                dft_fwd<ZR1>(a);
                dft_fwd<ZR1>(b);
#pragma unroll
                for (int i = 0; i < ZR1; ++i) r2c_pair(a[i], b[ZR1 - 1 - i], tw[k0 + ZR0 * i]);
#pragma unroll
                for (int i = 0; i < ZR1; ++i) { ba[i * PITCH] = a[i]; bb[i * PITCH] = b[i]; }
            }
        }
        ctx.sync();
    }
    if constexpr (!DO_Y) {
        // copy out (slot-major rows are contiguous in HBM), two columns = 16 bytes per store
        float4* So4 = reinterpret_cast<float4*>(So);
        for (int i = ctx.tid; i < NL * H / 2; i += ctx.nthr) {
            const int l = i / (H / 2), pc = 2 * (i - l * (H / 2));
            const float2 a = s[kz_swz(pc, y0 + l) * PITCH + l], b = s[kz_swz(pc + 1, y0 + l) * PITCH + l];
            So4[i] = make_float4(a.x, a.y, b.x, b.y);
        }
        // Nyquist plane: written transposed ([y][x]) so that the y pass can fetch it with TMA tiles
        float2* Qt = p.Q + (size_t)by * ((size_t)N * N);
        for (int l = ctx.tid; l < NL; l += ctx.nthr) Qt[(size_t)(y0 + l) * N + x] = s[H * PITCH + l];
    } else {
        static_assert(!DO_Y || Plan<N>::NS == 2, "fused planes use two-stage y plans");
        // C: r2c split fused into y stage 0.  One task owns the row pair (k, H-k) for R y-values.
        constexpr int RY = StageInfo<N, 0>::R, STY = StageInfo<N, 0>::ST;
        constexpr int TWMUL = 1;  // tw has length N: w_N^k = tw[k]
        for (int t = ctx.tid; t < (H / 2 + 1) * STY; t += ctx.nthr) {
            const int k = t / STY, q = t - k * STY;
            float2 a[RY], b[RY];
            int ra, rb;
            if (k == 0) {
                ra = 0; rb = H;
#pragma unroll
                for (int r = 0; r < RY; ++r) {
                    const float2 z = s[q + STY * r];
                    a[r] = make_float2(z.x + z.y, 0.f);
                    b[r] = make_float2(z.x - z.y, 0.f);
                }
            } else if (k == H / 2) {
                ra = rb = freq2pos<H>(k);
#pragma unroll
                for (int r = 0; r < RY; ++r) {
                    const float2 z = s[ra * PITCH + q + STY * r];
                    a[r] = make_float2(z.x, -z.y);
                    b[r] = a[r];
                }
            } else {
                ra = freq2pos<H>(k); rb = freq2pos<H>(H - k);
                const float2 w = tw[k * TWMUL];
#pragma unroll
                for (int r = 0; r < RY; ++r) {
                    a[r] = s[ra * PITCH + q + STY * r];
                    b[r] = s[rb * PITCH + q + STY * r];
                    r2c_pair(a[r], b[r], w);
                }
            }
            bfly_fwd<N, 0, N>(a, q, tw);
#pragma unroll
            for (int r = 0; r < RY; ++r) s[ra * PITCH + q + STY * r] = a[r];
            if (rb != ra) {
                bfly_fwd<N, 0, N>(b, q, tw);
#pragma unroll
                for (int r = 0; r < RY; ++r) s[rb * PITCH + q + STY * r] = b[r];
            }
        }
        ctx.sync();
        // D: last y stage smem -> registers -> global; lanes over kz slots (contiguous in HBM)
        constexpr int R1 = StageInfo<N, 1>::R;
        static_assert(StageInfo<N, 1>::ST == 1, "last stage");
        for (int t = ctx.tid; t < H * (N / R1); t += ctx.nthr) {
            const int blk = t / H, pz = t - blk * H;
            float2 v[R1];
#pragma unroll
            for (int r = 0; r < R1; ++r) v[r] = s[pz * PITCH + blk * R1 + r];
            dft_fwd<R1>(v);
#pragma unroll
            for (int r = 0; r < R1; ++r) So[(size_t)(blk * R1 + r) * H + kz_swz(pz, blk * R1 + r)] = v[r];
        }
        for (int blk = ctx.tid; blk < N / R1; blk += ctx.nthr) {  // Nyquist row
            float2 v[R1];
#pragma unroll
            for (int r = 0; r < R1; ++r) v[r] = s[H * PITCH + blk * R1 + r];
            dft_fwd<R1>(v);
#pragma unroll
            for (int r = 0; r < R1; ++r) Qo[blk * R1 + r] = v[r];
        }
    }
}

}  // namespace sap
