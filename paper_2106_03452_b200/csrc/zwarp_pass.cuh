// zwarp_pass.cuh -- forward z pass for N >= 256 (F1+F2 and B2+B3 of SURVEY 8(a)): real lines -> half spectrum, one tile of
// 32 z-lines per CTA, each WARP owning four of the lines from the first butterfly to the store.
//
// Replaces the [slot][line] tile of zy_pass.cuh for these sizes (that layout stays for the fused planes of N <= 128,
// where the y transform runs across the lines).  Here a line never meets another line after the rasterisation, so
//   - the tile is line-major and the only block barriers are the two around the rasterisation; the stages of a warp's
//     lines are separated by __syncwarp, and the warps of a CTA drift apart (one stores while another transforms),
//   - lanes run over the points of a line: the first stage reads 128 contiguous bytes per half-warp, the last stage
//     reads its 16 consecutive values with 16-byte accesses (a line is padded by 2 values per 16, which keeps those
//     aligned and conflict-free), and
//   - the Hermitian split happens on the way out: a half-warp takes the slot pair (k, H-k) for 16 consecutive k of
//     two blocks that are each other's mirror, so both stores are 128 contiguous bytes -- no separate split pass,
//     no transposing copy-out.
// Plans: H = N/2 = R0 x 16 with R0 = 8 (N = 256) or 16 (N = 512); stored order, column swizzle and the transposed
// Nyquist plane exactly as zy_pass.cuh writes them.  Equations: Eq.10-12, DESIGN.md "Backward".
#pragma once
#include "fft_core.cuh"
#include "zy_pass.cuh"

namespace sap {

template <int N> struct ZwCfg {
    static constexpr int H = N / 2, NL = 32, NT = 256, LPW = NL / (NT / 32);   // 4 lines per warp
    static constexpr int R0 = StageInfo<H, 0>::R, R1 = StageInfo<H, 1>::R;
    static_assert(Plan<H>::NS == 2 && R1 == 16 && StageInfo<H, 0>::ST == 16, "z plans are R0 x 16");
    // a line is padded by PAD values per 16: two at N = 256 (the 16 values of a last-stage butterfly stay 16-byte aligned:
    // 8 vector accesses, conflict-free), one at N = 512 (three CTAs still fit an SM; 16 conflict-free 8-byte accesses)
    static constexpr int PAD = (N == 256) ? 2 : 1, BS = 16 + PAD;
    static constexpr int LP = H + PAD * (H / 16);   // padded line pitch (complex values)
    static constexpr int GPL = R0 / 2;              // half-warp groups per line in the split: GPL - 1 block pairs + the special one
    static constexpr int MINB = (N == 256) ? 4 : 3;
    static constexpr size_t SMEM = ((size_t)NL * LP + H + (R0 - 1) * 16) * sizeof(float2);
};
// position of complex element e of a line inside the padded line
template <int PAD> SAP_HD int zw_pe(int e) { return e + PAD * (e >> 4); }

// r2c pair with packed arithmetic: za = Z[k], zb = Z[H-k], wh = exp(-2 pi i k / N) / 2  ->  xa = X[k], xb = X[H-k]
// (r2c_pair of fft_core.cuh: E = (za + conj zb)/2, D = (za - conj zb)/2, F = i w D, X[k] = E - F, X[H-k] = conj(E + F))
__device__ __forceinline__ void zw_r2c_pair(float2 za, float2 zb, float2 wh, float2& xa, float2& xb) {
    const float2 t = __fadd2_rn(za, make_float2(zb.x, -zb.y));    // 2 E
    const float2 u = __fadd2_rn(za, make_float2(-zb.x, zb.y));    // 2 D
    const float2 g = cmul(u, wh);                                  // w D
    const float2 half = make_float2(0.5f, 0.5f);
    xa = __ffma2_rn(t, half, make_float2(g.y, -g.x));              // E - i w D
    const float2 q = __ffma2_rn(t, half, make_float2(-g.y, g.x));  // E + i w D
    xb = make_float2(q.x, -q.y);
}

template <int N, int SRC>
__global__ void __launch_bounds__(ZwCfg<N>::NT, ZwCfg<N>::MINB) k_zw_fwd(const ZyFwdParams p) {
    using C = ZwCfg<N>;
    constexpr int H = C::H, NL = C::NL, NT = C::NT, LPW = C::LPW, R0 = C::R0, LP = C::LP, GPL = C::GPL, BS = C::BS;
    constexpr int NTY = N / NL, NBINS = N * NTY, M = N - 1;
    extern __shared__ __align__(16) float2 zw_smem[];
    float2* s = zw_smem;                 // [NL][LP]
    float2* tws = s + (size_t)NL * LP;   // [H]  split twiddles, halved: tws[k0 * 16 + j] = w_N^(k0 + R0 j) / 2
    float2* tw0 = tws + H;               // [(R0-1) * 16] stage-0 twiddles: tw0[(r-1) * 16 + q] = w_H^(r q)
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int bx = blockIdx.x, item = blockIdx.y;   // a CTA takes the p.nch channels of its tile one after the other
    pdl_wait();
    if (SRC == SRC_SPLAT && p.clear_cnt && bx == 0 && item == 0) {
        for (int i = tid; i < p.clear_n; i += NT) p.clear_cnt[i] = 0;
        if (tid == 0) p.clear_sync[0] = 0u;
    }
    const size_t V = (size_t)N * N * N;
    const size_t line0 = (size_t)bx * NL;  // global line index = x*N + y
    const int x = (int)(line0 / N), y0 = (int)(line0 % N), ty = y0 / NL;
    if (SRC == SRC_GBAR) {   // pull the tile of G (32 KB, contiguous) towards L2 while the points are rasterised
        const char* g = reinterpret_cast<const char*>(p.G + (size_t)item * V + line0 * N);
        for (int i = tid; i < NL * N * 4 / 128; i += NT) asm volatile("prefetch.global.L2 [%0];" ::"l"(g + (size_t)i * 128));
    }
    // bins that can touch lines [line0, line0 + NL): x-slabs {x, x-1} x y-tiles {ty, ty-1}
    const int* bs = p.bin_start + (size_t)item * (NBINS + 1);
    int b_lo[4], b_n[4], total = 0;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const int xb = (k & 1) ? ((x - 1) & M) : x;
        const int tb = (k & 2) ? ((ty + NTY - 1) % NTY) : ty;
        const int bin = xb * NTY + tb;
        b_lo[k] = bs[bin];
        b_n[k] = bs[bin + 1] - b_lo[k];
        total += b_n[k];
    }
    // the bins, the tables and the fixed-point scale are the same for every channel of the tile (the points come from L1
    // the second and third time)
    if (total > 0 || SRC == SRC_GBAR) {
        for (int i = tid; i < H; i += NT) { const float2 w = p.tw[(i >> 4) + R0 * (i & 15)]; tws[i] = make_float2(0.5f * w.x, 0.5f * w.y); }
        for (int i = tid; i < (R0 - 1) * 16; i += NT) tw0[i] = p.tw[2 * ((i >> 4) + 1) * (i & 15)];
    }
    const int lw = warp * LPW;
    const int hw = lane >> 4, j = lane & 15;
#pragma unroll 1
    for (int ch = 0; ch < p.nch; ++ch) {
    const int by = item * p.nch + ch;
    float2* So = p.S + (size_t)by * ((size_t)N * N * H) + line0 * H;
    float2* Qt = p.Q + (size_t)by * ((size_t)N * N);   // transposed Nyquist plane [y][x]
    if (SRC == SRC_SPLAT && total == 0) {  // nothing lands here: the spectrum of zeros is zeros
        // With the activity lists: in an ACTIVE plane the first stage of the y pass reads the rows of an inactive tile as zeros
        // whatever the spectrum holds there (nobody has to write them); an INACTIVE plane is not touched by the y pass (in place
        // on channels 0 and 1) and the x pass reads the zeros of channels 0 and 1 as the y pass's output -- nobody reads channel 2
        const bool skip_main = p.plane_act && (p.plane_act[(size_t)item * N + x] != 0 || ch == 2);
        float4* So4 = reinterpret_cast<float4*>(So);
        if (!skip_main)
            for (int i = tid; i < NL * H / 2; i += NT) So4[i] = make_float4(0.f, 0.f, 0.f, 0.f);
        for (int l = tid; l < NL; l += NT) Qt[(size_t)(y0 + l) * N + x] = make_float2(0.f, 0.f);
        continue;
    }
    if (ch > 0) __syncthreads();   // every warp is done with the previous channel's tile
    // GBAR tile that no point can touch: W = 0 there, Gbar' = s G (- the delta term) straight from HBM: no zero fill, no
    // rasterisation, one barrier less
    const bool has_pts = total > 0;
    if (has_pts) {
        float4* s4 = reinterpret_cast<float4*>(s);
        for (int i = tid; i < NL * LP / 2; i += NT) s4[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
    // fixed-point rasterisation (see zy_pass.cuh): scale 2^k with (points that can touch the tile) x (largest normal
    // component of the item) x 2^k < 2^30
    const float amax = (SRC == SRC_SPLAT) ? bits_u2f(p.nmax[item]) : 1.f;
    const FixScale fs = fix_scale((float)total * amax);
    if (has_pts) __syncthreads();
    if (has_pts) {
        int* si = reinterpret_cast<int*>(s);
        const float4* sp = p.spts + (size_t)item * p.P;
        const float4* sn = p.snrm + (size_t)item * p.P;
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            for (int i = b_lo[k] + tid; i < b_lo[k] + b_n[k]; i += NT) {
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
                            atomicAdd(si + (ly * LP + zw_pe<C::PAD>(z >> 1)) * 2 + (z & 1), fix_round(wxy * (dz ? fz : 1.f - fz)));
                        }
                    }
                }
            }
        }
    }
    __syncthreads();
    // ---- from here on a warp works on its own LPW lines ----
    // stage 0 (radix R0, stride 16): task = (line, q), q = lane & 15; fixed point -> float (GBAR: combined with G) on the way in
    {
        float cs_ = 0.f, cw = 0.f, c0 = 0.f;
        const float2* g2 = nullptr;
        if (SRC == SRC_GBAR) {
            g2 = reinterpret_cast<const float2*>(p.G + (size_t)item * V) + line0 * H;
            cs_ = p.bw[item * 4 + 0]; cw = p.bw[item * 4 + 1] * fs.invS; c0 = p.bw[item * 4 + 2];
        }
#pragma unroll 1
        for (int it = 0; it < LPW / 2; ++it) {
            const int l = lw + 2 * it + hw;
            float2* ls = s + l * LP + j;
            float2 v[R0];
            if (SRC == SRC_GBAR) {
#pragma unroll
                for (int r = 0; r < R0; ++r) v[r] = g2[l * H + j + 16 * r];
                if (has_pts) {
#pragma unroll
                    for (int r = 0; r < R0; ++r) {
                        const int2 iv = *reinterpret_cast<const int2*>(ls + BS * r);
                        v[r] = __ffma2_rn(make_float2(cs_, cs_), v[r], __fmul2_rn(make_float2(cw, cw), make_float2((float)iv.x, (float)iv.y)));
                    }
                } else {
#pragma unroll
                    for (int r = 0; r < R0; ++r) v[r] = cscale(cs_, v[r]);
                }
                if (line0 == 0 && l == 0 && j == 0) v[0].x -= c0;
            } else {
#pragma unroll
                for (int r = 0; r < R0; ++r) {
                    const int2 iv = *reinterpret_cast<const int2*>(ls + BS * r);
                    v[r] = __fmul2_rn(make_float2(fs.invS, fs.invS), make_float2((float)iv.x, (float)iv.y));
                }
            }
            dft_fwd<R0>(v);
#pragma unroll
            for (int r = 1; r < R0; ++r) v[r] = cmul(v[r], tw0[(r - 1) * 16 + j]);
#pragma unroll
            for (int r = 0; r < R0; ++r) ls[BS * r] = v[r];
        }
    }
    __syncwarp();
    // stage 1 (radix 16, stride 1): task = (line, block k0); 16 consecutive values = 8 x 16 bytes
    {
        constexpr int TPL = R0;                       // tasks per line
        constexpr int NIT = LPW * TPL / 32;           // 1 (N = 256) or 2 (N = 512)
#pragma unroll 1
        for (int it = 0; it < NIT; ++it) {
            const int t = it * 32 + lane, l = lw + t / TPL, k0 = t % TPL;
            float2* b2 = s + l * LP + BS * k0;
            float2 v[16];
            if constexpr (C::PAD == 2) {
                float4* b4 = reinterpret_cast<float4*>(b2);
#pragma unroll
                for (int r = 0; r < 8; ++r) {
                    const float4 u = b4[r];
                    v[2 * r] = make_float2(u.x, u.y);
                    v[2 * r + 1] = make_float2(u.z, u.w);
                }
                dft_fwd<16>(v);
#pragma unroll
                for (int r = 0; r < 8; ++r) b4[r] = make_float4(v[2 * r].x, v[2 * r].y, v[2 * r + 1].x, v[2 * r + 1].y);
            } else {
#pragma unroll
                for (int r = 0; r < 16; ++r) v[r] = b2[r];
                dft_fwd<16>(v);
#pragma unroll
                for (int r = 0; r < 16; ++r) b2[r] = v[r];
            }
        }
    }
    __syncwarp();
    // Hermitian split on the way out.  Slot p = 16 k0 + k1 holds Z[k], k = k0 + R0 k1, and Z[H - k] sits in block R0 - k0 at
    // index 15 - k1 (block 0: index 16 - k1): a half-warp takes k1 = j = 0..15 of the block pair (k0, R0 - k0) of one line,
    // reads the two blocks (one of them backwards), and stores X[k] and X[H - k] to the two mirrored 128-byte segments of
    // the line's row.  The blocks 0 and R0/2 are their own mirrors: they share a half-warp (lanes 1..7 and 8..15; lane 0
    // has k = 0 with the Nyquist value, and k = H/2).  A half-warp keeps its line while k0 runs: every address below is a
    // per-line base plus a compile-time offset.
#pragma unroll
    for (int a = 0; a < LPW / 2; ++a) {
        const int l = lw + 2 * a + hw, y = y0 + l, sw = y & 15;
        const float2* ls = s + l * LP;
        float2* row = So + (size_t)l * H;
        {   // block pairs (k0, R0 - k0), k0 = 1 .. R0/2 - 1
            const float2* la = ls + j;
            const float2* lb = ls + BS * R0 + 15 - j;
            float2* ra = row + (j ^ sw);
            float2* rb = row + R0 * 16 + ((15 - j) ^ sw);
            const float2* tj = tws + j;
#pragma unroll
            for (int k0 = 1; k0 < R0 / 2; ++k0) {
                const float2 za = la[BS * k0], zb = lb[-BS * k0];
                float2 xa, xb;
                zw_r2c_pair(za, zb, tj[16 * k0], xa, xb);   // k = k0 + R0 j
                ra[16 * k0] = xa;
                rb[-16 * k0] = xb;
            }
        }
        {   // the self-mirrored blocks 0 and KB = R0/2
            constexpr int KB = R0 / 2;
            const int blk = j >> 3, jj = j & 7;
            if (j == 0) {
                const float2 z = ls[0], zh = ls[8];
                row[sw] = make_float2(z.x + z.y, 0.f);
                Qt[(size_t)y * N + x] = make_float2(z.x - z.y, 0.f);
                row[8 ^ sw] = make_float2(zh.x, -zh.y);
            } else {
                const int ia = blk ? BS * KB + jj : jj, ib = blk ? BS * KB + 15 - jj : 16 - jj;
                const int ca = blk ? KB * 16 + (jj ^ sw) : (jj ^ sw), cb = blk ? KB * 16 + ((15 - jj) ^ sw) : ((16 - jj) ^ sw);
                float2 xa, xb;
                zw_r2c_pair(ls[ia], ls[ib], tws[blk ? KB * 16 + jj : jj], xa, xb);   // k = R0 jj  |  KB + R0 jj
                row[ca] = xa;
                row[cb] = xb;
            }
        }
    }
    }   // channels
}

}  // namespace sap
