// zwarp_inv.cuh -- inverse z pass for N >= 256 (F4 and B5 of SURVEY 8(a)): half spectrum -> real lines, the mirror of
// k_zw_fwd (zwarp_pass.cuh).  A WARP owns four z-lines from the load to the store; there is no block barrier and no ring:
// a CTA walks the tiles of 32 lines with its eight warps free of one another, and the loads of a warp's four lines (16 per
// lane, issued before the first use) are what keeps HBM busy.
//   1. inverse Hermitian split straight from HBM: a half-warp reads the slot pairs (k, H-k) of two mirrored 16-slot blocks
//      of its line (two 128-byte segments, the column swizzle undone on the way) and writes Z[k], Z[H-k] to the padded
//      line-major tile;
//   2. inverse of the last plan stage (radix 16, stride 1): a lane takes the 16 consecutive values of one block;
//   3. inverse stage 0 (radix R0, stride 16): lanes over q, 128 contiguous bytes per half-warp, registers -> HBM.
// Listed mode (sap_dpsr.cu, ActLists): the three vbar planes of the backward only on the tiles a point can touch.
// Equations: Eq.17; the 1/N^3 of the inverse transform is folded into the spectral multiplier.
#pragma once
#include "zwarp_pass.cuh"
#include "zline_pass.cuh"

namespace sap {

// c2r pair with packed arithmetic: xa = X[k], xb = X[H-k], wh = exp(-2 pi i k / N) / 2  ->  za = Z[k], zb = Z[H-k]
// (c2r_pair of fft_core.cuh: E = (xa + conj xb)/2, D = (xa - conj xb)/2, O = conj(w) D, Z[k] = E + i O, Z[H-k] = conj(E - i O))
__device__ __forceinline__ void zw_c2r_pair(float2 xa, float2 xb, float2 wh, float2& za, float2& zb) {
    const float2 t = __fadd2_rn(xa, make_float2(xb.x, -xb.y));    // 2 E
    const float2 u = __fadd2_rn(xa, make_float2(-xb.x, xb.y));    // 2 D
    const float2 o = cmulc(u, wh);                                 // conj(w) D
    const float2 half = make_float2(0.5f, 0.5f);
    za = __ffma2_rn(t, half, make_float2(-o.y, o.x));              // E + i O
    const float2 q = __ffma2_rn(t, half, make_float2(o.y, -o.x));  // E - i O
    zb = make_float2(q.x, -q.y);
}

template <int N>
__global__ void __launch_bounds__(ZwCfg<N>::NT, ZwCfg<N>::MINB) k_zw_inv(const ZlInvParams p) {
    using C = ZwCfg<N>;
    constexpr int H = C::H, NL = C::NL, NT = C::NT, LPW = C::LPW, R0 = C::R0, LP = C::LP, BS = C::BS;
    constexpr int TPP = N * N / NL;   // tiles per plane = bins per item (a bin tile is 32 lines)
    extern __shared__ __align__(16) float2 zwi_smem[];
    float2* s = zwi_smem;                // [NL][LP]
    float2* tws = s + (size_t)NL * LP;   // [H]  split twiddles, halved: tws[k0 * 16 + j] = w_N^(k0 + R0 j) / 2
    float2* tw0 = tws + H;               // [(R0-1) * 16] stage-0 twiddles: tw0[(r-1) * 16 + q] = w_H^(r q)
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    for (int i = tid; i < H; i += NT) { const float2 w = p.tw[(i >> 4) + R0 * (i & 15)]; tws[i] = make_float2(0.5f * w.x, 0.5f * w.y); }
    for (int i = tid; i < (R0 - 1) * 16; i += NT) tw0[i] = p.tw[2 * ((i >> 4) + 1) * (i & 15)];
    __syncthreads();   // the tables are constants of the handle; the only block barrier of the kernel
    pdl_wait();
    const bool listed = p.zlist != nullptr;
    const long long total = listed ? (long long)p.nact[0] * 3 : (long long)p.planes * TPP;
    const int lw = warp * LPW, hw = lane >> 4, j = lane & 15;
    for (long long v = blockIdx.x; v < total; v += gridDim.x) {
        // At 256^3 the pass before this one wrote the planes in ascending x and a spectrum is half the L2: walk them in
        // descending x (the planes written last are read first).  At 512^3 a spectrum is four times the L2: no gain.
        const long long vv = (N == 256) ? total - 1 - v : v;
        long long g;   // dense tile id: plane * TPP + tile
        if (listed) {
            const long long e = vv / 3;
            const int ch = (int)(vv - e * 3), id = p.zlist[e], item = id / p.nbins, bin = id - item * p.nbins;
            g = ((long long)item * 3 + ch) * TPP + bin;
        } else {
            g = vv;
        }
        const int y0 = (int)((g * NL) % N);
        const float2* So = p.S + (size_t)g * NL * H;
        const float2* Qo = p.Q + (size_t)g * NL;
        float2* out2 = reinterpret_cast<float2*>(p.out) + (size_t)g * NL * H;
        // 1. inverse split, HBM -> registers -> tile.  A half-warp keeps its line while k0 runs (constant offsets).
#pragma unroll
        for (int a = 0; a < LPW / 2; ++a) {
            const int l = lw + 2 * a + hw, sw = (y0 + l) & 15;
            const float2* row = So + (size_t)l * H;
            float2* ls = s + l * LP;
            constexpr int KB = R0 / 2;
            const int blk = j >> 3, jj = j & 7;
            // the loads of the line first: GPL - 1 block pairs + the self-mirrored blocks 0 and KB
            float2 xa[R0 / 2], xb[R0 / 2];
            {
                const float2* ra = row + (j ^ sw);
                const float2* rb = row + R0 * 16 + ((15 - j) ^ sw);
#pragma unroll
                for (int k0 = 1; k0 < R0 / 2; ++k0) { xa[k0] = __ldcs(ra + 16 * k0); xb[k0] = __ldcs(rb - 16 * k0); }
                if (j == 0) {
                    xa[0] = __ldcs(row + sw);                 // X[0]
                    xb[0] = __ldcs(row + (8 ^ sw));           // X[H/2]
                } else {
                    const int ca = blk ? KB * 16 + (jj ^ sw) : (jj ^ sw), cb = blk ? KB * 16 + ((15 - jj) ^ sw) : ((16 - jj) ^ sw);
                    xa[0] = __ldcs(row + ca);
                    xb[0] = __ldcs(row + cb);
                }
            }
            float xh = 0.f;
            if (j == 0) xh = __ldcs(Qo + l).x;                // X[H], the Nyquist value
            {
                float2* la = ls + j;
                float2* lb = ls + BS * R0 + 15 - j;
                const float2* tj = tws + j;
#pragma unroll
                for (int k0 = 1; k0 < R0 / 2; ++k0) {
                    float2 za, zb;
                    zw_c2r_pair(xa[k0], xb[k0], tj[16 * k0], za, zb);   // k = k0 + R0 j
                    la[BS * k0] = za;
                    lb[-BS * k0] = zb;
                }
            }
            if (j == 0) {
                ls[0] = make_float2(0.5f * (xa[0].x + xh), 0.5f * (xa[0].x - xh));
                ls[8] = make_float2(xb[0].x, -xb[0].y);
            } else {
                const int ia = blk ? BS * KB + jj : jj, ib = blk ? BS * KB + 15 - jj : 16 - jj;
                float2 za, zb;
                zw_c2r_pair(xa[0], xb[0], tws[blk ? KB * 16 + jj : jj], za, zb);   // k = R0 jj  |  KB + R0 jj
                ls[ia] = za;
                ls[ib] = zb;
            }
        }
        __syncwarp();
        // 2. inverse of the last plan stage: task = (line, block k0), 16 consecutive values
        {
            constexpr int TPL = R0, NIT = LPW * TPL / 32;
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
                    dft_inv<16>(v);
#pragma unroll
                    for (int r = 0; r < 8; ++r) b4[r] = make_float4(v[2 * r].x, v[2 * r].y, v[2 * r + 1].x, v[2 * r + 1].y);
                } else {
#pragma unroll
                    for (int r = 0; r < 16; ++r) v[r] = b2[r];
                    dft_inv<16>(v);
#pragma unroll
                    for (int r = 0; r < 16; ++r) b2[r] = v[r];
                }
            }
        }
        __syncwarp();
        // 3. inverse stage 0: task = (line, q = lane & 15), conjugate twiddle then the inverse radix-R0 butterfly; the R0 results
        //    are the complex values q + 16 r of the line = reals 2 (q + 16 r), + 1: 128 contiguous bytes per half-warp
#pragma unroll 1
        for (int it = 0; it < LPW / 2; ++it) {
            const int l = lw + 2 * it + hw;
            const float2* ls = s + l * LP + j;
            float2 v[R0];
#pragma unroll
            for (int r = 0; r < R0; ++r) v[r] = ls[BS * r];
#pragma unroll
            for (int r = 1; r < R0; ++r) v[r] = cmulc(v[r], tw0[(r - 1) * 16 + j]);
            dft_inv<R0>(v);
            float2* o = out2 + (size_t)l * H + j;
#pragma unroll
            for (int r = 0; r < R0; ++r) o[16 * r] = v[r];
        }
        __syncwarp();   // the tile is free for this warp's lines of the next tile
    }
}

}  // namespace sap
