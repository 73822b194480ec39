// fft_core.cuh -- in-shared-memory radix FFT building blocks for the DPSR kernels (sm_100a).
//
// All FFTs of the path (Eq.12/13/17) are power-of-two lengths 16..512 done on
// lines that live in shared memory.  The forward transform is decimation-in-frequency, in place,
// natural order in -> digit-reversed ("stored") order out; the inverse is the exact mirror
// (decimation-in-time, stored order in -> natural order out).  Because every butterfly reads and
// writes the same R slots, a stage has no intra-stage hazards: one block barrier between stages is
// all the synchronisation there is.  Spectra are kept in stored order in HBM on all three axes; only
// the spectral solve needs to know which frequency a slot holds (pos2freq).
//
// Most functions are __host__ __device__ (plain arithmetic; the host uses pos2freq to build the frequency
// table of the solve); the product only ever runs the butterflies on the device.
#pragma once
#include <cuda_runtime.h>

#define SAP_HD __host__ __device__ __forceinline__

namespace sap {

// Programmatic dependent launch (all kernels of the path are launched with it, see launch_pdl in sap_dpsr.cu):
// the launch of kernel n+1 is processed while kernel n runs; pdl_wait() blocks until kernel n has completed and
// its writes are visible.  Nothing written by a predecessor is touched before pdl_wait().  No kernel triggers its
// dependents early (griddepcontrol.launch_dependents on entry was measured 20% SLOWER at 128^3: the early CTAs
// take shared memory and issue slots from the running kernel), so the trigger is the implicit one at grid exit.
#ifdef __CUDACC__
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
#endif

// Complex arithmetic on float2 = (re, im).  On sm_100a these map to the packed FP32x2 instructions
// (FADD2 / FMUL2 / FFMA2): one issue slot per complex add, two per complex multiply.  The operand
// modifiers of those instructions (half swap, per-half negate, scalar broadcast) absorb mul_mi and conj.
#ifdef __CUDA_ARCH__
SAP_HD float2 cadd(float2 a, float2 b) { return __fadd2_rn(a, b); }
SAP_HD float2 csub(float2 a, float2 b) { return __fadd2_rn(a, make_float2(-b.x, -b.y)); }
SAP_HD float2 cmul(float2 a, float2 w) {
    return __ffma2_rn(make_float2(a.y, a.y), make_float2(-w.y, w.x), __fmul2_rn(make_float2(a.x, a.x), w));
}
// a * conj(w)
SAP_HD float2 cmulc(float2 a, float2 w) {
    return __ffma2_rn(make_float2(a.y, a.y), make_float2(w.y, w.x), __fmul2_rn(make_float2(a.x, a.x), make_float2(w.x, -w.y)));
}
// s * a (real scale)
SAP_HD float2 cscale(float s, float2 a) { return __fmul2_rn(make_float2(s, s), a); }
// c + s * a
SAP_HD float2 caxpy(float s, float2 a, float2 c) { return __ffma2_rn(make_float2(s, s), a, c); }
#else
SAP_HD float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
SAP_HD float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
SAP_HD float2 cmul(float2 a, float2 w) { return make_float2(a.x * w.x - a.y * w.y, a.x * w.y + a.y * w.x); }
// a * conj(w)
SAP_HD float2 cmulc(float2 a, float2 w) { return make_float2(a.x * w.x + a.y * w.y, a.y * w.x - a.x * w.y); }
SAP_HD float2 cscale(float s, float2 a) { return make_float2(s * a.x, s * a.y); }
SAP_HD float2 caxpy(float s, float2 a, float2 c) { return make_float2(c.x + s * a.x, c.y + s * a.y); }
#endif
// a * (-i)
SAP_HD float2 mul_mi(float2 a) { return make_float2(a.y, -a.x); }

// ---- radix plans: N = R0 * R1 * R2 -------------------------------------------------------------
template <int N> struct Plan;
template <> struct Plan<16>  { static constexpr int NS = 1, R0 = 16, R1 = 1,  R2 = 1; };
template <> struct Plan<32>  { static constexpr int NS = 2, R0 = 8,  R1 = 4,  R2 = 1; };
template <> struct Plan<64>  { static constexpr int NS = 2, R0 = 8,  R1 = 8,  R2 = 1; };
template <> struct Plan<128> { static constexpr int NS = 2, R0 = 8,  R1 = 16, R2 = 1; };
template <> struct Plan<256> { static constexpr int NS = 2, R0 = 16, R1 = 16, R2 = 1; };
template <> struct Plan<512> { static constexpr int NS = 3, R0 = 8,  R1 = 8,  R2 = 8; };

template <int N, int S> struct StageInfo {
    using P = Plan<N>;
    static constexpr int R = (S == 0) ? P::R0 : (S == 1) ? P::R1 : P::R2;
    // butterfly stride of stage S: N / (R0 * ... * RS)
    static constexpr int ST = (S == 0) ? N / P::R0 : (S == 1) ? N / (P::R0 * P::R1) : N / (P::R0 * P::R1 * P::R2);
};

// slot p (stored order) of a forward-transformed line holds frequency pos2freq<N>(p)
template <int N> SAP_HD int pos2freq(int p) {
    using P = Plan<N>;
    constexpr int st0 = N / P::R0;
    constexpr int st1 = st0 / P::R1;
    int k0 = p / st0;
    int r = p - k0 * st0;
    int k1 = r / st1;
    int k2 = r - k1 * st1;
    return k0 + P::R0 * (k1 + P::R1 * k2);
}
template <int N> SAP_HD int freq2pos(int k) {
    using P = Plan<N>;
    constexpr int st0 = N / P::R0;
    constexpr int st1 = st0 / P::R1;
    int k0 = k % P::R0;
    int r = k / P::R0;
    int k1 = r % P::R1;
    int k2 = r / P::R1;
    return k0 * st0 + k1 * st1 + k2;
}

// ---- register butterflies: forward DFT of R values, natural order in and out ------------------
template <int R> SAP_HD float2 unit_root(int k);  // exp(-2 pi i k / R), k < R/2
template <> SAP_HD float2 unit_root<8>(int k) {
    switch (k) {
        case 0: return make_float2(1.f, 0.f);
        case 1: return make_float2(0.70710678118654752f, -0.70710678118654752f);
        case 2: return make_float2(0.f, -1.f);
        default: return make_float2(-0.70710678118654752f, -0.70710678118654752f);
    }
}
template <> SAP_HD float2 unit_root<16>(int k) {
    switch (k) {
        case 0: return make_float2(1.f, 0.f);
        case 1: return make_float2(0.92387953251128674f, -0.38268343236508977f);
        case 2: return make_float2(0.70710678118654752f, -0.70710678118654752f);
        case 3: return make_float2(0.38268343236508977f, -0.92387953251128674f);
        case 4: return make_float2(0.f, -1.f);
        case 5: return make_float2(-0.38268343236508977f, -0.92387953251128674f);
        case 6: return make_float2(-0.70710678118654752f, -0.70710678118654752f);
        default: return make_float2(-0.92387953251128674f, -0.38268343236508977f);
    }
}

template <> SAP_HD float2 unit_root<32>(int k) {
    // exp(-2 pi i k / 32), k = 0..15
    const float c[16] = {1.f, 0.98078528040323043f, 0.92387953251128674f, 0.83146961230254524f, 0.70710678118654752f,
                         0.55557023301960218f, 0.38268343236508977f, 0.19509032201612825f, 0.f, -0.19509032201612825f,
                         -0.38268343236508977f, -0.55557023301960218f, -0.70710678118654752f, -0.83146961230254524f,
                         -0.92387953251128674f, -0.98078528040323043f};
    const float sn[16] = {0.f, 0.19509032201612825f, 0.38268343236508977f, 0.55557023301960218f, 0.70710678118654752f,
                          0.83146961230254524f, 0.92387953251128674f, 0.98078528040323043f, 1.f, 0.98078528040323043f,
                          0.92387953251128674f, 0.83146961230254524f, 0.70710678118654752f, 0.55557023301960218f,
                          0.38268343236508977f, 0.19509032201612825f};
    return make_float2(c[k], -sn[k]);
}

// Forward (INV = false, kernel exp(-2 pi i jk/R)) or unnormalised inverse (INV = true, exp(+...)) DFT of R
// values, natural order in and out.  The two differ only in the sign of i and the conjugated roots.
// a * (+i)
SAP_HD float2 mul_pi(float2 a) { return make_float2(-a.y, a.x); }
template <int R, bool INV> SAP_HD void dft_dir(float2 (&v)[R]) {
    if constexpr (R == 1) {
    } else if constexpr (R == 2) {
        float2 a = v[0], b = v[1];
        v[0] = cadd(a, b);
        v[1] = csub(a, b);
    } else if constexpr (R == 4) {
        float2 t0 = cadd(v[0], v[2]), t1 = csub(v[0], v[2]);
        float2 t2 = cadd(v[1], v[3]), d = csub(v[1], v[3]);
        float2 t3 = INV ? mul_pi(d) : mul_mi(d);
        v[0] = cadd(t0, t2);
        v[2] = csub(t0, t2);
        v[1] = cadd(t1, t3);
        v[3] = csub(t1, t3);
    } else {
        float2 e[R / 2], o[R / 2];
#pragma unroll
        for (int i = 0; i < R / 2; ++i) { e[i] = v[2 * i]; o[i] = v[2 * i + 1]; }
        dft_dir<R / 2, INV>(e);
        dft_dir<R / 2, INV>(o);
        // v[k] = e + t, v[k + R/2] = e - t with t = o w^k (forward) or o conj(w^k) (inverse).  The roots are compile-time
        // constants: written so that each enters as a SCALAR immediate of a packed instruction and the rotations +-i o as
        // operand modifiers (half swap + per-half negate).  A constant PAIR (wr, wi) would have to sit in two registers, and
        // at the register budget of these kernels the compiler rebuilt such pairs with two MOVs per use (10-12 % of all
        // executed instructions).  t = wr o + wi (i o) [forward; -i o inverse]:
        //   general root:            e +- t = fma(+-wi, rot, fma(+-wr, o, e))                     4 packed instructions
        //   w = c (+-1 - i) (k = R/8, 3R/8):  t = c s, s = rot' +- o,  e +- t = fma(+-c, s, e)    3 instead of 4
#pragma unroll
        for (int k = 0; k < R / 2; ++k) {
            if (k == 0) {
                v[k] = cadd(e[k], o[k]);
                v[k + R / 2] = csub(e[k], o[k]);
            } else if (k == R / 4) {
                const float2 t = INV ? mul_pi(o[k]) : mul_mi(o[k]);
                v[k] = cadd(e[k], t);
                v[k + R / 2] = csub(e[k], t);
            } else if (R >= 8 && (8 * k == R || 8 * k == 3 * R)) {
                constexpr float c = 0.70710678118654752f;
                const float2 r = INV ? mul_pi(o[k]) : mul_mi(o[k]);
                const float2 sm = (8 * k == R) ? cadd(r, o[k]) : csub(r, o[k]);
                v[k] = caxpy(c, sm, e[k]);
                v[k + R / 2] = caxpy(-c, sm, e[k]);
            } else {
                const float2 w = unit_root<R>(k);   // (wr, wi), folded to immediates (k is an unrolled constant)
                const float2 rot = INV ? mul_mi(o[k]) : mul_pi(o[k]);
                v[k] = caxpy(w.y, rot, caxpy(w.x, o[k], e[k]));
                v[k + R / 2] = caxpy(-w.y, rot, caxpy(-w.x, o[k], e[k]));
            }
        }
    }
}
template <int R> SAP_HD void dft_fwd(float2 (&v)[R]) { dft_dir<R, false>(v); }
template <int R> SAP_HD void dft_inv(float2 (&v)[R]) { dft_dir<R, true>(v); }

// ---- register-level stage butterflies --------------------------------------------------------------
// Stage S of the length-N plan on R values held in registers.  j is the butterfly's index inside its
// sub-transform (0 <= j < ST).  Forward (DIF): DFT_R then twiddle w_{R*ST}^{r j}; inverse (DIT): conjugate
// twiddle then inverse DFT_R.  tw = exp(-2 pi i t / TWN).
template <int N, int S, int TWN>
SAP_HD void bfly_fwd(float2 (&v)[StageInfo<N, S>::R], int j, const float2* tw) {
    constexpr int R = StageInfo<N, S>::R;
    constexpr int ST = StageInfo<N, S>::ST;
    constexpr int TWMUL = TWN / (R * ST);
    dft_fwd<R>(v);
    if (ST > 1) {
#pragma unroll
        for (int r = 1; r < R; ++r) v[r] = cmul(v[r], tw[r * j * TWMUL]);
    }
}
template <int N, int S, int TWN>
SAP_HD void bfly_inv(float2 (&v)[StageInfo<N, S>::R], int j, const float2* tw) {
    constexpr int R = StageInfo<N, S>::R;
    constexpr int ST = StageInfo<N, S>::ST;
    constexpr int TWMUL = TWN / (R * ST);
    if (ST > 1) {
#pragma unroll
        for (int r = 1; r < R; ++r) v[r] = cmulc(v[r], tw[r * j * TWMUL]);
    }
    dft_inv<R>(v);
}

// r2c / c2r pair formulas on single values (see r2c_split / c2r_split below for the derivation).
// w = exp(-2 pi i k / N).  In: a = Z[k], b = Z[H-k].  Out: a = X[k], b = X[H-k].
// Device path: packed (7 instructions instead of 12; bit-identical: the halvings are exact): t = a + conj b = 2 E,
// u = a - conj b = 2 D, g = (u / 2) w, X[k] = t / 2 - i g, X[H-k] = conj(t / 2 + i g).
#ifdef __CUDA_ARCH__
SAP_HD void r2c_pair(float2& a, float2& b, float2 w) {
    const float2 half = make_float2(0.5f, 0.5f);
    const float2 t = __fadd2_rn(a, make_float2(b.x, -b.y));
    const float2 u = __fadd2_rn(a, make_float2(-b.x, b.y));
    const float2 g = cmul(__fmul2_rn(u, half), w);
    a = __ffma2_rn(t, half, make_float2(g.y, -g.x));
    const float2 q = __ffma2_rn(t, half, make_float2(-g.y, g.x));
    b = make_float2(q.x, -q.y);
}
// t = a + conj b = 2 E, u = a - conj b = 2 D, o = (u / 2) conj w, Z[k] = t / 2 + i o, Z[H-k] = conj(t / 2 - i o)
SAP_HD void c2r_pair(float2& a, float2& b, float2 w) {
    const float2 half = make_float2(0.5f, 0.5f);
    const float2 t = __fadd2_rn(a, make_float2(b.x, -b.y));
    const float2 u = __fadd2_rn(a, make_float2(-b.x, b.y));
    const float2 o = cmulc(__fmul2_rn(u, half), w);
    a = __ffma2_rn(t, half, make_float2(-o.y, o.x));
    const float2 q = __ffma2_rn(t, half, make_float2(o.y, -o.x));
    b = make_float2(q.x, -q.y);
}
#else
SAP_HD void r2c_pair(float2& a, float2& b, float2 w) {
    float2 e = make_float2(0.5f * (a.x + b.x), 0.5f * (a.y - b.y));
    float2 d = make_float2(0.5f * (a.x - b.x), 0.5f * (a.y + b.y));
    float2 wd = cmul(d, w);
    float2 f = make_float2(-wd.y, wd.x);
    a = csub(e, f);
    float2 g = cadd(e, f);
    b = make_float2(g.x, -g.y);
}
// In: a = X[k], b = X[H-k].  Out: a = Z[k], b = Z[H-k].
SAP_HD void c2r_pair(float2& a, float2& b, float2 w) {
    float2 e = make_float2(0.5f * (a.x + b.x), 0.5f * (a.y - b.y));
    float2 d = make_float2(0.5f * (a.x - b.x), 0.5f * (a.y + b.y));
    float2 o = cmulc(d, w);
    float2 io = make_float2(-o.y, o.x);
    a = cadd(e, io);
    float2 g = csub(e, io);
    b = make_float2(g.x, -g.y);
}
#endif

// ---- one radix stage over a set of lines in shared memory --------------------------------------
// Element n of line l lives at s[l * LS + n * ES].  tw is the table exp(-2 pi i t / TWN), t < TWN,
// TWN a multiple of N.  LANES_LINES: consecutive threads take consecutive lines (same butterfly),
// else consecutive threads take consecutive butterflies of one line.
template <int N, int S, bool INV, int TWN, bool LANES_LINES>
SAP_HD void fft_stage(float2* s, int ES, int LS, int nlines, const float2* tw, int tid, int nthr) {
    constexpr int R = StageInfo<N, S>::R;
    constexpr int ST = StageInfo<N, S>::ST;
    constexpr int Q = N / R;               // butterflies per line
    constexpr int TWMUL = TWN / (R * ST);  // w_{R*ST}^e = tw[e * TWMUL]
    const int ntasks = nlines * Q;
    for (int t = tid; t < ntasks; t += nthr) {
        int line, q;
        if (LANES_LINES) { q = t / nlines; line = t - q * nlines; }
        else { line = t / Q; q = t - line * Q; }
        const int blk = q / ST;
        const int j = q - blk * ST;
        float2* base = s + line * LS + (blk * (R * ST) + j) * ES;
        float2 v[R];
#pragma unroll
        for (int r = 0; r < R; ++r) v[r] = base[r * ST * ES];
        if (!INV) {
            dft_fwd<R>(v);
            if (ST > 1) {
#pragma unroll
                for (int r = 1; r < R; ++r) v[r] = cmul(v[r], tw[r * j * TWMUL]);
            }
        } else {
            if (ST > 1) {
#pragma unroll
                for (int r = 1; r < R; ++r) v[r] = cmulc(v[r], tw[r * j * TWMUL]);
            }
            dft_inv<R>(v);
        }
#pragma unroll
        for (int r = 0; r < R; ++r) base[r * ST * ES] = v[r];
    }
}

// ---- real <-> half-complex split for a length-N real line done as an H = N/2 point complex FFT --
// After the forward H-point FFT, slot pos(k) holds Z[k] = E[k] + i O[k] (E, O = DFTs of the even and
// odd samples).  X[k] = E[k] + w^k O[k], w = exp(-2 pi i / N), k = 0..H.  In place: X[k] goes to slot
// pos(k) (k < H) and X[H] to the extra row H.  One task handles the pair (k, H-k).
// Rows are at s[row * RS + line * LS].
template <int N, int TWN, class Ctx>
SAP_HD void r2c_split(Ctx& ctx, float2* s, int RS, int LS, int nlines, const float2* tw) {
    constexpr int H = N / 2;
    constexpr int TWMUL = TWN / N;
    const int ntasks = nlines * (H / 2 + 1);
    for (int t = ctx.tid; t < ntasks; t += ctx.nthr) {
        const int k = t / nlines;
        const int line = t - k * nlines;
        float2* col = s + line * LS;
        if (k == 0) {
            float2 z = col[0];  // pos(0) = 0
            col[0] = make_float2(z.x + z.y, 0.f);
            col[H * RS] = make_float2(z.x - z.y, 0.f);
        } else if (k == H / 2) {
            float2* p = col + freq2pos<H>(k) * RS;
            float2 z = *p;
            *p = make_float2(z.x, -z.y);
        } else {
            float2* pa = col + freq2pos<H>(k) * RS;
            float2* pb = col + freq2pos<H>(H - k) * RS;
            float2 a = *pa, b = *pb;
            float2 e = make_float2(0.5f * (a.x + b.x), 0.5f * (a.y - b.y));  // (A + conj B)/2
            float2 d = make_float2(0.5f * (a.x - b.x), 0.5f * (a.y + b.y));  // (A - conj B)/2
            float2 wd = cmul(d, tw[k * TWMUL]);
            float2 f = make_float2(-wd.y, wd.x);  // i w^k D
            *pa = csub(e, f);                     // X[k]   = E - F
            float2 g = cadd(e, f);
            *pb = make_float2(g.x, -g.y);         // X[H-k] = conj(E + F)
        }
    }
}

}  // namespace sap
