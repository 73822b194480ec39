// spectral.cuh -- the spectral multiplier of the solve (Eq.3 / Eq.16) and the tile geometry
// of the strided-axis passes (ring_pass.cuh).
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
// 1 / x for x = |u|^2, an exact integer >= 1: the approximate reciprocal (one MUFU, 1 ulp) -- __frcp_rn brings a
// Newton step and a denormal slow path whose branches cost 8% of the solve kernel's instructions
SAP_HD float fast_rcp(float x) {
#ifdef __CUDA_ARCH__
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
#else
    return 1.f / x;
#endif
}
// f = cs g / q from three table entries (0 at DC); branch-free
SAP_HD float mult_f(const float4& ex, const float4& ey, const float4& ez, float cs) {
    const float q = ex.y + ey.y + ez.y;
    const float f = cs * (ex.z * ey.z) * ez.z * fast_rcp(q);
    return (q > 0.f) ? f : 0.f;
}
// the same with the column part (y and z slots: fixed for all butterflies of a thread) folded once per tile
struct MultCol {
    float qyz, gyz;   // |u_y|^2 + |u_z|^2,  cs g_y g_z
};
SAP_HD MultCol mult_col(const float4& ey, const float4& ez, float cs) { return MultCol{ey.y + ez.y, cs * ey.z * ez.z}; }
SAP_HD float mult_fc(const float4& ex, const MultCol& c) {
    const float q = ex.y + c.qyz;
    const float f = c.gyz * ex.z * fast_rcp(q);
    return (q > 0.f) ? f : 0.f;
}

// MODE_FWD3 / MODE_INV3: the y pass of the three field channels when it is a kernel of its own (N >= 256).  The y and z
// channels travel between the y pass and the x pass as ONE spectrum (u = h_y v~_y + h_z v~_z forward; B = the inverse x
// transform of -i f Gbar'~ backward, from which vbar_y and vbar_z differ only by factors that commute with the
// remaining transforms), which saves one spectrum write and one read in each direction.
enum { MODE_FWD = 0, MODE_INV = 1, MODE_SOLVE = 2, MODE_ADJ = 3, MODE_FWD3 = 4, MODE_INV3 = 5 };

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

}  // namespace sap
