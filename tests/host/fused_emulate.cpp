// Host emulation of the fused (latency-path) forward and backward of paper_2106_03452_b200/csrc/fused_small.cuh
// (compiled with g++, no GPU).  The phase bodies of that file are __host__ __device__ templates on a small context;
// here every "CTA" is run to the next grid barrier in turn, single-threaded, each with its own persistent
// "shared memory", so that the tile / slot / swizzle / bin index logic of the whole path is exercised end to end.
// Reads  : argv[1] = binary input  {int N, B, P; float sigma; float pts[B][P][3], nrm[B][P][3], G[B][N^3]}
// Writes : argv[2] = binary output {float chi[B][N^3], stats[B][4], gp[B][P][3], gn[B][P][3]}
// Used by tests/test_host_logic.py, which compares the output with the float64 oracle.  Not part of the product and
// not the oracle: it shares the product's arithmetic on purpose.
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <vector>
#include "fused_small.cuh"

using namespace sap;

struct HostCtx {
    int tid = 0, nthr = 1;
    void sync() const {}
    void atomic_add(int* p, int v) const { *p += v; }
    int atomic_inc(int* p) const { return (*p)++; }
    void gatomic_add(float* p, float v) const { *p += v; }
    void gatomic_add(double* p, double v) const { *p += v; }
    double gload(const double* p) const { return *p; }
    float gload(const float* p) const { return *p; }
    float block_sum(float x, float*) const { return x; }
    void stamp(int) const {}
    float block_sum_all(float x, float*) const { return x; }
};

template <int N> static int run(int B, int P, float sigma, const float* pts, const float* nrm, const float* G, FILE* fo) {
    using C = FusedCfg<N>;
    constexpr int H = N / 2;
    const int ncta = 148;
    if (B * N > ncta || B > C::MAXB) { fprintf(stderr, "batch too large for the fused path\n"); return 2; }
    const size_t V = (size_t)N * N * N, SP = (size_t)N * N * H, QP = (size_t)N * N;
    std::vector<float> chi(B * V), gp((size_t)B * P * 3, 7.f), gn((size_t)B * P * 3, 7.f), stats(B * 4), bw(B * 4);
    std::vector<float4> spts((size_t)B * P), snrm((size_t)B * P), ftab(N + H + 1);
    std::vector<int> bin_start(B * (N + 1)), hist((size_t)B * ncta * N);
    std::vector<float2> S3(B * 3 * SP), Q3(B * 3 * QP), S1(B * SP), Q1(B * QP), tw(N);
    std::vector<double> acc(2 * B, 0.0);
    std::vector<unsigned> sync(4, 0);
    for (int t = 0; t < N; ++t) {
        const double a = -2.0 * M_PI * t / N;
        tw[t] = make_float2((float)cos(a), (float)sin(a));
    }
    const float cg = 2.f * sigma * sigma / ((float)N * (float)N);
    for (int i = 0; i < N; ++i) ftab[i] = freq_entry_n<N>(i, cg);
    for (int i = 0; i <= H; ++i) ftab[N + i] = freq_entry_z<N>(i, cg);
    FusedParams p{};
    p.pts = pts; p.nrm = nrm; p.chi = chi.data(); p.G = G; p.gp = gp.data(); p.gn = gn.data(); p.P = P; p.B = B;
    p.spts = spts.data(); p.snrm = snrm.data(); p.bin_start = bin_start.data(); p.hist = hist.data();
    p.S3 = S3.data(); p.Q3 = Q3.data(); p.S1 = S1.data(); p.Q1 = Q1.data(); p.tw = tw.data(); p.ftab = ftab.data();
    p.acc = acc.data(); p.stats = stats.data(); p.bw = bw.data(); p.sync = sync.data(); p.stamps = nullptr;
    p.cs = (float)((2.0 / ((double)N * N * N)) / (-2.0 * M_PI));
    std::vector<std::vector<unsigned char>> smem(ncta, std::vector<unsigned char>(C::BYTES + 128));
    auto sm_of = [&](int cta) {
        unsigned char* b = smem[cta].data();
        b += (128 - ((size_t)b & 127)) & 127;
        return FusedSmem<N>(b);
    };
    HostCtx ctx;
    const int per = x_tiles<N>();
    // ---- forward ----
    for (int c = 0; c < ncta; ++c) { auto sm = sm_of(c); fused_tables<N>(ctx, p, sm); }
    for (int c = 0; c < ncta; ++c) { auto sm = sm_of(c); fwd_hist<N>(ctx, p, sm, c, ncta); }
    for (int c = 0; c < ncta; ++c) { auto sm = sm_of(c); fwd_scatter<N>(ctx, p, sm, c, ncta); }
    for (int c = 0; c < ncta; ++c) { auto sm = sm_of(c); for (int t = c; t < B * N; t += ncta) fwd_splat_zy<N>(ctx, p, sm, t); }
    for (int c = 0; c < ncta; ++c) {
        auto sm = sm_of(c);
        for (int g = 0; g < C::XNG; ++g) {
            float2* b0 = sm.big + (size_t)g * 2 * C::XBUF;
            for (int T = c * C::XNG + g; T < B * per; T += ncta * C::XNG) fwd_x_solve<N>(ctx, p, sm, b0, b0 + C::XBUF, T / per, T % per);
        }
    }
    for (int c = 0; c < B * N; ++c) { auto sm = sm_of(c); fwd_inv_mean<N>(ctx, p, sm, c); }
    for (int c = 0; c < B * N; ++c) { auto sm = sm_of(c); fwd_scale_store<N>(ctx, p, sm, c); }
    for (auto& a : acc) a = 0.0;
    // ---- backward ----
    for (int c = 0; c < ncta; ++c) { auto sm = sm_of(c); if (c < B * N) bwd_load_reduce<N>(ctx, p, sm, c); bwd_zero_grads(ctx, p, c, ncta); }
    for (int c = 0; c < B * N; ++c) { auto sm = sm_of(c); bwd_gbar_zy<N>(ctx, p, sm, c); }
    for (int c = 0; c < ncta; ++c) {
        auto sm = sm_of(c);
        for (int g = 0; g < C::XNG; ++g) {
            float2* b0 = sm.big + (size_t)g * 2 * C::XBUF;
            for (int T = c * C::XNG + g; T < B * per; T += ncta * C::XNG) bwd_x_adj<N>(ctx, p, sm, b0, b0 + C::XBUF, T / per, T % per);
        }
    }
    for (int c = 0; c < ncta; ++c) { auto sm = sm_of(c); for (int t = c; t < B * N; t += ncta) bwd_inv_gather<N>(ctx, p, sm, t); }
    fwrite(chi.data(), 4, chi.size(), fo);
    fwrite(stats.data(), 4, stats.size(), fo);
    fwrite(gp.data(), 4, gp.size(), fo);
    fwrite(gn.data(), 4, gn.size(), fo);
    return 0;
}

int main(int argc, char** argv) {
    if (argc < 3) return 1;
    FILE* fi = fopen(argv[1], "rb");
    if (!fi) return 1;
    int hdr[3];
    float sigma;
    if (fread(hdr, 4, 3, fi) != 3 || fread(&sigma, 4, 1, fi) != 1) return 1;
    const int N = hdr[0], B = hdr[1], P = hdr[2];
    const size_t V = (size_t)N * N * N;
    std::vector<float> pts((size_t)B * P * 3), nrm((size_t)B * P * 3), G(B * V);
    if (fread(pts.data(), 4, pts.size(), fi) != pts.size() || fread(nrm.data(), 4, nrm.size(), fi) != nrm.size() ||
        fread(G.data(), 4, G.size(), fi) != G.size()) return 1;
    fclose(fi);
    FILE* fo = fopen(argv[2], "wb");
    if (!fo) return 1;
    int rc = 2;
    if (N == 32) rc = run<32>(B, P, sigma, pts.data(), nrm.data(), G.data(), fo);
    else if (N == 64) rc = run<64>(B, P, sigma, pts.data(), nrm.data(), G.data(), fo);
    else if (N == 128) rc = run<128>(B, P, sigma, pts.data(), nrm.data(), G.data(), fo);
    fclose(fo);
    if (rc == 0) printf("OK\n");
    return rc;
}
