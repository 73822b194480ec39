// Host-side check of the radix-FFT building blocks of paper_2106_03452_b200/csrc/fft_core.cuh (compiled with g++, no GPU):
// every plan's stored order is a permutation (pos2freq / freq2pos inverse of each other) and the staged
// decimation-in-frequency transform followed by its decimation-in-time mirror reproduce a naive DFT and the input.
// Used by tests/test_host_logic.py.  Not part of the product.
#include <cmath>
#include <cstdio>
#include <vector>
#include "fft_core.cuh"

using namespace sap;

template <int N> static int check() {
    int bad = 0;
    for (int p = 0; p < N; ++p)
        if (freq2pos<N>(pos2freq<N>(p)) != p || pos2freq<N>(p) < 0 || pos2freq<N>(p) >= N) ++bad;
    std::vector<float2> tw(N), x(N), s(N);
    for (int t = 0; t < N; ++t) {
        const double a = -2.0 * M_PI * t / N;
        tw[t] = make_float2((float)cos(a), (float)sin(a));
        x[t] = make_float2((float)sin(0.37 * t + 0.1) + (t % 7) * 0.25f, (float)cos(1.3 * t) - (t % 5) * 0.5f);
    }
    s = x;
    // forward: stages 0..NS-1 on one line (element stride 1), single "thread"
    fft_stage<N, 0, false, N, false>(s.data(), 1, N, 1, tw.data(), 0, 1);
    if (Plan<N>::NS > 1) fft_stage<N, (Plan<N>::NS > 1 ? 1 : 0), false, N, false>(s.data(), 1, N, 1, tw.data(), 0, 1);
    if (Plan<N>::NS > 2) fft_stage<N, (Plan<N>::NS > 2 ? 2 : 0), false, N, false>(s.data(), 1, N, 1, tw.data(), 0, 1);
    double err = 0, ref = 0;
    for (int p = 0; p < N; ++p) {
        const int k = pos2freq<N>(p);
        double re = 0, im = 0;
        for (int j = 0; j < N; ++j) {
            const double a = -2.0 * M_PI * (double)((long long)k * j % N) / N;
            re += x[j].x * cos(a) - x[j].y * sin(a);
            im += x[j].x * sin(a) + x[j].y * cos(a);
        }
        err = fmax(err, fmax(fabs(re - s[p].x), fabs(im - s[p].y)));
        ref = fmax(ref, fmax(fabs(re), fabs(im)));
    }
    if (err > 2e-5 * ref) { printf("N=%d forward err %.3e (ref %.3e)\n", N, err, ref); ++bad; }
    // inverse mirror: stages NS-1..0
    if (Plan<N>::NS > 2) fft_stage<N, (Plan<N>::NS > 2 ? 2 : 0), true, N, false>(s.data(), 1, N, 1, tw.data(), 0, 1);
    if (Plan<N>::NS > 1) fft_stage<N, (Plan<N>::NS > 1 ? 1 : 0), true, N, false>(s.data(), 1, N, 1, tw.data(), 0, 1);
    fft_stage<N, 0, true, N, false>(s.data(), 1, N, 1, tw.data(), 0, 1);
    double e2 = 0, r2 = 0;
    for (int j = 0; j < N; ++j) {
        e2 = fmax(e2, fmax(fabs(s[j].x / N - x[j].x), fabs(s[j].y / N - x[j].y)));
        r2 = fmax(r2, fmax(fabs(x[j].x), fabs(x[j].y)));
    }
    if (e2 > 2e-5 * r2) { printf("N=%d round-trip err %.3e\n", N, e2); ++bad; }
    // Hermitian pair formulas: c2r_pair undoes r2c_pair
    for (int k = 1; k < N / 4; ++k) {
        float2 a = x[k], b = x[N / 2 - k], a0 = a, b0 = b;
        r2c_pair(a, b, tw[k]);
        c2r_pair(a, b, tw[k]);
        if (fabs(a.x - a0.x) + fabs(a.y - a0.y) + fabs(b.x - b0.x) + fabs(b.y - b0.y) > 1e-4) { printf("N=%d pair k=%d\n", N, k); ++bad; }
    }
    return bad;
}

int main() {
    int bad = check<16>() + check<32>() + check<64>() + check<128>() + check<256>() + check<512>();
    printf(bad ? "FAIL %d\n" : "OK\n", bad);
    return bad ? 1 : 0;
}
