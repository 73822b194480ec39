/*
 * dpsr_oracle.c -- float64 CPU ORACLE for the DPSR layer of "Shape As Points"
 * (arXiv 2106.03452).  Citations "PAPER.md:Lnnn" refer to /root/reference/PAPER.md.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code,
 * header, table or constant generator with the CUDA path under paper_2106_03452_b200/.
 *
 * It follows the algorithm step by step in the paper's order (rasterise -> FFT ->
 * spectral solve -> IFFT -> normalise), with the FFT replaced by its plain definition
 * (a naive separable DFT, O(N^4) per 3-D transform; itself pinned in tests against the
 * O(N^6) triple sum `oracle_dft3_direct` and against closed forms).  No blocking, no
 * fusion, no symmetry tricks: every 3-D transform is a full complex one.  OpenMP only
 * parallelises over independent lines/planes; each output element is still the plain
 * sequential sum over j = 0..N-1.
 *
 * Readings of the paper taken here:
 *   R1  unit cube [0,1)^3, origin 0, voxel 1/N, vertex j at j/N, periodic wrap.
 *   R2  neighbours floor(t), floor(t)+1 with weights (1-f, f).
 *   R3  derivative multiplier zeroed at the Nyquist index k_a = N/2 (|u|^2 and g keep (N/2)^2).
 *   R4  chi~(0) = 0.
 *   R5  shift by the point mean first, then scale by m/|chi'[0,0,0] - mu|.
 *   R6  Eq.3 literally, integer frequencies: g = exp(-2 sigma^2 |u|^2 / N^2).
 *   R8  forward DFT unnormalised, inverse 1/N^3.
 *
 * Pins: tests/test_oracle_*.py (-m "not gpu").  Exact numerical values of chi for the
 * paper's own data: PARITY UNPINNED -- the paper prints no worked numerical example
 * (only the closed forms / invariants in those tests and the definitions pin it).
 *
 * Layout everywhere: C order, z fastest: idx(jx,jy,jz) = (jx*N + jy)*N + jz.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include <stddef.h>

#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_PI 3.14159265358979323846264338327950288

static inline size_t idx3(int N, int jx, int jy, int jz) {
    return ((size_t)jx * N + jy) * N + jz;
}
static inline int wrap(int j, int N) {
    int r = j % N;
    return r < 0 ? r + N : r;
}

int oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ------------------------------------------------------------------------------------
 * Point rasterisation, Eq.10-11, readings R1/R2/R10.
 * t = c*N, j0 = floor(t), f = t - j0; the 8 neighbours (j0+d) mod N, d in {0,1}^3, get
 * weight prod_a (d_a ? f_a : 1-f_a).  v[ch][j] += w * n[ch];  W[j] += w  (W: the same
 * splat applied to the scalar 1; used by Eq.4's mean and by the backward).
 * points, normals: [P][3] double.  v: [3][N^3] (zeroed here).  W: [N^3] or NULL.
 * ---------------------------------------------------------------------------------- */
void oracle_splat(int N, long P, const double* points, const double* normals,
                  double* v, double* W) {
    size_t V = (size_t)N * N * N;
    memset(v, 0, 3 * V * sizeof(double));
    if (W) memset(W, 0, V * sizeof(double));
    for (long i = 0; i < P; ++i) {
        int j0[3];
        double f[3];
        for (int a = 0; a < 3; ++a) {
            double t = points[3 * i + a] * (double)N;
            double fl = floor(t);
            j0[a] = (int)fl;
            f[a] = t - fl;
        }
        for (int dx = 0; dx < 2; ++dx)
            for (int dy = 0; dy < 2; ++dy)
                for (int dz = 0; dz < 2; ++dz) {
                    double w = (dx ? f[0] : 1.0 - f[0]) * (dy ? f[1] : 1.0 - f[1]) *
                               (dz ? f[2] : 1.0 - f[2]);
                    size_t j = idx3(N, wrap(j0[0] + dx, N), wrap(j0[1] + dy, N),
                                    wrap(j0[2] + dz, N));
                    for (int ch = 0; ch < 3; ++ch) v[ch * V + j] += w * normals[3 * i + ch];
                    if (W) W[j] += w;
                }
    }
}

/* Trilinear sample of a scalar grid at the points with the splat's weights (R11):
 * out[i] = sum_corners w * grid[corner].  Eq.4 "chi'|x=c". */
void oracle_interp(int N, long P, const double* points, const double* grid, double* out) {
    for (long i = 0; i < P; ++i) {
        int j0[3];
        double f[3];
        for (int a = 0; a < 3; ++a) {
            double t = points[3 * i + a] * (double)N;
            double fl = floor(t);
            j0[a] = (int)fl;
            f[a] = t - fl;
        }
        double acc = 0.0;
        for (int dx = 0; dx < 2; ++dx)
            for (int dy = 0; dy < 2; ++dy)
                for (int dz = 0; dz < 2; ++dz) {
                    double w = (dx ? f[0] : 1.0 - f[0]) * (dy ? f[1] : 1.0 - f[1]) *
                               (dz ? f[2] : 1.0 - f[2]);
                    acc += w * grid[idx3(N, wrap(j0[0] + dx, N), wrap(j0[1] + dy, N),
                                         wrap(j0[2] + dz, N))];
                }
        out[i] = acc;
    }
}

/* ------------------------------------------------------------------------------------
 * Discrete Fourier transform, the discrete form of Eq.12/13, R8:
 *   sign = -1: out(k) =        sum_j in(j) exp(-2 pi i k.j / N)      (forward, unnormalised)
 *   sign = +1: out(k) = N^-3 * sum_j in(j) exp(+2 pi i k.j / N)      (inverse)
 * Separable: one naive O(N^2) DFT per line along x, then y, then z.
 * in_im may be NULL (real input).  All arrays [N^3].  Returns 0, or -1 on allocation failure.
 * ---------------------------------------------------------------------------------- */
static void twiddle_matrix(int N, int sign, double* wr, double* wi) {
    /* w[k][j] = exp(sign * 2 pi i * ((k*j) mod N) / N); the mod keeps the argument small. */
    for (int k = 0; k < N; ++k)
        for (int j = 0; j < N; ++j) {
            long m = ((long)k * j) % N;
            double ang = (double)sign * 2.0 * ORACLE_PI * (double)m / (double)N;
            wr[(size_t)k * N + j] = cos(ang);
            wi[(size_t)k * N + j] = sin(ang);
        }
}

int oracle_dft3(int N, const double* in_re, const double* in_im, double* out_re,
                double* out_im, int sign) {
    size_t V = (size_t)N * N * N;
    size_t NN = (size_t)N * N;
    double* wr = (double*)malloc(NN * sizeof(double));
    double* wi = (double*)malloc(NN * sizeof(double));
    double* ar = (double*)malloc(V * sizeof(double));
    double* ai = (double*)malloc(V * sizeof(double));
    double* br = (double*)malloc(V * sizeof(double));
    double* bi = (double*)malloc(V * sizeof(double));
    if (!wr || !wi || !ar || !ai || !br || !bi) {
        free(wr); free(wi); free(ar); free(ai); free(br); free(bi);
        return -1;
    }
    twiddle_matrix(N, sign, wr, wi);
    memcpy(ar, in_re, V * sizeof(double));
    if (in_im) memcpy(ai, in_im, V * sizeof(double));
    else memset(ai, 0, V * sizeof(double));

    /* axis x: b[kx][yz] = sum_jx w[kx][jx] * a[jx][yz]  (inner loop over the contiguous yz) */
#pragma omp parallel for schedule(static)
    for (int k = 0; k < N; ++k) {
        double* orr = br + (size_t)k * NN;
        double* oi = bi + (size_t)k * NN;
        for (size_t e = 0; e < NN; ++e) { orr[e] = 0.0; oi[e] = 0.0; }
        for (int j = 0; j < N; ++j) {
            double cr = wr[(size_t)k * N + j], ci = wi[(size_t)k * N + j];
            const double* xr = ar + (size_t)j * NN;
            const double* xi = ai + (size_t)j * NN;
            for (size_t e = 0; e < NN; ++e) {
                orr[e] += cr * xr[e] - ci * xi[e];
                oi[e] += cr * xi[e] + ci * xr[e];
            }
        }
    }
    /* axis y: a[x][ky][z] = sum_jy w[ky][jy] * b[x][jy][z] */
#pragma omp parallel for schedule(static) collapse(2)
    for (int x = 0; x < N; ++x)
        for (int k = 0; k < N; ++k) {
            double* orr = ar + ((size_t)x * N + k) * N;
            double* oi = ai + ((size_t)x * N + k) * N;
            for (int e = 0; e < N; ++e) { orr[e] = 0.0; oi[e] = 0.0; }
            for (int j = 0; j < N; ++j) {
                double cr = wr[(size_t)k * N + j], ci = wi[(size_t)k * N + j];
                const double* xr = br + ((size_t)x * N + j) * N;
                const double* xi = bi + ((size_t)x * N + j) * N;
                for (int e = 0; e < N; ++e) {
                    orr[e] += cr * xr[e] - ci * xi[e];
                    oi[e] += cr * xi[e] + ci * xr[e];
                }
            }
        }
    /* axis z: out[line][kz] = sum_jz w[jz][kz] * a[line][jz]   (w is symmetric: w[j][k] = w[k][j]) */
    double scale = (sign > 0) ? 1.0 / ((double)N * (double)N * (double)N) : 1.0;
#pragma omp parallel for schedule(static)
    for (size_t line = 0; line < NN; ++line) {
        double* orr = br + line * N;
        double* oi = bi + line * N;
        const double* xr = ar + line * N;
        const double* xi = ai + line * N;
        for (int k = 0; k < N; ++k) { orr[k] = 0.0; oi[k] = 0.0; }
        for (int j = 0; j < N; ++j) {
            const double* cr = wr + (size_t)j * N;
            const double* ci = wi + (size_t)j * N;
            double vr = xr[j], vi = xi[j];
            for (int k = 0; k < N; ++k) {
                orr[k] += cr[k] * vr - ci[k] * vi;
                oi[k] += cr[k] * vi + ci[k] * vr;
            }
        }
    }
    for (size_t e = 0; e < V; ++e) {
        out_re[e] = br[e] * scale;
        out_im[e] = bi[e] * scale;
    }
    free(wr); free(wi); free(ar); free(ai); free(br); free(bi);
    return 0;
}

/* The O(N^6) definition itself: a direct triple sum per output element, no separability.
 * Only for tiny N (8): pins oracle_dft3 in tests (north_star: "a direct O(N^6) DFT on 8^3"). */
void oracle_dft3_direct(int N, const double* in_re, const double* in_im, double* out_re,
                        double* out_im, int sign) {
    double scale = (sign > 0) ? 1.0 / ((double)N * (double)N * (double)N) : 1.0;
    for (int kx = 0; kx < N; ++kx)
        for (int ky = 0; ky < N; ++ky)
            for (int kz = 0; kz < N; ++kz) {
                double sr = 0.0, si = 0.0;
                for (int jx = 0; jx < N; ++jx)
                    for (int jy = 0; jy < N; ++jy)
                        for (int jz = 0; jz < N; ++jz) {
                            double ang = (double)sign * 2.0 * ORACLE_PI *
                                         (double)(kx * jx + ky * jy + kz * jz) / (double)N;
                            double c = cos(ang), s = sin(ang);
                            size_t j = idx3(N, jx, jy, jz);
                            double xr = in_re[j], xi = in_im ? in_im[j] : 0.0;
                            sr += c * xr - s * xi;
                            si += c * xi + s * xr;
                        }
                out_re[idx3(N, kx, ky, kz)] = sr * scale;
                out_im[idx3(N, kx, ky, kz)] = si * scale;
            }
}

/* ------------------------------------------------------------------------------------
 * Spectral multiplier of Eq.3 / Eq.14-16, readings R3/R4/R6/R7:
 *   u_a = k_a if k_a < N/2 else k_a - N           (integer signed frequency)
 *   q   = u_x^2 + u_y^2 + u_z^2                    (|u|^2; Nyquist counts (N/2)^2)
 *   g   = exp(-2 sigma^2 q / N^2)
 *   uh_a = u_a, except uh_a = 0 where k_a = N/2    (R3)
 *   M_c(k) = g * i * uh_c / (-2 pi q),  M_c(0) = 0 (R4)
 * Returns the REAL number m_c with M_c = i * m_c, i.e. m_c = g * uh_c / (-2 pi q).
 * ---------------------------------------------------------------------------------- */
static inline void multiplier(int N, double sigma, int kx, int ky, int kz, double m[3]) {
    int k[3] = {kx, ky, kz};
    double u[3], uh[3], q = 0.0;
    for (int a = 0; a < 3; ++a) {
        u[a] = (k[a] < N / 2) ? (double)k[a] : (double)(k[a] - N);
        uh[a] = (2 * k[a] == N) ? 0.0 : u[a];
        q += u[a] * u[a];
    }
    if (q == 0.0) { m[0] = m[1] = m[2] = 0.0; return; }
    double g = exp(-2.0 * sigma * sigma * q / ((double)N * (double)N));
    for (int a = 0; a < 3; ++a) m[a] = g * uh[a] / (-2.0 * ORACLE_PI * q);
}

void oracle_multiplier(int N, double sigma, int kx, int ky, int kz, double* m3) {
    multiplier(N, sigma, kx, ky, kz, m3);
}

/* chi~(k) = sum_c M_c(k) v~_c(k) = i * sum_c m_c v~_c   (Eq.3).  vt_*: [3][N^3]. */
void oracle_spectral_solve(int N, double sigma, const double* vt_re, const double* vt_im,
                           double* ct_re, double* ct_im) {
    size_t V = (size_t)N * N * N;
#pragma omp parallel for schedule(static)
    for (int kx = 0; kx < N; ++kx)
        for (int ky = 0; ky < N; ++ky)
            for (int kz = 0; kz < N; ++kz) {
                double m[3];
                multiplier(N, sigma, kx, ky, kz, m);
                size_t k = idx3(N, kx, ky, kz);
                double dr = 0.0, di = 0.0; /* d = sum_c m_c * v~_c */
                for (int c = 0; c < 3; ++c) {
                    dr += m[c] * vt_re[c * V + k];
                    di += m[c] * vt_im[c * V + k];
                }
                ct_re[k] = -di; /* i * (dr + i di) = -di + i dr */
                ct_im[k] = dr;
            }
}

/* Transposed multiplier (backward): vbar~_c(k) = conj(M_c(k)) * gt(k) = -i m_c * gt(k). */
void oracle_spectral_adjoint(int N, double sigma, const double* gt_re, const double* gt_im,
                             double* vb_re, double* vb_im) {
    size_t V = (size_t)N * N * N;
#pragma omp parallel for schedule(static)
    for (int kx = 0; kx < N; ++kx)
        for (int ky = 0; ky < N; ++ky)
            for (int kz = 0; kz < N; ++kz) {
                double m[3];
                multiplier(N, sigma, kx, ky, kz, m);
                size_t k = idx3(N, kx, ky, kz);
                for (int c = 0; c < 3; ++c) {
                    /* -i m (gr + i gi) = m gi - i m gr */
                    vb_re[c * V + k] = m[c] * gt_im[k];
                    vb_im[c * V + k] = -m[c] * gt_re[k];
                }
            }
}

/* ------------------------------------------------------------------------------------
 * DPSR forward, Eq.2-4 == Eq.10-18 of Suppl. A (L341-L388).
 * points, normals [P][3] double (callers pass the fp32-rounded values promoted to double).
 * Outputs (any may be NULL except chi): chi [N^3]; chi_prime [N^3]; v [3][N^3]; W [N^3];
 * stats[4] = {mu, a, s, max|Im IDFT| / max|Re IDFT|}.
 * Returns 0 ok, -1 allocation failure, -2 bad argument.
 * ---------------------------------------------------------------------------------- */
int oracle_dpsr_forward(int N, double sigma, long P, const double* points,
                        const double* normals, double* chi, double* chi_prime, double* v_out,
                        double* W_out, double* stats) {
    if (N <= 0 || (N & 1) || P <= 0 || !points || !normals || !chi) return -2;
    const double m_scale = 0.5; /* "we fix the overall scale to m = 0.5" */
    size_t V = (size_t)N * N * N;
    int rc = -1;
    double* v = (double*)malloc(3 * V * sizeof(double));
    double* W = (double*)malloc(V * sizeof(double));
    double* vt_re = (double*)malloc(3 * V * sizeof(double));
    double* vt_im = (double*)malloc(3 * V * sizeof(double));
    double* ct_re = (double*)malloc(V * sizeof(double));
    double* ct_im = (double*)malloc(V * sizeof(double));
    double* cp_re = (double*)malloc(V * sizeof(double));
    double* cp_im = (double*)malloc(V * sizeof(double));
    double* samp = (double*)malloc((size_t)P * sizeof(double));
    if (!v || !W || !vt_re || !vt_im || !ct_re || !ct_im || !cp_re || !cp_im || !samp) goto done;

    /* 1. rasterise (Eq.10-11) */
    oracle_splat(N, P, points, normals, v, W);
    /* 2. v~ = FFT(v) per channel (Eq.12) */
    for (int c = 0; c < 3; ++c)
        if (oracle_dft3(N, v + c * V, NULL, vt_re + c * V, vt_im + c * V, -1)) goto done;
    /* 3. chi~ = g (i u . v~) / (-2 pi |u|^2) (Eq.3 / Eq.16) */
    oracle_spectral_solve(N, sigma, vt_re, vt_im, ct_re, ct_im);
    /* 4. chi' = IFFT(chi~) (Eq.17); keep the real part, report the imaginary residue */
    if (oracle_dft3(N, ct_re, ct_im, cp_re, cp_im, +1)) goto done;
    double max_re = 0.0, max_im = 0.0;
    for (size_t e = 0; e < V; ++e) {
        if (fabs(cp_re[e]) > max_re) max_re = fabs(cp_re[e]);
        if (fabs(cp_im[e]) > max_im) max_im = fabs(cp_im[e]);
    }
    /* 5. normalise (Eq.4 / Eq.18, reading R5) */
    oracle_interp(N, P, points, cp_re, samp);
    double mu = 0.0;
    for (long i = 0; i < P; ++i) mu += samp[i];
    mu /= (double)P;
    double a = cp_re[0] - mu;          /* chi'|x=0 after the shift */
    double s = m_scale / fabs(a);
    for (size_t e = 0; e < V; ++e) chi[e] = s * (cp_re[e] - mu);

    if (chi_prime) memcpy(chi_prime, cp_re, V * sizeof(double));
    if (v_out) memcpy(v_out, v, 3 * V * sizeof(double));
    if (W_out) memcpy(W_out, W, V * sizeof(double));
    if (stats) {
        stats[0] = mu; stats[1] = a; stats[2] = s;
        stats[3] = (max_re > 0.0) ? max_im / max_re : 0.0;
    }
    rc = 0;
done:
    free(v); free(W); free(vt_re); free(vt_im); free(ct_re); free(ct_im);
    free(cp_re); free(cp_im); free(samp);
    return rc;
}

/* ------------------------------------------------------------------------------------
 * DPSR backward: the exact adjoint of the forward above ("differentiable", PAPER.md:L17;
 * third factor of Eq.5).  The paper gives no formulas; derivation in DESIGN.md
 * ("Backward") and SURVEY.md 8(c):
 *   S0 = sum G, S1 = sum G chi, beta = S1/a - s S0
 *   Gbar' = s G + (beta/P) W - (S1/a) delta_{j,0}                (= dL/dchi')
 *   vbar_c = Re IDFT( conj(M_c) DFT(Gbar') ) * N^3 ... see note  (= dL/dv_c)
 *   dL/dn_i[c] = sum_corners w vbar_c[corner]
 *   dL/dc_i[a] = sum_corners (dw/dc_a) ( n_i . vbar[corner] + (beta/P) chi'[corner] )
 * Note on constants: forward chi' = IDFT(M . DFT(v)) with IDFT carrying 1/N^3.  Its transpose is
 * vbar = DFT^T( M^T IDFT^T Gbar' ) = conj-free: DFT and IDFT matrices are symmetric, so
 * vbar_c = DFT( M_c . IDFT(Gbar') ), which equals IDFT( M_c(-k) . DFT(Gbar') ) after the index
 * flip k -> -k, and M_c(-k) = -M_c(k) = conj(M_c(k)).  So: vbar_c = IDFT( conj(M_c) DFT(Gbar') ).
 * Inputs: chi_prime, W, stats = {mu,a,s} from oracle_dpsr_forward; G [N^3].
 * Outputs: grad_points, grad_normals [P][3]; optional gbar [N^3], vbar [3][N^3].
 * ---------------------------------------------------------------------------------- */
int oracle_dpsr_backward(int N, double sigma, long P, const double* points,
                         const double* normals, const double* chi_prime, const double* W,
                         const double* stats, const double* G, double* grad_points,
                         double* grad_normals, double* gbar_out, double* vbar_out) {
    if (N <= 0 || (N & 1) || P <= 0 || !points || !normals || !chi_prime || !W || !stats || !G ||
        !grad_points || !grad_normals)
        return -2;
    size_t V = (size_t)N * N * N;
    double mu = stats[0], a = stats[1], s = stats[2];
    int rc = -1;
    double* gbar = (double*)malloc(V * sizeof(double));
    double* gt_re = (double*)malloc(V * sizeof(double));
    double* gt_im = (double*)malloc(V * sizeof(double));
    double* vb_re = (double*)malloc(3 * V * sizeof(double));
    double* vb_im = (double*)malloc(3 * V * sizeof(double));
    double* vbar = (double*)malloc(3 * V * sizeof(double));
    double* tmp_im = (double*)malloc(V * sizeof(double));
    if (!gbar || !gt_re || !gt_im || !vb_re || !vb_im || !vbar || !tmp_im) goto done;

    double S0 = 0.0, S1 = 0.0;
    for (size_t e = 0; e < V; ++e) {
        double chi = s * (chi_prime[e] - mu);
        S0 += G[e];
        S1 += G[e] * chi;
    }
    double beta = S1 / a - s * S0;
    for (size_t e = 0; e < V; ++e) gbar[e] = s * G[e] + (beta / (double)P) * W[e];
    gbar[0] -= S1 / a;

    if (oracle_dft3(N, gbar, NULL, gt_re, gt_im, -1)) goto done;
    oracle_spectral_adjoint(N, sigma, gt_re, gt_im, vb_re, vb_im);
    for (int c = 0; c < 3; ++c)
        if (oracle_dft3(N, vb_re + c * V, vb_im + c * V, vbar + c * V, tmp_im, +1)) goto done;

    for (long i = 0; i < P; ++i) {
        int j0[3];
        double f[3];
        for (int ax = 0; ax < 3; ++ax) {
            double t = points[3 * i + ax] * (double)N;
            double fl = floor(t);
            j0[ax] = (int)fl;
            f[ax] = t - fl;
        }
        double gn[3] = {0, 0, 0}, gc[3] = {0, 0, 0};
        for (int dx = 0; dx < 2; ++dx)
            for (int dy = 0; dy < 2; ++dy)
                for (int dz = 0; dz < 2; ++dz) {
                    double wx = dx ? f[0] : 1.0 - f[0];
                    double wy = dy ? f[1] : 1.0 - f[1];
                    double wz = dz ? f[2] : 1.0 - f[2];
                    size_t j = idx3(N, wrap(j0[0] + dx, N), wrap(j0[1] + dy, N),
                                    wrap(j0[2] + dz, N));
                    double w = wx * wy * wz;
                    double dot = 0.0;
                    for (int c = 0; c < 3; ++c) {
                        gn[c] += w * vbar[c * V + j];
                        dot += normals[3 * i + c] * vbar[c * V + j];
                    }
                    double val = dot + (beta / (double)P) * chi_prime[j];
                    /* dw/dc_a = N * (d_a ? +1 : -1) * prod_{b != a} w_b */
                    gc[0] += (double)N * (dx ? 1.0 : -1.0) * wy * wz * val;
                    gc[1] += (double)N * (dy ? 1.0 : -1.0) * wx * wz * val;
                    gc[2] += (double)N * (dz ? 1.0 : -1.0) * wx * wy * val;
                }
        for (int c = 0; c < 3; ++c) {
            grad_normals[3 * i + c] = gn[c];
            grad_points[3 * i + c] = gc[c];
        }
    }
    if (gbar_out) memcpy(gbar_out, gbar, V * sizeof(double));
    if (vbar_out) memcpy(vbar_out, vbar, 3 * V * sizeof(double));
    rc = 0;
done:
    free(gbar); free(gt_re); free(gt_im); free(vb_re); free(vb_im); free(vbar); free(tmp_im);
    return rc;
}

/* ------------------------------------------------------------------------------------
 * One spectral coefficient of chi' straight from the points, without any grid:
 *   v~_c(k) = sum_i n_i[c] sum_corners w exp(-2 pi i k.(j0+d)/N)        (Eq.10-12)
 *   chi~(k) = i sum_c m_c(k) v~_c(k)                                     (Eq.3)
 * O(8P) per frequency.  Used for parity at sizes where the O(N^4) DFT is too slow
 * (512^3): the test transforms the GPU's chi at sampled k and compares with s * chi~(k).
 * out[2] = {Re, Im}.
 * ---------------------------------------------------------------------------------- */
void oracle_chi_tilde_at(int N, double sigma, long P, const double* points,
                         const double* normals, int kx, int ky, int kz, double* out) {
    double vt_re[3] = {0, 0, 0}, vt_im[3] = {0, 0, 0};
    for (long i = 0; i < P; ++i) {
        int j0[3];
        double f[3];
        for (int a = 0; a < 3; ++a) {
            double t = points[3 * i + a] * (double)N;
            double fl = floor(t);
            j0[a] = (int)fl;
            f[a] = t - fl;
        }
        double er = 0.0, ei = 0.0;
        for (int dx = 0; dx < 2; ++dx)
            for (int dy = 0; dy < 2; ++dy)
                for (int dz = 0; dz < 2; ++dz) {
                    double w = (dx ? f[0] : 1.0 - f[0]) * (dy ? f[1] : 1.0 - f[1]) *
                               (dz ? f[2] : 1.0 - f[2]);
                    long ph = (long)kx * wrap(j0[0] + dx, N) + (long)ky * wrap(j0[1] + dy, N) +
                              (long)kz * wrap(j0[2] + dz, N);
                    double ang = -2.0 * ORACLE_PI * (double)(ph % N) / (double)N;
                    er += w * cos(ang);
                    ei += w * sin(ang);
                }
        for (int c = 0; c < 3; ++c) {
            vt_re[c] += normals[3 * i + c] * er;
            vt_im[c] += normals[3 * i + c] * ei;
        }
    }
    double m[3];
    multiplier(N, sigma, kx, ky, kz, m);
    double dr = 0.0, di = 0.0;
    for (int c = 0; c < 3; ++c) { dr += m[c] * vt_re[c]; di += m[c] * vt_im[c]; }
    out[0] = -di;
    out[1] = dr;
}
