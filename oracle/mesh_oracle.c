/*
 * mesh_oracle.c -- float64 CPU ORACLE for the mesh side of the optimisation-based pipeline of "Shape As Points"
 * (arXiv 2106.03452, Sec.3.2): Marching Cubes on the indicator grid, the surrogate gradient of
 * Eq.6 and the bi-directional L2 Chamfer distance.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT (same rules as dpsr_oracle.c): only tests/, smoke() and bench.py's
 * cpu_baseline legs may load it; it shares no code, header or table with the CUDA path.  Plain loops, float64,
 * single-threaded.
 *
 * Readings of the paper taken here (M1-M6; the paper gives no formulas for this part and calls
 * a library for Marching Cubes, footnote PAPER.md:L248):
 *   M1  level set chi = 0; a node is INSIDE iff chi < 0 (R9: outward normals give chi < 0 inside); cells are the
 *       (N-1)^3 cubes between nodes, no periodic wrap for the mesh.
 *   M2  one vertex per grid edge whose end nodes differ in INSIDE, at the linear zero crossing
 *       p = (j + t e_a) / N, t = chi0 / (chi0 - chi1).
 *   M3  triangulation of a cube by RULE, not by a copied table: on every cube face the crossed face-edges are joined
 *       pairwise (two crossed edges: one segment; four -- the ambiguous face -- : the two INSIDE corners are cut off
 *       separately); the segments of the six faces close into loops; a loop is oriented so that its normal points to
 *       OUTSIDE (increasing chi), rotated to start at its smallest cube-edge id, and fan-triangulated from that
 *       vertex; loops are ordered by their smallest edge id.  The face rule depends on the face's four corner signs
 *       only, so neighbouring cubes agree and the mesh is watertight.
 *   M4  n_mesh of a vertex = normalised gradient of chi at the vertex: central differences (periodic, like chi
 *       itself) at the two end nodes of its edge, linearly interpolated with t.  Points to increasing chi.
 *   M5  Eq.6, dp_mesh/dchi = -n_mesh, with "chi at p_mesh" the trilinear interpolant of the grid (R11): a vertex
 *       sits on a grid edge, so  G[node0] += (1-t) g_v,  G[node1] += t g_v,  g_v = -(dL/dp_v . n_v).
 *   M6  Chamfer: L = mean_i min_k |a_i - b_k|^2 + mean_k min_i |b_k - a_i|^2 (squared L2, both directions, first index
 *       wins a tie); the mesh samples are the mesh vertices.
 *
 * Cube conventions: corner c has offsets (c & 1, (c >> 1) & 1, (c >> 2) & 1) along (x, y, z).  Cube edge
 * e = 4 a + k runs along axis a; k = u + 2 v with (u, v) the offsets along the two OTHER axes in increasing axis order.
 * Grid layout: C order, z fastest: node(jx,jy,jz) = (jx*N + jy)*N + jz.
 *
 * Pins: tests/test_oracle_mesh.py (-m "not gpu"): a linear field reproduces its plane exactly; sphere / torus: closed
 * oriented 2-manifold, Euler characteristic 2 / 0, vertices within O(h^2) of the surface, enclosed volume; every one of
 * the 256 sign configurations embedded in a grid gives a closed surface; Chamfer against hand-computed values and
 * finite differences; Eq.6 against a hand-built single-vertex case.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>

/* ---- cube tables, derived from the rule M3 ---------------------------------------------------------------------- */
static void corner_off(int c, int* o) { o[0] = c & 1; o[1] = (c >> 1) & 1; o[2] = (c >> 2) & 1; }
static int corner_id(const int* o) { return o[0] | (o[1] << 1) | (o[2] << 2); }
static void other_axes(int a, int* b1, int* b2) { *b1 = (a == 0) ? 1 : 0; *b2 = (a == 2) ? 1 : 2; }
/* end corners of cube edge e */
static void edge_ends(int e, int* c0, int* c1) {
    int a = e / 4, k = e % 4, b1, b2, o[3];
    other_axes(a, &b1, &b2);
    o[a] = 0; o[b1] = k & 1; o[b2] = k >> 1;
    *c0 = corner_id(o);
    o[a] = 1;
    *c1 = corner_id(o);
}
/* cube edge joining two adjacent corners */
static int edge_between(int ca, int cb) {
    int oa[3], ob[3], a = -1, b1, b2;
    corner_off(ca, oa); corner_off(cb, ob);
    for (int d = 0; d < 3; ++d) if (oa[d] != ob[d]) a = d;
    other_axes(a, &b1, &b2);
    return 4 * a + (oa[b1] | (oa[b2] << 1));
}

#define MC_MAX_TRI 12
/* triangles of sign configuration `cfg` (bit c set: corner c INSIDE) as triples of cube-edge ids; returns their number */
static int cube_case(int cfg, int tris[MC_MAX_TRI][3]) {
    int nb[12][2], deg[12], crossed[12];
    for (int e = 0; e < 12; ++e) {
        int c0, c1;
        edge_ends(e, &c0, &c1);
        crossed[e] = ((cfg >> c0) & 1) != ((cfg >> c1) & 1);
        deg[e] = 0;
    }
    /* faces: normal axis a, side s; corner cycle (0,0),(1,0),(1,1),(0,1) in the (b1,b2) plane */
    for (int a = 0; a < 3; ++a)
        for (int s = 0; s < 2; ++s) {
            int b1, b2, cyc[4], fe[4], in[4], ncross = 0;
            static const int cu[4] = {0, 1, 1, 0}, cv[4] = {0, 0, 1, 1};
            other_axes(a, &b1, &b2);
            for (int i = 0; i < 4; ++i) {
                int o[3];
                o[a] = s; o[b1] = cu[i]; o[b2] = cv[i];
                cyc[i] = corner_id(o);
                in[i] = (cfg >> cyc[i]) & 1;
            }
            for (int i = 0; i < 4; ++i) {
                fe[i] = edge_between(cyc[i], cyc[(i + 1) & 3]);   /* face-edge i joins corners i and i+1 */
                ncross += in[i] != in[(i + 1) & 3];
            }
            if (ncross == 2) {
                int x[2], n = 0;
                for (int i = 0; i < 4; ++i) if (in[i] != in[(i + 1) & 3]) x[n++] = fe[i];
                nb[x[0]][deg[x[0]]++] = x[1];
                nb[x[1]][deg[x[1]]++] = x[0];
            } else if (ncross == 4) {
                for (int i = 0; i < 4; ++i)
                    if (in[i]) {   /* cut INSIDE corner i off: join the face-edges on either side of it */
                        int ea = fe[(i + 3) & 3], eb = fe[i];
                        nb[ea][deg[ea]++] = eb;
                        nb[eb][deg[eb]++] = ea;
                    }
            }
        }
    /* walk the loops */
    int used[12] = {0}, nt = 0;
    int loops[4][12], len[4], first[4], nl = 0;
    for (int e0 = 0; e0 < 12; ++e0) {
        if (!crossed[e0] || used[e0]) continue;
        int L[12], n = 0, prev = -1, cur = e0;   /* e0 is the smallest edge id of its loop */
        do {
            L[n++] = cur;
            used[cur] = 1;
            int nx = (nb[cur][0] != prev) ? nb[cur][0] : nb[cur][1];
            if (n == 1) nx = nb[cur][0];
            prev = cur;
            cur = nx;
        } while (cur != e0);
        /* orientation: Newell normal of the loop (edge midpoints) against the mean INSIDE -> OUTSIDE direction */
        double nrm[3] = {0, 0, 0}, dir[3] = {0, 0, 0}, mid[12][3];
        for (int i = 0; i < n; ++i) {
            int c0, c1, o0[3], o1[3];
            edge_ends(L[i], &c0, &c1);
            corner_off(c0, o0); corner_off(c1, o1);
            int c0_in = (cfg >> c0) & 1;
            for (int d = 0; d < 3; ++d) {
                mid[i][d] = 0.5 * (o0[d] + o1[d]);
                dir[d] += c0_in ? (o1[d] - o0[d]) : (o0[d] - o1[d]);
            }
        }
        for (int i = 0; i < n; ++i) {
            const double* p = mid[i];
            const double* q = mid[(i + 1) % n];
            nrm[0] += (p[1] - q[1]) * (p[2] + q[2]);
            nrm[1] += (p[2] - q[2]) * (p[0] + q[0]);
            nrm[2] += (p[0] - q[0]) * (p[1] + q[1]);
        }
        int flip = (nrm[0] * dir[0] + nrm[1] * dir[1] + nrm[2] * dir[2]) < 0;
        loops[nl][0] = L[0];
        for (int i = 1; i < n; ++i) loops[nl][i] = flip ? L[n - i] : L[i];
        len[nl] = n;
        first[nl] = e0;
        ++nl;
    }
    (void)first;   /* loops are found in increasing order of their smallest edge id */
    for (int l = 0; l < nl; ++l)
        for (int i = 1; i + 1 < len[l]; ++i) {
            tris[nt][0] = loops[l][0]; tris[nt][1] = loops[l][i]; tris[nt][2] = loops[l][i + 1];
            ++nt;
        }
    return nt;
}

/* table export: ntri[256], tris[256][MC_MAX_TRI][3] (cube-edge ids, -1 padded); returns the largest triangle count */
int mesh_oracle_mc_table(int* ntri, int* tris) {
    int mx = 0;
    for (int cfg = 0; cfg < 256; ++cfg) {
        int t[MC_MAX_TRI][3];
        int n = cube_case(cfg, t);
        ntri[cfg] = n;
        if (n > mx) mx = n;
        for (int i = 0; i < MC_MAX_TRI; ++i)
            for (int k = 0; k < 3; ++k) tris[(cfg * MC_MAX_TRI + i) * 3 + k] = (i < n) ? t[i][k] : -1;
    }
    return mx;
}

/* ---- Marching Cubes on the grid (M1-M4) --------------------------------------------------------------------------- */
static long node_of(int N, int x, int y, int z) { return ((long)x * N + y) * N + z; }

void mesh_oracle_mc_count(int N, const double* chi, long* nverts, long* ntris) {
    long nv = 0, nt = 0;
    int t[MC_MAX_TRI][3];
    for (int x = 0; x < N; ++x)
        for (int y = 0; y < N; ++y)
            for (int z = 0; z < N; ++z) {
                const int j[3] = {x, y, z};
                const int in0 = chi[node_of(N, x, y, z)] < 0.0;
                for (int a = 0; a < 3; ++a) {
                    if (j[a] + 1 >= N) continue;
                    int k[3] = {x, y, z};
                    k[a] += 1;
                    nv += in0 != (chi[node_of(N, k[0], k[1], k[2])] < 0.0);
                }
                if (x + 1 < N && y + 1 < N && z + 1 < N) {
                    int cfg = 0;
                    for (int c = 0; c < 8; ++c) cfg |= (chi[node_of(N, x + (c & 1), y + ((c >> 1) & 1), z + ((c >> 2) & 1))] < 0.0) << c;
                    nt += cube_case(cfg, t);
                }
            }
    *nverts = nv;
    *ntris = nt;
}

static void grad_at(int N, const double* chi, int x, int y, int z, double* g) {
    const int M = N - 1;   /* N is a power of two on this path; periodic wrap like chi itself */
    g[0] = 0.5 * N * (chi[node_of(N, (x + 1) & M, y, z)] - chi[node_of(N, (x - 1) & M, y, z)]);
    g[1] = 0.5 * N * (chi[node_of(N, x, (y + 1) & M, z)] - chi[node_of(N, x, (y - 1) & M, z)]);
    g[2] = 0.5 * N * (chi[node_of(N, x, y, (z + 1) & M)] - chi[node_of(N, x, y, (z - 1) & M)]);
}

/* verts/normals [V][3]; vnode [V] = linear index of the edge's first node, vaxis [V], vt [V]; tris [T][3] vertex ids.
 * Vertices in increasing (node, axis) order, triangles in increasing cell order then in the order of M3. */
void mesh_oracle_mc_extract(int N, const double* chi, double* verts, double* normals, long* vnode, int* vaxis, double* vt,
                            long* tris) {
    const long V3 = 3L * N * N * N;
    long* vid = (long*)malloc(sizeof(long) * (size_t)V3);
    for (long i = 0; i < V3; ++i) vid[i] = -1;
    long nv = 0, nt = 0;
    for (int x = 0; x < N; ++x)
        for (int y = 0; y < N; ++y)
            for (int z = 0; z < N; ++z) {
                const int j[3] = {x, y, z};
                const long n0 = node_of(N, x, y, z);
                const double c0 = chi[n0];
                for (int a = 0; a < 3; ++a) {
                    if (j[a] + 1 >= N) continue;
                    int k[3] = {x, y, z};
                    k[a] += 1;
                    const double c1 = chi[node_of(N, k[0], k[1], k[2])];
                    if ((c0 < 0.0) == (c1 < 0.0)) continue;
                    const double t = c0 / (c0 - c1);
                    double g0[3], g1[3], g[3], nn = 0.0;
                    grad_at(N, chi, x, y, z, g0);
                    grad_at(N, chi, k[0], k[1], k[2], g1);
                    for (int d = 0; d < 3; ++d) {
                        verts[3 * nv + d] = (j[d] + (d == a ? t : 0.0)) / N;
                        g[d] = (1.0 - t) * g0[d] + t * g1[d];
                        nn += g[d] * g[d];
                    }
                    nn = sqrt(nn);
                    for (int d = 0; d < 3; ++d) normals[3 * nv + d] = (nn > 0.0) ? g[d] / nn : 0.0;
                    vnode[nv] = n0; vaxis[nv] = a; vt[nv] = t;
                    vid[3 * n0 + a] = nv;
                    ++nv;
                }
            }
    int t3[MC_MAX_TRI][3];
    for (int x = 0; x + 1 < N; ++x)
        for (int y = 0; y + 1 < N; ++y)
            for (int z = 0; z + 1 < N; ++z) {
                int cfg = 0;
                for (int c = 0; c < 8; ++c) cfg |= (chi[node_of(N, x + (c & 1), y + ((c >> 1) & 1), z + ((c >> 2) & 1))] < 0.0) << c;
                const int n = cube_case(cfg, t3);
                for (int i = 0; i < n; ++i) {
                    for (int k = 0; k < 3; ++k) {
                        const int e = t3[i][k], a = e / 4, kk = e % 4;
                        int b1, b2, o[3];
                        other_axes(a, &b1, &b2);
                        o[a] = 0; o[b1] = kk & 1; o[b2] = kk >> 1;
                        tris[3 * nt + k] = vid[3 * node_of(N, x + o[0], y + o[1], z + o[2]) + a];
                    }
                    ++nt;
                }
            }
    free(vid);
}

/* ---- Eq.6 (M5): G[N^3] from dL/dp_v --------------------------------------------------------------------------------- */
void mesh_oracle_eq6_backward(int N, long V, const long* vnode, const int* vaxis, const double* vt, const double* normals,
                              const double* dLdp, double* G) {
    const long stride[3] = {(long)N * N, N, 1};
    memset(G, 0, sizeof(double) * (size_t)N * N * N);
    for (long v = 0; v < V; ++v) {
        const double g = -(dLdp[3 * v] * normals[3 * v] + dLdp[3 * v + 1] * normals[3 * v + 1] + dLdp[3 * v + 2] * normals[3 * v + 2]);
        G[vnode[v]] += (1.0 - vt[v]) * g;
        G[vnode[v] + stride[vaxis[v]]] += vt[v] * g;
    }
}

/* ---- bi-directional squared-L2 Chamfer distance (M6), brute force ------------------------------------------------ */
void mesh_oracle_chamfer(long na, const double* a, long nb, const double* b, long* nn_a, long* nn_b, double* dist_a,
                         double* dist_b, double* loss, double* grad_a, double* grad_b) {
    double la = 0.0, lb = 0.0;
    for (long i = 0; i < na; ++i) {
        double best = INFINITY; long bk = -1;
        for (long k = 0; k < nb; ++k) {
            const double dx = a[3 * i] - b[3 * k], dy = a[3 * i + 1] - b[3 * k + 1], dz = a[3 * i + 2] - b[3 * k + 2];
            const double d = dx * dx + dy * dy + dz * dz;
            if (d < best) { best = d; bk = k; }
        }
        nn_a[i] = bk; dist_a[i] = best; la += best;
    }
    for (long k = 0; k < nb; ++k) {
        double best = INFINITY; long bi = -1;
        for (long i = 0; i < na; ++i) {
            const double dx = a[3 * i] - b[3 * k], dy = a[3 * i + 1] - b[3 * k + 1], dz = a[3 * i + 2] - b[3 * k + 2];
            const double d = dx * dx + dy * dy + dz * dz;
            if (d < best) { best = d; bi = i; }
        }
        nn_b[k] = bi; dist_b[k] = best; lb += best;
    }
    *loss = la / (double)na + lb / (double)nb;
    if (grad_a) {
        memset(grad_a, 0, sizeof(double) * 3 * (size_t)na);
        for (long i = 0; i < na; ++i)
            for (int d = 0; d < 3; ++d) grad_a[3 * i + d] += 2.0 / (double)na * (a[3 * i + d] - b[3 * nn_a[i] + d]);
        for (long k = 0; k < nb; ++k)
            for (int d = 0; d < 3; ++d) grad_a[3 * nn_b[k] + d] += 2.0 / (double)nb * (a[3 * nn_b[k] + d] - b[3 * k + d]);
    }
    if (grad_b) {
        memset(grad_b, 0, sizeof(double) * 3 * (size_t)nb);
        for (long k = 0; k < nb; ++k)
            for (int d = 0; d < 3; ++d) grad_b[3 * k + d] += 2.0 / (double)nb * (b[3 * k + d] - a[3 * nn_b[k] + d]);
        for (long i = 0; i < na; ++i)
            for (int d = 0; d < 3; ++d) grad_b[3 * nn_a[i] + d] += 2.0 / (double)na * (b[3 * nn_a[i] + d] - a[3 * i + d]);
    }
}
