// sap_mesh.cu -- the mesh side of the optimisation-based pipeline (include/sap_mesh.h): Marching Cubes on the indicator
// grid, the surrogate gradient of Eq.6 (L113-L117) and the bi-directional L2 Chamfer distance (L102),
// all on the device with data-dependent sizes kept in device memory.  Readings M1-M6: DESIGN.md / sap_mesh.h.
//
//   Marching Cubes: classify (per node: which of its 3 owned edges cross, sign configuration and triangle count of its
//   cell; per-block totals) -> exclusive scan of the block totals -> emit vertices (per-node offsets from an in-block
//   scan; position, normal, t) -> emit triangles (vertex ids looked up through the per-node offsets).  No atomics, so
//   vertex and triangle order are fixed: increasing (node, axis) and increasing cell.
//   Eq.6: owner-computes gather per grid node over its <= 6 incident edges (no atomics, no memset, deterministic).
//   Chamfer: exact nearest neighbours, lowest index wins an exact tie: exhaustive search through shared-memory tiles up to
//   2e10 pairs, above that a counting sort of each set into a uniform cell grid and a ring search.
#include <cuda_runtime.h>
#include <math.h>
#include <stdio.h>
#include <atomic>
#include <mutex>
#include <new>
#include <string>

#include "../../include/sap_mesh.h"

namespace sapm {

// ---- cube triangulation by rule M3, built on the host --------------------------------------------------------------
constexpr int MAX_TRI = 12;
struct CubeTables {
    unsigned char ntri[256];
    signed char tri[256][MAX_TRI * 3];
    int max_tri;
};
static int ins_bit(int v, int pos, int bit) { return (v & ((1 << pos) - 1)) | (bit << pos) | ((v >> pos) << (pos + 1)); }
static int del_bit(int v, int pos) { return (v & ((1 << pos) - 1)) | ((v >> (pos + 1)) << pos); }
static int edge_of(int ca, int cb) {   // cube edge joining two adjacent corners
    const int d = ca ^ cb;
    const int a = (d == 1) ? 0 : (d == 2) ? 1 : 2;
    return 4 * a + del_bit(ca, a);
}
static void build_case(int cfg, CubeTables& T) {
    int link[12][2], nlink[12];
    bool cut[12];
    for (int e = 0; e < 12; ++e) {
        const int a = e >> 2, c0 = ins_bit(e & 3, a, 0), c1 = c0 | (1 << a);
        cut[e] = (((cfg >> c0) ^ (cfg >> c1)) & 1) != 0;
        nlink[e] = 0;
    }
    auto join = [&](int ea, int eb) { link[ea][nlink[ea]++] = eb; link[eb][nlink[eb]++] = ea; };
    static const int gray[4] = {0, 1, 3, 2};   // (u, v) = (0,0), (1,0), (1,1), (0,1)
    for (int a = 0; a < 3; ++a)
        for (int side = 0; side < 2; ++side) {
            int corner[4], fedge[4], inside[4], ncut = 0;
            for (int i = 0; i < 4; ++i) {
                corner[i] = ins_bit(gray[i], a, side);
                inside[i] = (cfg >> corner[i]) & 1;
            }
            for (int i = 0; i < 4; ++i) {
                fedge[i] = edge_of(corner[i], corner[(i + 1) & 3]);
                ncut += inside[i] != inside[(i + 1) & 3];
            }
            if (ncut == 2) {
                int first = -1;
                for (int i = 0; i < 4; ++i)
                    if (inside[i] != inside[(i + 1) & 3]) {
                        if (first < 0) first = fedge[i];
                        else join(first, fedge[i]);
                    }
            } else if (ncut == 4) {
                for (int i = 0; i < 4; ++i)
                    if (inside[i]) join(fedge[(i + 3) & 3], fedge[i]);   // cut each INSIDE corner off on its own
            }
        }
    bool done[12] = {};
    int nt = 0;
    for (int start = 0; start < 12; ++start) {
        if (!cut[start] || done[start]) continue;
        int loop[12], n = 0;
        for (int prev = -1, cur = start;;) {
            loop[n++] = cur;
            done[cur] = true;
            const int next = (n == 1 || link[cur][0] != prev) ? link[cur][0] : link[cur][1];
            prev = cur;
            cur = next;
            if (cur == start) break;
        }
        // orientation: loop normal (Newell, edge midpoints) must agree with the mean INSIDE -> OUTSIDE direction
        double mid[12][3], out_dir[3] = {0, 0, 0}, nrm[3] = {0, 0, 0};
        for (int i = 0; i < n; ++i) {
            const int a = loop[i] >> 2, c0 = ins_bit(loop[i] & 3, a, 0);
            for (int d = 0; d < 3; ++d) mid[i][d] = (d == a) ? 0.5 : (double)((c0 >> d) & 1);
            out_dir[a] += ((cfg >> c0) & 1) ? 1.0 : -1.0;
        }
        for (int i = 0; i < n; ++i) {
            const double* p = mid[i];
            const double* q = mid[(i + 1) % n];
            for (int d = 0; d < 3; ++d) {
                const int d1 = (d + 1) % 3, d2 = (d + 2) % 3;
                nrm[d] += (p[d1] - q[d1]) * (p[d2] + q[d2]);
            }
        }
        const bool reverse = nrm[0] * out_dir[0] + nrm[1] * out_dir[1] + nrm[2] * out_dir[2] < 0.0;
        for (int i = 1; i + 1 < n; ++i) {
            const int v1 = reverse ? loop[n - i] : loop[i], v2 = reverse ? loop[n - i - 1] : loop[i + 1];
            T.tri[cfg][3 * nt] = (signed char)loop[0];
            T.tri[cfg][3 * nt + 1] = (signed char)v1;
            T.tri[cfg][3 * nt + 2] = (signed char)v2;
            ++nt;
        }
    }
    T.ntri[cfg] = (unsigned char)nt;
    for (int i = 3 * nt; i < 3 * MAX_TRI; ++i) T.tri[cfg][i] = -1;
}
static const CubeTables& cube_tables() {
    static CubeTables T;
    static bool built = false;
    if (!built) {
        T.max_tri = 0;
        for (int cfg = 0; cfg < 256; ++cfg) {
            build_case(cfg, T);
            if (T.ntri[cfg] > T.max_tri) T.max_tri = T.ntri[cfg];
        }
        built = true;
    }
    return T;
}

__constant__ unsigned char c_ntri[256];
__constant__ signed char c_tri[256 * MAX_TRI * 3];

// ---- Marching Cubes kernels ----------------------------------------------------------------------------------------
constexpr int MC_BLOCK = 256;
struct Node { int x, y, z; };
__device__ __forceinline__ Node node_xyz(unsigned n, int N, int lg) { return Node{(int)(n >> (2 * lg)), (int)((n >> lg) & (N - 1)), (int)(n & (N - 1))}; }
__device__ __forceinline__ unsigned long long pack(unsigned nv, unsigned nt) { return ((unsigned long long)nt << 32) | nv; }

// per node: code = crossing mask of its 3 owned edges (bit a: the edge towards +axis a) | triangle count of its cell << 3;
// cfg = sign configuration of its cell; per block: (vertices, triangles) of its nodes
__global__ void k_mc_classify(const float* __restrict__ chi, int N, int lg, unsigned char* __restrict__ code,
                              unsigned char* __restrict__ cfg_out, unsigned long long* __restrict__ blocksum) {
    __shared__ unsigned long long wsum[MC_BLOCK / 32];
    const unsigned n = blockIdx.x * MC_BLOCK + threadIdx.x;   // N^3 is a multiple of MC_BLOCK
    const Node j = node_xyz(n, N, lg);
    const int sx = N * N, sy = N;
    const bool hx = j.x + 1 < N, hy = j.y + 1 < N, hz = j.z + 1 < N;
    const bool in0 = chi[n] < 0.f;
    unsigned mask = 0, cfg = 0, nt = 0;
    const bool i1 = hx && chi[n + sx] < 0.f, i2 = hy && chi[n + sy] < 0.f, i4 = hz && chi[n + 1] < 0.f;
    if (hx && i1 != in0) mask |= 1u;
    if (hy && i2 != in0) mask |= 2u;
    if (hz && i4 != in0) mask |= 4u;
    if (hx && hy && hz) {
        cfg = (unsigned)in0 | ((unsigned)i1 << 1) | ((unsigned)i2 << 2) | ((unsigned)(chi[n + sx + sy] < 0.f) << 3) | ((unsigned)i4 << 4) |
              ((unsigned)(chi[n + sx + 1] < 0.f) << 5) | ((unsigned)(chi[n + sy + 1] < 0.f) << 6) | ((unsigned)(chi[n + sx + sy + 1] < 0.f) << 7);
        nt = c_ntri[cfg];
    }
    code[n] = (unsigned char)(mask | (nt << 3));
    cfg_out[n] = (unsigned char)cfg;
    unsigned long long s = pack(__popc(mask), nt);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0) wsum[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned long long t = 0;
        for (int w = 0; w < MC_BLOCK / 32; ++w) t += wsum[w];
        blocksum[blockIdx.x] = t;
    }
}
// one block: exclusive scan of the block totals in place; counts = {V, T}
__global__ void k_mc_scan_blocks(unsigned long long* __restrict__ blocksum, int nb, int* __restrict__ counts) {
    __shared__ unsigned long long part[1024];
    const int tid = threadIdx.x, per = (nb + 1023) / 1024;
    const int lo = tid * per, hi = min(lo + per, nb);
    unsigned long long s = 0;
    for (int i = lo; i < hi; ++i) s += blocksum[i];
    part[tid] = s;
    __syncthreads();
    for (int d = 1; d < 1024; d <<= 1) {   // Hillis-Steele, inclusive
        const unsigned long long v = (tid >= d) ? part[tid - d] : 0ull;
        __syncthreads();
        part[tid] += v;
        __syncthreads();
    }
    unsigned long long run = part[tid] - s;
    for (int i = lo; i < hi; ++i) {
        const unsigned long long v = blocksum[i];
        blocksum[i] = run;
        run += v;
    }
    if (tid == 1023) {
        counts[0] = (int)(part[1023] & 0xffffffffull);
        counts[1] = (int)(part[1023] >> 32);
    }
}
// exclusive scan of one packed value per thread over the block (MC_BLOCK threads)
__device__ __forceinline__ unsigned long long block_excl_scan(unsigned long long v, unsigned long long* wsum) {
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    unsigned long long inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const unsigned long long t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    if (lane == 31) wsum[w] = inc;
    __syncthreads();
    unsigned long long base = 0;
    for (int i = 0; i < w; ++i) base += wsum[i];
    return base + inc - v;
}
__global__ void k_mc_emit_verts(const float* __restrict__ chi, int N, int lg, const unsigned char* __restrict__ code,
                                const unsigned long long* __restrict__ blockoff, unsigned* __restrict__ vprefix,
                                unsigned* __restrict__ tprefix, float* __restrict__ verts, float* __restrict__ normals,
                                float* __restrict__ vt, int max_v) {
    __shared__ unsigned long long wsum[MC_BLOCK / 32];
    const unsigned n = blockIdx.x * MC_BLOCK + threadIdx.x;
    const unsigned cd = code[n], mask = cd & 7u;
    const unsigned long long off = blockoff[blockIdx.x] + block_excl_scan(pack(__popc(mask), cd >> 3), wsum);
    unsigned v = (unsigned)(off & 0xffffffffull);
    vprefix[n] = v;
    tprefix[n] = (unsigned)(off >> 32);
    if (!mask) return;
    const Node j = node_xyz(n, N, lg);
    const int M = N - 1;
    const float c0 = chi[n], hN = 0.5f * (float)N, inv = 1.f / (float)N;
    auto at = [&](int x, int y, int z) { return chi[((unsigned)(x & M) << (2 * lg)) | ((unsigned)(y & M) << lg) | (unsigned)(z & M)]; };
    auto grad = [&](int x, int y, int z, float* g) {   // central differences, periodic like chi itself (M4)
        g[0] = hN * (at(x + 1, y, z) - at(x - 1, y, z));
        g[1] = hN * (at(x, y + 1, z) - at(x, y - 1, z));
        g[2] = hN * (at(x, y, z + 1) - at(x, y, z - 1));
    };
    float g0[3];
    grad(j.x, j.y, j.z, g0);
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        if (!(mask & (1u << a))) continue;
        const int kx = j.x + (a == 0), ky = j.y + (a == 1), kz = j.z + (a == 2);
        const float c1 = at(kx, ky, kz);
        const float t = c0 / (c0 - c1);
        if ((int)v < max_v) {
            float g1[3], g[3];
            grad(kx, ky, kz, g1);
            float nn = 0.f;
#pragma unroll
            for (int d = 0; d < 3; ++d) { g[d] = (1.f - t) * g0[d] + t * g1[d]; nn += g[d] * g[d]; }
            const float rn = nn > 0.f ? 1.f / sqrtf(nn) : 0.f;
            const float p[3] = {(float)j.x, (float)j.y, (float)j.z};
#pragma unroll
            for (int d = 0; d < 3; ++d) {
                verts[3 * (size_t)v + d] = (p[d] + (d == a ? t : 0.f)) * inv;
                normals[3 * (size_t)v + d] = g[d] * rn;
            }
            vt[v] = t;
        }
        ++v;
    }
}
__global__ void k_mc_emit_tris(int N, int lg, const unsigned char* __restrict__ code, const unsigned char* __restrict__ cfgs,
                               const unsigned* __restrict__ vprefix, const unsigned* __restrict__ tprefix, int* __restrict__ tris,
                               int max_t) {
    const unsigned n = blockIdx.x * MC_BLOCK + threadIdx.x;
    const unsigned nt = code[n] >> 3;
    if (!nt) return;
    const unsigned cfg = cfgs[n], t0 = tprefix[n];
    // vertex id on cube edge e of this cell: owned by node n + offset, axis a
    auto vid = [&](int e) {
        const int a = e >> 2, k = e & 3;
        const int lo = k & 1, hi = k >> 1;
        const int ox = (a == 0) ? 0 : lo, oy = (a == 1) ? 0 : (a == 0 ? lo : hi), oz = (a == 2) ? 0 : hi;
        const unsigned m = n + ((unsigned)ox << (2 * lg)) + ((unsigned)oy << lg) + (unsigned)oz;
        return (int)(vprefix[m] + __popc(code[m] & ((1u << a) - 1u)));
    };
    for (unsigned i = 0; i < nt; ++i) {
        if ((int)(t0 + i) >= max_t) break;
        const signed char* tr = c_tri + (cfg * MAX_TRI + i) * 3;
        int* o = tris + 3 * (size_t)(t0 + i);
        o[0] = vid(tr[0]); o[1] = vid(tr[1]); o[2] = vid(tr[2]);
    }
}
// Eq.6 (M5), owner computes: node n gathers from its 3 owned edges (weight 1 - t) and the 3 edges that end in it (t)
__global__ void k_mc_eq6(int N, int lg, const unsigned char* __restrict__ code, const unsigned* __restrict__ vprefix,
                         const float* __restrict__ vt, const float* __restrict__ gv, const float* __restrict__ nrm,
                         float* __restrict__ G, int max_v) {
    const unsigned n = blockIdx.x * MC_BLOCK + threadIdx.x;
    const Node j = node_xyz(n, N, lg);
    const int jj[3] = {j.x, j.y, j.z};
    const unsigned stride[3] = {1u << (2 * lg), 1u << lg, 1u};
    float acc = 0.f;
    auto contrib = [&](unsigned m, int a, bool head) {
        const unsigned cm = code[m];
        if (!(cm & (1u << a))) return;
        const unsigned v = vprefix[m] + __popc(cm & ((1u << a) - 1u));
        if ((int)v >= max_v) return;
        const float g = -(gv[3 * (size_t)v] * nrm[3 * (size_t)v] + gv[3 * (size_t)v + 1] * nrm[3 * (size_t)v + 1] + gv[3 * (size_t)v + 2] * nrm[3 * (size_t)v + 2]);
        const float t = vt[v];
        acc += (head ? 1.f - t : t) * g;
    };
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        contrib(n, a, true);
        if (jj[a] >= 1) contrib(n - stride[a], a, false);
    }
    G[n] = acc;
}

// ---- Chamfer kernels -------------------------------------------------------------------------------------------------
constexpr int GC_MAX = 64;   // cells per axis of the largest grid (the workspace is sized for it)
__device__ __forceinline__ int count_of(int n, const int* n_dev) { return n_dev ? min(*n_dev, n) : n; }
// Cells per axis for a set of n points: about 2 points per cell on average (a surface fills O(Gc^2) of the Gc^3 cells
// with ~2 Gc / 3 points each).  Computed ON THE DEVICE from the actual count -- the size of a mesh is only known there --
// identically in every kernel that touches the grid, so a small set gets a coarse grid and a far query few rings.
__device__ __forceinline__ int grid_cells(int n) { return min(max((int)cbrtf(0.5f * (float)n), 2), GC_MAX); }
__device__ __forceinline__ int cell_coord(float c, int Gc) { return min(max((int)floorf(c * (float)Gc), 0), Gc - 1); }
__global__ void k_cell_count(const float* __restrict__ pts, int n, const int* n_dev, int* __restrict__ cnt) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int Gc = grid_cells(count_of(n, n_dev));
    if (i >= count_of(n, n_dev)) return;
    const int c = (cell_coord(pts[3 * i], Gc) * Gc + cell_coord(pts[3 * i + 1], Gc)) * Gc + cell_coord(pts[3 * i + 2], Gc);
    atomicAdd(cnt + c, 1);
}
// one block: start = exclusive scan of cnt over ncell entries (+ total at [ncell]); cursor = start
__global__ void k_cell_scan(int* __restrict__ cnt, int n, const int* n_dev, int* __restrict__ start, int* __restrict__ cursor) {
    __shared__ int part[1024];
    const int Gc = grid_cells(count_of(n, n_dev)), ncell = Gc * Gc * Gc;
    const int tid = threadIdx.x, per = (ncell + 1023) / 1024;
    const int lo = tid * per, hi = min(lo + per, ncell);
    int s = 0;
    for (int i = lo; i < hi; ++i) s += cnt[i];
    part[tid] = s;
    __syncthreads();
    for (int d = 1; d < 1024; d <<= 1) {
        const int v = (tid >= d) ? part[tid - d] : 0;
        __syncthreads();
        part[tid] += v;
        __syncthreads();
    }
    int run = part[tid] - s;
    for (int i = lo; i < hi; ++i) {
        const int c = cnt[i];
        start[i] = run;
        cursor[i] = run;
        cnt[i] = 0;              // the counters are zero again for the next grid
        run += c;
    }
    if (tid == 1023) start[ncell] = part[1023];
}
__global__ void k_cell_scatter(const float* __restrict__ pts, int n, const int* n_dev, int* __restrict__ cursor,
                               float4* __restrict__ sorted) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int Gc = grid_cells(count_of(n, n_dev));
    if (i >= count_of(n, n_dev)) return;
    const float x = pts[3 * i], y = pts[3 * i + 1], z = pts[3 * i + 2];
    const int c = (cell_coord(x, Gc) * Gc + cell_coord(y, Gc)) * Gc + cell_coord(z, Gc);
    sorted[atomicAdd(cursor + c, 1)] = make_float4(x, y, z, __int_as_float(i));
}
// exact nearest neighbour of every query in the binned set: rings of cells of growing Chebyshev radius r around the
// query's cell; every point not yet visited after ring r is at least r / Gc away, so the search stops once best <= (r/Gc)^2
__global__ void k_nn_query(const float* __restrict__ q, int nq, const int* nq_dev, const int* __restrict__ start,
                           const float4* __restrict__ sorted, int ntarget, const int* ntarget_dev, int* __restrict__ nn,
                           float* __restrict__ d2out) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= count_of(nq, nq_dev)) return;
    if (count_of(ntarget, ntarget_dev) <= 0) { nn[i] = -1; d2out[i] = 0.f; return; }
    const int Gc = grid_cells(count_of(ntarget, ntarget_dev));
    const float px = q[3 * i], py = q[3 * i + 1], pz = q[3 * i + 2];
    const int cx = cell_coord(px, Gc), cy = cell_coord(py, Gc), cz = cell_coord(pz, Gc);
    const float h = 1.f / (float)Gc;
    float best = INFINITY;
    int bi = 0x7fffffff;
    for (int r = 0; r < Gc; ++r) {
        const int x0 = max(cx - r, 0), x1 = min(cx + r, Gc - 1), y0 = max(cy - r, 0), y1 = min(cy + r, Gc - 1);
        const int z0 = max(cz - r, 0), z1 = min(cz + r, Gc - 1);
        for (int x = x0; x <= x1; ++x)
            for (int y = y0; y <= y1; ++y) {
                const bool shell_xy = (abs(x - cx) == r) || (abs(y - cy) == r);
                for (int z = z0; z <= z1; z += (shell_xy || r == 0) ? 1 : max(z1 - z0, 1)) {
                    if (!shell_xy && abs(z - cz) != r) continue;   // interior of the cube of radius r: visited by earlier rings
                    const int c = (x * Gc + y) * Gc + z;
                    for (int k = start[c]; k < start[c + 1]; ++k) {
                        const float4 t = sorted[k];
                        const float dx = px - t.x, dy = py - t.y, dz = pz - t.z;
                        const float d = dx * dx + dy * dy + dz * dz;
                        const int ti = __float_as_int(t.w);
                        if (d < best || (d == best && ti < bi)) { best = d; bi = ti; }
                    }
                }
            }
        const float reach = (float)r * h;
        if (best <= reach * reach) break;
    }
    nn[i] = bi;
    d2out[i] = best;
}
// Exact nearest neighbour by exhaustive search: the targets stream through shared memory in tiles, every thread keeps
// the best of its query.  O(nq nt), but regular and latency-free: at the sizes of the optimisation loop (1e5 mesh
// vertices x 2e4 input points = 2e9 pairs, ~0.3 ms) it beats the ring search by 3-20x, most of all while the mesh is
// still far from the cloud (the ring search then walks thousands of empty cells per query).  Targets are visited in
// index order and a candidate must be strictly closer, so the lowest index wins an exact tie.
constexpr int BF_TILE = 1024;
// A tile holds the targets two by two: tile[3 k2 .. 3 k2 + 2] = (x, x'), (y, y'), (z, z') of targets 2 k2 and 2 k2 + 1, so that the
// three differences, the square and the two fused multiply-adds of a PAIR of targets are six packed FP32x2 instructions; the
// two candidates are then examined in index order (strictly closer wins: the lowest index keeps an exact tie).  The sum is
// formed as fma(dz, dz, fma(dy, dy, dx dx)), what the scalar expression dx dx + dy dy + dz dz contracts to.
__device__ __forceinline__ void bf_fill_tile(float2* tile, const float* __restrict__ t, int t0, int m) {
    for (int k2 = threadIdx.x; 2 * k2 < m; k2 += blockDim.x) {
        const int k = 2 * k2;
        const bool two = k + 1 < m;   // an odd tail gets a far-away partner that can never win
        const float* a = t + 3 * (size_t)(t0 + k);
        tile[3 * k2 + 0] = make_float2(a[0], two ? a[3] : 3.0e18f);
        tile[3 * k2 + 1] = make_float2(a[1], two ? a[4] : 3.0e18f);
        tile[3 * k2 + 2] = make_float2(a[2], two ? a[5] : 3.0e18f);
    }
}
__device__ __forceinline__ void bf_scan_tile(const float2* tile, int m, int t0, float px, float py, float pz, float& best, int& bi) {
    const float2 px2 = make_float2(px, px), py2 = make_float2(py, py), pz2 = make_float2(pz, pz);
    const int m2 = (m + 1) >> 1;
#pragma unroll 4
    for (int k2 = 0; k2 < m2; ++k2) {
        const float2 cx = tile[3 * k2], cy = tile[3 * k2 + 1], cz = tile[3 * k2 + 2];
        const float2 dx = __fadd2_rn(px2, make_float2(-cx.x, -cx.y));
        const float2 dy = __fadd2_rn(py2, make_float2(-cy.x, -cy.y));
        const float2 dz = __fadd2_rn(pz2, make_float2(-cz.x, -cz.y));
        const float2 d = __ffma2_rn(dz, dz, __ffma2_rn(dy, dy, __fmul2_rn(dx, dx)));
        if (d.x < best) { best = d.x; bi = t0 + 2 * k2; }
        if (d.y < best) { best = d.y; bi = t0 + 2 * k2 + 1; }
    }
}
__global__ void __launch_bounds__(256) k_nn_brute(const float* __restrict__ q, int nq, const int* nq_dev, const float* __restrict__ t, int nt,
                                                  const int* nt_dev, int* __restrict__ nn, float* __restrict__ d2out) {
    __shared__ float2 tile[3 * BF_TILE / 2];
    const int n_q = count_of(nq, nq_dev), n_t = count_of(nt, nt_dev);
    if ((int)(blockIdx.x * blockDim.x) >= n_q) return;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const bool live = i < n_q;
    const float px = live ? q[3 * i] : 0.f, py = live ? q[3 * i + 1] : 0.f, pz = live ? q[3 * i + 2] : 0.f;
    float best = INFINITY;
    int bi = -1;
    for (int t0 = 0; t0 < n_t; t0 += BF_TILE) {
        const int m = min(BF_TILE, n_t - t0);
        __syncthreads();
        bf_fill_tile(tile, t, t0, m);
        __syncthreads();
        bf_scan_tile(tile, m, t0, px, py, pz, best, bi);
    }
    if (live) { nn[i] = bi; d2out[i] = (bi >= 0) ? best : 0.f; }
}

// The same search with the TARGETS split into gridDim.y chunks as well (few queries against many targets -- 20,000 input
// points against 100,000 mesh vertices -- would leave most SMs idle with one block per 256 queries).  A block keeps the
// best of its chunk per query and merges it with atomicMin on the 64-bit key (distance bits << 32 | index): distances are
// non-negative floats, so the keys order like (distance, index) and the lowest index still wins an exact tie.  keys must
// be all ones on entry; k_nn_finish unpacks them.
__global__ void __launch_bounds__(256) k_nn_brute_chunks(const float* __restrict__ q, int nq, const int* nq_dev, const float* __restrict__ t, int nt,
                                                         const int* nt_dev, unsigned long long* __restrict__ keys) {
    __shared__ float2 tile[3 * BF_TILE / 2];
    const int n_q = count_of(nq, nq_dev), n_t = count_of(nt, nt_dev);
    if ((int)(blockIdx.x * blockDim.x) >= n_q) return;
    const int ntiles = (n_t + BF_TILE - 1) / BF_TILE, per = (ntiles + (int)gridDim.y - 1) / (int)gridDim.y;
    const int t_lo = (int)blockIdx.y * per * BF_TILE, t_hi = min(n_t, t_lo + per * BF_TILE);
    if (t_lo >= t_hi) return;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const bool live = i < n_q;
    const float px = live ? q[3 * i] : 0.f, py = live ? q[3 * i + 1] : 0.f, pz = live ? q[3 * i + 2] : 0.f;
    float best = INFINITY;
    int bi = -1;
    for (int t0 = t_lo; t0 < t_hi; t0 += BF_TILE) {
        const int m = min(BF_TILE, t_hi - t0);
        __syncthreads();
        bf_fill_tile(tile, t, t0, m);
        __syncthreads();
        bf_scan_tile(tile, m, t0, px, py, pz, best, bi);
    }
    if (live && bi >= 0) atomicMin(keys + i, ((unsigned long long)__float_as_uint(best) << 32) | (unsigned)bi);
}
__global__ void k_nn_finish(const unsigned long long* __restrict__ keys, int nq, const int* nq_dev, int* __restrict__ nn, float* __restrict__ d2out) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= count_of(nq, nq_dev)) return;
    const unsigned long long k = keys[i];
    const bool found = k != ~0ull;
    nn[i] = found ? (int)(unsigned)(k & 0xffffffffull) : -1;
    d2out[i] = found ? __uint_as_float((unsigned)(k >> 32)) : 0.f;
}

__device__ __forceinline__ float block_sum_f(float x, float* sh) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = x;
    __syncthreads();
    float r = 0.f;
    if (threadIdx.x < 32) {
        r = (threadIdx.x < (blockDim.x >> 5)) ? sh[threadIdx.x] : 0.f;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) r += __shfl_xor_sync(0xffffffffu, r, o);
    }
    return r;
}
// a side: loss += d2 / na, grad_a[i] = (2 / na) (a_i - b_nn(i))
__global__ void k_chamfer_a(const float* __restrict__ a, int na, const int* na_dev, const float* __restrict__ b, const int* __restrict__ nn_a,
                            const float* __restrict__ d2, float* __restrict__ grad_a, double* __restrict__ lacc) {
    __shared__ float sh[32];
    const int n = count_of(na, na_dev), i = blockIdx.x * blockDim.x + threadIdx.x;
    float l = 0.f;
    if (i < n) {
        const int k = nn_a[i];
        l = d2[i] / (float)n;
        if (grad_a) {
            const float s = 2.f / (float)n;
#pragma unroll
            for (int d = 0; d < 3; ++d) grad_a[3 * i + d] = (k >= 0) ? s * (a[3 * i + d] - b[3 * k + d]) : 0.f;
        }
    }
    const float t = block_sum_f(l, sh);
    if (threadIdx.x == 0 && t != 0.f) atomicAdd(lacc, (double)t);
}
// b side: loss += d2 / nb, grad_a[nn_b(k)] += (2 / nb) (a_nn - b_k)
__global__ void k_chamfer_b(const float* __restrict__ a, int na, const int* na_dev, const float* __restrict__ b, int nb,
                            const int* __restrict__ nn_b, const float* __restrict__ d2, float* __restrict__ grad_a, double* __restrict__ lacc) {
    __shared__ float sh[32];
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    float l = 0.f;
    if (k < nb && count_of(na, na_dev) > 0) {
        const int i = nn_b[k];
        l = d2[k] / (float)nb;
        if (grad_a && i >= 0) {
            const float s = 2.f / (float)nb;
#pragma unroll
            for (int d = 0; d < 3; ++d) atomicAdd(grad_a + 3 * i + d, s * (a[3 * i + d] - b[3 * k + d]));
        }
    }
    const float t = block_sum_f(l, sh);
    if (threadIdx.x == 0 && t != 0.f) atomicAdd(lacc, (double)t);
}
__global__ void k_loss_store(double* __restrict__ lacc, float* __restrict__ loss) {
    *loss = (float)*lacc;
    *lacc = 0.0;
}

}  // namespace sapm

// ================================================================================================
struct sap_mesh {
    int N = 0, lg = 0, max_v = 0, max_t = 0, max_p = 0, device = 0, launches = 0;
    int nn_mode = SAP_NN_AUTO;
    unsigned char* code = nullptr;       // [N^3]
    unsigned char* cfg = nullptr;        // [N^3]
    unsigned long long* blocksum = nullptr;  // [N^3 / MC_BLOCK]
    unsigned* vprefix = nullptr;         // [N^3]
    unsigned* tprefix = nullptr;         // [N^3]
    float* vt = nullptr;                 // [max_v]
    int* counts_dev = nullptr;           // [2] of the last extract (device copy kept for the backward)
    // Chamfer
    int* cell_cnt = nullptr;             // [GC_MAX^3], zero between uses
    int* cell_start = nullptr;           // [GC_MAX^3 + 1]
    int* cell_cursor = nullptr;          // [GC_MAX^3]
    float4* sorted = nullptr;            // [max_p]
    int* nn_tmp_a = nullptr;             // [max_p]
    int* nn_tmp_b = nullptr;             // [max_p]
    float* d2_a = nullptr;               // [max_p]
    float* d2_b = nullptr;               // [max_p]
    double* lacc = nullptr;              // [1]
    unsigned long long* nn_keys = nullptr;  // [max_p] (distance, index) keys of the chunked exhaustive search
    int num_sms = 148;
    bool extracted = false;
    size_t ws_bytes = 0;
    std::string err;
};

namespace sapm {
static thread_local std::string g_err;
static bool ok(sap_mesh* h, cudaError_t e, const char* what) {
    if (e == cudaSuccess) return true;
    char buf[384];
    snprintf(buf, sizeof buf, "%s: %s", what, cudaGetErrorString(e));
    if (h) h->err = buf; else g_err = buf;
    return false;
}
template <class T> static cudaError_t alloc(sap_mesh* h, T** p, size_t n) {
    const cudaError_t e = cudaMalloc((void**)p, n * sizeof(T));
    if (e == cudaSuccess) h->ws_bytes += n * sizeof(T);
    return e;
}
static void free_all(sap_mesh* h) {
    cudaFree(h->code); cudaFree(h->cfg); cudaFree(h->blocksum); cudaFree(h->vprefix); cudaFree(h->tprefix); cudaFree(h->vt);
    cudaFree(h->counts_dev); cudaFree(h->cell_cnt); cudaFree(h->cell_start); cudaFree(h->cell_cursor); cudaFree(h->sorted);
    cudaFree(h->nn_tmp_a); cudaFree(h->nn_tmp_b); cudaFree(h->d2_a); cudaFree(h->d2_b); cudaFree(h->lacc); cudaFree(h->nn_keys);
}
static sap_status_t check(sap_mesh* h) {
    if (!h) return SAP_ERR_INVALID_ARG;
    h->err.clear();
    h->launches = 0;
    int dev = -1;
    if (!ok(h, cudaGetDevice(&dev), "cudaGetDevice")) return SAP_ERR_CUDA;
    if (dev != h->device) { h->err = "current CUDA device is not the one the handle was created on"; return SAP_ERR_INVALID_ARG; }
    return SAP_OK;
}
#define MESH_LAUNCH_CHECK(h, name)                                   \
    do {                                                             \
        ++(h)->launches;                                             \
        if (!ok((h), cudaGetLastError(), name)) return SAP_ERR_CUDA; \
    } while (0)
}  // namespace sapm
using namespace sapm;

extern "C" int sap_mc_table(int* ntri, int* tris) {
    const CubeTables& T = cube_tables();
    for (int c = 0; c < 256; ++c) {
        if (ntri) ntri[c] = T.ntri[c];
        if (tris) for (int i = 0; i < MAX_TRI * 3; ++i) tris[c * MAX_TRI * 3 + i] = T.tri[c][i];
    }
    return T.max_tri;
}

extern "C" sap_status_t sap_mesh_create(int N, int max_vertices, int max_triangles, int max_points, sap_mesh_t** out) {
    g_err.clear();
    if (!out) { g_err = "out is NULL"; return SAP_ERR_INVALID_ARG; }
    if (N <= 0 || max_vertices <= 0 || max_triangles <= 0 || max_points <= 0) { g_err = "sizes must be positive"; return SAP_ERR_INVALID_ARG; }
    int lg = 0;
    while ((1 << lg) < N) ++lg;
    if ((1 << lg) != N || N < 8 || N > 512) { g_err = "N must be a power of two in [8, 512]"; return SAP_ERR_UNSUPPORTED; }
    int dev = 0;
    if (!ok(nullptr, cudaGetDevice(&dev), "cudaGetDevice")) return SAP_ERR_CUDA;
    cudaDeviceProp prop;
    if (!ok(nullptr, cudaGetDeviceProperties(&prop, dev), "cudaGetDeviceProperties")) return SAP_ERR_CUDA;
    if (prop.major != 10) { g_err = "device is not sm_100 (Blackwell B200); this library has no other code path"; return SAP_ERR_UNSUPPORTED; }
    sap_mesh* h = new (std::nothrow) sap_mesh;
    if (!h) { g_err = "host allocation failed"; return SAP_ERR_OOM; }
    h->N = N; h->lg = lg; h->max_v = max_vertices; h->max_t = max_triangles; h->max_p = max_points; h->device = dev;
    const size_t V = (size_t)N * N * N, C = (size_t)GC_MAX * GC_MAX * GC_MAX;
    cudaError_t e = cudaSuccess;
    auto upd = [&](cudaError_t x) { if (e == cudaSuccess) e = x; };
    upd(alloc(h, &h->code, V)); upd(alloc(h, &h->cfg, V)); upd(alloc(h, &h->blocksum, V / MC_BLOCK));
    upd(alloc(h, &h->vprefix, V)); upd(alloc(h, &h->tprefix, V)); upd(alloc(h, &h->vt, (size_t)max_vertices));
    upd(alloc(h, &h->counts_dev, (size_t)2));
    upd(alloc(h, &h->cell_cnt, C)); upd(alloc(h, &h->cell_start, C + 1)); upd(alloc(h, &h->cell_cursor, C));
    upd(alloc(h, &h->sorted, (size_t)max_points));
    upd(alloc(h, &h->nn_tmp_a, (size_t)max_points)); upd(alloc(h, &h->nn_tmp_b, (size_t)max_points));
    upd(alloc(h, &h->d2_a, (size_t)max_points)); upd(alloc(h, &h->d2_b, (size_t)max_points));
    upd(alloc(h, &h->lacc, (size_t)1));
    upd(alloc(h, &h->nn_keys, (size_t)max_points));
    h->num_sms = prop.multiProcessorCount;
    if (e == cudaSuccess) upd(cudaMemset(h->lacc, 0, sizeof(double)));
    if (e == cudaSuccess) upd(cudaMemset(h->cell_cnt, 0, sizeof(int) * C));
    if (e == cudaSuccess) upd(cudaMemset(h->counts_dev, 0, 2 * sizeof(int)));
    if (e == cudaSuccess) {
        const CubeTables& T = cube_tables();
        upd(cudaMemcpyToSymbol(c_ntri, T.ntri, sizeof(T.ntri)));
        upd(cudaMemcpyToSymbol(c_tri, T.tri, sizeof(T.tri)));
    }
    if (e != cudaSuccess) {
        ok(nullptr, e, "sap_mesh_create");
        const bool oom = e == cudaErrorMemoryAllocation;
        free_all(h); delete h; cudaGetLastError();
        return oom ? SAP_ERR_OOM : SAP_ERR_CUDA;
    }
    *out = h;
    return SAP_OK;
}

extern "C" sap_status_t sap_mc_extract(sap_mesh_t* h, const float* chi, float* verts, float* normals, int* tris, int* counts,
                                       void* stream) {
    sap_status_t st = check(h);
    if (st != SAP_OK) return st;
    if (!chi || !verts || !normals || !tris || !counts) { h->err = "null pointer argument"; return SAP_ERR_INVALID_ARG; }
    cudaStream_t s = (cudaStream_t)stream;
    const int N = h->N, nb = (int)(((size_t)N * N * N) / MC_BLOCK);
    k_mc_classify<<<nb, MC_BLOCK, 0, s>>>(chi, N, h->lg, h->code, h->cfg, h->blocksum);
    MESH_LAUNCH_CHECK(h, "k_mc_classify");
    k_mc_scan_blocks<<<1, 1024, 0, s>>>(h->blocksum, nb, h->counts_dev);
    MESH_LAUNCH_CHECK(h, "k_mc_scan_blocks");
    k_mc_emit_verts<<<nb, MC_BLOCK, 0, s>>>(chi, N, h->lg, h->code, h->blocksum, h->vprefix, h->tprefix, verts, normals, h->vt, h->max_v);
    MESH_LAUNCH_CHECK(h, "k_mc_emit_verts");
    k_mc_emit_tris<<<nb, MC_BLOCK, 0, s>>>(N, h->lg, h->code, h->cfg, h->vprefix, h->tprefix, tris, h->max_t);
    MESH_LAUNCH_CHECK(h, "k_mc_emit_tris");
    if (!ok(h, cudaMemcpyAsync(counts, h->counts_dev, 2 * sizeof(int), cudaMemcpyDeviceToDevice, s), "copy counts")) return SAP_ERR_CUDA;
    h->extracted = true;
    return SAP_OK;
}

extern "C" sap_status_t sap_mc_backward(sap_mesh_t* h, const float* grad_verts, const float* normals, float* grad_chi, void* stream) {
    sap_status_t st = check(h);
    if (st != SAP_OK) return st;
    if (!grad_verts || !normals || !grad_chi) { h->err = "null pointer argument"; return SAP_ERR_INVALID_ARG; }
    if (!h->extracted) { h->err = "sap_mc_backward must follow sap_mc_extract on this handle"; return SAP_ERR_INVALID_ARG; }
    const int N = h->N, nb = (int)(((size_t)N * N * N) / MC_BLOCK);
    k_mc_eq6<<<nb, MC_BLOCK, 0, (cudaStream_t)stream>>>(N, h->lg, h->code, h->vprefix, h->vt, grad_verts, normals, grad_chi, h->max_v);
    MESH_LAUNCH_CHECK(h, "k_mc_eq6");
    return SAP_OK;
}

extern "C" sap_status_t sap_chamfer(sap_mesh_t* h, const float* a, int na, const int* na_dev, const float* b, int nb, float* loss,
                                    float* grad_a, int* nn_a, int* nn_b, void* stream) {
    sap_status_t st = check(h);
    if (st != SAP_OK) return st;
    if (!a || !b || !loss) { h->err = "null pointer argument"; return SAP_ERR_INVALID_ARG; }
    if (na < 0 || nb < 1 || na > h->max_p || nb > h->max_p) { h->err = "point counts out of range (0 <= na <= max_points, 1 <= nb <= max_points)"; return SAP_ERR_INVALID_ARG; }
    cudaStream_t s = (cudaStream_t)stream;
    int* nna = nn_a ? nn_a : h->nn_tmp_a;
    int* nnb = nn_b ? nn_b : h->nn_tmp_b;
    if (na == 0) {
        if (!ok(h, cudaMemsetAsync(loss, 0, sizeof(float), s), "memset loss")) return SAP_ERR_CUDA;
        return SAP_OK;
    }
    const int ga = (na + 255) / 256, gb = (nb + 255) / 256;
    // exhaustive search while the number of pairs is moderate (na is the capacity when the count lives on the device)
    const bool brute = h->nn_mode == SAP_NN_BRUTE || (h->nn_mode == SAP_NN_AUTO && (double)na * (double)nb <= 2.0e10);
    if (brute) {
        // one block per 256 queries; when that leaves SMs idle the targets are split over gridDim.y chunks as well
        auto nn_brute = [&](const float* q, int nq, const int* nq_dev, int gq, const float* t, int nt, const int* nt_dev, int* nn, float* d2) -> bool {
            const int ntiles = (nt + BF_TILE - 1) / BF_TILE;
            int chunks = (6 * h->num_sms + gq - 1) / gq;
            if (chunks > ntiles) chunks = ntiles;
            if (chunks <= 1) {
                k_nn_brute<<<gq, 256, 0, s>>>(q, nq, nq_dev, t, nt, nt_dev, nn, d2);
                return cudaGetLastError() == cudaSuccess;
            }
            if (cudaMemsetAsync(h->nn_keys, 0xff, sizeof(unsigned long long) * (size_t)nq, s) != cudaSuccess) return false;
            k_nn_brute_chunks<<<dim3(gq, chunks), 256, 0, s>>>(q, nq, nq_dev, t, nt, nt_dev, h->nn_keys);
            k_nn_finish<<<gq, 256, 0, s>>>(h->nn_keys, nq, nq_dev, nn, d2);
            h->launches += 1;
            return cudaGetLastError() == cudaSuccess;
        };
        if (!nn_brute(a, na, na_dev, ga, b, nb, nullptr, nna, h->d2_a)) { ok(h, cudaGetLastError(), "k_nn_brute"); h->err = "k_nn_brute launch failed"; return SAP_ERR_CUDA; }
        MESH_LAUNCH_CHECK(h, "k_nn_brute");
        k_chamfer_a<<<ga, 256, 0, s>>>(a, na, na_dev, b, nna, h->d2_a, grad_a, h->lacc);
        MESH_LAUNCH_CHECK(h, "k_chamfer_a");
        if (!nn_brute(b, nb, nullptr, gb, a, na, na_dev, nnb, h->d2_b)) { h->err = "k_nn_brute launch failed"; return SAP_ERR_CUDA; }
        MESH_LAUNCH_CHECK(h, "k_nn_brute");
        k_chamfer_b<<<gb, 256, 0, s>>>(a, na, na_dev, b, nb, nnb, h->d2_b, grad_a, h->lacc);
        MESH_LAUNCH_CHECK(h, "k_chamfer_b");
    } else {
        // grid over b, queries a
        k_cell_count<<<gb, 256, 0, s>>>(b, nb, nullptr, h->cell_cnt);
        MESH_LAUNCH_CHECK(h, "k_cell_count");
        k_cell_scan<<<1, 1024, 0, s>>>(h->cell_cnt, nb, nullptr, h->cell_start, h->cell_cursor);
        MESH_LAUNCH_CHECK(h, "k_cell_scan");
        k_cell_scatter<<<gb, 256, 0, s>>>(b, nb, nullptr, h->cell_cursor, h->sorted);
        MESH_LAUNCH_CHECK(h, "k_cell_scatter");
        k_nn_query<<<ga, 256, 0, s>>>(a, na, na_dev, h->cell_start, h->sorted, nb, nullptr, nna, h->d2_a);
        MESH_LAUNCH_CHECK(h, "k_nn_query");
        k_chamfer_a<<<ga, 256, 0, s>>>(a, na, na_dev, b, nna, h->d2_a, grad_a, h->lacc);
        MESH_LAUNCH_CHECK(h, "k_chamfer_a");
        // grid over a, queries b
        k_cell_count<<<ga, 256, 0, s>>>(a, na, na_dev, h->cell_cnt);
        MESH_LAUNCH_CHECK(h, "k_cell_count");
        k_cell_scan<<<1, 1024, 0, s>>>(h->cell_cnt, na, na_dev, h->cell_start, h->cell_cursor);
        MESH_LAUNCH_CHECK(h, "k_cell_scan");
        k_cell_scatter<<<ga, 256, 0, s>>>(a, na, na_dev, h->cell_cursor, h->sorted);
        MESH_LAUNCH_CHECK(h, "k_cell_scatter");
        k_nn_query<<<gb, 256, 0, s>>>(b, nb, nullptr, h->cell_start, h->sorted, na, na_dev, nnb, h->d2_b);
        MESH_LAUNCH_CHECK(h, "k_nn_query");
        k_chamfer_b<<<gb, 256, 0, s>>>(a, na, na_dev, b, nb, nnb, h->d2_b, grad_a, h->lacc);
        MESH_LAUNCH_CHECK(h, "k_chamfer_b");
    }
    k_loss_store<<<1, 1, 0, s>>>(h->lacc, loss);
    MESH_LAUNCH_CHECK(h, "k_loss_store");
    return SAP_OK;
}

// eta = move / (N max|gp|);  points <- clip(points - eta gp, 0, 1 - 1e-6);  normals <- normals - eta gn
namespace sapm {
__global__ void k_absmax(const float* __restrict__ g, int n, unsigned* __restrict__ out) {
    __shared__ float sh[32];
    float m = 0.f;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) m = fmaxf(m, fabsf(g[i]));
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = m;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < (int)(blockDim.x >> 5); ++w) m = fmaxf(m, sh[w]);
        atomicMax(out, __float_as_uint(m));   // non-negative floats order like their bit patterns
    }
}
__global__ void k_sgd_apply(float* __restrict__ pts, float* __restrict__ nrm, const float* __restrict__ gp, const float* __restrict__ gn,
                            int n, float move_over_N, unsigned* __restrict__ gmax) {
    const float eta = move_over_N / fmaxf(__uint_as_float(*gmax), 1e-20f);
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) {
        pts[i] = fminf(fmaxf(pts[i] - eta * gp[i], 0.f), 1.f - 1e-6f);
        nrm[i] -= eta * gn[i];
    }
}
__global__ void k_zero_u32(unsigned* p) { *p = 0u; }
}  // namespace sapm
extern "C" sap_status_t sap_points_sgd_step(float* points, float* normals, const float* grad_points, const float* grad_normals,
                                            int count, int N, float move, unsigned* scratch, void* stream) {
    if (!points || !normals || !grad_points || !grad_normals || !scratch || count < 1 || N < 1) return SAP_ERR_INVALID_ARG;
    cudaStream_t s = (cudaStream_t)stream;
    const int nb = (count + 255) / 256;
    k_zero_u32<<<1, 1, 0, s>>>(scratch);
    k_absmax<<<nb < 296 ? nb : 296, 256, 0, s>>>(grad_points, count, scratch);
    k_sgd_apply<<<nb, 256, 0, s>>>(points, normals, grad_points, grad_normals, count, move / (float)N, scratch);
    return cudaGetLastError() == cudaSuccess ? SAP_OK : SAP_ERR_CUDA;
}

extern "C" sap_status_t sap_chamfer_set_search(sap_mesh_t* h, int mode) {
    if (!h) return SAP_ERR_INVALID_ARG;
    h->err.clear();
    if (mode != SAP_NN_AUTO && mode != SAP_NN_BRUTE && mode != SAP_NN_GRID) { h->err = "unknown search mode"; return SAP_ERR_INVALID_ARG; }
    h->nn_mode = mode;
    return SAP_OK;
}

// ---- nearest-neighbour search without a handle and without an allocation (sap_chamfer_nn_static, sap_mesh.h) ---------------
// The scratch of the chunked exhaustive search (k_nn_brute_chunks: one (distance, index) key per query) as a file-scope
// device array: part of the module image, so every GPU that loads the library holds these 2 MiB until the process exits
// and nobody calls cudaMalloc for them.  In HOST code the name below is a host-side stand-in, not a device address: the
// entry point resolves the address once per device with cudaGetSymbolAddress (that device current) and hands the pointer
// to the kernels.  Every call on a GPU shares the array; it keeps the keys of the last call, so a call resets the keys
// it uses first, and calls that overlap on the GPU race on it.
namespace sapm {
static __device__ __align__(256) unsigned long long g_nn_static_keys[SAP_NN_STATIC_MAX_QUERIES];
constexpr int NN_STATIC_MAX_DEVICES = 64;
struct NnStaticDevice {
    std::atomic<int> ready{0};             // 0: not set up, 1: set up, -1: not an sm_100 device
    unsigned long long* keys = nullptr;    // device address of g_nn_static_keys on this device
    int num_sms = 0;
};
static NnStaticDevice g_nn_static[NN_STATIC_MAX_DEVICES];
static std::mutex g_nn_static_mu;
// keys of this call <- all ones (= "no candidate yet", larger than every (distance, index) key)
__global__ void k_nn_static_reset(unsigned long long* __restrict__ keys, int nq) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < nq) keys[i] = ~0ull;
}
// set-up of the current device: once per device, no allocation (attribute queries + the symbol's address)
static sap_status_t nn_static_device(NnStaticDevice** out) {
    int dev = -1;
    if (!ok(nullptr, cudaGetDevice(&dev), "cudaGetDevice")) return SAP_ERR_CUDA;
    if (dev < 0 || dev >= NN_STATIC_MAX_DEVICES) { g_err = "sap_chamfer_nn_static: device ordinal beyond the per-device table (64)"; return SAP_ERR_UNSUPPORTED; }
    NnStaticDevice& d = g_nn_static[dev];
    int st = d.ready.load(std::memory_order_acquire);
    if (st == 0) {
        std::lock_guard<std::mutex> lock(g_nn_static_mu);
        st = d.ready.load(std::memory_order_acquire);
        if (st == 0) {
            int major = 0, sms = 0;
            if (!ok(nullptr, cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev), "cudaDeviceGetAttribute")) return SAP_ERR_CUDA;
            if (!ok(nullptr, cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev), "cudaDeviceGetAttribute")) return SAP_ERR_CUDA;
            if (major != 10) {
                d.ready.store(-1, std::memory_order_release);
                st = -1;
            } else {
                unsigned long long* ptr = nullptr;
                if (!ok(nullptr, cudaGetSymbolAddress((void**)&ptr, g_nn_static_keys), "cudaGetSymbolAddress(g_nn_static_keys)")) return SAP_ERR_CUDA;
                if (!ptr) { g_err = "cudaGetSymbolAddress returned a null address for g_nn_static_keys"; return SAP_ERR_CUDA; }
                d.keys = ptr;
                d.num_sms = sms > 0 ? sms : 148;
                d.ready.store(1, std::memory_order_release);
                st = 1;
            }
        }
    }
    if (st < 0) { g_err = "device is not sm_100 (Blackwell B200); this library has no other code path"; return SAP_ERR_UNSUPPORTED; }
    *out = &d;
    return SAP_OK;
}
}  // namespace sapm

extern "C" sap_status_t sap_chamfer_nn_static(const float* queries, int nq, const float* targets, int nt, int* nn, float* d2, void* stream) {
    g_err.clear();
    if (!queries || !targets || !nn || !d2) { g_err = "null pointer argument"; return SAP_ERR_INVALID_ARG; }
    if (nq < 0 || nt < 1) { g_err = "point counts out of range (nq >= 0, nt >= 1)"; return SAP_ERR_INVALID_ARG; }
    if (nq > SAP_NN_STATIC_MAX_QUERIES) {
        char buf[256];
        snprintf(buf, sizeof buf, "nq = %d exceeds SAP_NN_STATIC_MAX_QUERIES = %d, the size of the library's static scratch array "
                 "(use sap_chamfer with a handle for larger sets)", nq, SAP_NN_STATIC_MAX_QUERIES);
        g_err = buf;
        return SAP_ERR_INVALID_ARG;
    }
    if (nq == 0) return SAP_OK;
    NnStaticDevice* d = nullptr;
    const sap_status_t st = nn_static_device(&d);
    if (st != SAP_OK) return st;
    cudaStream_t s = (cudaStream_t)stream;
    // the launch shape of sap_chamfer's exhaustive search: one block per 256 queries, the targets split over gridDim.y
    // chunks while that leaves SMs idle; here always through the keys (a single chunk included)
    const int gq = (nq + 255) / 256, ntiles = (nt + BF_TILE - 1) / BF_TILE;
    int chunks = (6 * d->num_sms + gq - 1) / gq;
    if (chunks > ntiles) chunks = ntiles;
    if (chunks < 1) chunks = 1;
    k_nn_static_reset<<<gq, 256, 0, s>>>(d->keys, nq);
    if (!ok(nullptr, cudaGetLastError(), "k_nn_static_reset")) return SAP_ERR_CUDA;
    k_nn_brute_chunks<<<dim3(gq, chunks), 256, 0, s>>>(queries, nq, nullptr, targets, nt, nullptr, d->keys);
    if (!ok(nullptr, cudaGetLastError(), "k_nn_brute_chunks")) return SAP_ERR_CUDA;
    k_nn_finish<<<gq, 256, 0, s>>>(d->keys, nq, nullptr, nn, d2);
    if (!ok(nullptr, cudaGetLastError(), "k_nn_finish")) return SAP_ERR_CUDA;
    return SAP_OK;
}

extern "C" void sap_mesh_destroy(sap_mesh_t* h) {
    if (!h) return;
    free_all(h);
    delete h;
}
extern "C" const char* sap_mesh_last_error(const sap_mesh_t* h) { return h ? h->err.c_str() : g_err.c_str(); }
extern "C" size_t sap_mesh_workspace_bytes(const sap_mesh_t* h) { return h ? h->ws_bytes : 0; }
extern "C" int sap_mesh_last_launch_count(const sap_mesh_t* h) { return h ? h->launches : 0; }
