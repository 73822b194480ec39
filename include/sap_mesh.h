/*
 * sap_mesh.h -- C ABI of the mesh side of the optimisation-based pipeline of Shape As Points (arXiv 2106.03452,
 * Sec.3.2), the steps that close the loop around the DPSR layer (include/sap_dpsr.h) on the device:
 *
 *   chi --Marching Cubes (L100)--> mesh {p_mesh, n_mesh} --Chamfer to the input cloud (L102)--> dL/dp_mesh
 *       --Eq.6, dp_mesh/dchi = -n_mesh (L113-L117)--> dL/dchi  (= grad_chi of sap_dpsr_backward)
 *
 * The paper calls a CPU library for Marching Cubes (footnote, L248) and gives no formulas for this part; the readings
 * M1-M6 taken here are listed in DESIGN.md and in oracle/mesh_oracle.c (the float64 oracle the kernels are tested
 * against):
 *   M1  level set chi = 0, a node is INSIDE iff chi < 0; cells are the (N-1)^3 cubes between nodes (no wrap).
 *   M2  one vertex per sign-changing grid edge at the linear zero crossing, p = (j + t e_a) / N in the unit cube.
 *   M3  cube triangulation by rule (face segments -> loops -> fans; ambiguous faces cut the INSIDE corners off), built
 *       at library load, not a copied table; watertight across cubes; triangles wind so that their normal points OUTSIDE.
 *   M4  n_mesh = normalised central-difference gradient of chi (periodic), interpolated along the edge.
 *   M5  Eq.6 through the trilinear interpolant: G[node0] += (1-t) g, G[node1] += t g, g = -(dL/dp . n_mesh).
 *   M6  Chamfer = mean_i min_k |a_i - b_k|^2 + mean_k min_i |b_k - a_i|^2; the mesh samples are the mesh vertices.
 *
 * Conventions as in sap_dpsr.h: status codes, "dev" pointers on the handle's device, work enqueued on `stream` and not
 * synchronised, the caller owns every buffer it passes, the handle owns its workspace (allocated in sap_mesh_create;
 * no call allocates).  Mesh sizes are data dependent and stay ON THE DEVICE: counts[2] = {V, T} is written by
 * sap_mc_extract and read by the other calls, so the whole loop can be enqueued (or graph-captured) without a host
 * round trip.  If V > max_vertices or T > max_triangles the arrays are filled up to their capacity and counts holds
 * the sizes that would have been needed: the caller checks counts against its capacities when it reads them.
 */
#ifndef SAP_MESH_H
#define SAP_MESH_H

#include "sap_dpsr.h"

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sap_mesh sap_mesh_t; /* opaque */

/*
 * Workspace for grids of N^3 nodes (N a power of two, 8 <= N <= 512), meshes of at most max_vertices / max_triangles
 * and Chamfer point sets of at most max_points points on either side (the mesh vertices count as one side, so
 * max_points >= max_vertices is advisable).  About 9 bytes per node + 40 bytes per point.
 */
sap_status_t sap_mesh_create(int N, int max_vertices, int max_triangles, int max_points, sap_mesh_t** out);

/*
 * Marching Cubes (M1-M4).
 *   chi      dev [N][N][N] float (the output of sap_dpsr_forward, one item)
 *   verts    dev [max_vertices][3] float   vertex positions in the unit cube, in increasing (node, axis) order
 *   normals  dev [max_vertices][3] float   n_mesh, unit length (0 where the gradient vanishes)
 *   tris     dev [max_triangles][3] int    vertex ids, in increasing cell order
 *   counts   dev [2] int                   {V, T} (see above)
 * The handle remembers, per vertex, its grid edge and interpolation parameter t for sap_mc_backward.
 */
sap_status_t sap_mc_extract(sap_mesh_t* h, const float* chi, float* verts, float* normals, int* tris, int* counts,
                            void* stream);

/*
 * Eq.6 (M5): dL/dchi from dL/dp_mesh.  Must follow the sap_mc_extract whose mesh it differentiates.
 *   grad_verts dev [max_vertices][3] float   dL/dp_mesh (rows >= V are ignored)
 *   normals    dev [max_vertices][3] float   the normals sap_mc_extract returned
 *   grad_chi   dev [N][N][N] float           overwritten (every node: owner-computes gather, no atomics, deterministic)
 */
sap_status_t sap_mc_backward(sap_mesh_t* h, const float* grad_verts, const float* normals, float* grad_chi, void* stream);

/*
 * Bi-directional squared-L2 Chamfer distance (M6) between point sets a and b in the unit cube [0,1)^3 with EXACT nearest
 * neighbours (the lowest index wins an exact tie).  Two searches: exhaustive through shared-memory tiles (regular, no
 * set-up; the default up to 2e10 pairs -- 1e5 mesh vertices against 2e4 input points take ~0.3 ms) and a uniform cell grid
 * with a ring search (cost grows with the distance between the sets; the default above that).
 *   a, na, na_dev  dev [>= na][3] float; the number of points is *na_dev if na_dev != NULL (a device int, e.g.
 *                  counts of sap_mc_extract; then na is only the capacity used to size the launches), else na
 *   b, nb          dev [nb][3] float (the input cloud)
 *   loss           dev [1] float, overwritten
 *   grad_a         dev [>= na][3] float or NULL   dL/da, overwritten
 *   nn_a, nn_b     dev [>= na] / [nb] int or NULL  index of the nearest neighbour of a_i in b / of b_k in a
 * An empty set (na == 0) gives loss = 0 and no gradients.
 */
sap_status_t sap_chamfer(sap_mesh_t* h, const float* a, int na, const int* na_dev, const float* b, int nb, float* loss,
                         float* grad_a, int* nn_a, int* nn_b, void* stream);

/* Nearest-neighbour search of sap_chamfer: SAP_NN_AUTO (default, by the number of pairs), or force one of the two. */
enum { SAP_NN_AUTO = 0, SAP_NN_BRUTE = 1, SAP_NN_GRID = 2 };
sap_status_t sap_chamfer_set_search(sap_mesh_t* h, int mode);

/*
 * The exhaustive nearest-neighbour search of sap_chamfer (M6: nn[i] = argmin_k |q_i - t_k|^2, the lowest index wins an
 * exact tie) for callers that cannot allocate: code under CUDA graph capture, serving loops and harnesses that forbid
 * cudaMalloc.  NO HANDLE AND NO ALLOCATION: the only scratch of the search -- one 64-bit (distance, index) key per query,
 * merged with atomicMin by the blocks that scan different chunks of the targets -- lives in a file-scope device array of
 * the library, SAP_NN_STATIC_MAX_QUERIES keys = 2 MiB, which every GPU that loads the library holds until the process
 * exits.  The call makes no cudaMalloc / cudaFree and calls no allocating routine; it enqueues three kernels on `stream`
 * (reset the keys of this call, scan, unpack) and does not synchronise.  The first call on a device also resolves the
 * array's device address (cudaGetSymbolAddress, once per device, with that device current): make one call before a
 * stream capture begins.
 *   queries, nq   dev [nq][3] float, 0 <= nq <= SAP_NN_STATIC_MAX_QUERIES (nq == 0: nothing is enqueued)
 *   targets, nt   dev [nt][3] float, nt >= 1
 *   nn            dev [nq] int    index of the nearest target, overwritten
 *   d2            dev [nq] float  its squared distance, overwritten
 * Returns SAP_ERR_INVALID_ARG for null pointers, nt < 1, nq < 0 and for nq > SAP_NN_STATIC_MAX_QUERIES (the message of
 * sap_mesh_last_error(NULL) names the limit; larger sets go through sap_chamfer and a handle), SAP_ERR_UNSUPPORTED when the
 * device is not sm_100, SAP_ERR_CUDA for a failed launch.
 * The array is SHARED by every call of the process on that GPU and keeps the keys of the last call: a call first resets
 * the nq keys it uses, so consecutive calls on one stream (or otherwise ordered) are independent of one another, but two
 * calls that OVERLAP on the GPU (different streams without an event between them, two host threads) race on it and give
 * wrong neighbours.  Results are bit-identical to the nn_a / nn_b of sap_chamfer in SAP_NN_BRUTE mode.
 */
#define SAP_NN_STATIC_MAX_QUERIES 262144
sap_status_t sap_chamfer_nn_static(const float* queries, int nq, const float* targets, int nt, int* nn, float* d2, void* stream);

/*
 * The plain point update of BASELINE.json configs[3] ("iterations with a point update between them") and of the
 * fixed-gradient mode of the coarse-to-fine driver, as two small kernels instead of a dozen framework ops:
 *   eta = move / (N max |grad_points|);  points <- clip(points - eta grad_points, 0, 1 - 1e-6);  normals <- normals - eta grad_normals
 * i.e. the largest point step is `move` cells of an N^3 grid.  All arrays dev float [count] (count = batch * P * 3),
 * scratch dev [1] unsigned.  (The paper's own loop uses Adam, L396: that stays with the host framework.)
 */
sap_status_t sap_points_sgd_step(float* points, float* normals, const float* grad_points, const float* grad_normals,
                                 int count, int N, float move, unsigned* scratch, void* stream);

/* The cube triangulation built at load (M3), for tests: ntri[256], tris[256][12][3] cube-edge ids (-1 padded).
 * Cube corner c has offsets (c & 1, (c >> 1) & 1, (c >> 2) & 1); cube edge 4 a + k runs along axis a, k = u + 2 v with
 * (u, v) the offsets along the two other axes in increasing order.  Returns the largest triangle count of a cube. */
int sap_mc_table(int* ntri, int* tris);

void sap_mesh_destroy(sap_mesh_t* h);
const char* sap_mesh_last_error(const sap_mesh_t* h);
size_t sap_mesh_workspace_bytes(const sap_mesh_t* h);
int sap_mesh_last_launch_count(const sap_mesh_t* h);

#ifdef __cplusplus
}
#endif
#endif /* SAP_MESH_H */
