/*
 * sap_dpsr.h -- C ABI of the B200-native DPSR layer (Shape As Points, arXiv 2106.03452).
 *
 * DPSR = differentiable Poisson surface reconstruction: an oriented point cloud {(c_i, n_i)} is
 * mapped to an indicator grid chi in R^{N x N x N} (Sec.3.1; Suppl. A, L337-L388)
 * and the map is differentiable w.r.t. points and normals (L17; third factor of Eq.5).
 * "PAPER.md:Lnnn" cites /root/reference/PAPER.md.  Readings R1..R14 of the paper: DESIGN.md.
 *
 * Every step runs in hand-written sm_100a CUDA kernels inside libsap_dpsr.so; there is no CPU or
 * library (cuFFT) fallback.  All entry points return a status code and never throw or abort.
 *
 * Conventions
 *   - Layout: C order, z fastest.  chi[b][jx][jy][jz] is the value at position (jx, jy, jz)/N of
 *     the unit cube [0,1)^3 (R1: origin 0, voxel 1/N, periodic).
 *   - Pointers marked "dev" are CUDA device pointers valid on the handle's device; "host" are
 *     ordinary host pointers (pinned memory makes the *_host calls asynchronous copies).
 *   - The caller owns every buffer it passes and the stream.  The handle owns its workspace,
 *     allocated once in sap_dpsr_create; sap_dpsr_forward / sap_dpsr_backward never allocate.  The
 *     fused-loss and host-buffer variants need extra buffers: allocate them up front with
 *     sap_dpsr_reserve (then those calls never allocate either and can be captured in a CUDA graph
 *     from their first call); without it they allocate on their first use.
 *   - Every call must be made with the handle's device current (the one that was current in
 *     sap_dpsr_create); otherwise SAP_ERR_INVALID_ARG.
 *   - Work is enqueued on `stream` (a cudaStream_t cast to void*, NULL = default stream) and NOT
 *     synchronised, except where stated.  Device-side faults surface at the caller's next sync.
 *   - Preconditions not checked on the device: coordinates finite and in [0,1) (indices are wrapped
 *     mod N, nothing is ever written out of bounds).  If the shifted corner value a = chi'[0,0,0]-mu
 *     is 0 the scale is inf and chi is inf/NaN as IEEE dictates.
 *   - A handle is not thread-safe; use one handle per stream.
 */
#ifndef SAP_DPSR_H
#define SAP_DPSR_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sap_dpsr sap_dpsr_t; /* opaque */

typedef enum {
    SAP_OK = 0,
    SAP_ERR_INVALID_ARG = 1, /* null pointer, non-positive size, sigma < 0 or non-finite, num_points out of range */
    SAP_ERR_UNSUPPORTED = 2, /* N not in {32, 64, 128, 256, 512}; device is not sm_100 */
    SAP_ERR_OOM = 3,         /* workspace allocation failed */
    SAP_ERR_CUDA = 4         /* launch / runtime error; see sap_dpsr_last_error */
} sap_status_t;

/*
 * Create a solver for grids of N^3 (N in {32,64,128,256,512}: the resolutions of the paper's
 * coarse-to-fine schedule, plus 512), Gaussian bandwidth sigma >= 0 of Eq.3
 * (sigma = 0 means no filter, L460), `batch` independent shapes per call (the
 * learning setting uses 32, L419) and at most max_points points per shape.  The scale m of Eq.2 is
 * fixed to 0.5 (L77).  Allocates the workspace (about 8 N^3 floats per batch item) on the current
 * CUDA device.  *out is set only on SAP_OK.
 */
sap_status_t sap_dpsr_create(int N, float sigma, int batch, int max_points, sap_dpsr_t** out);

/*
 * Forward, Eq.2-4 = Eq.10-18 (L341-L388):
 *   splat normals with trilinear weights (Eq.10-11) -> 3 real-to-complex 3-D FFTs (Eq.12) ->
 *   chi~ = g_sigma(u) * i u.v~ / (-2 pi |u|^2), chi~(0) = 0 (Eq.3/16) -> inverse FFT (Eq.17) ->
 *   chi = s (chi' - mu), mu = mean over the points of the trilinear sample of chi',
 *   s = 0.5 / |chi'[0,0,0] - mu| (Eq.4/18, reading R5).
 *   points   dev [batch][num_points][3] float, coordinates in [0,1)
 *   normals  dev [batch][num_points][3] float, any magnitude (L494)
 *   num_points 1 <= num_points <= max_points, the same for every item of the batch
 *   chi      dev [batch][N][N][N] float, overwritten
 * The handle remembers (mu, a, s) per item and the points sorted into bins (with their original index)
 * for the backward, which re-rasterises the point density W from them.
 */
sap_status_t sap_dpsr_forward(sap_dpsr_t* h, const float* points, const float* normals,
                              int num_points, float* chi, void* stream);

/*
 * Backward: the exact adjoint of sap_dpsr_forward (dL/dpoints, dL/dnormals from dL/dchi); must
 * follow, on the same handle, the forward call it differentiates, with that call's chi, unmodified,
 * and NO other forward variant on the handle in between: the backward works from the state the
 * forward left in the handle (points and normals sorted into bins, mu, a, s).  `points` and `normals`
 * are accepted for symmetry with the forward and must be that call's inputs; they are not read
 * again.  A caller that interleaves forwards (two shapes per step, an evaluation forward inside a
 * training step) detects a stale handle with sap_dpsr_epoch / sap_dpsr_check_epoch below, or uses
 * one handle per live forward.  Derivation: DESIGN.md "Backward".
 *   chi          dev [batch][N][N][N]   forward output
 *   grad_chi     dev [batch][N][N][N]   dL/dchi
 *   grad_points  dev [batch][num_points][3], overwritten
 *   grad_normals dev [batch][num_points][3], overwritten
 */
sap_status_t sap_dpsr_backward(sap_dpsr_t* h, const float* points, const float* normals,
                               int num_points, const float* chi, const float* grad_chi,
                               float* grad_points, float* grad_normals, void* stream);

/*
 * Learning-based setting (Sec.3.3, Eq.9): L_DPSR = || chi - chi_gt ||^2, one value per item.
 * sap_dpsr_forward_mse is sap_dpsr_forward whose normalisation pass also evaluates the loss and its gradient
 * G = dL/dchi = 2 (chi - chi_gt) together with the grid reductions of the backward; G stays inside the handle
 * (one more N^3 grid per item, allocated on first use), so it never makes a round trip through the caller.
 *   chi_gt  dev [batch][N][N][N] float   target indicator grid
 *   chi     dev [batch][N][N][N] float   overwritten with the prediction (needed by the backward)
 *   loss    dev [batch] float            overwritten with the squared L2 distance of each item
 * sap_dpsr_backward_mse returns dL/dpoints and dL/dnormals of that loss; it must follow, on the same handle, the
 * sap_dpsr_forward_mse it differentiates, with the same points/normals and that call's chi, unmodified.
 */
sap_status_t sap_dpsr_forward_mse(sap_dpsr_t* h, const float* points, const float* normals,
                                  int num_points, const float* chi_gt, float* chi, float* loss,
                                  void* stream);
sap_status_t sap_dpsr_backward_mse(sap_dpsr_t* h, const float* points, const float* normals,
                                   int num_points, const float* chi, float* grad_points,
                                   float* grad_normals, void* stream);

/*
 * Host-buffer variants (the end-to-end path): the same computation with HOST pointers.  Inputs are
 * copied to handle-owned device staging buffers with cudaMemcpyAsync on `stream`, the kernels run,
 * and the outputs are copied back; the call returns after synchronising `stream`.
 * sap_dpsr_forward_host keeps chi on the device inside the handle for the backward that follows;
 * chi_host may be NULL to skip the device->host copy of chi.
 */
sap_status_t sap_dpsr_forward_host(sap_dpsr_t* h, const float* points_host,
                                   const float* normals_host, int num_points, float* chi_host,
                                   void* stream);
sap_status_t sap_dpsr_backward_host(sap_dpsr_t* h, const float* grad_chi_host,
                                    float* grad_points_host, float* grad_normals_host,
                                    void* stream);

/*
 * Every forward variant increments the handle's epoch.  sap_dpsr_epoch returns the epoch of the last
 * forward (0: none yet); sap_dpsr_check_epoch returns SAP_ERR_INVALID_ARG when `epoch` is not the
 * current one, i.e. when a backward for the forward that returned `epoch` would silently use another
 * call's bins and statistics.  The Python autograd wrapper keeps the epoch with the saved tensors.
 */
unsigned long long sap_dpsr_epoch(const sap_dpsr_t* h);
sap_status_t sap_dpsr_check_epoch(sap_dpsr_t* h, unsigned long long epoch);

/*
 * Allocates up front the optional buffers of the fused-loss path (SAP_RESERVE_MSE: one N^3 grid per
 * item) and / or of the host-buffer path (SAP_RESERVE_HOST: device staging for points, normals,
 * chi, dL/dchi and the gradients).  `what` is an OR of the flags.  Idempotent.
 */
enum { SAP_RESERVE_MSE = 1, SAP_RESERVE_HOST = 2 };
sap_status_t sap_dpsr_reserve(sap_dpsr_t* h, int what);

/*
 * Two implementations of the same path live in the library:
 *   SAP_PATH_THROUGHPUT  one kernel per pass (11 launches per forward+backward for N <= 128, 15 for N >= 256), persistent TMA rings:
 *                        every size, any batch;
 *   SAP_PATH_LATENCY     the whole forward and the whole backward as ONE cooperative kernel each, phases separated by grid
 *                        barriers, planes kept in shared memory across them (N <= 128 and batch * N <= number of SMs:
 *                        the 32^3 / 64^3 / 128^3 levels of the coarse-to-fine schedule, at batch 1).
 * SAP_PATH_AUTO (default) takes the latency path where it measured faster (eligible handles with N <= 64), else the
 * throughput path; SAP_PATH_LATENCY forces it on any eligible handle (else SAP_ERR_UNSUPPORTED).  Both leave the same state in the
 handle, so a forward on one path may be followed by the backward on the other.  sap_dpsr_get_path returns the path
 * the next call will take.  The fused-loss entry points always use the throughput path.
 */
enum { SAP_PATH_AUTO = 0, SAP_PATH_THROUGHPUT = 1, SAP_PATH_LATENCY = 2 };
sap_status_t sap_dpsr_set_path(sap_dpsr_t* h, int path);
int sap_dpsr_get_path(const sap_dpsr_t* h);

/*
 * Latency path only: device time between the grid barriers of the last forward and backward, stamped by CTA 0
 * (microseconds in us[i], static labels in names[i]; either may be NULL).  Blocking (device -> host copy on the
 * legacy stream).  Returns the number of entries written (at most cap).
 */
int sap_dpsr_get_fused_phases(sap_dpsr_t* h, float* us, const char** names, int cap);

/* Copies the per-item statistics of the last forward to host: stats_host[batch][3] = {mu, a, s}.
 * Synchronises `stream`. */
sap_status_t sap_dpsr_get_stats(sap_dpsr_t* h, float* stats_host, void* stream);

/*
 * Activity lists (on by default).  The binning of a forward also records which 32-line tiles (whole x-planes for
 * N <= 128) and which x-planes a point can touch at all (Eq.10-11: a point reaches the 8 grid nodes
 * around it).  The splatted field is identically zero elsewhere and the gather of the backward reads nothing there, so
 * the y and z passes of the three-channel spectra (forward y pass and inverse y pass for N >= 256, inverse z pass of
 * the backward for every N) only load, transform and store what is active; results are unchanged.
 * sap_dpsr_set_sparse(h, 0) makes every pass process every tile (for measurements); takes effect at the next forward.
 * sap_dpsr_get_activity copies the counts of the last throughput-path forward to host, summed over the batch:
 * out_host[4] = {active tiles, tiles, active planes, planes}; synchronises `stream`.  SAP_ERR_INVALID_ARG when the
 * lists are off or the last forward took the latency path (which keeps no lists).
 */
sap_status_t sap_dpsr_set_sparse(sap_dpsr_t* h, int on);
sap_status_t sap_dpsr_get_activity(sap_dpsr_t* h, int* out_host, void* stream);

/* Frees the workspace and the handle.  NULL is allowed. */
void sap_dpsr_destroy(sap_dpsr_t* h);

/* Message of the last error on this handle ("" if none); the string is owned by the handle.
 * With h == NULL returns the message of the last failed sap_dpsr_create on this thread. */
const char* sap_dpsr_last_error(const sap_dpsr_t* h);

/* Bytes of device workspace owned by the handle. */
size_t sap_dpsr_workspace_bytes(const sap_dpsr_t* h);

/* Number of kernel launches the last forward / backward call enqueued (for bench.py's gpu_launches). */
int sap_dpsr_last_launch_count(const sap_dpsr_t* h);

/*
 * Per-kernel timing for the bench (off by default).  When on, forward/backward record a CUDA event on
 * the caller's stream before their first launch and after every launch.  sap_dpsr_get_profile waits
 * for the last event of the most recent forward or backward call and writes, for each of its
 * launches in order, the device time in milliseconds between the surrounding events (ms[i]) and a
 * static kernel label (names[i]; either array may be NULL).  Returns the number of entries written
 * (at most cap), 0 if profiling is off or nothing was recorded.
 */
sap_status_t sap_dpsr_set_profiling(sap_dpsr_t* h, int on);
int sap_dpsr_get_profile(sap_dpsr_t* h, float* ms, const char** names, int cap);

#ifdef __cplusplus
}
#endif
#endif /* SAP_DPSR_H */
