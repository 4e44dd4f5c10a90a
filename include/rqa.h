/*
 * rqa.h — C ABI of librqa.so: the data-parallel hot path of averaged recurrence quantification analysis
 * (Panis, Adamek & Marwan, arXiv 2208.09136) on one NVIDIA B200 (sm_100a).
 *
 * Citations are lines of the paper's text and the readings S1..S18 listed in DESIGN.md.
 *
 * The path (sec. 2, 3, 5):
 *   rqa_embed       delay-coordinate embedding x_i[c] = y[i + c*tau]
 *   rqa_eps_for_rr  thresholds eps_k that realise K target recurrence rates:          PAPER.md:78, Eq. 3 (:63)
 *                   eps_k = the ceil(RR_k*P)-th smallest of the P = N'(N'-1)/2
 *                   pairwise distances (exact order statistic, readings S4-S6)
 *   rqa_line_hist   diagonal-line-length histograms P_k(l) of the recurrence plot     PAPER.md:69-72 (Eq. 4), :125
 *                   R_ij = (d_ij <= eps_k), all K thresholds in one pass, upper
 *                   triangle only, R never stored
 *   rqa_det_avg     DET_k (Eq. 4) and its average over the K recurrence rates (Eq. 5)
 * On top of it: rqa_det_prefix_avg (Eq. 5 for every cut-off), rqa_line_measures (L, L_max, RR from the
 * histogram) and rqa_sorting_rate_host (Eq. 6).
 *
 * Conventions (BASELINE.json north_star):
 *   - distances are fp32: maximum norm max_c |x_i[c]-x_j[c]|, or the Euclidean norm computed
 *     as sqrtf(((t0*t0 + t1*t1) + ...)) in the order c = 0..m-1, every operation rounded to fp32, no FMA;
 *   - recurrence means d <= eps (S1); the main diagonal is excluded and only pairs i<j are counted (S2);
 *   - "N" of the paper is N' = N - (m-1)*tau embedded points everywhere (S3);
 *   - runs that touch the border of the plot count with their truncated length (S8);
 *   - counts are exact uint64; RR and DET are fp64 ratios of exact integers.
 *
 * Workspace size: rqa_workspace_bytes sizes for the worst case of the shape (the recurrence rates are not known then): about
 * 0.9 GB per series of 1e5 points at K = 20 (candidate list of the threshold select, up to 6 % of the pairs; segment
 * summaries of the scans), 126 MB per series of 2e4 points at K = 32, linear in the batch.
 *
 * Memory and ownership: every buffer is owned by the caller.  Pointers named d_* are DEVICE pointers,
 * h_* are HOST pointers.  The library keeps no device allocation and no global state between calls (the only
 * process-wide datum is the monotone launch counter behind rqa_launch_count()), with ONE stated exception: the static
 * scratch array of rqa_line_hist_static, the entry point for callers that cannot allocate (see there).
 * Every call enqueues its work on `stream` (a cudaStream_t passed as void*; NULL = the legacy default
 * stream) and returns without synchronising; outputs are valid once the stream has been synchronised.
 *
 * Errors: a status code is returned, never an exception or an abort.  Argument errors are detected
 * before anything is launched.  rqa_last_error() gives a thread-local detail string.  Conditions that can
 * only be seen on the device (NaN/Inf in the series) are recorded in the workspace and reported by
 * rqa_workspace_status().
 *
 * There is no CPU fallback: without a CUDA device every compute call returns RQA_ERR_CUDA.
 */
#ifndef RQA_H
#define RQA_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define RQA_MAX_K 128 /* maximum number of thresholds per call */
#define RQA_MAX_M 16  /* maximum embedding dimension */

typedef enum {
    RQA_OK = 0,
    RQA_ERR_INVALID_ARG = 1,
    RQA_ERR_NONFINITE_INPUT = 2,
    RQA_ERR_WORKSPACE_TOO_SMALL = 3,
    RQA_ERR_UNSUPPORTED = 4,
    RQA_ERR_CUDA = 5
} rqa_status;

typedef enum { RQA_NORM_MAX = 0, RQA_NORM_EUCLID = 1 } rqa_norm;

/*
 * A batch of point sets, as a strided view of fp32 device memory:
 *     x_i[c] of series b = data[b*batch_stride + i*point_stride + c*coord_stride],  0<=i<n_points, 0<=c<m.
 * Delay view of raw series (what rqa_embed returns when d_X == NULL): point_stride = 1, coord_stride = tau.
 * Materialised row-major X[batch][n_points][m]:                       point_stride = m, coord_stride = 1.
 * All series of a batch share n_points, m and the strides.  Strides are in elements and must be >= 1.
 * theiler = w > 1 excludes the diagonals j - i < w as well (temporally correlated neighbours; the paper uses none,
 * reading S9): every "P" below is then P_w = (N'-w)(N'-w+1)/2, the number of pairs with j - i >= w, and lines are
 * counted on the diagonals j - i = w..N'-1.  w <= N'-1.
 */
typedef struct rqa_points {
    const float* data; /* device pointer */
    int64_t n_points;  /* N' >= 2 */
    int32_t m;         /* 1..RQA_MAX_M */
    int32_t batch;     /* >= 1 */
    int64_t point_stride;
    int64_t coord_stride;
    int64_t batch_stride;
    int64_t theiler;   /* Theiler window w: only pairs with j - i >= w are counted; 0 or 1 = the main diagonal only */
} rqa_points;

const char* rqa_status_string(rqa_status s);
const char* rqa_last_error(void);
/* "major.minor sm_100a" build tag; never NULL. */
const char* rqa_version(void);

/*
 * Bytes of device workspace that rqa_eps_for_rr / rqa_line_hist / rqa_vert_hist need for this shape (the largest).
 * The workspace is scratch: its contents need not survive between calls, except that rqa_workspace_status()
 * reads the status block the last call wrote.  It must be 256-byte aligned.
 */
rqa_status rqa_workspace_bytes(const rqa_points* pts, int32_t K, size_t* bytes);

/*
 * Synchronises `stream`, then returns what the last call that used this workspace recorded on the device:
 * RQA_OK, RQA_ERR_NONFINITE_INPUT (a NaN or Inf among the points; outputs are then undefined) or
 * RQA_ERR_CUDA.
 */
rqa_status rqa_workspace_status(const void* d_ws, void* stream);

/*
 * Delay embedding (forward indexing, reading S7).  N' = N - (m-1)*tau must be >= 2.
 *   d_series  [batch] series of N samples, series b at d_series + b*series_stride
 *   d_X       NULL: nothing is copied, *view_out describes the strided delay view of d_series;
 *             else: [batch][N'][m] row-major, written by the call, and *view_out describes it.
 */
rqa_status rqa_embed(const float* d_series, int64_t N, int32_t batch, int64_t series_stride, int32_t m,
                     int64_t tau, float* d_X, rqa_points* view_out, void* stream);

/*
 * Thresholds for target recurrence rates (readings S4-S6).
 *   h_rr            HOST array of K target rates, each in (0, 1], any order, duplicates allowed
 *   d_eps           [batch][K] eps_k = the r_k-th smallest pairwise distance, r_k = ceil(rr_k * P) evaluated
 *                   in fp64 and clamped to [1, P], P = N'(N'-1)/2 — in the caller's order of h_rr
 *   d_count         [batch][K] C_k = #{i<j : d_ij <= eps_k}  (>= r_k when there are ties)
 *   d_rr_realised   [batch][K] (double)C_k / (double)P
 * 1 <= K <= RQA_MAX_K.
 */
rqa_status rqa_eps_for_rr(const rqa_points* pts, rqa_norm norm, const double* h_rr, int32_t K, float* d_eps,
                          uint64_t* d_count, double* d_rr_realised, void* d_ws, size_t ws_bytes, void* stream);

/*
 * Diagonal-line histograms at K thresholds.
 *   d_eps   [batch][K] thresholds (device), any order, duplicates allowed, each finite and >= 0
 *   d_hist  [batch][K][n_points] uint64, overwritten: d_hist[b][k][l] = number of maximal runs of exactly l
 *           consecutive recurrent cells (d <= eps_k) along the diagonals j-i = 1..N'-1; [..][0] = 0.
 * Invariant tying it to rqa_eps_for_rr: sum_l l*d_hist[b][k][l] == C_k.
 * The strict Heaviside of the paper's Eq. 2 (H(0) = 0, recurrence means d < eps) needs no other kernel:
 * fp32 distances are discrete, so d < eps is d <= nextafterf(eps, -inf) for eps > 0; pass those thresholds.
 */
rqa_status rqa_line_hist(const rqa_points* pts, rqa_norm norm, const float* d_eps, int32_t K, uint64_t* d_hist,
                         void* d_ws, size_t ws_bytes, void* stream);

/*
 * DET_k = sum_{l>=l_min} l*P_k(l) / sum_{l>=1} l*P_k(l)  (Eq. 4; 0 if the denominator is 0) and
 * mean_b = (1/K) * sum_{k=0}^{K-1} DET_k, summed left to right in fp64 (Eq. 5; reading S11).
 *   d_hist      [batch][K][n_points] from rqa_line_hist
 *   d_det       [batch][K]     d_det_mean  [batch]
 */
rqa_status rqa_det_avg(const uint64_t* d_hist, int32_t batch, int32_t K, int64_t n_points, int64_t l_min,
                       double* d_det, double* d_det_mean, void* stream);

/*
 * Eq. 5 as a curve ("we test the averaging for RR* in [1, 2, 3, ..., 99]"): the averaged determinism
 * for every cut-off, d_prefix[b][k] = (d_det[b][0] + ... + d_det[b][k]) / (k+1), summed left to right in fp64, in the
 * caller's order of the recurrence rates (pass them ascending for the paper's curve).  d_prefix[b][0] = d_det[b][0]
 * ("the average of one value is the value itself"); d_prefix[b][K-1] = rqa_det_avg's mean.
 *   d_det     [batch][K] from rqa_det_avg        d_prefix  [batch][K]
 */
rqa_status rqa_det_prefix_avg(const double* d_det, int32_t batch, int32_t K, double* d_prefix, void* stream);

/*
 * The other measures the paper derives from the same histogram ("DET, L, L_max and RR"):
 *   d_L        [batch][K] average diagonal line length  sum_{l>=l_min} l*P_k(l) / sum_{l>=l_min} P_k(l)  (0 if no line)
 *   d_Lmax     [batch][K] longest diagonal line  max{ l : P_k(l) > 0 }  (0 if none)
 *   d_rr_hist  [batch][K] recurrence rate from the histogram  sum_{l>=1} l*P_k(l) / P,  P = N'(N'-1)/2 (or P_w for the
 *              Theiler window `theiler` the histogram was built with; 0 or 1 = none)
 * and, as one of the "other RQA measures" the averaging applies to (not defined in the paper itself),
 *   d_entr     [batch][K] Shannon entropy of the line-length distribution  -sum_{l>=l_min} p(l) ln p(l),
 *              p(l) = P_k(l) / sum_{l>=l_min} P_k(l)  (0 if no line), computed as ln T - (1/T) sum P ln P in fp64.
 * Any of the four outputs may be NULL.  Integer sums are exact uint64; L and RR are one fp64 division.
 */
rqa_status rqa_line_measures(const uint64_t* d_hist, int32_t batch, int32_t K, int64_t n_points, int64_t l_min,
                             int64_t theiler, double* d_L, uint64_t* d_Lmax, double* d_rr_hist, double* d_entr,
                             void* stream);

/*
 * Vertical-line histograms at K thresholds ("this approach can also be applied for other RQA measures": the
 * vertical-line measures laminarity and trapping time; the paper defines none itself, reading S19).
 *   d_vhist  [batch][K][n_points] uint64, overwritten: d_vhist[b][k][v] = number of maximal runs of exactly v recurrent
 *            cells (d <= eps_k) down the columns of the FULL symmetric N' x N' matrix.  The cells with
 *            |i - j| < w (w = 1: the main diagonal; w = pts->theiler > 1: the Theiler window) are not recurrent and split
 *            a column in two; runs touching the border of the plot or that band count with their truncated length.
 * Every recurrent pair i<j lies in column j and in column i: sum_v v*d_vhist[b][k][v] == 2*C_k.
 * Arguments, workspace (rqa_workspace_bytes covers it) and errors as rqa_line_hist; N'^2 cells are visited.
 */
rqa_status rqa_vert_hist(const rqa_points* pts, rqa_norm norm, const float* d_eps, int32_t K, uint64_t* d_vhist,
                         void* d_ws, size_t ws_bytes, void* stream);

/*
 * Laminarity and trapping time from the vertical-line histogram (the definitions of the paper's ref. [2], which
 * PAPER.md:86 points to; not written out in the paper):
 *   d_lam  [batch][K]  LAM_k = sum_{v>=v_min} v*P_k(v) / sum_{v>=1} v*P_k(v)            (0 if the denominator is 0)
 *   d_tt   [batch][K]  TT_k  = sum_{v>=v_min} v*P_k(v) / sum_{v>=v_min} P_k(v)          (0 if there is no such line)
 * Exact uint64 sums, one fp64 division each.  Either output may be NULL.  Their averages over the recurrence rates (Eq. 5
 * applied to LAM / TT) are rqa_det_prefix_avg on d_lam / d_tt.
 */
rqa_status rqa_lam_tt(const uint64_t* d_vhist, int32_t batch, int32_t K, int64_t n_points, int64_t v_min, double* d_lam,
                      double* d_tt, void* stream);

/*
 * Sorting rate S (Eq. 6), the paper's evaluation score; plain host arithmetic on R*n numbers.
 *   h_measure  HOST [R][n]: the measure (DET or averaged DET) of n series given in their natural order (y_j = j, the
 *              order the measure is expected to increase in), for R realisations
 *   h_S        HOST: (W - D) / W with D = sum_i sum_j |x_j - y_j|, x_j = place of series j when the n values of one
 *              realisation are ordered ascending (equal values keep the given order), and W = R * sum_j |n+1-2j|
 *              (= 500 for n = R = 10).  1 = perfectly sorted, 0 = reversed.
 */
rqa_status rqa_sorting_rate_host(const double* h_measure, int32_t R, int32_t n, double* h_S);

/*
 * The whole path for HOST buffers (what bench.py's `e2e` times): copies the series to the device workspace,
 * runs rqa_embed (view) -> rqa_eps_for_rr -> rqa_line_hist -> rqa_det_avg on `stream`, copies the results
 * back and synchronises the stream before returning.
 *   h_series  [batch][N] fp32 (pinned memory gives asynchronous copies)
 *   h_eps, h_count, h_rr_realised, h_det  [batch][K];  h_det_mean [batch];  h_hist [batch][K][N'] or NULL
 *   d_ws      device workspace of at least rqa_sweep_workspace_bytes(...) bytes
 */
rqa_status rqa_sweep_workspace_bytes(int64_t N, int32_t batch, int32_t m, int64_t tau, int32_t K, size_t* bytes);
rqa_status rqa_sweep_host(const float* h_series, int64_t N, int32_t batch, int32_t m, int64_t tau, rqa_norm norm,
                          const double* h_rr, int32_t K, int64_t l_min, float* h_eps, uint64_t* h_count,
                          double* h_rr_realised, double* h_det, double* h_det_mean, uint64_t* h_hist, void* d_ws,
                          size_t ws_bytes, void* stream);

/*
 * Number of kernel launches the library has enqueued from this process so far (monotone counter; bench.py
 * reports the difference over its timed region as `gpu_launches`).
 */
uint64_t rqa_launch_count(void);

/*
 * Per-call options (expert / testing knobs and the multi-GPU split).  The library keeps NO global state: the plain
 * calls above are the `_opt` calls below with opt = NULL (every field 0 = automatic).  Options change how a result is
 * computed, never the result (every path of rqa_eps_for_rr is exact).  Workspace sizes depend on them: pass the same
 * options to rqa_workspace_bytes_opt and to the call that uses the workspace.
 *   select_path   rqa_eps_for_rr: 0 automatic, 1 = materialise all distances (small P), 2 = sample-bracket + one
 *                 counting pass, 3 = four radix passes.  The radix passes serve views the tiled passes cannot stage
 *                 (coordinate span above 4096 elements, very wide points) and are the automatic recovery of a bracket
 *                 miss; they recompute every distance from global memory four times and cost about 20 x the bracket path
 *                 (88 ms instead of 4 ms per series of 1e5 points on a B200).  4 = one thread block per series, three
 *                 walks over the triangle with shared-memory histograms, nothing materialised (P <= 2^22 only; otherwise
 *                 automatic).  Automatic: series of at most 8192 pairs are sorted whole in shared memory, P <= 2^22
 *                 takes path 4 for batches of at least 12 series and path 1 below, everything else path 2.
 *   sample_size   bracket path: number of sampled pair distances per series
 *   cand_cap      bracket path: capacity of the candidate list per series (overflow falls back to the radix passes)
 *   line_chunk    rqa_line_hist / rqa_vert_hist: chunk length along the diagonals / columns, 1..1023
 *   line_segment  rqa_line_hist: consecutive chunks of one diagonal block that a block walks with the run state
 *                 carried in place (only segment borders are joined by the stitch kernel), >= 1
 *   line_buffers  rqa_line_hist: 1 = one set of series windows per block, staged by plain loads; 2 = two sets, the next
 *                 chunk's windows fetched by bulk asynchronous copies while the current chunk is scanned
 *   group_size    thresholds (targets) per pass of the grouped kernels of all three heavy calls, 1..32; 0 automatic: K <= 32
 *                 in one pass, more in groups of 20 (a pass over at most 20 thresholds keeps two blocks per SM; 7 % faster
 *                 and a third less workspace than groups of 32 at K = 99)
 *   line_path     rqa_line_hist / rqa_vert_hist: 0 automatic, 1 = the tiled scan, 2 = one thread block per series walking
 *                 every diagonal / column once for all K thresholds (P <= 2^22 only; otherwise automatic).  Automatic: series of at most 8192
 *                 pairs take their one-block kernel, P <= 2^22 takes path 2 when the batch is large enough to fill the
 *                 GPU with such blocks (batch x ceil(K/32) >= 192), everything else the tiled scan.
 *   part_index, part_count
 *                 split of ONE call over part_count processes (one GPU each): this process visits
 *                 only its share of the tiles of the triangle (diagonal blocks part_index, part_index + part_count,
 *                 ...), and every exact integer counter that must be summed over the parts before the next step can
 *                 use it (level counts and digit bins of rqa_eps_for_rr; line aggregates and the histogram of
 *                 rqa_line_hist) is handed to `reduce`.  After the call every part holds the complete, identical
 *                 outputs.  part_count <= 1: the whole job, `reduce` is not called.
 *   reduce        int reduce(ctx, d_counters, n, stream): sum the n uint64 device counters at d_counters element-wise
 *                 over all parts, in place, ordered on `stream` (e.g. ncclAllReduce(ncclUint64, ncclSum), or
 *                 torch.distributed.all_reduce on a tensor wrapping the pointer); return 0 on success.  Every part
 *                 makes the same sequence of reduce calls with the same n.
 *   ev_kernel_begin, ev_kernel_end
 *                 measurement hooks (NULL = none): two cudaEvent_t created by the caller, recorded on `stream` just before
 *                 and just after the launch(es) of the call's dominant kernel — the counting pass over all cells of
 *                 rqa_eps_for_rr (first group of 32 targets), the diagonal scan of rqa_line_hist (first group of 32
 *                 thresholds) — so that a caller can time that kernel alone without a profiler.  Not recorded when the call
 *                 takes a path without that kernel (small P, strided fallback).
 */
typedef int (*rqa_reduce_fn)(void* ctx, uint64_t* d_counters, size_t n, void* stream);
typedef struct rqa_options {
    int32_t select_path;
    int32_t line_chunk;
    int32_t line_segment;
    int32_t part_index;
    int32_t part_count;
    int32_t line_buffers;
    int64_t sample_size;
    int64_t cand_cap;
    rqa_reduce_fn reduce;
    void* reduce_ctx;
    void* ev_kernel_begin;
    void* ev_kernel_end;
    int32_t line_path;
    int32_t group_size;
} rqa_options;

rqa_status rqa_workspace_bytes_opt(const rqa_points* pts, int32_t K, const rqa_options* opt, size_t* bytes);
rqa_status rqa_eps_for_rr_opt(const rqa_points* pts, rqa_norm norm, const double* h_rr, int32_t K, float* d_eps,
                              uint64_t* d_count, double* d_rr_realised, void* d_ws, size_t ws_bytes, void* stream,
                              const rqa_options* opt);
rqa_status rqa_line_hist_opt(const rqa_points* pts, rqa_norm norm, const float* d_eps, int32_t K, uint64_t* d_hist,
                             void* d_ws, size_t ws_bytes, void* stream, const rqa_options* opt);
rqa_status rqa_vert_hist_opt(const rqa_points* pts, rqa_norm norm, const float* d_eps, int32_t K, uint64_t* d_vhist,
                             void* d_ws, size_t ws_bytes, void* stream, const rqa_options* opt);

/*
 * rqa_line_hist for callers that cannot allocate device memory (code under CUDA-graph capture,
 * tight serving loops, harnesses that forbid cudaMalloc): same arguments minus the workspace, same kernels, same
 * results bit for bit.  The scratch is a static device array of RQA_STATIC_SCRATCH_BYTES inside the library; the call
 * makes no cudaMalloc / cudaFree / allocating library call and is asynchronous on `stream` like rqa_line_hist.
 *   - every GPU on which the process uses this call holds RQA_STATIC_SCRATCH_BYTES of device memory until exit;
 *   - a shape whose scan needs more scratch returns RQA_ERR_UNSUPPORTED (nothing launched; the message states the
 *     bytes needed).  The scan's scratch grows with the number of tiles it cuts the triangle into, not simply with N:
 *     BASELINE.json's configs 1-3 fit (6 series of 10^4 points at K = 20 need 113 MiB), one series of 10^4 points fits
 *     at any K, one series of 10^5 points does not (207 MiB); a batch that runs as one block per series (line_path
 *     above) needs none at all, e.g. 900 series of 10^3 points at K = 99;
 *   - all calls on one device share the array and it keeps the last call's contents: calls in stream order are
 *     independent (the path clears what must start at zero), calls that OVERLAP on the GPU race — serialise them or use
 *     rqa_line_hist with one workspace per stream;
 *   - a non-finite point or a bad threshold is recorded in the scratch as in a workspace; there is no
 *     rqa_workspace_status for it (validate inputs with the workspace calls where that matters).
 * Errors: as rqa_line_hist, plus RQA_ERR_UNSUPPORTED as above and RQA_ERR_CUDA if the scratch address cannot be got.
 */
#define RQA_STATIC_SCRATCH_BYTES (128u << 20)
rqa_status rqa_line_hist_static(const rqa_points* pts, rqa_norm norm, const float* d_eps, int32_t K, uint64_t* d_hist,
                                void* stream);

#ifdef __cplusplus
}
#endif
#endif /* RQA_H */
