// rqa_api.cu — the C ABI of librqa.so (include/rqa.h): argument validation, workspace carving, and the
// small kernels of the path (embedding gather, finite check, DET reduction).  The two heavy steps live in
// rqa_select.cu (thresholds) and rqa_line.cu (line histograms).
#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>

#include "rqa_common.cuh"

namespace rqa {

static thread_local char t_err[512] = "";
std::atomic<uint64_t> g_launches{0};

rqa_status make_options(const rqa_options* in, Options* out, const char* who) {
    *out = Options{};
    if (!in) return RQA_OK;
    if (in->select_path < 0 || in->select_path > 4) { set_error("%s: options.select_path is 0..4", who); return RQA_ERR_INVALID_ARG; }
    if (in->line_chunk < 0 || in->line_chunk > 1023) { set_error("%s: options.line_chunk is 0..1023", who); return RQA_ERR_INVALID_ARG; }
    if (in->line_buffers < 0 || in->line_buffers > 2) { set_error("%s: options.line_buffers is 0..2", who); return RQA_ERR_INVALID_ARG; }
    if (in->line_path < 0 || in->line_path > 2) { set_error("%s: options.line_path is 0..2", who); return RQA_ERR_INVALID_ARG; }
    if (in->group_size < 0 || in->group_size > 32) { set_error("%s: options.group_size is 0..32", who); return RQA_ERR_INVALID_ARG; }
    if (in->line_segment < 0) { set_error("%s: options.line_segment must be >= 0", who); return RQA_ERR_INVALID_ARG; }
    if (in->sample_size < 0 || in->cand_cap < 0) { set_error("%s: options.sample_size and cand_cap must be >= 0", who); return RQA_ERR_INVALID_ARG; }
    if (in->part_count < 0 || in->part_index < 0 || (in->part_count > 0 && in->part_index >= in->part_count) ||
        (in->part_count == 0 && in->part_index != 0)) {
        set_error("%s: options need 0 <= part_index < part_count", who);
        return RQA_ERR_INVALID_ARG;
    }
    if (in->part_count > 1 && !in->reduce) { set_error("%s: options.part_count > 1 needs a reduce callback", who); return RQA_ERR_INVALID_ARG; }
    out->select_path = in->select_path;
    out->line_chunk = in->line_chunk;
    out->line_segment = in->line_segment;
    out->line_buffers = in->line_buffers;
    out->line_path = in->line_path;
    out->group_size = in->group_size;
    out->sample_size = in->sample_size;
    out->cand_cap = in->cand_cap;
    out->parts = in->part_count > 1 ? in->part_count : 1;
    out->part = in->part_count > 1 ? in->part_index : 0;
    out->reduce = in->reduce;
    out->reduce_ctx = in->reduce_ctx;
    out->ev_begin = in->ev_kernel_begin;
    out->ev_end = in->ev_kernel_end;
    return RQA_OK;
}

int sm_count() {
    static thread_local int cached_dev = -1, cached = 148;
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return 148; }
    if (dev != cached_dev) {
        int n = 0;
        if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && n > 0) cached = n;
        else { cudaGetLastError(); cached = 148; }
        cached_dev = dev;
    }
    return cached;
}

void set_error(const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(t_err, sizeof(t_err), fmt, ap);
    va_end(ap);
}

rqa_status validate_points(const rqa_points* p, const char* who) {
    if (!p) { set_error("%s: pts is NULL", who); return RQA_ERR_INVALID_ARG; }
    if (!p->data) { set_error("%s: pts->data is NULL", who); return RQA_ERR_INVALID_ARG; }
    if (p->n_points < 2) { set_error("%s: n_points = %lld < 2", who, (long long)p->n_points); return RQA_ERR_INVALID_ARG; }
    if (p->n_points > (int64_t)1 << 24) { set_error("%s: n_points = %lld > 2^24 unsupported", who, (long long)p->n_points); return RQA_ERR_UNSUPPORTED; }
    if (p->m < 1 || p->m > RQA_MAX_M) { set_error("%s: m = %d outside 1..%d", who, p->m, RQA_MAX_M); return RQA_ERR_INVALID_ARG; }
    if (p->batch < 1) { set_error("%s: batch = %d < 1", who, p->batch); return RQA_ERR_INVALID_ARG; }
    if (p->batch > 65535) { set_error("%s: batch = %d > 65535 unsupported (one grid row per series)", who, p->batch); return RQA_ERR_UNSUPPORTED; }
    if (p->point_stride < 1 || p->coord_stride < 1 || p->batch_stride < 0) { set_error("%s: strides must be >= 1", who); return RQA_ERR_INVALID_ARG; }
    if (p->batch > 1 && p->batch_stride < 1) { set_error("%s: batch_stride must be >= 1 when batch > 1", who); return RQA_ERR_INVALID_ARG; }
    if (p->theiler < 0 || p->theiler > p->n_points - 1) { set_error("%s: theiler = %lld outside 0..n_points-1", who, (long long)p->theiler); return RQA_ERR_INVALID_ARG; }
    return RQA_OK;
}

// ------------------------------------------------------------------------------------------- kernels
__global__ void embed_kernel(const float* __restrict__ y, int64_t N, int64_t series_stride, int m, int64_t tau,
                             int64_t n, float* __restrict__ X) {
    int b = blockIdx.y;
    int64_t total = n * m;
    for (int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; q < total; q += (int64_t)gridDim.x * blockDim.x) {
        int64_t i = q / m;
        int c = (int)(q - i * m);
        X[(int64_t)b * total + q] = y[(int64_t)b * series_stride + i + c * tau];
    }
}

__global__ void finite_check_kernel(View v, WsStatus* st) {
    int b = blockIdx.y;
    const float* yb = v.data + (int64_t)b * v.bs;
    int64_t total = v.n * v.m;
    bool bad = false;
    for (int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; q < total; q += (int64_t)gridDim.x * blockDim.x) {
        int64_t i = q / v.m;
        int c = (int)(q - i * v.m);
        float x = yb[i * v.ps + c * v.cs];
        bad |= !isfinite(x);
    }
    if (__syncthreads_or(bad) && threadIdx.x == 0) atomicExch(&st->nonfinite, 1);
}

__global__ void status_reset_kernel(WsStatus* st) {
    if (threadIdx.x < 64) ((int32_t*)st)[threadIdx.x] = 0;
}

// One block per (k, b): exact uint64 sums of l*P(l) (Eq. 4).
__global__ void det_kernel(const uint64_t* __restrict__ hist, int K, int64_t n, int64_t l_min, double* __restrict__ det) {
    int k = blockIdx.x, b = blockIdx.y;
    const uint64_t* h = hist + ((int64_t)b * K + k) * n;
    unsigned long long num = 0, den = 0;
    for (int64_t l = 1 + threadIdx.x; l < n; l += blockDim.x) {
        unsigned long long w = (unsigned long long)l * h[l];
        den += w;
        if (l >= l_min) num += w;
    }
    __shared__ unsigned long long s_num[32], s_den[32];
    for (int off = 16; off; off >>= 1) {
        num += __shfl_down_sync(0xffffffffu, num, off);
        den += __shfl_down_sync(0xffffffffu, den, off);
    }
    int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (lane == 0) { s_num[w] = num; s_den[w] = den; }
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned long long a = 0, c = 0;
        for (int q = 0; q < (int)(blockDim.x >> 5); ++q) { a += s_num[q]; c += s_den[q]; }
        det[(int64_t)b * K + k] = c ? (double)a / (double)c : 0.0;
    }
}

// Short rows (the many-short-series regime of the paper's grid): one WARP per (k, b) row, eight rows per block.
__global__ void __launch_bounds__(256) det_rows_kernel(const uint64_t* __restrict__ hist, int64_t rows, int64_t n, int64_t l_min,
                                                       double* __restrict__ det) {
    const int64_t row = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (row >= rows) return;
    const uint64_t* h = hist + row * n;
    unsigned long long num = 0, den = 0;
    for (int64_t l = 1 + (threadIdx.x & 31); l < n; l += 32) {
        unsigned long long w = (unsigned long long)l * h[l];
        den += w;
        if (l >= l_min) num += w;
    }
    for (int off = 16; off; off >>= 1) {
        num += __shfl_down_sync(0xffffffffu, num, off);
        den += __shfl_down_sync(0xffffffffu, den, off);
    }
    if ((threadIdx.x & 31) == 0) det[row] = den ? (double)num / (double)den : 0.0;
}

// Eq. 5: mean over the K rates, summed k = 0..K-1 left to right in fp64 (reading S11).
__global__ void det_mean_kernel(const double* __restrict__ det, int K, int batch, double* __restrict__ mean) {
    int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= batch) return;
    double s = 0.0;
    for (int k = 0; k < K; ++k) s += det[(int64_t)b * K + k];
    mean[b] = s / (double)K;
}

rqa_status launch_finite_check(const View& v, WsStatus* st, cudaStream_t s) {
    status_reset_kernel<<<1, 64, 0, s>>>(st);
    RQA_LAUNCH_CHECK();
    int64_t total = v.n * v.m;
    int blocks = (int)std::min<int64_t>((total + 255) / 256, 1024);
    finite_check_kernel<<<dim3(blocks, v.batch), 256, 0, s>>>(v, st);
    RQA_LAUNCH_CHECK();
    return RQA_OK;
}

}  // namespace rqa

using namespace rqa;

extern "C" {

const char* rqa_status_string(rqa_status s) {
    switch (s) {
        case RQA_OK: return "RQA_OK";
        case RQA_ERR_INVALID_ARG: return "RQA_ERR_INVALID_ARG";
        case RQA_ERR_NONFINITE_INPUT: return "RQA_ERR_NONFINITE_INPUT";
        case RQA_ERR_WORKSPACE_TOO_SMALL: return "RQA_ERR_WORKSPACE_TOO_SMALL";
        case RQA_ERR_UNSUPPORTED: return "RQA_ERR_UNSUPPORTED";
        case RQA_ERR_CUDA: return "RQA_ERR_CUDA";
    }
    return "RQA_ERR_UNKNOWN";
}

const char* rqa_last_error(void) { return t_err; }
const char* rqa_version(void) { return "0.1 sm_100a"; }
uint64_t rqa_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }

rqa_status rqa_workspace_bytes_opt(const rqa_points* pts, int32_t K, const rqa_options* opt, size_t* bytes) {
    if (!bytes) { set_error("rqa_workspace_bytes: bytes is NULL"); return RQA_ERR_INVALID_ARG; }
    if (!pts) { set_error("rqa_workspace_bytes: pts is NULL"); return RQA_ERR_INVALID_ARG; }
    if (K < 1 || K > RQA_MAX_K) { set_error("rqa_workspace_bytes: K = %d outside 1..%d", K, RQA_MAX_K); return RQA_ERR_INVALID_ARG; }
    Options o;
    rqa_status st = make_options(opt, &o, "rqa_workspace_bytes");
    if (st != RQA_OK) return st;
    // data pointer is not needed for sizing
    rqa_points p = *pts;
    if (!p.data) p.data = (const float*)(uintptr_t)256;
    st = validate_points(&p, "rqa_workspace_bytes");
    if (st != RQA_OK) return st;
    View v = make_view(p);
    size_t a = select_workspace_bytes(v, K, o), b = line_workspace_bytes(v, K, o), c = vert_workspace_bytes(v, K, o);
    *bytes = sizeof(WsStatus) + std::max(a, std::max(b, c));
    return RQA_OK;
}

rqa_status rqa_workspace_bytes(const rqa_points* pts, int32_t K, size_t* bytes) {
    return rqa_workspace_bytes_opt(pts, K, nullptr, bytes);
}

rqa_status rqa_workspace_status(const void* d_ws, void* stream) {
    if (!d_ws) { set_error("rqa_workspace_status: d_ws is NULL"); return RQA_ERR_INVALID_ARG; }
    cudaStream_t s = (cudaStream_t)stream;
    WsStatus h;
    RQA_CUDA_TRY(cudaMemcpyAsync(&h, d_ws, sizeof(h), cudaMemcpyDeviceToHost, s));
    RQA_CUDA_TRY(cudaStreamSynchronize(s));
    if (h.nonfinite) { set_error("non-finite value (NaN or Inf) among the input points"); return RQA_ERR_NONFINITE_INPUT; }
    if (h.bad_eps) { set_error("rqa_line_hist: a threshold is NaN, Inf or negative"); return RQA_ERR_INVALID_ARG; }
    if (h.internal) { set_error("internal inconsistency recorded on the device"); return RQA_ERR_CUDA; }
    return RQA_OK;
}

rqa_status rqa_embed(const float* d_series, int64_t N, int32_t batch, int64_t series_stride, int32_t m, int64_t tau,
                     float* d_X, rqa_points* view_out, void* stream) {
    if (!d_series || !view_out) { set_error("rqa_embed: NULL argument"); return RQA_ERR_INVALID_ARG; }
    if (m < 1 || m > RQA_MAX_M || tau < 1 || batch < 1) { set_error("rqa_embed: need 1 <= m <= %d, tau >= 1, batch >= 1", RQA_MAX_M); return RQA_ERR_INVALID_ARG; }
    if (batch > 1 && series_stride < N) { set_error("rqa_embed: series_stride < N"); return RQA_ERR_INVALID_ARG; }
    int64_t n = N - (int64_t)(m - 1) * tau;
    if (n < 2) { set_error("rqa_embed: N' = N - (m-1)*tau = %lld < 2", (long long)n); return RQA_ERR_INVALID_ARG; }
    rqa_points v;
    v.n_points = n; v.m = m; v.batch = batch; v.theiler = 0;
    if (!d_X) {
        v.data = d_series; v.point_stride = 1; v.coord_stride = tau; v.batch_stride = series_stride;
    } else {
        cudaStream_t s = (cudaStream_t)stream;
        int blocks = (int)std::min<int64_t>((n * m + 255) / 256, 2048);
        embed_kernel<<<dim3(blocks, batch), 256, 0, s>>>(d_series, N, series_stride, m, tau, n, d_X);
        RQA_LAUNCH_CHECK();
        v.data = d_X; v.point_stride = m; v.coord_stride = 1; v.batch_stride = n * m;
    }
    *view_out = v;
    return RQA_OK;
}

rqa_status rqa_eps_for_rr(const rqa_points* pts, rqa_norm norm, const double* h_rr, int32_t K, float* d_eps,
                          uint64_t* d_count, double* d_rr_realised, void* d_ws, size_t ws_bytes, void* stream) {
    return rqa_eps_for_rr_opt(pts, norm, h_rr, K, d_eps, d_count, d_rr_realised, d_ws, ws_bytes, stream, nullptr);
}

rqa_status rqa_eps_for_rr_opt(const rqa_points* pts, rqa_norm norm, const double* h_rr, int32_t K, float* d_eps,
                              uint64_t* d_count, double* d_rr_realised, void* d_ws, size_t ws_bytes, void* stream,
                              const rqa_options* opt) {
    rqa_status st = validate_points(pts, "rqa_eps_for_rr");
    if (st != RQA_OK) return st;
    Options o;
    st = make_options(opt, &o, "rqa_eps_for_rr");
    if (st != RQA_OK) return st;
    if (norm != RQA_NORM_MAX && norm != RQA_NORM_EUCLID) { set_error("rqa_eps_for_rr: unknown norm %d", (int)norm); return RQA_ERR_INVALID_ARG; }
    if (K < 1 || K > RQA_MAX_K) { set_error("rqa_eps_for_rr: K = %d outside 1..%d", K, RQA_MAX_K); return RQA_ERR_INVALID_ARG; }
    if (!h_rr || !d_eps || !d_count || !d_rr_realised || !d_ws) { set_error("rqa_eps_for_rr: NULL argument"); return RQA_ERR_INVALID_ARG; }
    if (((uintptr_t)d_ws & 255) != 0) { set_error("rqa_eps_for_rr: workspace must be 256-byte aligned"); return RQA_ERR_INVALID_ARG; }
    View v = make_view(*pts);
    uint64_t P = n_pairs(v);
    uint64_t rank[RQA_MAX_K];
    for (int k = 0; k < K; ++k) {
        double rr = h_rr[k];
        if (!(rr > 0.0) || !(rr <= 1.0)) { set_error("rqa_eps_for_rr: rr[%d] = %g outside (0, 1]", k, rr); return RQA_ERR_INVALID_ARG; }
        // the literal fp64 expression ceil(rr * (double)P), clamped to [1, P] (reading S5)
        double r = std::ceil(rr * (double)P);
        rank[k] = !(r >= 1.0) ? 1 : (r >= (double)P ? P : (uint64_t)r);
    }
    size_t need = sizeof(WsStatus) + select_workspace_bytes(v, K, o);
    if (ws_bytes < need) { set_error("rqa_eps_for_rr: workspace %zu < %zu bytes", ws_bytes, need); return RQA_ERR_WORKSPACE_TOO_SMALL; }
    cudaStream_t s = (cudaStream_t)stream;
    Arena ws(d_ws, ws_bytes);
    WsStatus* status = ws.take<WsStatus>(1);
    st = launch_finite_check(v, status, s);
    if (st != RQA_OK) return st;
    return run_select(v, (int)norm, rank, K, d_eps, d_count, d_rr_realised, ws, s, o);
}

rqa_status rqa_line_hist(const rqa_points* pts, rqa_norm norm, const float* d_eps, int32_t K, uint64_t* d_hist,
                         void* d_ws, size_t ws_bytes, void* stream) {
    return rqa_line_hist_opt(pts, norm, d_eps, K, d_hist, d_ws, ws_bytes, stream, nullptr);
}

rqa_status rqa_line_hist_opt(const rqa_points* pts, rqa_norm norm, const float* d_eps, int32_t K, uint64_t* d_hist,
                             void* d_ws, size_t ws_bytes, void* stream, const rqa_options* opt) {
    rqa_status st = validate_points(pts, "rqa_line_hist");
    if (st != RQA_OK) return st;
    Options o;
    st = make_options(opt, &o, "rqa_line_hist");
    if (st != RQA_OK) return st;
    if (norm != RQA_NORM_MAX && norm != RQA_NORM_EUCLID) { set_error("rqa_line_hist: unknown norm %d", (int)norm); return RQA_ERR_INVALID_ARG; }
    if (K < 1 || K > RQA_MAX_K) { set_error("rqa_line_hist: K = %d outside 1..%d", K, RQA_MAX_K); return RQA_ERR_INVALID_ARG; }
    if (!d_eps || !d_hist || !d_ws) { set_error("rqa_line_hist: NULL argument"); return RQA_ERR_INVALID_ARG; }
    if (((uintptr_t)d_ws & 255) != 0) { set_error("rqa_line_hist: workspace must be 256-byte aligned"); return RQA_ERR_INVALID_ARG; }
    View v = make_view(*pts);
    size_t need = sizeof(WsStatus) + line_workspace_bytes(v, K, o);
    if (ws_bytes < need) { set_error("rqa_line_hist: workspace %zu < %zu bytes", ws_bytes, need); return RQA_ERR_WORKSPACE_TOO_SMALL; }
    cudaStream_t s = (cudaStream_t)stream;
    Arena ws(d_ws, ws_bytes);
    WsStatus* status = ws.take<WsStatus>(1);
    st = launch_finite_check(v, status, s);
    if (st != RQA_OK) return st;
    return run_line_hist(v, (int)norm, d_eps, K, d_hist, ws, s, o);
}

rqa_status rqa_vert_hist(const rqa_points* pts, rqa_norm norm, const float* d_eps, int32_t K, uint64_t* d_vhist,
                         void* d_ws, size_t ws_bytes, void* stream) {
    return rqa_vert_hist_opt(pts, norm, d_eps, K, d_vhist, d_ws, ws_bytes, stream, nullptr);
}

rqa_status rqa_vert_hist_opt(const rqa_points* pts, rqa_norm norm, const float* d_eps, int32_t K, uint64_t* d_vhist,
                             void* d_ws, size_t ws_bytes, void* stream, const rqa_options* opt) {
    rqa_status st = validate_points(pts, "rqa_vert_hist");
    if (st != RQA_OK) return st;
    Options o;
    st = make_options(opt, &o, "rqa_vert_hist");
    if (st != RQA_OK) return st;
    if (norm != RQA_NORM_MAX && norm != RQA_NORM_EUCLID) { set_error("rqa_vert_hist: unknown norm %d", (int)norm); return RQA_ERR_INVALID_ARG; }
    if (K < 1 || K > RQA_MAX_K) { set_error("rqa_vert_hist: K = %d outside 1..%d", K, RQA_MAX_K); return RQA_ERR_INVALID_ARG; }
    if (!d_eps || !d_vhist || !d_ws) { set_error("rqa_vert_hist: NULL argument"); return RQA_ERR_INVALID_ARG; }
    if (((uintptr_t)d_ws & 255) != 0) { set_error("rqa_vert_hist: workspace must be 256-byte aligned"); return RQA_ERR_INVALID_ARG; }
    View v = make_view(*pts);
    size_t need = sizeof(WsStatus) + vert_workspace_bytes(v, K, o);
    if (ws_bytes < need) { set_error("rqa_vert_hist: workspace %zu < %zu bytes", ws_bytes, need); return RQA_ERR_WORKSPACE_TOO_SMALL; }
    cudaStream_t s = (cudaStream_t)stream;
    Arena ws(d_ws, ws_bytes);
    WsStatus* status = ws.take<WsStatus>(1);
    st = launch_finite_check(v, status, s);
    if (st != RQA_OK) return st;
    return run_vert_hist(v, (int)norm, d_eps, K, d_vhist, ws, s, o);
}

rqa_status rqa_det_avg(const uint64_t* d_hist, int32_t batch, int32_t K, int64_t n_points, int64_t l_min,
                       double* d_det, double* d_det_mean, void* stream) {
    if (!d_hist || !d_det || !d_det_mean) { set_error("rqa_det_avg: NULL argument"); return RQA_ERR_INVALID_ARG; }
    if (batch < 1 || K < 1 || K > RQA_MAX_K || n_points < 2 || l_min < 1) { set_error("rqa_det_avg: need batch >= 1, 1 <= K <= %d, n_points >= 2, l_min >= 1", RQA_MAX_K); return RQA_ERR_INVALID_ARG; }
    cudaStream_t s = (cudaStream_t)stream;
    if (n_points <= 2048) {
        const int64_t rows = (int64_t)K * batch;
        det_rows_kernel<<<(unsigned)((rows + 7) / 8), 256, 0, s>>>(d_hist, rows, n_points, l_min, d_det);
    } else {
        det_kernel<<<dim3(K, batch), 256, 0, s>>>(d_hist, K, n_points, l_min, d_det);
    }
    RQA_LAUNCH_CHECK();
    det_mean_kernel<<<(batch + 127) / 128, 128, 0, s>>>(d_det, K, batch, d_det_mean);
    RQA_LAUNCH_CHECK();
    return RQA_OK;
}

// ------------------------------------------------------------------------------------ host-buffer sweep
namespace {
struct SweepLayout {
    size_t series, eps, count, rr, det, mean, hist, inner, total;
};
SweepLayout sweep_layout(int64_t N, int batch, int m, int64_t tau, int K, size_t inner_ws) {
    int64_t n = N - (int64_t)(m - 1) * tau;
    SweepLayout L;
    size_t o = 0;
    L.series = o; o += align_up(sizeof(float) * (size_t)batch * N);
    L.eps = o;    o += align_up(sizeof(float) * (size_t)batch * K);
    L.count = o;  o += align_up(sizeof(uint64_t) * (size_t)batch * K);
    L.rr = o;     o += align_up(sizeof(double) * (size_t)batch * K);
    L.det = o;    o += align_up(sizeof(double) * (size_t)batch * K);
    L.mean = o;   o += align_up(sizeof(double) * (size_t)batch);
    L.hist = o;   o += align_up(sizeof(uint64_t) * (size_t)batch * K * n);
    L.inner = o;  o += inner_ws;
    L.total = o;
    return L;
}
}  // namespace

rqa_status rqa_sweep_workspace_bytes(int64_t N, int32_t batch, int32_t m, int64_t tau, int32_t K, size_t* bytes) {
    if (!bytes) { set_error("rqa_sweep_workspace_bytes: bytes is NULL"); return RQA_ERR_INVALID_ARG; }
    if (m < 1 || m > RQA_MAX_M || tau < 1 || batch < 1 || N - (int64_t)(m - 1) * tau < 2) { set_error("rqa_sweep_workspace_bytes: bad shape"); return RQA_ERR_INVALID_ARG; }
    rqa_points p;
    p.data = nullptr; p.n_points = N - (int64_t)(m - 1) * tau; p.m = m; p.batch = batch;
    p.point_stride = 1; p.coord_stride = tau; p.batch_stride = N; p.theiler = 0;
    size_t inner = 0;
    rqa_status st = rqa_workspace_bytes(&p, K, &inner);
    if (st != RQA_OK) return st;
    *bytes = sweep_layout(N, batch, m, tau, K, align_up(inner)).total;
    return RQA_OK;
}

rqa_status rqa_sweep_host(const float* h_series, int64_t N, int32_t batch, int32_t m, int64_t tau, rqa_norm norm,
                          const double* h_rr, int32_t K, int64_t l_min, float* h_eps, uint64_t* h_count,
                          double* h_rr_realised, double* h_det, double* h_det_mean, uint64_t* h_hist, void* d_ws,
                          size_t ws_bytes, void* stream) {
    if (!h_series || !h_rr || !h_eps || !h_count || !h_rr_realised || !h_det || !h_det_mean || !d_ws) { set_error("rqa_sweep_host: NULL argument"); return RQA_ERR_INVALID_ARG; }
    size_t total = 0;
    rqa_status st = rqa_sweep_workspace_bytes(N, batch, m, tau, K, &total);
    if (st != RQA_OK) return st;
    if (ws_bytes < total) { set_error("rqa_sweep_host: workspace %zu < %zu bytes", ws_bytes, total); return RQA_ERR_WORKSPACE_TOO_SMALL; }
    if (((uintptr_t)d_ws & 255) != 0) { set_error("rqa_sweep_host: workspace must be 256-byte aligned"); return RQA_ERR_INVALID_ARG; }
    int64_t n = N - (int64_t)(m - 1) * tau;
    rqa_points p;
    p.data = nullptr; p.n_points = n; p.m = m; p.batch = batch; p.point_stride = 1; p.coord_stride = tau; p.batch_stride = N;
    p.theiler = 0;
    size_t inner = 0;
    rqa_workspace_bytes(&p, K, &inner);
    inner = align_up(inner);
    SweepLayout L = sweep_layout(N, batch, m, tau, K, inner);
    char* w = (char*)d_ws;
    cudaStream_t s = (cudaStream_t)stream;
    float* d_series = (float*)(w + L.series);
    float* d_eps = (float*)(w + L.eps);
    uint64_t* d_count = (uint64_t*)(w + L.count);
    double* d_rr = (double*)(w + L.rr);
    double* d_det = (double*)(w + L.det);
    double* d_mean = (double*)(w + L.mean);
    uint64_t* d_hist = (uint64_t*)(w + L.hist);
    void* d_inner = w + L.inner;
    RQA_CUDA_TRY(cudaMemcpyAsync(d_series, h_series, sizeof(float) * (size_t)batch * N, cudaMemcpyHostToDevice, s));
    rqa_points view;
    st = rqa_embed(d_series, N, batch, N, m, tau, nullptr, &view, stream);
    if (st != RQA_OK) return st;
    st = rqa_eps_for_rr(&view, norm, h_rr, K, d_eps, d_count, d_rr, d_inner, inner, stream);
    if (st != RQA_OK) return st;
    st = rqa_line_hist(&view, norm, d_eps, K, d_hist, d_inner, inner, stream);
    if (st != RQA_OK) return st;
    st = rqa_det_avg(d_hist, batch, K, n, l_min, d_det, d_mean, stream);
    if (st != RQA_OK) return st;
    size_t bk = (size_t)batch * K;
    RQA_CUDA_TRY(cudaMemcpyAsync(h_eps, d_eps, sizeof(float) * bk, cudaMemcpyDeviceToHost, s));
    RQA_CUDA_TRY(cudaMemcpyAsync(h_count, d_count, sizeof(uint64_t) * bk, cudaMemcpyDeviceToHost, s));
    RQA_CUDA_TRY(cudaMemcpyAsync(h_rr_realised, d_rr, sizeof(double) * bk, cudaMemcpyDeviceToHost, s));
    RQA_CUDA_TRY(cudaMemcpyAsync(h_det, d_det, sizeof(double) * bk, cudaMemcpyDeviceToHost, s));
    RQA_CUDA_TRY(cudaMemcpyAsync(h_det_mean, d_mean, sizeof(double) * (size_t)batch, cudaMemcpyDeviceToHost, s));
    if (h_hist) RQA_CUDA_TRY(cudaMemcpyAsync(h_hist, d_hist, sizeof(uint64_t) * bk * n, cudaMemcpyDeviceToHost, s));
    return rqa_workspace_status(d_inner, stream);
}

}  // extern "C"
