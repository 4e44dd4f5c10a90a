// rqa_common.cuh — internal declarations shared by the translation units of librqa.so.
// Not part of the public ABI (that is include/rqa.h) and not shared with the oracle.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include <atomic>

#include "rqa.h"

namespace rqa {

// ---------------------------------------------------------------------------------------------- errors
void set_error(const char* fmt, ...);
extern std::atomic<uint64_t> g_launches;

#define RQA_CUDA_TRY(expr)                                                                         \
    do {                                                                                           \
        cudaError_t e__ = (expr);                                                                  \
        if (e__ != cudaSuccess) {                                                                  \
            rqa::set_error("%s failed: %s (%s:%d)", #expr, cudaGetErrorString(e__), __FILE__, __LINE__); \
            return RQA_ERR_CUDA;                                                                   \
        }                                                                                          \
    } while (0)

// counts the launch and checks cudaGetLastError
#define RQA_LAUNCH_CHECK()                                                                         \
    do {                                                                                           \
        rqa::g_launches.fetch_add(1, std::memory_order_relaxed);                                   \
        cudaError_t e__ = cudaGetLastError();                                                      \
        if (e__ != cudaSuccess) {                                                                  \
            rqa::set_error("kernel launch failed: %s (%s:%d)", cudaGetErrorString(e__), __FILE__, __LINE__); \
            return RQA_ERR_CUDA;                                                                   \
        }                                                                                          \
    } while (0)

// --------------------------------------------------------------------------------------------- options
// Validated per-call copy of rqa_options (include/rqa.h); every field 0 = automatic.  There is no process-wide state.
struct Options {
    int select_path = 0;      // 0 auto, 1 direct (materialise all distances), 2 bracket (sample + one counting pass), 3 radix
    int line_chunk = 0;       // diagonal scan: chunk length L (<= 1023)
    int line_segment = 0;     // diagonal scan: chunks per segment
    int line_buffers = 0;     // diagonal scan: window sets per block (1 plain loads, 2 bulk-copy double buffer)
    int line_path = 0;        // 0 auto, 1 tiled scan, 2 one block per series (P <= 2^22)
    int group_size = 0;       // thresholds per pass of the grouped kernels (0 auto)
    int part = 0, parts = 1;  // this process' share of the tiles (multi-GPU split of one call)
    int64_t sample_size = 0;  // bracket path: sample size S
    int64_t cand_cap = 0;     // bracket path: candidate capacity per series
    rqa_reduce_fn reduce = nullptr;
    void* reduce_ctx = nullptr;
    void* ev_begin = nullptr;  // cudaEvent_t recorded just before / after the call's dominant kernel (bench.py's roofline)
    void* ev_end = nullptr;
};
rqa_status make_options(const rqa_options* in, Options* out, const char* who);

// Sum n uint64 device counters over the parts of a split call (no-op for a single part).
inline rqa_status reduce_parts(const Options& o, void* d_counters, size_t n, cudaStream_t s) {
    if (o.parts <= 1) return RQA_OK;
    if (o.reduce(o.reduce_ctx, (uint64_t*)d_counters, n, (void*)s) != 0) {
        set_error("the reduce callback of rqa_options failed");
        return RQA_ERR_CUDA;
    }
    return RQA_OK;
}

// Thresholds (targets) per pass of the grouped kernels (counting pass, diagonal scan, column scan; at most GK = 32).
// More than 32 go in groups of 20 (a pass over at most 20 thresholds keeps two blocks per SM): measured on 10 series
// of 1e5 points at K = 99, rqa_line_hist 553 -> 503 ms, rqa_eps_for_rr 283 -> 278 ms, workspace 13.2 -> 8.5 GB; groups
// of 25 or 10 are slower (810 / 1248 ms for both calls), and K = 32 in two groups of 16 is slower than in one pass
// (config 5: 71 -> 103 ms).
inline int group_size_for(int K, const Options& opt) {
    if (opt.group_size > 0) return opt.group_size < 32 ? opt.group_size : 32;
    return K <= 32 ? 32 : 20;
}

// ------------------------------------------------------------------------------------------------ view
// Device-side copy of rqa_points (x_i[c] of series b = data[b*bs + i*ps + c*cs]).
struct View {
    const float* data;
    int64_t n;   // N'
    int32_t m;
    int32_t batch;
    int64_t ps, cs, bs;
    int64_t w;   // first diagonal counted (Theiler window), >= 1
};

inline View make_view(const rqa_points& p) {
    View v;
    v.data = p.data;
    v.n = p.n_points;
    v.m = p.m;
    v.batch = p.batch;
    v.ps = p.point_stride;
    v.cs = p.coord_stride;
    v.bs = p.batch_stride;
    v.w = p.theiler > 1 ? p.theiler : 1;
    return v;
}

inline uint64_t n_pairs(int64_t n) { return (uint64_t)n * (uint64_t)(n - 1) / 2; }
// With a Theiler window w the diagonals w..n-1 are counted: the same triangle as for n_diag = n - w + 1 points.
inline int64_t n_diag(const View& v) { return v.n - v.w + 1; }
inline uint64_t n_pairs(const View& v) { return n_pairs(n_diag(v)); }

rqa_status validate_points(const rqa_points* pts, const char* who);

// ------------------------------------------------------------------------------------------- workspace
// Status block at the start of every workspace (256 bytes reserved).
struct WsStatus {
    int32_t nonfinite;   // set to 1 by the finite check when a NaN/Inf is seen
    int32_t internal;    // set to 1 on an internal inconsistency (should never happen)
    int32_t bad_eps;     // set to 1 by rqa_line_hist when a threshold is NaN, Inf or negative
    int32_t pad[61];
};
static_assert(sizeof(WsStatus) == 256, "status block is 256 bytes");

inline size_t align_up(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }

// Simple bump allocator over the caller's workspace.
struct Arena {
    char* base;
    size_t size, off;
    Arena(void* p, size_t n) : base((char*)p), size(n), off(0) {}
    template <typename T>
    T* take(size_t count) {
        size_t bytes = align_up(count * sizeof(T));
        T* r = (T*)(base + off);
        off += bytes;
        return r;
    }
    bool ok() const { return off <= size; }
};

// ------------------------------------------------------------------------------------ internal launchers
rqa_status launch_finite_check(const View& v, WsStatus* st, cudaStream_t s);

size_t select_workspace_bytes(const View& v, int K, const Options& opt);
rqa_status run_select(const View& v, int norm, const uint64_t* h_rank, int K, float* d_eps, uint64_t* d_count,
                      double* d_rr, Arena& ws, cudaStream_t s, const Options& opt);

size_t line_workspace_bytes(const View& v, int K, const Options& opt);
rqa_status run_line_hist(const View& v, int norm, const float* d_eps, int K, uint64_t* d_hist, Arena& ws,
                         cudaStream_t s, const Options& opt);

// Short series (at most 8192 counted pairs): one block per series, everything in shared memory (rqa_small.cu).
bool small_series(const View& v);
bool small_line_fits(const View& v, int K);
rqa_status run_select_small(const View& v, int norm, const uint64_t* h_rank, int K, float* d_eps, uint64_t* d_count,
                            double* d_rr, cudaStream_t s);
rqa_status run_line_small(const View& v, int norm, const float* d_eps, int K, uint64_t* d_hist, WsStatus* status,
                          cudaStream_t s);

// Many series of moderate length (P <= 2^22 counted pairs): one block selects all thresholds of a series (rqa_block.cu).
// A series it cannot finish (massive ties) gets *(int32_t*)((char*)d_fallback + b*fallback_stride) = 1.
bool block_select_fits(const View& v, int K);
rqa_status run_select_block(const View& v, int norm, const uint64_t* h_rank, int K, float* d_eps, uint64_t* d_count,
                            double* d_rr, int32_t* d_fallback, size_t fallback_stride, cudaStream_t s);

bool block_line_fits(const View& v, int K);
rqa_status run_line_block(const View& v, int norm, const float* d_eps, int K, uint64_t* d_hist, WsStatus* status,
                          cudaStream_t s, bool vertical = false);   // vertical: the columns of the full matrix (rqa_vert_hist)

size_t vert_workspace_bytes(const View& v, int K, const Options& opt);
rqa_status run_vert_hist(const View& v, int norm, const float* d_eps, int K, uint64_t* d_vhist, Arena& ws,
                         cudaStream_t s, const Options& opt);

// Number of SMs of the current device (cached per thread; 148 on a B200).
int sm_count();

// ---------------------------------------------------------------------------------------- device helpers
#ifdef __CUDACC__
// Distance between embedded points i and j of one series (yb = series base).  Max norm: PAPER.md:50.
// Euclid: fixed order c = 0..m-1, every operation individually rounded (no FMA) — DESIGN.md reading S13.
template <int NORM>
__device__ __forceinline__ float point_distance(const float* __restrict__ yb, int64_t i, int64_t j, int m,
                                                int64_t ps, int64_t cs) {
    const float* a = yb + i * ps;
    const float* b = yb + j * ps;
    if (NORM == RQA_NORM_MAX) {
        float d = 0.0f;
        for (int c = 0; c < m; ++c) d = fmaxf(d, fabsf(__fsub_rn(a[c * cs], b[c * cs])));
        return d;
    } else {
        float t = __fsub_rn(a[0], b[0]);
        float s = __fmul_rn(t, t);
        for (int c = 1; c < m; ++c) {
            t = __fsub_rn(a[c * cs], b[c * cs]);
            s = __fadd_rn(s, __fmul_rn(t, t));
        }
        return __fsqrt_rn(s);
    }
}
#endif

}  // namespace rqa
