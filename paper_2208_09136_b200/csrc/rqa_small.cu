// rqa_small.cu — short series (at most 8192 counted pairs, i.e. N' <= 128): one thread block does a whole series.
//
// Half of the paper's experiment grid is series of 10^2 and 10^3 points (900 series per length).  For
// N' <= 128 the tiled passes of rqa_select.cu / rqa_line.cu are the wrong shape (a tile is 512 diagonals wide) and a
// sweep is a chain of ~45 launches; here every distance of a series fits in shared memory, so
//   sel_small_kernel   computes the P distances once, sorts their bit patterns in shared memory (bitonic network) and
//                      reads eps_k = sorted[r_k - 1], C_k = #{d <= eps_k} (readings S4-S6) — the plain
//                      definition;
//   line_small_kernel  computes the distances once, then one thread per diagonal walks it with a stack of the nested
//                      thresholds' runs and counts line lengths into a shared-memory difference array;
//                      the block writes the whole P_k(l) row set itself (no global atomics, no memset).
// Both are exact and are covered by the same parity tests as the general paths (which explicit option knobs still
// select for any size).
#include <algorithm>

#include "rqa_tiles.cuh"

namespace rqa {

namespace {

constexpr int SMALL_MAX_PAIRS = 8192;
constexpr int SMALL_THREADS = 512;
constexpr int SMALL_MAX_N = 129;         // 8192 pairs: at most 128 diagonals (N' <= 128, or more points under a wide Theiler window)

struct SmallRanks {
    unsigned long long r[RQA_MAX_K];
};

// The counted triangle (diagonals o = w..n-1, nd = n - w of them) is enumerated diagonal by diagonal: pair number p lies on
// diagonal o = w + q at position i = p - off(q), off(q) = q*nd - q(q-1)/2 cells on the diagonals before it.  One flat
// loop over p (all threads busy, the loads of many pairs in flight), q found from a table of the offsets.
__device__ __forceinline__ void small_diag_offsets(int nd, int* s_off) {
    for (int q = threadIdx.x; q <= nd; q += SMALL_THREADS) s_off[q] = q * nd - q * (q - 1) / 2;
}
__device__ __forceinline__ int small_diag_of(const int* s_off, int nd, int p) {
    int lo = 0, hi = nd;                                       // last q with off(q) <= p
    while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (s_off[mid] <= p) lo = mid; else hi = mid;
    }
    return lo;
}
template <int NORM>
__device__ __forceinline__ void small_distances(const View& v, const float* yb, const int* s_off, int P, float* out) {
    const int w = (int)v.w, nd = (int)v.n - w;
    for (int p = threadIdx.x; p < P; p += SMALL_THREADS) {
        const int q = small_diag_of(s_off, nd, p), i = p - s_off[q];
        out[p] = point_distance<NORM>(yb, i, i + w + q, v.m, v.ps, v.cs);
    }
}

template <int NORM>
__global__ void __launch_bounds__(SMALL_THREADS) sel_small_kernel(View v, SmallRanks ranks, int K, unsigned int P, int P2,
                                                                 float* __restrict__ eps,
                                                                 unsigned long long* __restrict__ count,
                                                                 double* __restrict__ rr) {
    extern __shared__ uint32_t s_key[];                      // [P2] bit patterns (non-negative floats order like them)
    __shared__ int s_off[SMALL_MAX_N + 1];
    const int b = blockIdx.x, tid = threadIdx.x;
    const float* yb = v.data + (int64_t)b * v.bs;
    small_diag_offsets((int)(v.n - v.w), s_off);
    __syncthreads();
    small_distances<NORM>(v, yb, s_off, (int)P, (float*)s_key);
    for (int q = (int)P + tid; q < P2; q += SMALL_THREADS) s_key[q] = 0xffffffffu;      // padding sorts last
    __syncthreads();
    // bitonic network: every thread handles whole compare-exchange pairs (q, q | j), q without bit j
    for (int k = 2; k <= P2; k <<= 1) {
        for (int j = k >> 1; j > 0; j >>= 1) {
            for (int t = tid; t < P2 / 2; t += SMALL_THREADS) {
                const int q = 2 * t - (t & (j - 1)), p = q | j;
                const uint32_t a = s_key[q], c = s_key[p];
                const bool up = (q & k) == 0;
                if ((a > c) == up) { s_key[q] = c; s_key[p] = a; }
            }
            __syncthreads();
        }
    }
    for (int k = tid; k < K; k += SMALL_THREADS) {
        const uint32_t e = s_key[ranks.r[k] - 1];            // the r_k-th smallest
        int lo = 0, hi = (int)P;                              // first index with key > e
        while (lo < hi) {
            const int mid = (lo + hi) >> 1;
            if (s_key[mid] <= e) lo = mid + 1; else hi = mid;
        }
        eps[(int64_t)b * K + k] = __uint_as_float(e);
        count[(int64_t)b * K + k] = (unsigned long long)lo;
        rr[(int64_t)b * K + k] = (double)lo / (double)P;
    }
}

// One thread per diagonal.  Thresholds are nested, so after a cell of level v (= number of distinct thresholds below
// its distance) exactly the thresholds j >= v are inside a run, and the runs of all thresholds form a stack of
// (lowest threshold, start) entries ordered by start: a lower level pushes one entry, a higher level pops the entries it
// ends, each giving ONE line length for a whole range [a, b) of thresholds, counted as D[a][len]++, D[b][len]-- in a
// difference array over the thresholds.  Work per cell does not depend on K (the same idea as the tiled scan, in its
// plainest form: lines of every length are emitted, nothing is deferred).
// Shared memory: uint8 level[P] diagonal by diagonal | then 32-bit words: D[(K+1)][n] | eps sorted distinct [K+1] | j_of[K] | 2 x scratch[K] |
// stacks [LINE_SMALL_THREADS][K+1] uint16 (lo << 8 | start).
constexpr int LINE_SMALL_THREADS = 256;

__host__ __device__ inline size_t line_small_smem(int64_t P, int K, int64_t n) {
    return 4 * (((size_t)P + 3) / 4 + (size_t)(K + 1) * (size_t)n + (size_t)(K + 1) + 3 * (size_t)K) +
           2 * (size_t)(SMALL_MAX_N) * (size_t)(K + 2);
}

template <int NORM>
__global__ void __launch_bounds__(LINE_SMALL_THREADS) line_small_kernel(View v, const float* __restrict__ eps, int K,
                                                                       unsigned long long* __restrict__ hist,
                                                                       WsStatus* status) {
    extern __shared__ uint32_t s_mem[];
    __shared__ int s_off[SMALL_MAX_N + 1];
    __shared__ int s_J;
    const int b = blockIdx.x, tid = threadIdx.x;
    const int n = (int)v.n, w = (int)v.w, nd = n - w;
    const int P = nd * (nd + 1) / 2;
    uint8_t* s_lev = (uint8_t*)s_mem;                         // level of every cell, diagonal by diagonal
    int* s_D = (int*)(s_mem + (P + 3) / 4);
    float* s_eps = (float*)(s_D + (K + 1) * n);
    int* s_jof = (int*)(s_eps + (K + 1));
    float* s_san = (float*)(s_jof + K);                      // thresholds with NaN / negative / infinite values replaced by 0
    int* s_first = (int*)(s_san + K);
    uint16_t* s_stk = (uint16_t*)(s_first + K) + (size_t)tid * (K + 2);
    const float* yb = v.data + (int64_t)b * v.bs;
    const float* e = eps + (int64_t)b * K;

    for (int q = tid; q <= nd; q += LINE_SMALL_THREADS) s_off[q] = q * nd - q * (q - 1) / 2;
    for (int q = tid; q < (K + 1) * n; q += LINE_SMALL_THREADS) s_D[q] = 0;
    // the K thresholds sorted, duplicates removed: distinct index j_of[k] of caller threshold k
    bool bad = false;
    for (int k = tid; k < K; k += LINE_SMALL_THREADS) {
        float x = e[k];
        if (!(x >= 0.0f) || isinf(x)) { bad = true; x = 0.0f; }
        s_san[k] = x;
    }
    if (bad) atomicExch(&status->bad_eps, 1);
    if (tid == 0) s_J = 0;
    __syncthreads();
    for (int k = tid; k < K; k += LINE_SMALL_THREADS) {      // first occurrence of its value?
        int first = 1;
        for (int u = 0; u < k; ++u) first &= s_san[u] != s_san[k];
        s_first[k] = first;
    }
    __syncthreads();
    for (int k = tid; k < K; k += LINE_SMALL_THREADS) {
        int below = 0;                                       // distinct values below this threshold
        for (int q = 0; q < K; ++q) below += s_first[q] && s_san[q] < s_san[k];
        s_jof[k] = below;
        s_eps[below] = s_san[k];                             // equal thresholds write the same value to the same slot
        atomicMax(&s_J, below + 1);
    }
    __syncthreads();
    const int J = s_J;
    // every cell's level = number of distinct thresholds below its distance (all threads, one flat loop over the pairs)
    for (int p = tid; p < P; p += LINE_SMALL_THREADS) {
        int lo = 0, hi = nd;                                  // diagonal of pair p: last q with off(q) <= p
        while (hi - lo > 1) {
            const int mid = (lo + hi) >> 1;
            if (s_off[mid] <= p) lo = mid; else hi = mid;
        }
        const int i = p - s_off[lo];
        const float x = point_distance<NORM>(yb, i, i + w + lo, v.m, v.ps, v.cs);
        int a = 0, c = J;
        while (a < c) {
            const int mid = (a + c) >> 1;
            if (s_eps[mid] < x) a = mid + 1; else c = mid;
        }
        s_lev[p] = (uint8_t)a;
    }
    __syncthreads();
    for (int q = tid; q < nd; q += LINE_SMALL_THREADS) {     // diagonal o = w + q, len = nd - q cells
        const uint8_t* lev = s_lev + s_off[q];
        const int len = nd - q;
        int top = 0, pv = J;
        auto ended = [&](int vnew, int t) {                  // the thresholds [pv, vnew) end their runs before cell t
            while (top > 0) {
                const uint32_t en = s_stk[top - 1];
                const int lo = (int)(en >> 8), start = (int)(en & 255u);
                const int hi = top > 1 ? (int)(s_stk[top - 2] >> 8) : J;
                const int upto = hi < vnew ? hi : vnew;
                atomicAdd(&s_D[lo * n + (t - start)], 1);
                atomicSub(&s_D[upto * n + (t - start)], 1);
                if (hi <= vnew) {
                    --top;
                    if (hi == vnew) break;
                } else {
                    s_stk[top - 1] = (uint16_t)((vnew << 8) | start);   // the rest of the entry lives on
                    break;
                }
            }
        };
        for (int t = 0; t < len; ++t) {
            const int lo = lev[t];
            if (lo < pv) s_stk[top++] = (uint16_t)((lo << 8) | t);
            else if (lo > pv) ended(lo, t);
            pv = lo;
        }
        if (pv < J) ended(J, len);
    }
    __syncthreads();
    // prefix sums of D over the thresholds turn every column into the histogram of the distinct thresholds
    for (int l = tid; l < n; l += LINE_SMALL_THREADS) {
        int acc = 0;
        for (int j = 0; j < J; ++j) {
            acc += s_D[j * n + l];
            s_D[j * n + l] = acc;
        }
    }
    __syncthreads();
    unsigned long long* out = hist + (int64_t)b * K * n;
    for (int q = tid; q < K * n; q += LINE_SMALL_THREADS) {
        const int k = q / n, l = q - k * n;
        out[q] = l == 0 ? 0ull : (unsigned long long)(unsigned int)s_D[s_jof[k] * n + l];
    }
}

constexpr size_t SMALL_SMEM_MAX = 200 * 1024;

}  // namespace

bool small_series(const View& v) { return n_pairs(v) <= (uint64_t)SMALL_MAX_PAIRS && n_diag(v) <= SMALL_MAX_N; }

bool small_line_fits(const View& v, int K) {
    return small_series(v) && v.n <= 255 && line_small_smem((int64_t)n_pairs(v), K, v.n) <= SMALL_SMEM_MAX;
}

rqa_status run_select_small(const View& v, int norm, const uint64_t* h_rank, int K, float* d_eps, uint64_t* d_count,
                            double* d_rr, cudaStream_t s) {
    SmallRanks ranks;
    for (int k = 0; k < K; ++k) ranks.r[k] = h_rank[k];
    const unsigned int P = (unsigned int)n_pairs(v);
    int P2 = 2;
    while ((unsigned int)P2 < P) P2 <<= 1;
    const size_t smem = sizeof(uint32_t) * (size_t)P2;
    if (norm == RQA_NORM_MAX)
        sel_small_kernel<RQA_NORM_MAX><<<v.batch, SMALL_THREADS, smem, s>>>(v, ranks, K, P, P2, d_eps, (unsigned long long*)d_count, d_rr);
    else
        sel_small_kernel<RQA_NORM_EUCLID><<<v.batch, SMALL_THREADS, smem, s>>>(v, ranks, K, P, P2, d_eps, (unsigned long long*)d_count, d_rr);
    RQA_LAUNCH_CHECK();
    return RQA_OK;
}

rqa_status run_line_small(const View& v, int norm, const float* d_eps, int K, uint64_t* d_hist, WsStatus* status,
                          cudaStream_t s) {
    const size_t smem = line_small_smem((int64_t)n_pairs(v), K, v.n);
    auto kern = norm == RQA_NORM_MAX ? line_small_kernel<RQA_NORM_MAX> : line_small_kernel<RQA_NORM_EUCLID>;
    static thread_local bool attr_set[8][2] = {};
    int dev = 0;
    RQA_CUDA_TRY(cudaGetDevice(&dev));
    const int which = norm == RQA_NORM_MAX ? 0 : 1;
    if (dev >= 8 || !attr_set[dev][which]) {
        RQA_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMALL_SMEM_MAX));
        if (dev < 8) attr_set[dev][which] = true;
    }
    kern<<<v.batch, LINE_SMALL_THREADS, smem, s>>>(v, d_eps, K, (unsigned long long*)d_hist, status);
    RQA_LAUNCH_CHECK();
    return RQA_OK;
}

}  // namespace rqa
