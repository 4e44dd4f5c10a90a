// rqa_select.cu — rqa_eps_for_rr: exact multi-target order statistics of the P = N'(N'-1)/2 pairwise
// distances ("preselect RR and use the corresponding eps"; readings S4-S6).
//
// The N'^2 distance matrix is never stored: every pass recomputes d_ij tile by tile.
// Non-negative fp32 values order like their uint32 bit patterns, so the select works on patterns.
//
// v0 (this file, generic fallback): classic most-significant-digit radix select, 4 passes of 8 bits, all K
// targets resolved in each pass; targets that share a prefix share one 256-bin histogram ("group").
#include "rqa_common.cuh"

namespace rqa {

namespace {

struct SelBatch {
    int32_t G;                        // number of live groups (distinct prefixes)
    int32_t pad;
    uint32_t gprefix[RQA_MAX_K];      // distinct prefixes, ascending (determined high bits, low bits zero)
    int32_t group_of[RQA_MAX_K];      // target -> group
    uint32_t prefix[RQA_MAX_K];       // target -> prefix
    uint64_t resid[RQA_MAX_K];        // 1-based residual rank inside the prefix range
    uint64_t below[RQA_MAX_K];        // number of distances strictly below the prefix range
};

struct Ranks {
    uint64_t r[RQA_MAX_K];
};

constexpr int SEL_W = 128;            // diagonals per block (= threads)
constexpr int SEL_L = 512;            // positions per tile

__global__ void select_init_kernel(SelBatch* st, Ranks ranks, int K) {
    SelBatch& s = st[blockIdx.x];
    int k = threadIdx.x;
    if (k == 0) { s.G = 1; s.gprefix[0] = 0; }
    if (k < K) {
        s.group_of[k] = 0;
        s.prefix[k] = 0;
        s.resid[k] = ranks.r[k];
        s.below[k] = 0;
    }
}

// One pass: digit histogram of the cells whose determined high bits match a live prefix.
// grid = (o-blocks, chunks, batch); thread t walks diagonal o0+t over positions [i0, i0+L).
template <int NORM>
__global__ void __launch_bounds__(SEL_W) radix_pass_kernel(View v, int pass, const SelBatch* __restrict__ st,
                                                           unsigned long long* __restrict__ bins, int K) {
    extern __shared__ uint32_t sbins[];      // [G][256]
    __shared__ uint32_t s_gprefix[RQA_MAX_K];
    const int b = blockIdx.z;
    const int64_t o0 = 1 + (int64_t)blockIdx.x * SEL_W;
    const int64_t i0 = (int64_t)blockIdx.y * SEL_L;
    if (i0 >= v.n - o0) return;              // empty tile (beyond the hypotenuse)
    const SelBatch& s = st[b];
    const int G = s.G;
    for (int q = threadIdx.x; q < G * 256; q += blockDim.x) sbins[q] = 0;
    for (int q = threadIdx.x; q < G; q += blockDim.x) s_gprefix[q] = s.gprefix[q];
    __syncthreads();

    const float* yb = v.data + (int64_t)b * v.bs;
    const int64_t o = o0 + threadIdx.x;
    const int shift = 24 - 8 * pass;
    const uint32_t himask = pass == 0 ? 0u : (0xFFFFFFFFu << (32 - 8 * pass));
    if (o < v.n) {
        int64_t iend = min(i0 + (int64_t)SEL_L, v.n - o);
        for (int64_t i = i0; i < iend; ++i) {
            float d = point_distance<NORM>(yb, i, i + o, v.m, v.ps, v.cs);
            uint32_t key = __float_as_uint(d);
            uint32_t hi = key & himask;
            int lo = 0, hiq = G;             // first group with gprefix >= hi
            while (lo < hiq) {
                int mid = (lo + hiq) >> 1;
                if (s_gprefix[mid] < hi) lo = mid + 1; else hiq = mid;
            }
            if (lo < G && s_gprefix[lo] == hi) atomicAdd(&sbins[lo * 256 + ((key >> shift) & 255u)], 1u);
        }
    }
    __syncthreads();
    unsigned long long* gb = bins + (int64_t)b * K * 256;
    for (int q = threadIdx.x; q < G * 256; q += blockDim.x) {
        uint32_t c = sbins[q];
        if (c) atomicAdd(&gb[q], (unsigned long long)c);
    }
}

// One block per series: every target picks its digit, then the groups are rebuilt and the bins cleared.
__global__ void __launch_bounds__(256) radix_resolve_kernel(SelBatch* st, unsigned long long* bins, int K, int pass,
                                                            unsigned long long P, float* __restrict__ eps,
                                                            unsigned long long* __restrict__ count,
                                                            double* __restrict__ rr) {
    const int b = blockIdx.x;
    SelBatch& s = st[b];
    unsigned long long* gb = bins + (int64_t)b * K * 256;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nwarps = blockDim.x >> 5;
    const int shift = 24 - 8 * pass;
    __shared__ uint32_t s_prefix[RQA_MAX_K];
    __shared__ int s_first[RQA_MAX_K];

    for (int k = warp; k < K; k += nwarps) {
        const unsigned long long* h = gb + s.group_of[k] * 256;
        unsigned long long c[8], sum = 0;
        for (int q = 0; q < 8; ++q) { c[q] = h[lane * 8 + q]; sum += c[q]; }
        unsigned long long incl = sum;
        for (int off = 1; off < 32; off <<= 1) {
            unsigned long long t = __shfl_up_sync(0xffffffffu, incl, off);
            if (lane >= off) incl += t;
        }
        const unsigned long long resid = s.resid[k];
        unsigned ball = __ballot_sync(0xffffffffu, incl >= resid);
        int src = ball ? (__ffs(ball) - 1) : 31;      // ball == 0 cannot happen (resid <= group total)
        unsigned long long excl = incl - sum;
        int digit = 0;
        unsigned long long e = excl, ties = 0;
        if (lane == src) {
            for (int q = 0; q < 8; ++q) {
                if (e + c[q] >= resid) { digit = lane * 8 + q; ties = c[q]; break; }
                e += c[q];
            }
        }
        digit = __shfl_sync(0xffffffffu, digit, src);
        e = __shfl_sync(0xffffffffu, e, src);
        ties = __shfl_sync(0xffffffffu, ties, src);
        if (lane == 0) {
            uint32_t p = s.prefix[k] | ((uint32_t)digit << shift);
            s.prefix[k] = p;
            s_prefix[k] = p;
            unsigned long long below = s.below[k] + e;
            s.below[k] = below;
            s.resid[k] = resid - e;
            if (pass == 3) {
                eps[(int64_t)b * K + k] = __uint_as_float(p);
                unsigned long long cnt = below + ties;
                count[(int64_t)b * K + k] = cnt;
                rr[(int64_t)b * K + k] = (double)cnt / (double)P;
            }
        }
    }
    __syncthreads();
    // regroup: distinct prefixes, ascending
    for (int k = threadIdx.x; k < K; k += blockDim.x) {
        int first = 1;
        for (int j = 0; j < k; ++j) first &= (s_prefix[j] != s_prefix[k]);
        s_first[k] = first;
    }
    __syncthreads();
    for (int k = threadIdx.x; k < K; k += blockDim.x) {
        int less = 0;
        for (int j = 0; j < K; ++j) less += (s_first[j] && s_prefix[j] < s_prefix[k]);
        s.group_of[k] = less;
        if (s_first[k]) s.gprefix[less] = s_prefix[k];
    }
    if (threadIdx.x == 0) {
        int G = 0;
        for (int j = 0; j < K; ++j) G += s_first[j];
        s.G = G;
    }
    for (int q = threadIdx.x; q < K * 256; q += blockDim.x) gb[q] = 0ull;
}

}  // namespace

size_t select_workspace_bytes(const View& v, int K) {
    return align_up(sizeof(SelBatch) * (size_t)v.batch) + align_up(sizeof(uint64_t) * (size_t)v.batch * K * 256);
}

rqa_status run_select(const View& v, int norm, const uint64_t* h_rank, int K, float* d_eps, uint64_t* d_count,
                      double* d_rr, Arena& ws, cudaStream_t s) {
    SelBatch* st = ws.take<SelBatch>(v.batch);
    unsigned long long* bins = (unsigned long long*)ws.take<uint64_t>((size_t)v.batch * K * 256);
    if (!ws.ok()) { set_error("run_select: workspace too small"); return RQA_ERR_WORKSPACE_TOO_SMALL; }
    Ranks ranks;
    for (int k = 0; k < K; ++k) ranks.r[k] = h_rank[k];
    RQA_CUDA_TRY(cudaMemsetAsync(bins, 0, sizeof(uint64_t) * (size_t)v.batch * K * 256, s));
    select_init_kernel<<<v.batch, RQA_MAX_K, 0, s>>>(st, ranks, K);
    RQA_LAUNCH_CHECK();
    const size_t smem = (size_t)K * 256 * sizeof(uint32_t);
    auto kern = norm == RQA_NORM_MAX ? radix_pass_kernel<RQA_NORM_MAX> : radix_pass_kernel<RQA_NORM_EUCLID>;
    if (smem > 48 * 1024) RQA_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    dim3 grid((unsigned)((v.n - 1 + SEL_W - 1) / SEL_W), (unsigned)((v.n - 1 + SEL_L - 1) / SEL_L), (unsigned)v.batch);
    const unsigned long long P = n_pairs(v.n);
    for (int pass = 0; pass < 4; ++pass) {
        kern<<<grid, SEL_W, smem, s>>>(v, pass, st, bins, K);
        RQA_LAUNCH_CHECK();
        radix_resolve_kernel<<<v.batch, 256, 0, s>>>(st, bins, K, pass, P, d_eps, (unsigned long long*)d_count, d_rr);
        RQA_LAUNCH_CHECK();
    }
    return RQA_OK;
}

}  // namespace rqa
