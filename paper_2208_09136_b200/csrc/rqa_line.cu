// rqa_line.cu — rqa_line_hist: diagonal-line-length histograms P_k(l) at K thresholds
// (Eq. 4 and the sentence under it; PAPER.md:125 upper triangle, R computed on the fly).
//
// v0 (this file): one thread per diagonal, K run counters, global atomics.  Correct and simple; the fused
// tiled kernel replaces it.
#include "rqa_common.cuh"

namespace rqa {

namespace {

template <int NORM>
__global__ void __launch_bounds__(128) line_naive_kernel(View v, const float* __restrict__ eps, int K,
                                                         unsigned long long* __restrict__ hist) {
    const int b = blockIdx.y;
    const int64_t o = 1 + (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (o >= v.n) return;
    const float* yb = v.data + (int64_t)b * v.bs;
    const float* e = eps + (int64_t)b * K;
    unsigned long long* h = hist + (int64_t)b * K * v.n;
    uint32_t run[RQA_MAX_K];
    for (int k = 0; k < K; ++k) run[k] = 0;
    for (int64_t i = 0; i + o < v.n; ++i) {
        float d = point_distance<NORM>(yb, i, i + o, v.m, v.ps, v.cs);
        for (int k = 0; k < K; ++k) {
            if (d <= e[k]) {
                ++run[k];
            } else if (run[k]) {
                atomicAdd(&h[(int64_t)k * v.n + run[k]], 1ull);
                run[k] = 0;
            }
        }
    }
    for (int k = 0; k < K; ++k)
        if (run[k]) atomicAdd(&h[(int64_t)k * v.n + run[k]], 1ull);
}

}  // namespace

size_t line_workspace_bytes(const View&, int) { return 256; }

rqa_status run_line_hist(const View& v, int norm, const float* d_eps, int K, uint64_t* d_hist, Arena&, cudaStream_t s) {
    RQA_CUDA_TRY(cudaMemsetAsync(d_hist, 0, sizeof(uint64_t) * (size_t)v.batch * K * v.n, s));
    dim3 grid((unsigned)((v.n - 1 + 127) / 128), (unsigned)v.batch);
    if (norm == RQA_NORM_MAX)
        line_naive_kernel<RQA_NORM_MAX><<<grid, 128, 0, s>>>(v, d_eps, K, (unsigned long long*)d_hist);
    else
        line_naive_kernel<RQA_NORM_EUCLID><<<grid, 128, 0, s>>>(v, d_eps, K, (unsigned long long*)d_hist);
    RQA_LAUNCH_CHECK();
    return RQA_OK;
}

}  // namespace rqa
