// rqa_measures.cu — the cheap reductions that sit on top of the line histograms:
//   rqa_det_prefix_avg     Eq. 5 as a curve: the averaged determinism for every cut-off RR*
//   rqa_line_measures      "the histogram is used for the calculation of (DET, L, L_max and RR)",
//                          plus the entropy of the line-length distribution (one of the "other RQA measures")
//   rqa_lam_tt             laminarity and trapping time from the vertical-line histogram
//   rqa_sorting_rate_host  Eq. 6, the paper's evaluation score (host arithmetic on a few numbers)
#include "rqa_common.cuh"

namespace rqa {
namespace {

// prefix[b][k] = (det[b][0] + ... + det[b][k]) / (k+1), summed left to right in fp64 (reading S11).
__global__ void det_prefix_kernel(const double* __restrict__ det, int K, int batch, double* __restrict__ prefix) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= batch) return;
    double sum = 0.0;
    for (int k = 0; k < K; ++k) {
        sum += det[(int64_t)b * K + k];
        prefix[(int64_t)b * K + k] = sum / (double)(k + 1);
    }
}

// One block per (threshold, series): exact uint64 sums over the histogram row.
__global__ void __launch_bounds__(256) line_measures_kernel(const uint64_t* __restrict__ hist, int K, int64_t n, int64_t l_min,
                                                            int64_t w,
                                                            double* __restrict__ L, uint64_t* __restrict__ Lmax,
                                                            double* __restrict__ rr, double* __restrict__ entr) {
    const int k = blockIdx.x, b = blockIdx.y;
    const uint64_t* row = hist + ((int64_t)b * K + k) * n;
    unsigned long long pts = 0, lpts = 0, lines = 0, lmax = 0;
    double hlogh = 0.0;                                      // sum h ln h: ENTR = ln T - (1/T) sum h ln h, T = #lines
    for (int64_t l = 1 + threadIdx.x; l < n; l += blockDim.x) {
        const unsigned long long h = row[l];
        pts += (unsigned long long)l * h;
        if (l >= l_min) {
            lpts += (unsigned long long)l * h;
            lines += h;
            if (entr && h > 1) hlogh += (double)h * log((double)h);
        }
        if (h) lmax = (unsigned long long)l;                 // l increases along the loop
    }
    __shared__ unsigned long long s[4][8];
    __shared__ double s_e[8];
    for (int off = 16; off; off >>= 1) {
        pts += __shfl_down_sync(0xffffffffu, pts, off);
        lpts += __shfl_down_sync(0xffffffffu, lpts, off);
        lines += __shfl_down_sync(0xffffffffu, lines, off);
        lmax = max(lmax, __shfl_down_sync(0xffffffffu, lmax, off));
        hlogh += __shfl_down_sync(0xffffffffu, hlogh, off);
    }
    if ((threadIdx.x & 31) == 0) {
        const int w = threadIdx.x >> 5;
        s[0][w] = pts; s[1][w] = lpts; s[2][w] = lines; s[3][w] = lmax; s_e[w] = hlogh;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        pts = lpts = lines = lmax = 0;
        hlogh = 0.0;
        for (int w = 0; w < 8; ++w) { pts += s[0][w]; lpts += s[1][w]; lines += s[2][w]; lmax = max(lmax, s[3][w]); hlogh += s_e[w]; }
        const int64_t o = (int64_t)b * K + k;
        if (L) L[o] = lines ? (double)lpts / (double)lines : 0.0;
        if (Lmax) Lmax[o] = lmax;
        if (rr) rr[o] = (double)pts / (double)((unsigned long long)(n - w) * (unsigned long long)(n - w + 1) / 2);
        if (entr) entr[o] = lines ? log((double)lines) - hlogh / (double)lines : 0.0;
    }
}

// One block per (threshold, series): LAM and TT from the vertical-line histogram, exact uint64 sums.
__global__ void __launch_bounds__(256) lam_tt_kernel(const uint64_t* __restrict__ vhist, int K, int64_t n, int64_t v_min,
                                                     double* __restrict__ lam, double* __restrict__ tt) {
    const int k = blockIdx.x, b = blockIdx.y;
    const uint64_t* row = vhist + ((int64_t)b * K + k) * n;
    unsigned long long all = 0, num = 0, lines = 0;
    for (int64_t v = 1 + threadIdx.x; v < n; v += blockDim.x) {
        const unsigned long long h = row[v];
        all += (unsigned long long)v * h;
        if (v >= v_min) { num += (unsigned long long)v * h; lines += h; }
    }
    __shared__ unsigned long long s[3][8];
    for (int off = 16; off; off >>= 1) {
        all += __shfl_down_sync(0xffffffffu, all, off);
        num += __shfl_down_sync(0xffffffffu, num, off);
        lines += __shfl_down_sync(0xffffffffu, lines, off);
    }
    if ((threadIdx.x & 31) == 0) { const int w = threadIdx.x >> 5; s[0][w] = all; s[1][w] = num; s[2][w] = lines; }
    __syncthreads();
    if (threadIdx.x == 0) {
        all = num = lines = 0;
        for (int w = 0; w < 8; ++w) { all += s[0][w]; num += s[1][w]; lines += s[2][w]; }
        const int64_t o = (int64_t)b * K + k;
        if (lam) lam[o] = all ? (double)num / (double)all : 0.0;
        if (tt) tt[o] = lines ? (double)num / (double)lines : 0.0;
    }
}

}  // namespace
}  // namespace rqa

using namespace rqa;

extern "C" {

rqa_status rqa_det_prefix_avg(const double* d_det, int32_t batch, int32_t K, double* d_prefix, void* stream) {
    if (!d_det || !d_prefix) { set_error("rqa_det_prefix_avg: NULL argument"); return RQA_ERR_INVALID_ARG; }
    if (batch < 1 || K < 1 || K > RQA_MAX_K) { set_error("rqa_det_prefix_avg: need batch >= 1, 1 <= K <= %d", RQA_MAX_K); return RQA_ERR_INVALID_ARG; }
    det_prefix_kernel<<<(batch + 127) / 128, 128, 0, (cudaStream_t)stream>>>(d_det, K, batch, d_prefix);
    RQA_LAUNCH_CHECK();
    return RQA_OK;
}

rqa_status rqa_line_measures(const uint64_t* d_hist, int32_t batch, int32_t K, int64_t n_points, int64_t l_min,
                             int64_t theiler, double* d_L, uint64_t* d_Lmax, double* d_rr_hist, double* d_entr,
                             void* stream) {
    if (!d_hist) { set_error("rqa_line_measures: d_hist is NULL"); return RQA_ERR_INVALID_ARG; }
    if (batch < 1 || K < 1 || K > RQA_MAX_K || n_points < 2 || l_min < 1 || theiler < 0 || theiler > n_points - 1) { set_error("rqa_line_measures: need batch >= 1, 1 <= K <= %d, n_points >= 2, l_min >= 1, 0 <= theiler <= n_points-1", RQA_MAX_K); return RQA_ERR_INVALID_ARG; }
    line_measures_kernel<<<dim3(K, batch), 256, 0, (cudaStream_t)stream>>>(d_hist, K, n_points, l_min, theiler > 1 ? theiler : 1, d_L,
                                                                          d_Lmax, d_rr_hist, d_entr);
    RQA_LAUNCH_CHECK();
    return RQA_OK;
}

rqa_status rqa_lam_tt(const uint64_t* d_vhist, int32_t batch, int32_t K, int64_t n_points, int64_t v_min, double* d_lam,
                      double* d_tt, void* stream) {
    if (!d_vhist) { set_error("rqa_lam_tt: d_vhist is NULL"); return RQA_ERR_INVALID_ARG; }
    if (batch < 1 || K < 1 || K > RQA_MAX_K || n_points < 2 || v_min < 1) { set_error("rqa_lam_tt: need batch >= 1, 1 <= K <= %d, n_points >= 2, v_min >= 1", RQA_MAX_K); return RQA_ERR_INVALID_ARG; }
    lam_tt_kernel<<<dim3(K, batch), 256, 0, (cudaStream_t)stream>>>(d_vhist, K, n_points, v_min, d_lam, d_tt);
    RQA_LAUNCH_CHECK();
    return RQA_OK;
}

rqa_status rqa_sorting_rate_host(const double* h_measure, int32_t R, int32_t n, double* h_S) {
    if (!h_measure || !h_S) { set_error("rqa_sorting_rate_host: NULL argument"); return RQA_ERR_INVALID_ARG; }
    if (R < 1 || n < 2) { set_error("rqa_sorting_rate_host: need R >= 1 realisations of n >= 2 series"); return RQA_ERR_INVALID_ARG; }
    // y_j = j (the series are given in their natural order), z = y reversed, x_j = place of series j when the
    // n series of one realisation are ordered by the measure (ascending; equal values keep their given order).
    long long worst = 0, dep = 0;
    for (int j = 1; j <= n; ++j) worst += llabs((long long)(n + 1 - j) - j);
    worst *= R;
    for (int i = 0; i < R; ++i) {
        const double* mrow = h_measure + (int64_t)i * n;
        for (int j = 0; j < n; ++j) {
            int x = 1;
            for (int q = 0; q < n; ++q) x += (mrow[q] < mrow[j]) || (mrow[q] == mrow[j] && q < j);
            dep += llabs((long long)x - (j + 1));
        }
    }
    *h_S = (double)(worst - dep) / (double)worst;
    return RQA_OK;
}

}  // extern "C"
