// rqa_block.cu — thresholds for MANY series of moderate length (8192 < P <= 2^22 counted pairs, N' up to ~2900) in one
// call: one thread block selects all K thresholds of a series, nothing is materialised in global memory.
//
// The paper's experiment grid is 900 series per length at N = 10^2, 10^3 with K = 99 recurrence rates
// (PAPER.md:82-84).  For N = 10^3 the materialise-then-radix-select path of rqa_select.cu reads the 1.8 GB of
// distances of such a batch eight times with a prefix search per element (18 ms); here every series is one block that
// recomputes its distances from a shared-memory copy of the series in three walks over the triangle:
//   walk 1  histogram of all P distances over BLK_NB1 equal-width bins of [0, bound]   (bound >= every distance)
//           -> per target: its bin, the count below the bin, the residual rank inside it
//   walk 2  for the cells that fall into a target's bin: histogram over its BLK_SUB equal sub-bins
//           -> per target: its (bin, sub-bin) cell, count below, residual rank
//   walk 3  the cells that fall into a target's (bin, sub-bin) cell are collected (a few per target), sorted by their
//           fp32 bit patterns in shared memory, and eps_k = the residual-rank-th of its cell, C_k = #{d <= eps_k}
// (readings S4-S6: exact order statistic, ties counted).  The bin of a distance is floor(d * scale), a
// monotone function of d, so everything in a lower bin is strictly smaller than everything in a higher one and equal
// values share a bin: the selection is exact.  A series whose target cells hold more than BLK_CAP distances (massive
// ties: a constant or coarsely quantised series) is flagged and done by the radix passes of rqa_select.cu.
#include <algorithm>
#include <cmath>

#include "rqa_tiles.cuh"

namespace rqa {

namespace {

constexpr int BLK_THREADS = 1024;
constexpr int BLK_NB1 = 4096;            // bins of walk 1
constexpr int BLK_SUB = 128;             // sub-bins of walk 2 (128: two blocks per SM fit at K = 99)
constexpr int BLK_CAP = 8192;            // collected distances of walk 3 (sorted in shared memory)
constexpr uint32_t BLK_MARK = 0x80000000u;
constexpr size_t BLK_SMEM_MAX = 227 * 1024 - 4096;   // opt-in limit minus the static arrays below

struct BlockTargets {
    unsigned long long r[RQA_MAX_K];     // ranks, ascending
    int32_t k_of[RQA_MAX_K];             // caller's index of the target
};

// Distance provider.  M > 0: a delay view (point stride 1) with m == M whose samples sit in shared memory at byte
// address `sa`: shared-memory loads with compile-time trip counts.  M == 0: any view, through a generic pointer (the
// shared copy when it fits, the global series otherwise).
template <int NORM, int M>
struct BlockDist {
    uint32_t sa;
    int cs4;                     // 4 * coordinate stride (bytes)
    const float* yb;
    int m, ps, cs;
    __device__ __forceinline__ float at(int i, int o) const {
        if (M > 0) {
            const uint32_t a = sa + 4u * (uint32_t)i, b = a + 4u * (uint32_t)o;
            if (NORM == RQA_NORM_MAX) {
                float d = 0.0f;
#pragma unroll
                for (int c = 0; c < M; ++c) d = fmaxf(d, fabsf(__fsub_rn(lds_f32(a + c * cs4), lds_f32(b + c * cs4))));
                return d;
            }
            float t = __fsub_rn(lds_f32(a), lds_f32(b));
            float s = __fmul_rn(t, t);
#pragma unroll
            for (int c = 1; c < M; ++c) {
                t = __fsub_rn(lds_f32(a + c * cs4), lds_f32(b + c * cs4));
                s = __fadd_rn(s, __fmul_rn(t, t));
            }
            return __fsqrt_rn(s);
        }
        const float* pa = yb + (size_t)i * ps;
        const float* pb = pa + (size_t)o * ps;
        if (NORM == RQA_NORM_MAX) {
            float d = 0.0f;
            for (int c = 0; c < m; ++c) d = fmaxf(d, fabsf(__fsub_rn(pa[c * cs], pb[c * cs])));
            return d;
        }
        float t = __fsub_rn(pa[0], pb[0]);
        float s = __fmul_rn(t, t);
        for (int c = 1; c < m; ++c) {
            t = __fsub_rn(pa[c * cs], pb[c * cs]);
            s = __fadd_rn(s, __fmul_rn(t, t));
        }
        return __fsqrt_rn(s);
    }
};

// Every counted cell (i, j = i + o), o = w..n-1, exactly once.  Diagonal w + q is paired with diagonal n - 1 - q: every
// pair has n - w + 1 cells.  A pair is cut into `split` equal ranges so that the items fill the block; the lanes of a
// warp sit on adjacent diagonals at the same i (x_i is a broadcast, x_j a run of consecutive addresses).
template <class D, class F>
__device__ __forceinline__ void walk_triangle(const D& dist, int n, int w, int split, F&& f) {
    const int nd = n - w, nq = (nd + 1) / 2, items = nq * split;
    for (int it = threadIdx.x; it < items; it += BLK_THREADS) {
        const int h = it / nq, q = it - h * nq;
        const int o1 = w + q, o2 = n - 1 - q, len1 = n - o1, len = len1 + (o2 != o1 ? n - o2 : 0);
        const int a = (int)((long long)len * h / split), b = (int)((long long)len * (h + 1) / split);
        const int e1 = b < len1 ? b : len1;
#pragma unroll 8
        for (int i = a; i < e1; ++i) f(dist.at(i, o1));
        const int a2 = (a > len1 ? a : len1) - len1, e2 = b - len1;
#pragma unroll 8
        for (int i = a2; i < e2; ++i) f(dist.at(i, o2));
    }
}

__device__ __forceinline__ int bin_of(float t) {               // t >= 0 (a NaN converts to 0, +inf to INT_MAX)
    return min((int)t, BLK_NB1 - 1);
}
__device__ __forceinline__ int sub_of(float t, int bin) {
    const int s = (int)(__fmul_rn(__fsub_rn(t, (float)bin), (float)BLK_SUB));   // t - bin is exact for t < BLK_NB1
    return min(max(s, 0), BLK_SUB - 1);
}

// Shared memory: hist1 [BLK_NB1] | hist2 [K][BLK_SUB] | cand [BLK_CAP] (32-bit words) | slot1 [BLK_NB1] bytes |
// the series (stage_floats floats, optional)
__host__ __device__ inline size_t block_smem_bytes(int K, size_t stage_floats) {
    return 4 * ((size_t)BLK_NB1 + (size_t)K * BLK_SUB + (size_t)BLK_CAP + stage_floats) + (size_t)BLK_NB1;
}

template <int NORM, int M>
__global__ void __launch_bounds__(BLK_THREADS) sel_block_kernel(View v, BlockTargets tg, int K, unsigned int P,
                                                                int stage_floats, int split, int32_t* fallback,
                                                                size_t fallback_stride, float* __restrict__ eps,
                                                                unsigned long long* __restrict__ count,
                                                                double* __restrict__ rr) {
    extern __shared__ __align__(16) uint32_t s_mem[];
    __shared__ float s_red[2][BLK_THREADS / 32];
    __shared__ uint32_t s_scan[BLK_THREADS / 32];
    __shared__ int s_bin[RQA_MAX_K], s_slot[RQA_MAX_K], s_sub[RQA_MAX_K];
    __shared__ uint32_t s_below[RQA_MAX_K], s_rho[RQA_MAX_K], s_before[RQA_MAX_K];
    __shared__ uint32_t s_ncand, s_total;
    __shared__ float s_scale;
    uint32_t* hist1 = s_mem;
    uint32_t* hist2 = hist1 + BLK_NB1;
    uint32_t* cand = hist2 + (size_t)K * BLK_SUB;
    uint8_t* slot1 = (uint8_t*)(cand + BLK_CAP);
    float* stage = (float*)(slot1 + BLK_NB1);

    const int b = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int n = (int)v.n, w = (int)v.w, m = v.m, ps = (int)v.ps, cs = (int)v.cs;
    const float* yb = v.data + (int64_t)b * v.bs;

    // the series' value range bounds every distance: |a - b| <= max - min per coordinate (Euclid: times sqrt(m))
    const int ny = (n - 1) * ps + (m - 1) * cs + 1;
    float lo = __int_as_float(0x7f800000), hi = -lo;
    for (int q = tid; q < ny; q += BLK_THREADS) {
        const float x = yb[q];
        if (stage_floats) stage[q] = x;
        lo = fminf(lo, x);
        hi = fmaxf(hi, x);
    }
    for (int off = 16; off; off >>= 1) {
        lo = fminf(lo, __shfl_xor_sync(0xffffffffu, lo, off));
        hi = fmaxf(hi, __shfl_xor_sync(0xffffffffu, hi, off));
    }
    if (lane == 0) { s_red[0][warp] = lo; s_red[1][warp] = hi; }
    for (int q = tid; q < BLK_NB1; q += BLK_THREADS) { hist1[q] = 0; slot1[q] = 0; }
    for (int q = tid; q < K * BLK_SUB; q += BLK_THREADS) hist2[q] = 0;
    if (tid == 0) s_ncand = 0;
    __syncthreads();
    if (tid == 0) {
        float a = s_red[0][0], c = s_red[1][0];
        for (int q = 1; q < BLK_THREADS / 32; ++q) { a = fminf(a, s_red[0][q]); c = fmaxf(c, s_red[1][q]); }
        float bound = c - a;
        if (NORM != RQA_NORM_MAX) bound *= sqrtf((float)m);
        s_scale = bound > 0.0f && bound < __int_as_float(0x7f800000) ? (float)BLK_NB1 / bound : 0.0f;
    }
    __syncthreads();
    if (stage_floats) yb = stage;
    const float scale = s_scale;
    BlockDist<NORM, M> dist;
    dist.sa = smem_addr(stage);
    dist.cs4 = 4 * cs;
    dist.yb = yb; dist.m = m; dist.ps = ps; dist.cs = cs;

    // ---- walk 1: all distances into BLK_NB1 bins
    walk_triangle(dist, n, w, split, [&](float d) { atomicAdd(&hist1[bin_of(__fmul_rn(d, scale))], 1u); });
    __syncthreads();
    {   // inclusive prefix sums of hist1 in place (four bins per thread)
        uint32_t c[BLK_NB1 / BLK_THREADS], sum = 0;
#pragma unroll
        for (int q = 0; q < BLK_NB1 / BLK_THREADS; ++q) { sum += hist1[tid * (BLK_NB1 / BLK_THREADS) + q]; c[q] = sum; }
        uint32_t incl = sum;
        for (int off = 1; off < 32; off <<= 1) {
            const uint32_t u = __shfl_up_sync(0xffffffffu, incl, off);
            if (lane >= off) incl += u;
        }
        if (lane == 31) s_scan[warp] = incl;
        __syncthreads();
        if (warp == 0) {
            uint32_t x = s_scan[lane];
            for (int off = 1; off < 32; off <<= 1) {
                const uint32_t u = __shfl_up_sync(0xffffffffu, x, off);
                if (lane >= off) x += u;
            }
            s_scan[lane] = x;
        }
        __syncthreads();
        const uint32_t base = incl - sum + (warp ? s_scan[warp - 1] : 0u);
#pragma unroll
        for (int q = 0; q < BLK_NB1 / BLK_THREADS; ++q) hist1[tid * (BLK_NB1 / BLK_THREADS) + q] = base + c[q];
    }
    __syncthreads();
    if (tid < K) {                                             // target tid: first bin whose cumulative count reaches its rank
        const uint32_t r = (uint32_t)tg.r[tid];
        int a = 0, c = BLK_NB1 - 1;
        while (a < c) {
            const int mid = (a + c) >> 1;
            if (hist1[mid] >= r) c = mid; else a = mid + 1;
        }
        const uint32_t below = a ? hist1[a - 1] : 0u;
        s_bin[tid] = a;
        s_below[tid] = below;
        s_rho[tid] = r - below;
    }
    __syncthreads();
    if (tid == 0) {                                            // distinct target bins, ascending (ranks are ascending)
        int slot = 0;
        for (int t = 0; t < K; ++t) {
            if (t > 0 && s_bin[t] != s_bin[t - 1]) ++slot;
            s_slot[t] = slot;
            slot1[s_bin[t]] = (uint8_t)(slot + 1);
        }
    }
    __syncthreads();

    // ---- walk 2: the cells of the target bins into BLK_SUB sub-bins each
    walk_triangle(dist, n, w, split, [&](float d) {
        const float t = __fmul_rn(d, scale);
        const int bin = bin_of(t), s = slot1[bin];
        if (s) atomicAdd(&hist2[(s - 1) * BLK_SUB + sub_of(t, bin)], 1u);
    });
    __syncthreads();
    if (tid < K) {
        const uint32_t* h = hist2 + s_slot[tid] * BLK_SUB;
        const uint32_t rho = s_rho[tid];
        uint32_t acc = 0;
        int sub = 0;
        for (; sub < BLK_SUB - 1; ++sub) {
            if (acc + h[sub] >= rho) break;
            acc += h[sub];
        }
        s_sub[tid] = sub;
        s_below[tid] += acc;
        s_rho[tid] = rho - acc;
    }
    __syncthreads();
    if (tid == 0) {                                            // distinct target cells, ascending: offsets in the sorted list
        uint32_t before = 0, prev_count = 0;
        for (int t = 0; t < K; ++t) {
            const int cell = s_slot[t] * BLK_SUB + s_sub[t];
            if (t > 0 && cell != s_slot[t - 1] * BLK_SUB + s_sub[t - 1]) before += prev_count;
            prev_count = hist2[cell] & ~BLK_MARK;
            hist2[cell] |= BLK_MARK;
            s_before[t] = before;
        }
        s_total = before + prev_count;
    }
    __syncthreads();
    const uint32_t total = s_total;
    if (total > (uint32_t)BLK_CAP) {                          // massive ties: the radix passes redo this series
        if (tid == 0) *(int32_t*)((char*)fallback + (size_t)b * fallback_stride) = 1;
        return;
    }

    // ---- walk 3: collect the distances of the target cells, sort them
    walk_triangle(dist, n, w, split, [&](float d) {
        const float t = __fmul_rn(d, scale);
        const int bin = bin_of(t), s = slot1[bin];
        if (s && (hist2[(s - 1) * BLK_SUB + sub_of(t, bin)] & BLK_MARK)) {
            const uint32_t at = atomicAdd(&s_ncand, 1u);
            if (at < (uint32_t)BLK_CAP) cand[at] = __float_as_uint(d);
        }
    });
    int P2 = 2;
    while ((uint32_t)P2 < total) P2 <<= 1;
    __syncthreads();
    for (int q = (int)total + tid; q < P2; q += BLK_THREADS) cand[q] = 0xffffffffu;      // padding sorts last
    __syncthreads();
    for (int k = 2; k <= P2; k <<= 1) {
        for (int j = k >> 1; j > 0; j >>= 1) {
            for (int t = tid; t < P2 / 2; t += BLK_THREADS) {
                const int q = 2 * t - (t & (j - 1)), p = q | j;
                const uint32_t a = cand[q], c = cand[p];
                const bool up = (q & k) == 0;
                if ((a > c) == up) { cand[q] = c; cand[p] = a; }
            }
            __syncthreads();
        }
    }
    if (tid < K) {
        const uint32_t e = cand[s_before[tid] + s_rho[tid] - 1];
        int a = 0, c = (int)total;                              // first index with key > e
        while (a < c) {
            const int mid = (a + c) >> 1;
            if (cand[mid] <= e) a = mid + 1; else c = mid;
        }
        const unsigned long long C = (unsigned long long)s_below[tid] + ((uint32_t)a - s_before[tid]);
        const int64_t at = (int64_t)b * K + tg.k_of[tid];
        eps[at] = __uint_as_float(e);
        count[at] = C;
        rr[at] = (double)C / (double)P;
    }
}


// ------------------------------------------------------------------------------------------- diagonal lines
// rqa_line_hist for the same regime: one block per series, one thread per pair of diagonals.
// Thresholds are nested, so after a cell of level v (= number of distinct thresholds below its distance) exactly the
// thresholds j >= v are inside a run, and the runs of all thresholds on a diagonal form a stack of (lowest threshold,
// start) entries: a lower level pushes one entry, a higher level pops the entries it ends, each giving ONE line length for
// a whole range [a, b) of thresholds, counted as D[a][len]++, D[b][len]-- in a shared-memory difference array over the
// thresholds (lengths below LB_LCAP; longer lines use the histogram rows themselves as the difference array).  Work per cell
// does not depend on K: all K = 99 thresholds of the paper's sweep in ONE walk, where the tiled scan takes one pass per
// group of 32.  The level of a cell: a bucket table over [0, eps_max] gives the thresholds in lower buckets, a short
// loop adds those of the cell's own bucket.
constexpr int LB_THREADS = 512;
constexpr int LB_LCAP = 128;             // line lengths counted in shared memory
constexpr int LB_NB = 4096;              // buckets of the level table

__host__ __device__ inline size_t line_block_smem_bytes(int K, size_t stage_floats) {
    return 4 * ((size_t)(K + 1) * LB_LCAP + stage_floats) + (size_t)LB_NB;
}

// VERT: the same walk down the COLUMNS of the full symmetric matrix (rqa_vert_hist, reading S19): one thread per
// column j, rows i = 0..n-1, the cells with |i - j| < w excluded (not recurrent at any threshold; they split a column).
template <int NORM, int M, bool VERT>
__global__ void __launch_bounds__(LB_THREADS, 3) line_block_kernel(View v, const float* __restrict__ eps, int K,
                                                                  int stage_floats,
                                                                  unsigned long long* __restrict__ hist,
                                                                  WsStatus* status) {
    extern __shared__ __align__(16) uint32_t s_mem[];
    __shared__ float s_eps[RQA_MAX_K + 1], s_san[RQA_MAX_K];
    __shared__ int s_jof[RQA_MAX_K], s_first[RQA_MAX_K];
    __shared__ int s_J;
    int* s_D = (int*)s_mem;                                   // [(K + 1)][LB_LCAP]
    uint8_t* lut = (uint8_t*)(s_D + (size_t)(K + 1) * LB_LCAP);
    float* stage = (float*)(lut + LB_NB);

    const int b = blockIdx.x, tid = threadIdx.x;
    const int n = (int)v.n, w = (int)v.w, m = v.m, ps = (int)v.ps, cs = (int)v.cs;
    const float* yb = v.data + (int64_t)b * v.bs;
    const float* e = eps + (int64_t)b * K;
    unsigned long long* out = hist + (int64_t)b * K * n;

    if (stage_floats) {
        const int ny = (n - 1) * ps + (m - 1) * cs + 1;
        for (int q = tid; q < ny; q += LB_THREADS) stage[q] = yb[q];
        yb = stage;
    }
    for (int q = tid; q < (K + 1) * LB_LCAP; q += LB_THREADS) s_D[q] = 0;
    // the histogram rows beyond the shared-memory lengths start at zero (written before the walk's atomics)
    if (n > LB_LCAP)
        for (int q = tid; q < K * (n - LB_LCAP); q += LB_THREADS) {
            const int k = q / (n - LB_LCAP), l = LB_LCAP + (q - k * (n - LB_LCAP));
            out[(int64_t)k * n + l] = 0ull;
        }
    // the K thresholds sorted, duplicates removed: distinct index j_of[k] of caller threshold k
    bool bad = false;
    for (int k = tid; k < K; k += LB_THREADS) {
        float x = e[k];
        if (!(x >= 0.0f) || isinf(x)) { bad = true; x = 0.0f; }
        s_san[k] = x;
    }
    if (bad) atomicExch(&status->bad_eps, 1);
    if (tid == 0) s_J = 0;
    __syncthreads();
    for (int k = tid; k < K; k += LB_THREADS) {
        int first = 1;
        for (int u = 0; u < k; ++u) first &= s_san[u] != s_san[k];
        s_first[k] = first;
    }
    __syncthreads();
    for (int k = tid; k < K; k += LB_THREADS) {
        int below = 0;
        for (int q = 0; q < K; ++q) below += s_first[q] && s_san[q] < s_san[k];
        s_jof[k] = below;
        s_eps[below] = s_san[k];
        atomicMax(&s_J, below + 1);
    }
    __syncthreads();
    const int J = s_J;
    const float emax = s_eps[J - 1];
    const float scale = emax > 0.0f ? (float)LB_NB / emax : 0.0f;
    // lut[q] = thresholds whose bucket is below q (all of them are below every distance of bucket q)
    for (int q = tid; q < LB_NB; q += LB_THREADS) {
        int a = 0, c = J;
        while (a < c) {
            const int mid = (a + c) >> 1;
            if (min((int)__fmul_rn(s_eps[mid], scale), LB_NB - 1) < q) a = mid + 1; else c = mid;
        }
        lut[q] = (uint8_t)a;
    }
    __syncthreads();

    BlockDist<NORM, M> dist;
    dist.sa = smem_addr(stage);
    dist.cs4 = 4 * cs;
    dist.yb = yb; dist.m = m; dist.ps = ps; dist.cs = cs;

    uint32_t stk[RQA_MAX_K + 1];                              // (lowest threshold << 16 | start), top = smallest threshold
    auto emit = [&](int lo, int upto, int len) {              // one line of `len` cells for the thresholds [lo, upto)
        if (len < LB_LCAP) {
            atomicAdd(&s_D[lo * LB_LCAP + len], 1);
            atomicSub(&s_D[upto * LB_LCAP + len], 1);
        } else {
            // long lines: the same difference array in the histogram rows themselves (row j = distinct threshold j for
            // now; 64-bit wrap-around arithmetic; no row is needed for upto == J)
            atomicAdd(&out[(int64_t)lo * n + len], 1ull);
            if (upto < J) atomicAdd(&out[(int64_t)upto * n + len], ~0ull);
        }
    };
    // Every lane is a small state machine over its two diagonals: one step either takes the next cell (level, maybe a
    // push) or ends ONE stack entry of a pending level rise.  A rise that ends several entries spreads over several
    // steps while the other lanes go on with their cells, so the warp never waits for the longest pop sequence of a
    // cell (lanes drift apart along their diagonals; the walk's loads are then plain shared-memory gathers).
    const int nd = n - w, nq = VERT ? n : (nd + 1) / 2;
    for (int q = tid; q < nq; q += LB_THREADS) {
        const int o1 = VERT ? q : w + q, o2 = VERT ? q : n - 1 - q;      // VERT: o = the column
        int o = o1, len = VERT ? n : n - o1, t = 0;
        int depth = 0, pv = J;                                 // top entry in `cur`, the entries below in stk[0 .. depth-2]
        uint32_t cur = 0;
        int vnew = -1, tend = 0;                               // pending rise: the thresholds [.., vnew) end before cell tend
        bool second = o2 == o1;                                // no second diagonal for the middle one (VERT: never)
        while (true) {
            if (vnew >= 0) {                                   // end one entry
                const uint32_t nxt = depth > 1 ? stk[depth - 2] : ((uint32_t)J << 16);
                const int lo = (int)(cur >> 16), start = (int)(cur & 0xffffu), hi = (int)(nxt >> 16);
                emit(lo, hi < vnew ? hi : vnew, tend - start);
                if (hi <= vnew) {
                    --depth;
                    cur = nxt;
                    if (hi == vnew || depth == 0) vnew = -1;
                } else {
                    cur = ((uint32_t)vnew << 16) | (uint32_t)start;            // the rest of the entry lives on
                    vnew = -1;
                }
            } else if (t < len) {                              // next cell
                int lev = J;
                const int gap = VERT ? (t > o ? t - o : o - t) : w;
                if (gap >= w) {
                    const float d = VERT ? dist.at(t < o ? t : o, gap) : dist.at(t, o);
                    lev = lut[min((int)__fmul_rn(d, scale), LB_NB - 1)];
                    while (lev < J && s_eps[lev] < d) ++lev;
                }
                if (lev < pv) {
                    if (depth > 0) stk[depth - 1] = cur;
                    cur = ((uint32_t)lev << 16) | (uint32_t)t;
                    ++depth;
                } else if (lev > pv) {
                    vnew = lev;
                    tend = t;
                }
                pv = lev;
                ++t;
            } else if (pv < J) {                               // end of the diagonal: every open run ends
                vnew = J;
                tend = len;
                pv = J;
            } else if (!second) {                              // on to the partner diagonal
                second = true;
                o = o2; len = n - o2; t = 0;
            } else {
                break;
            }
        }
    }
    __syncthreads();
    // prefix sums of D over the thresholds turn every column into the histogram of the distinct thresholds
    const int ncol = n < LB_LCAP ? n : LB_LCAP;
    for (int l = tid; l < ncol; l += LB_THREADS) {
        int acc = 0;
        for (int j = 0; j < J; ++j) {
            acc += s_D[j * LB_LCAP + l];
            s_D[j * LB_LCAP + l] = acc;
        }
    }
    __syncthreads();
    for (int q = tid; q < K * ncol; q += LB_THREADS) {
        const int k = q / ncol, l = q - k * ncol;
        out[(int64_t)k * n + l] = l == 0 ? 0ull : (unsigned long long)(unsigned int)s_D[s_jof[k] * LB_LCAP + l];
    }
    // the long lengths: prefix sums over the distinct thresholds, then row k of the caller = row j_of[k] (a column is
    // read completely by its thread before it is rewritten)
    for (int l = LB_LCAP + tid; l < n; l += LB_THREADS) {
        unsigned long long acc = 0;
        for (int j = 0; j < J; ++j) {
            acc += out[(int64_t)j * n + l];
            stk[j] = (uint32_t)acc;
        }
        for (int k = 0; k < K; ++k) out[(int64_t)k * n + l] = (unsigned long long)stk[s_jof[k]];
    }
}

}  // namespace

bool block_select_fits(const View& v, int K) {
    const uint64_t P = n_pairs(v);
    return P > 0 && P <= (1ull << 22) && v.n <= (1 << 20) && v.ps <= 64 && v.cs <= (1 << 16) &&
           block_smem_bytes(K, 0) <= BLK_SMEM_MAX;
}

rqa_status run_select_block(const View& v, int norm, const uint64_t* h_rank, int K, float* d_eps, uint64_t* d_count,
                            double* d_rr, int32_t* d_fallback, size_t fallback_stride, cudaStream_t s) {
    int order[RQA_MAX_K];
    for (int k = 0; k < K; ++k) order[k] = k;
    std::stable_sort(order, order + K, [&](int a, int b) { return h_rank[a] < h_rank[b]; });
    BlockTargets tg{};
    for (int t = 0; t < K; ++t) { tg.r[t] = h_rank[order[t]]; tg.k_of[t] = order[t]; }
    // the series is copied to shared memory when it fits beside the histograms
    const size_t ny = (size_t)(v.n - 1) * v.ps + (size_t)(v.m - 1) * v.cs + 1;
    const size_t stage = block_smem_bytes(K, ny) <= BLK_SMEM_MAX ? ny : 0;
    const size_t smem = block_smem_bytes(K, stage);
    // cut the diagonal pairs so that the work items fill the block's threads evenly
    const int nq = (int)((v.n - v.w + 1) / 2);
    int split = 1;
    double best = 0.0;
    for (int c = 1; c <= 8; ++c) {
        const double items = (double)nq * c, eff = items / (std::ceil(items / BLK_THREADS) * BLK_THREADS);
        if (eff > best + 0.02) { best = eff; split = c; }
    }
    // compiled-in embedding for staged delay views of the common dimensions
    const int M = (stage && v.ps == 1 && (v.m == 1 || v.m == 3)) ? v.m : 0;
    using Kern = void (*)(View, BlockTargets, int, unsigned int, int, int, int32_t*, size_t, float*, unsigned long long*, double*);
    const bool mx = norm == RQA_NORM_MAX;
    Kern kern = M == 1 ? (mx ? sel_block_kernel<RQA_NORM_MAX, 1> : sel_block_kernel<RQA_NORM_EUCLID, 1>)
              : M == 3 ? (mx ? sel_block_kernel<RQA_NORM_MAX, 3> : sel_block_kernel<RQA_NORM_EUCLID, 3>)
                       : (mx ? sel_block_kernel<RQA_NORM_MAX, 0> : sel_block_kernel<RQA_NORM_EUCLID, 0>);
    static thread_local bool attr_set[8][6] = {};
    int dev = 0;
    RQA_CUDA_TRY(cudaGetDevice(&dev));
    const int which = (mx ? 0 : 1) + 2 * (M == 1 ? 1 : M == 3 ? 2 : 0);
    if (dev >= 8 || !attr_set[dev][which]) {
        RQA_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)BLK_SMEM_MAX));
        if (dev < 8) attr_set[dev][which] = true;
    }
    kern<<<v.batch, BLK_THREADS, smem, s>>>(v, tg, K, (unsigned int)n_pairs(v), (int)stage, split, d_fallback, fallback_stride,
                                            d_eps, (unsigned long long*)d_count, d_rr);
    RQA_LAUNCH_CHECK();
    return RQA_OK;
}

bool block_line_fits(const View& v, int K) {
    const uint64_t P = n_pairs(v);
    return P > 0 && P <= (1ull << 22) && v.n < 65536 && v.ps <= 64 && v.cs <= (1 << 16) &&
           line_block_smem_bytes(K, 0) <= 100 * 1024;
}

rqa_status run_line_block(const View& v, int norm, const float* d_eps, int K, uint64_t* d_hist, WsStatus* status,
                          cudaStream_t s, bool vertical) {
    const size_t ny = (size_t)(v.n - 1) * v.ps + (size_t)(v.m - 1) * v.cs + 1;
    const size_t stage = line_block_smem_bytes(K, ny) <= 74 * 1024 ? ny : 0;      // three blocks per SM
    const size_t smem = line_block_smem_bytes(K, stage);
    const int M = (stage && v.ps == 1 && (v.m == 1 || v.m == 3)) ? v.m : 0;
    using Kern = void (*)(View, const float*, int, int, unsigned long long*, WsStatus*);
    const bool mx = norm == RQA_NORM_MAX;
    Kern kern;
    if (!vertical)
        kern = M == 1 ? (mx ? line_block_kernel<RQA_NORM_MAX, 1, false> : line_block_kernel<RQA_NORM_EUCLID, 1, false>)
             : M == 3 ? (mx ? line_block_kernel<RQA_NORM_MAX, 3, false> : line_block_kernel<RQA_NORM_EUCLID, 3, false>)
                      : (mx ? line_block_kernel<RQA_NORM_MAX, 0, false> : line_block_kernel<RQA_NORM_EUCLID, 0, false>);
    else
        kern = M == 1 ? (mx ? line_block_kernel<RQA_NORM_MAX, 1, true> : line_block_kernel<RQA_NORM_EUCLID, 1, true>)
             : M == 3 ? (mx ? line_block_kernel<RQA_NORM_MAX, 3, true> : line_block_kernel<RQA_NORM_EUCLID, 3, true>)
                      : (mx ? line_block_kernel<RQA_NORM_MAX, 0, true> : line_block_kernel<RQA_NORM_EUCLID, 0, true>);
    static thread_local bool attr_set[8][12] = {};
    int dev = 0;
    RQA_CUDA_TRY(cudaGetDevice(&dev));
    const int which = (mx ? 0 : 1) + 2 * (M == 1 ? 1 : M == 3 ? 2 : 0) + (vertical ? 6 : 0);
    if (dev >= 8 || !attr_set[dev][which]) {
        RQA_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 110 * 1024));
        if (dev < 8) attr_set[dev][which] = true;
    }
    kern<<<v.batch, LB_THREADS, smem, s>>>(v, d_eps, K, (int)stage, (unsigned long long*)d_hist, status);
    RQA_LAUNCH_CHECK();
    return RQA_OK;
}

}  // namespace rqa
