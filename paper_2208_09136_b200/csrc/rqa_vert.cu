// rqa_vert.cu — rqa_vert_hist: VERTICAL-line-length histograms of the recurrence plot at K thresholds in one pass
// ("this approach can also be applied for other RQA measures": laminarity LAM and trapping time TT are
// the vertical-line counterparts of DET and L; the paper defines no vertical-line measure itself, reading S19
// fixes the convention).
//
// Reading S19: a vertical line is a maximal run of recurrent cells down a column of the FULL symmetric N' x N' matrix
// (PAPER.md:57); the cells with |i - j| < w are excluded (w = 1: the main diagonal, S2; w > 1: the Theiler window,
// S9) and split a column in two; runs touching the border of the plot or the excluded band count with their truncated
// length (S8).  Every recurrent pair i<j is one cell of column j and one of column i: sum_v v*P_k(v) = 2*C_k.
//
// Work decomposition: a tile = 512 adjacent COLUMNS (one per thread) x a chunk of <= 1023 rows.  The lanes of a warp sit
// on 32 adjacent columns at the same row i, so the row point x_i is a shared-memory broadcast (kept in a register ring)
// and the thread's own point x_j lives in registers for the whole item: one shared-memory load per cell.  Everything
// after the distance — level table, monotone run stack, deferred events, aggregates for P(1..3), in-place carry across
// the chunks of a segment, (prefix, suffix) summaries at segment borders — is the machinery of the diagonal scan
// (rqa_scan.cuh), fed by another distance provider.  The full matrix has N'^2 cells: twice the work of rqa_line_hist.
#include <algorithm>
#include <cmath>

#include "rqa_scan.cuh"

namespace rqa {

namespace {

// Distances down one column.  W = warm-up cells before the chunk.  M > 0: compile-time (M, TAU), the row samples
// y[i .. i+S-1] in a register ring (one new sample per cell), the column's coordinates y[j + c*TAU] in registers.
// M == 0: run-time (m, tau) and point stride ps, recomputed from the two windows for every cell.
template <int NORM, int M, int TAU, int W>
struct ColDist {
    static constexpr int S = M > 0 ? (M - 1) * TAU + 1 : 1;
    float ring[S];
    float bj[M > 0 ? M : 1];
    uint32_t ya;                // cursor: shared-window address of the row sample of the current super-step's first cell
    uint32_t yb;                // shared-window address of the column's point in the column window
    int m, tau, ps;             // M == 0: run-time dimension, coordinate stride, point stride (floats)
    int rel_org;                // (first row of the chunk) - (column) + w - 1
    int rel;                    // the same for the cursor's row: cell R is excluded iff (unsigned)(rel + R) < band
    uint32_t band;              // 2w - 1

    __device__ __forceinline__ int pstride() const { return M > 0 ? 1 : ps; }
    __device__ __forceinline__ void seek(uint32_t ya_org, uint32_t yb_org, int t0) {
        ya = ya_org + 4 * (t0 + W) * pstride();
        yb = yb_org;
        rel = rel_org + t0;
    }
    __device__ __forceinline__ void advance(int cells) { ya += 4 * cells * pstride(); rel += cells; }
    __device__ __forceinline__ void prime() {
#pragma unroll
        for (int x = 0; x < (M > 0 ? S - 1 : 0); ++x) ring[x] = lds_f32(ya + 4 * x);
    }
    template <int R>
    __device__ __forceinline__ void push() {
        if (M > 0) ring[(R + S - 1) % S] = lds_f32(ya + 4 * (R + S - 1));
    }
    template <int R>
    __device__ __forceinline__ float distance() const {
        float d;
        if (M == 0) {
            float t0 = __fsub_rn(lds_f32(ya + 4 * R * ps), lds_f32(yb));
            d = NORM == RQA_NORM_MAX ? fabsf(t0) : __fmul_rn(t0, t0);
            for (int c = 1; c < m; ++c) {
                float t = __fsub_rn(lds_f32(ya + 4 * (R * ps + c * tau)), lds_f32(yb + 4 * c * tau));
                d = NORM == RQA_NORM_MAX ? fmaxf(d, fabsf(t)) : __fadd_rn(d, __fmul_rn(t, t));
            }
        } else {
            float t0 = __fsub_rn(ring[R % S], bj[0]);
            d = NORM == RQA_NORM_MAX ? fabsf(t0) : __fmul_rn(t0, t0);
#pragma unroll
            for (int c = 1; c < M; ++c) {
                float t = __fsub_rn(ring[(R + c * TAU) % S], bj[c]);
                d = NORM == RQA_NORM_MAX ? fmaxf(d, fabsf(t)) : __fadd_rn(d, __fmul_rn(t, t));
            }
        }
        if (NORM != RQA_NORM_MAX) d = __fsqrt_rn(d);
        // the excluded band |i - j| < w: not recurrent at any threshold
        return (uint32_t)(rel + R) < band ? __int_as_float(0x7f800000) : d;
    }
};

template <int NORM, int M, int TAU, int NP, bool MULTI>
using ColScanner = ScannerT<ColDist<NORM, M, TAU, 2>, NP, MULTI>;

struct VertArgs {
    View v;
    int g, NG, K, L, S;         // threshold group, groups, thresholds, rows per chunk, chunks per segment
    int part, parts, n_cbl;     // this process' column blocks: cb = part + q*parts, q < n_cbl
    const LineGroup* groups;
    unsigned long long* hist;   // [batch][K][n]
    unsigned long long* agg;    // [batch][NG][3][GK+1]
    uint32_t* pre;              // [batch][n_cbl][segs][2*NP][LW]
    uint32_t* suf;
    uint32_t* carry;            // [gridDim.x][2*NP][LW]
    unsigned int* counter;
    uint32_t segs;              // segments per column block = ceil(n / (S*L))
    int m, tau;
};

__host__ __device__ inline int col_window(int span, int ps) { return (LW * ps + span + 3 + 4) & ~3; }

template <int NORM, int M, int TAU, int NP>
__global__ void __launch_bounds__(LW, (NP <= 10 ? 2 : 1)) vert_scan_kernel(VertArgs a) {
    using SM = ScanSmem<NP>;
    extern __shared__ __align__(16) char smem[];
    __shared__ unsigned int s_item;
    __shared__ int s_rep[GK];

    const int tid = threadIdx.x;
    uint8_t* lut_s = (uint8_t*)(smem + SM::off_lut);
    float* eps_s = (float*)(smem + SM::off_eps);
    uint32_t* tot_s = (uint32_t*)(smem + SM::off_tot);
    uint32_t* agg_s = (uint32_t*)(smem + SM::off_agg);
    int32_t* sh_s = (int32_t*)(smem + SM::off_sh);
    uint16_t* stk_s = (uint16_t*)(smem + SM::off_stk);
    const int span = M > 0 ? (M - 1) * TAU : (a.m - 1) * a.tau;
    const int ps = M > 0 ? 1 : (int)a.v.ps;
    const int L = a.L;
    const int LA = window_la(L, span, 2, ps), LB = col_window(span, ps);
    float* ya_s = (float*)(smem + SM::off_ya);
    float* yb_s = ya_s + LA;
    const int64_t n = a.v.n;
    const int64_t T = (int64_t)a.S * L;
    const int64_t ny = (n - 1) * ps + span + 1;
    uint32_t* carry_col = a.carry + ((size_t)blockIdx.x * (2 * NP)) * LW + tid;
    const unsigned int per_series = a.segs * (unsigned)a.n_cbl;
    const unsigned int n_items = per_series * (unsigned)a.v.batch;

    stk_s[tid] = 0;
    for (int q = tid; q < SM::NLEV * LW; q += LW) agg_s[q] = 0;
    for (int q = tid; q < SM::NLEV * LS; q += LW) sh_s[q] = 0;
    if (tid < 3 * (GK + 1)) tot_s[tid] = 0;
    int cur_b = -1, J = 0;
    __syncthreads();

    while (true) {
        if (tid == 0) s_item = atomicAdd(a.counter, 1u);
        __syncthreads();
        const unsigned int item = s_item;
        if (item >= n_items) break;
        const int b = (int)(item / per_series);
        const uint32_t r_item = item - (uint32_t)b * per_series;
        const int q_cb = (int)(r_item / a.segs);
        const int seg = (int)(r_item - (uint32_t)q_cb * a.segs);
        const LineGroup& G = a.groups[(int64_t)b * a.NG + a.g];
        if (b != cur_b) {
            J = G.J;
            for (int q = tid; q < NB / 4; q += LW) ((uint32_t*)lut_s)[q] = ((const uint32_t*)G.lut)[q];
            if (tid <= GK) eps_s[tid] = G.epsd[tid];
            if (tid < GK) s_rep[tid] = G.rep_k[tid];
            stk_s[tid] = (uint16_t)J;
            cur_b = b;
        }
        const int64_t j0 = (int64_t)LW * (a.part + (int64_t)q_cb * a.parts);
        const int64_t j = j0 + tid;
        const bool valid = j < n;
        const int64_t seg_s = (int64_t)seg * T;                // first row of the segment
        const int c_end = (int)min((int64_t)a.S, (n - seg_s + L - 1) / L);
        const float* y = a.v.data + (int64_t)b * a.v.bs;
        unsigned long long* grow = a.hist + (int64_t)b * a.K * n;
        const size_t out_row = ((((size_t)b * a.n_cbl + q_cb) * a.segs + seg) * (2 * NP)) * LW + tid;
        for (int jj = 0; jj < J; ++jj) carry_col[jj * LW] = CARRY_SEG;
        // the columns' points: staged once per item
        for (int x = tid; x < LB; x += LW) {
            const int64_t gi = j0 * ps + x;
            yb_s[x] = gi < ny ? y[gi] : 0.0f;
        }
        for (int c = 0; c < c_end; ++c) {
            const int64_t s = seg_s + (int64_t)c * L;          // first row of the chunk
            for (int x = tid; x < LA; x += LW) {
                const int64_t gi = (s - 2) * ps + x;
                ya_s[x] = (gi >= 0 && gi < ny) ? y[gi] : 0.0f;
            }
            __syncthreads();
            const int cnt = valid ? (int)min((int64_t)L, n - s) : 0;
            const int cnt_hi = __shfl_sync(FULL, cnt, 0);
            const int cnt_lo = __shfl_sync(FULL, cnt, 31);
            if (cnt_hi > 0) {
                const uint32_t yb_org = pin(smem_addr(yb_s) + 4 * tid * ps);
                auto setup = [&](auto& sc) {
                    sc.ya_org = smem_addr(ya_s);
                    sc.lut = pin(smem_addr(lut_s) - BUCKET_MAGIC_BITS);
                    sc.eps = smem_addr(eps_s);
                    sc.agg = pin(smem_addr(agg_s) + 4 * tid);
                    sc.sh = smem_addr(sh_s);
                    sc.stk = pin(smem_addr(stk_s) + 2 * tid);
                    sc.q0 = pin(smem_addr(smem + SM::off_q) + 2 * tid);
                    sc.grow = (unsigned long long*)pin64((unsigned long long)grow);
                    sc.rep = G.rep_k;
                    sc.carry = carry_col;
                    sc.pre_out = a.pre + out_row;
                    sc.scale = G.scale;
                    sc.dcap = G.dcap;
                    sc.J4 = 4u * (uint32_t)J;
                    sc.m = a.m;
                    sc.tau = a.tau;
                    sc.ps = ps;
                    sc.n = (int64_t)pin64((unsigned long long)n);
                    sc.v1 = sc.v2 = sc.J4;
                    sc.w2a = sc.w2b = sc.J4;
                    sc.xa = sc.xb = 0;
                    sc.A = 0; sc.ts = 0; sc.top = sc.stk;
                    sc.rel_org = (int)(s - j + a.v.w - 1);
                    sc.band = (uint32_t)(2 * a.v.w - 1);
                    if (M > 0) {
#pragma unroll
                        for (int cc = 0; cc < (M > 0 ? M : 1); ++cc) sc.bj[cc] = yb_s[tid + cc * (M > 0 ? TAU : 1)];
                    }
                };
                const int first_real = -(int)min((int64_t)2, s);   // rows before the plot do not exist
                if (G.multi) {
                    ColScanner<NORM, M, TAU, NP, true> sc;
                    setup(sc);
                    scan_chunk(sc, cnt, cnt_lo, cnt_hi, first_real, yb_org);
                } else {
                    ColScanner<NORM, M, TAU, NP, false> sc;
                    setup(sc);
                    scan_chunk(sc, cnt, cnt_lo, cnt_hi, first_real, yb_org);
                }
            }
            __syncthreads();
            reduce_chunk_aggregates(agg_s, tot_s, J);
            __syncthreads();
        }
        // end of the segment: the runs still alive (and the prefix runs that never ended) for the stitch kernel
        if (valid) {
            for (int jj = 0; jj < J; ++jj) {
                const uint32_t cj = carry_col[jj * LW];
                if (cj & CARRY_SEG) a.pre[out_row + (size_t)jj * LW] = cj & ~CARRY_SEG;
                a.suf[out_row + (size_t)jj * LW] = cj & ~CARRY_SEG;
            }
        }
        flush_item(tot_s, sh_s, J, a.agg + ((int64_t)b * a.NG + a.g) * 3 * (GK + 1), grow, s_rep, n);
        __syncthreads();
    }
}

// One thread per (column, distinct threshold): join the (prefix, suffix) summaries of consecutive segments and emit the
// lines of length >= 4 that touch a segment border (including the two ends of the column).
struct VStitchArgs {
    int64_t n, T;
    int g, NG, K, NP, part, parts, n_cbl;
    const LineGroup* groups;
    unsigned long long* hist;
    const uint32_t* pre;
    const uint32_t* suf;
    uint32_t segs;
};

__global__ void __launch_bounds__(LW) vert_stitch_kernel(VStitchArgs a) {
    const int q_cb = blockIdx.x, jj = blockIdx.y, b = blockIdx.z;
    const LineGroup& G = a.groups[(int64_t)b * a.NG + a.g];
    if (jj >= G.J) return;
    const int tid = threadIdx.x;
    const int64_t col = (int64_t)LW * (a.part + (int64_t)q_cb * a.parts) + tid;
    if (col >= a.n) return;
    unsigned long long* row = a.hist + ((int64_t)b * a.K + G.rep_k[jj]) * a.n;
    const int64_t stride = (int64_t)(2 * a.NP) * LW;
    const int64_t base = ((((int64_t)b * a.n_cbl + q_cb) * a.segs) * (2 * a.NP) + jj) * LW + tid;
    uint32_t carry = 0;
    for (uint32_t c = 0; c < a.segs; ++c) {
        const uint32_t p = a.pre[base + (int64_t)c * stride], sf = a.suf[base + (int64_t)c * stride];
        const uint32_t cntc = (uint32_t)min(a.T, a.n - (int64_t)c * a.T);
        if (p == cntc) {
            carry += cntc;
        } else {
            const uint32_t tot = carry + p;
            if (tot >= (uint32_t)LMIN_EXPLICIT) atomicAdd(&row[tot], 1ull);
            carry = sf;
        }
    }
    if (carry >= (uint32_t)LMIN_EXPLICIT) atomicAdd(&row[carry], 1ull);
}

// General strided views the tiles cannot stage: one thread per column, K run counters, global atomics.
template <int NORM>
__global__ void __launch_bounds__(128) vert_strided_kernel(View v, const float* __restrict__ eps, int K,
                                                           unsigned long long* __restrict__ hist, int part, int parts) {
    const int b = blockIdx.y;
    if ((int)(blockIdx.x % (unsigned)parts) != part) return;
    const int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= v.n) return;
    const float* yb = v.data + (int64_t)b * v.bs;
    const float* e = eps + (int64_t)b * K;
    unsigned long long* h = hist + (int64_t)b * K * v.n;
    uint32_t run[RQA_MAX_K];
    for (int k = 0; k < K; ++k) run[k] = 0;
    for (int64_t i = 0; i < v.n; ++i) {
        const int64_t gap = i > j ? i - j : j - i;
        const float d = gap < v.w ? __int_as_float(0x7f800000) : point_distance<NORM>(yb, min(i, j), max(i, j), v.m, v.ps, v.cs);
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

__global__ void vert_eps_check_kernel(const float* __restrict__ eps, int64_t count, WsStatus* status) {
    bool bad = false;
    for (int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; q < count; q += (int64_t)gridDim.x * blockDim.x) {
        const float x = eps[q];
        bad |= !(x >= 0.0f) || isinf(x);
    }
    if (bad) atomicExch(&status->bad_eps, 1);
}

// ------------------------------------------------------------------------------------------ host side
constexpr size_t SMEM_PER_BLOCK_MAX = 227 * 1024 - 256;
constexpr size_t SMEM_PER_SM = 228 * 1024, SMEM_BLOCK_RESERVED = 1024;

struct VertPlan {
    bool scan;
    int L, S, NG, NP, gs, span, blocks_per_sm;
    int n_cb, n_cbl;            // column blocks of the plot / of this part
    uint32_t segs;
    unsigned grid;
    size_t smem;
};

size_t vert_smem_bytes(int NP, int L, int span, int ps) {
    const size_t fixed = NP == 5 ? ScanSmem<5>::off_ya : (NP == 10 ? ScanSmem<10>::off_ya : ScanSmem<16>::off_ya);
    return fixed + 4 * ((size_t)window_la(L, span, 2, ps) + col_window(span, ps));
}

VertPlan make_vert_plan(const View& v, int K, const Options& opt) {
    VertPlan p{};
    p.span = (int)std::min<int64_t>((int64_t)(v.m - 1) * v.cs, (int64_t)MAX_SPAN + 1);
    p.gs = group_size_for(K, opt);
    p.NG = (K + p.gs - 1) / p.gs;
    p.NP = scan_pairs_for(std::min(K, p.gs));
    p.blocks_per_sm = p.NP <= 10 ? 2 : 1;
    const int ps = (int)std::min<int64_t>(v.ps, 1 << 20);
    p.scan = p.span <= MAX_SPAN && vert_smem_bytes(p.NP, 32, p.span, ps) <= SMEM_PER_BLOCK_MAX;
    const unsigned slots = (unsigned)(sm_count() * p.blocks_per_sm);
    const double cells = (double)v.n * (double)v.n * (double)v.batch / (double)opt.parts;
    int64_t L = (int64_t)std::ceil(cells / ((double)LW * slots * 4.0));
    p.L = (int)std::max<int64_t>(32, std::min<int64_t>(LMAX, L));
    if (opt.line_chunk > 0) p.L = (int)std::min<int64_t>(LMAX, opt.line_chunk);
    const size_t budget = std::min(SMEM_PER_SM / p.blocks_per_sm - SMEM_BLOCK_RESERVED, SMEM_PER_BLOCK_MAX);
    while (p.scan && p.L > 32 && vert_smem_bytes(p.NP, p.L, p.span, ps) > budget) p.L = std::max(32, p.L - 16);
    while (p.scan && p.L > 32 && vert_smem_bytes(p.NP, p.L, p.span, ps) > SMEM_PER_BLOCK_MAX) p.L = std::max(32, p.L / 2);
    p.n_cb = (int)((v.n + LW - 1) / LW);
    p.n_cbl = p.n_cb > opt.part ? (p.n_cb - opt.part + opt.parts - 1) / opt.parts : 0;
    const uint64_t chunks = (uint64_t)((v.n + p.L - 1) / p.L) * (uint64_t)p.n_cbl * (uint64_t)v.batch;
    int64_t S = (int64_t)(chunks / ((uint64_t)slots * 8));
    p.S = (int)std::max<int64_t>(1, std::min<int64_t>(8, S));
    if (opt.line_segment > 0) p.S = opt.line_segment;
    p.segs = (uint32_t)((v.n + (int64_t)p.S * p.L - 1) / ((int64_t)p.S * p.L));
    const uint64_t items = (uint64_t)p.segs * (uint64_t)p.n_cbl * (uint64_t)v.batch;
    p.grid = (unsigned)std::max<uint64_t>(1, std::min<uint64_t>(items, slots));
    p.smem = vert_smem_bytes(p.NP, p.L, p.span, ps);
    return p;
}

template <int NORM, int M, int TAU, int NP>
rqa_status launch_vscan(const VertArgs& a, const VertPlan& p, cudaStream_t s) {
    auto kern = vert_scan_kernel<NORM, M, TAU, NP>;
    static thread_local bool attr_set[8] = {false};
    int dev = 0;
    RQA_CUDA_TRY(cudaGetDevice(&dev));
    if (dev >= 8 || !attr_set[dev]) {
        RQA_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_PER_BLOCK_MAX));
        if (dev < 8) attr_set[dev] = true;
    }
    kern<<<p.grid, LW, p.smem, s>>>(a);
    RQA_LAUNCH_CHECK();
    return RQA_OK;
}

template <int NORM, int NP>
rqa_status dispatch_vembedding(const VertArgs& a, const VertPlan& p, cudaStream_t s) {
    const bool delay = a.v.ps == 1;
    if (delay && a.m == 1) return launch_vscan<NORM, 1, 1, NP>(a, p, s);
    if (delay && a.m == 3 && a.tau == 1) return launch_vscan<NORM, 3, 1, NP>(a, p, s);
    if (delay && a.m == 3 && a.tau == 3) return launch_vscan<NORM, 3, 3, NP>(a, p, s);
    if (delay && a.m == 5 && a.tau == 2) return launch_vscan<NORM, 5, 2, NP>(a, p, s);
    return launch_vscan<NORM, 0, 0, NP>(a, p, s);
}

template <int NORM>
rqa_status dispatch_vpairs(const VertArgs& a, const VertPlan& p, cudaStream_t s) {
    if (p.NP == 5) return dispatch_vembedding<NORM, 5>(a, p, s);
    if (p.NP == 10) return dispatch_vembedding<NORM, 10>(a, p, s);
    return dispatch_vembedding<NORM, 16>(a, p, s);
}

struct VertWs {
    LineGroup* groups;
    unsigned long long* agg;
    unsigned int* counters;
    uint32_t *pre, *suf, *carry;
};
VertWs carve_vert(Arena& ws, const View& v, const VertPlan& p) {
    VertWs w{};
    w.groups = ws.take<LineGroup>((size_t)v.batch * p.NG);
    w.agg = (unsigned long long*)ws.take<uint64_t>((size_t)v.batch * p.NG * 3 * (GK + 1));
    w.counters = ws.take<unsigned int>((size_t)p.NG);
    const size_t rows = (size_t)v.batch * p.n_cbl * p.segs * 2 * p.NP * LW;
    w.pre = ws.take<uint32_t>(rows);
    w.suf = ws.take<uint32_t>(rows);
    w.carry = ws.take<uint32_t>((size_t)p.grid * 2 * p.NP * LW);
    return w;
}

}  // namespace

size_t vert_workspace_bytes(const View& v, int K, const Options& opt) {
    VertPlan p = make_vert_plan(v, K, opt);
    if (!p.scan) return 256;
    Arena a(nullptr, ~(size_t)0);
    carve_vert(a, v, p);
    return a.off;
}

rqa_status run_vert_hist(const View& v, int norm, const float* d_eps, int K, uint64_t* d_vhist, Arena& ws, cudaStream_t s,
                         const Options& opt) {
    WsStatus* status = (WsStatus*)ws.base;
    const size_t hist_words = (size_t)v.batch * K * v.n;
    // many series of moderate length: one block per series walks every column once for all K thresholds (rqa_block.cu)
    // (N'^2 cells per block: only where the plot itself is moderate, whatever the Theiler window leaves of it)
    if (opt.parts == 1 && block_line_fits(v, K) && v.n <= 4096 &&
        (opt.line_path == 2 || (opt.line_path == 0 && opt.line_chunk == 0 && (int64_t)v.batch * ((K + GK - 1) / GK) >= 192)))
        return run_line_block(v, norm, d_eps, K, d_vhist, status, s, true);
    RQA_CUDA_TRY(cudaMemsetAsync(d_vhist, 0, sizeof(uint64_t) * hist_words, s));
    VertPlan p = make_vert_plan(v, K, opt);
    if (!p.scan) {
        vert_eps_check_kernel<<<1, 256, 0, s>>>(d_eps, (int64_t)v.batch * K, status);
        RQA_LAUNCH_CHECK();
        dim3 grid((unsigned)((v.n + 127) / 128), (unsigned)v.batch);
        if (norm == RQA_NORM_MAX)
            vert_strided_kernel<RQA_NORM_MAX><<<grid, 128, 0, s>>>(v, d_eps, K, (unsigned long long*)d_vhist, opt.part, opt.parts);
        else
            vert_strided_kernel<RQA_NORM_EUCLID><<<grid, 128, 0, s>>>(v, d_eps, K, (unsigned long long*)d_vhist, opt.part, opt.parts);
        RQA_LAUNCH_CHECK();
        return reduce_parts(opt, d_vhist, hist_words, s);
    }
    VertWs w = carve_vert(ws, v, p);
    if (!ws.ok()) { set_error("rqa_vert_hist: workspace too small"); return RQA_ERR_WORKSPACE_TOO_SMALL; }
    const size_t agg_words = (size_t)v.batch * p.NG * 3 * (GK + 1);
    RQA_CUDA_TRY(cudaMemsetAsync(w.agg, 0, sizeof(uint64_t) * agg_words, s));
    RQA_CUDA_TRY(cudaMemsetAsync(w.counters, 0, sizeof(unsigned int) * (size_t)p.NG, s));
    rqa_status st = launch_line_groups(d_eps, K, p.NG, p.gs, v.batch, w.groups, status, s);
    if (st != RQA_OK) return st;
    for (int g = 0; g < p.NG && p.n_cbl > 0; ++g) {
        VertArgs a;
        a.v = v; a.g = g; a.NG = p.NG; a.K = K; a.L = p.L; a.S = p.S;
        a.part = opt.part; a.parts = opt.parts; a.n_cbl = p.n_cbl;
        a.groups = w.groups; a.hist = (unsigned long long*)d_vhist; a.agg = w.agg;
        a.pre = w.pre; a.suf = w.suf; a.carry = w.carry; a.counter = w.counters + g; a.segs = p.segs;
        a.m = v.m; a.tau = (int)v.cs;
        if (g == 0 && opt.ev_begin) RQA_CUDA_TRY(cudaEventRecord((cudaEvent_t)opt.ev_begin, s));
        st = norm == RQA_NORM_MAX ? dispatch_vpairs<RQA_NORM_MAX>(a, p, s) : dispatch_vpairs<RQA_NORM_EUCLID>(a, p, s);
        if (st != RQA_OK) return st;
        if (g == 0 && opt.ev_end) RQA_CUDA_TRY(cudaEventRecord((cudaEvent_t)opt.ev_end, s));
        VStitchArgs sa;
        sa.n = v.n; sa.T = (int64_t)p.S * p.L; sa.g = g; sa.NG = p.NG; sa.K = K; sa.NP = p.NP;
        sa.part = opt.part; sa.parts = opt.parts; sa.n_cbl = p.n_cbl;
        sa.groups = w.groups; sa.hist = (unsigned long long*)d_vhist; sa.pre = w.pre; sa.suf = w.suf; sa.segs = p.segs;
        vert_stitch_kernel<<<dim3((unsigned)p.n_cbl, (unsigned)(2 * p.NP), (unsigned)v.batch), LW, 0, s>>>(sa);
        RQA_LAUNCH_CHECK();
    }
    st = reduce_parts(opt, d_vhist, hist_words, s);
    if (st != RQA_OK) return st;
    st = reduce_parts(opt, w.agg, agg_words, s);
    if (st != RQA_OK) return st;
    return launch_line_finalize(v.n, p.NG, p.NP, K, v.batch, w.groups, w.agg, (unsigned long long*)d_vhist, status, s);
}

}  // namespace rqa
