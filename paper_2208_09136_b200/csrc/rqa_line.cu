// rqa_line.cu — rqa_line_hist: diagonal-line-length histograms P_k(l) at K thresholds in ONE pass over the
// upper triangle (Eq. 4 and the sentence under it; upper triangle only, R_ij
// computed on the fly, never stored).  Design notes: DESIGN.md "Kernel: diagonal scan".
//
// Work decomposition
//   tile   = 512 adjacent diagonals (one per thread) x one chunk of <= 1023 positions; a thread walks its
//            chunk of its diagonal sequentially, lanes of a warp read y[i] (broadcast) and y[i+o+lane]
//            (consecutive) from two windows of the series staged in shared memory.
//   cell   : distance d (sliding window over e_i = |y_i - y_{i+o}| for the max norm), then its LEVEL
//            v = #{distinct thresholds < d} by one table lookup + one exact compare (thresholds are nested:
//            the cell is recurrent at threshold j iff v <= j).
//   runs   : thresholds are nested, so the runs of all thresholds along a diagonal form a monotone stack of
//            (lowest threshold, start position); it changes only when the maximum level of the last 4 cells
//            changes, and one popped entry is one line length for a whole RANGE of thresholds, counted in a
//            difference array over the thresholds.  The work per cell does not depend on K.  In the bulk of a
//            chunk a thread only notes the changes in a small queue; all lanes replay their queues together
//            every 24 cells, so that the divergent stack code runs with most lanes busy.
//   lines  : P_j(1), P_j(2), P_j(3) are NOT emitted line by line.  The kernel histograms the level of every
//            cell and the window maxima of 2 and 3 consecutive levels (thread-private shared-memory words of three
//            10-bit counters, no conflicts; a chunk has <= 1023 cells); their prefix sums over the level are
//            C_j = sum l*P_j(l), Q2_j = sum (l-1)*P_j(l) and Q3_j = sum_{l>=3} (l-2)*P_j(l), from which the
//            finalize kernel solves P_j(1..3) exactly.
//            Lines of length >= 4 that lie inside a chunk go to the shared-memory difference array (l < 128) or
//            to global atomics (longer).  Runs touching a chunk border are written as (prefix, suffix) summaries
//            and joined along each diagonal by the stitch kernel.

#include "rqa_tiles.cuh"

namespace rqa {

namespace {

constexpr int LMAX = 1023;       // longest chunk: cell positions fit the 10 bits of a stack entry, counters 10 bits
constexpr int LS = 128;          // lines shorter than this are counted in shared memory
constexpr int LMIN_EXPLICIT = 4; // lines of length >= 4 are emitted one by one; 1..3 come from the aggregates
constexpr int QCELLS = 24;       // cells between two drains of the per-thread event queues (= their capacity)

// Everything the scan needs to know about one group of <= 32 thresholds of one series.
struct LineGroup {
    int32_t J;            // number of distinct thresholds in the group, 1..32
    int32_t multi;        // 1 if some table bucket holds two or more distinct thresholds (refine by a loop)
    int32_t kcount;       // caller thresholds in this group
    int32_t pad;
    float scale;          // bucket(d) = bucket_of(d, dcap, scale) (rqa_tiles.cuh): one FMA, exact rounding
    float dcap;
    float epsd[GK + 1];   // distinct thresholds ascending, epsd[J] = +inf
    int32_t k_of[GK];     // sorted position -> caller's index k
    int32_t j_of[GK];     // sorted position -> distinct index j
    int32_t rep_k[GK];    // distinct index j -> the caller index whose histogram row accumulates the counts
    uint8_t lut[NB];      // bucket -> 4 * #{distinct thresholds in lower buckets}
};

// One block per series: sort the K thresholds, split them into groups of 32, build each group's table.
__global__ void __launch_bounds__(128) line_groups_kernel(const float* __restrict__ eps, int K, int NG,
                                                          LineGroup* __restrict__ groups, WsStatus* status) {
    const int b = blockIdx.x;
    const float* e = eps + (int64_t)b * K;
    __shared__ float s_sorted[RQA_MAX_K];
    __shared__ int s_korder[RQA_MAX_K];
    __shared__ int s_bad;
    if (threadIdx.x == 0) s_bad = 0;
    __syncthreads();
    for (int k = threadIdx.x; k < K; k += blockDim.x) {
        float x = e[k];
        if (!(x >= 0.0f) || isinf(x)) { s_bad = 1; x = 0.0f; }
        int pos = 0;
        for (int q = 0; q < K; ++q) {
            float z = e[q];
            if (!(z >= 0.0f) || isinf(z)) z = 0.0f;
            pos += (z < x) || (z == x && q < k);
        }
        s_sorted[pos] = x;
        s_korder[pos] = k;
    }
    __syncthreads();
    if (threadIdx.x == 0 && s_bad) atomicExch(&status->bad_eps, 1);
    for (int g = 0; g < NG; ++g) {
        LineGroup& G = groups[(int64_t)b * NG + g];
        const int base = g * GK;
        const int kc = min(GK, K - base);
        __shared__ int s_J;
        __shared__ float s_scale, s_dcap;
        if (threadIdx.x == 0) {
            int J = 0;
            for (int q = 0; q < kc; ++q) {
                float x = s_sorted[base + q];
                if (q == 0 || x != s_sorted[base + q - 1]) { G.epsd[J] = x; G.rep_k[J] = s_korder[base + q]; ++J; }
                G.k_of[q] = s_korder[base + q];
                G.j_of[q] = J - 1;
            }
            for (int q = J; q <= GK; ++q) G.epsd[q] = __int_as_float(0x7f800000);
            G.J = J;
            G.kcount = kc;
            G.pad = 0;
            // bucket function: linear in d up to just above the largest threshold, NB-1 buckets wide
            float emax = s_sorted[base + kc - 1];
            float dcap = emax >= 3.0e38f ? 3.4028234e38f : nextafterf(emax, __int_as_float(0x7f800000));
            float scale = bucket_scale(dcap);
            G.scale = scale;
            G.dcap = dcap;
            s_J = J; s_scale = scale; s_dcap = dcap;
        }
        __syncthreads();
        const int J = s_J;
        const float scale = s_scale, dcap = s_dcap;
        int multi = 0;
        for (int q = threadIdx.x; q < NB; q += blockDim.x) {
            int below = 0, inside = 0;
            for (int j = 0; j < J; ++j) {
                uint32_t bj = bucket_of(G.epsd[j], dcap, scale);
                below += bj < (uint32_t)q;
                inside += bj == (uint32_t)q;
            }
            G.lut[q] = (uint8_t)(4 * below);
            multi |= inside > 1;
        }
        multi = __syncthreads_or(multi);
        if (threadIdx.x == 0) G.multi = multi;
        __syncthreads();
    }
}

// tile_start[ob] = number of tiles of the diagonal blocks before ob; diagonal block ob = diagonals
// 1 + 256*ob .. 256 + 256*ob, its longest diagonal has n - 1 - 256*ob cells, cut into chunks of L.
__global__ void __launch_bounds__(1024) tile_table_kernel(int64_t n, int L, int n_ob, uint32_t* __restrict__ tile_start) {
    __shared__ uint32_t s_part[1024];
    const int per = (n_ob + 1023) / 1024;
    const int lo = threadIdx.x * per, hi = min(n_ob, lo + per);
    uint32_t sum = 0;
    for (int ob = lo; ob < hi; ++ob) sum += (uint32_t)((n - 1 - (int64_t)LW * ob + L - 1) / L);
    s_part[threadIdx.x] = sum;
    __syncthreads();
    for (int off = 1; off < 1024; off <<= 1) {
        uint32_t t = threadIdx.x >= off ? s_part[threadIdx.x - off] : 0;
        __syncthreads();
        s_part[threadIdx.x] += t;
        __syncthreads();
    }
    uint32_t run = s_part[threadIdx.x] - sum;
    for (int ob = lo; ob < hi; ++ob) {
        tile_start[ob] = run;
        run += (uint32_t)((n - 1 - (int64_t)LW * ob + L - 1) / L);
    }
    if (threadIdx.x == 1023) tile_start[n_ob] = s_part[1023];
}

// ------------------------------------------------------------------------------------------ the scan
// Cell distances: CellDist (rqa_tiles.cuh) with two warm-up cells before the chunk.
// Shared-memory plan of the scan kernel (bytes); NP: the group has J <= 2*NP distinct thresholds.
// The two series windows come last because their length depends on the run-time span (m-1)*tau.
template <int NP>
struct ScanSmem {
    static constexpr int NLEV = 2 * NP + 1;                   // levels 0..2NP
    static constexpr int off_lut = 0;
    static constexpr int off_eps = off_lut + NB;
    static constexpr int off_agg = off_eps + 4 * (GK + 4);
    static constexpr int agg_row = 4 * LW;                    // one level: a word per thread = three 10-bit counters
    static constexpr int off_sh = off_agg + NLEV * agg_row;   // int32 D[NLEV][LS]: difference array over the thresholds
    static constexpr int stk_row = 2 * LW;                    // one stack depth: a 16-bit entry per thread
    static constexpr int off_stk = off_sh + 4 * NLEV * LS;    // uint16 stack[NLEV][LW]
    static constexpr int off_q = off_stk + NLEV * stk_row;    // uint16 queue[QCELLS][LW]: deferred stack events
    static constexpr int off_ya = off_q + QCELLS * stk_row;
};
struct ScanArgs {
    View v;
    int g, NG, K, L, n_ob;
    const LineGroup* groups;
    const uint32_t* tile_start;
    unsigned long long* hist;   // [batch][K][n]
    unsigned long long* agg;    // [batch][NG][3][GK+1]
    uint16_t* pre;              // [batch][tiles][2*NP][LW]  prefix run of every threshold (recurrent since the chunk start)
    uint16_t* suf;              // [batch][tiles][2*NP][LW]  run alive at the chunk end
    uint32_t tiles;
    int m, tau;                 // run-time embedding (used by the M == 0 variant)
};

// Run state of one diagonal.  Thresholds are nested, so after a cell of level v exactly the thresholds j >= v are
// inside a run, and the start of that run does not increase with j: the runs of all thresholds form a monotone stack.
// Only runs that matter for explicit emission are kept: thresholds j >= A = max(level of the last 4 cells) have a run
// of >= 4 cells (shorter lines come from the aggregates).  Entry = (lo, start) covers the thresholds [lo, lo of the
// entry below); the top entry (lo = A) lives in registers, the others in a per-thread shared-memory column as
// uint16 (start << 6 | lo), bottom-most a sentinel with lo = J.  Cells before the chunk count as level 0, so the
// initial entry (0, start 0) stands for "recurrent since the chunk start" (prefix runs; start 0 marks them).
// Per cell the state changes only when A changes: a higher level pops the entries it ends (one line length for a
// whole range of thresholds -> D[lo][len]++, D[hi][len]--), a lower A pushes one entry.  Cost independent of K.
template <int NORM, int M, int TAU, int NP, bool MULTI>
struct Scanner : CellDist<NORM, M, TAU, 2> {
    using CD = CellDist<NORM, M, TAU, 2>;
    static constexpr int S = CD::S;
    using SM = ScanSmem<NP>;

    // per-thread state
    uint32_t v1, v2;            // 4*level of the previous two cells (real cells, also before the chunk)
    uint32_t w2a, w2b;          // max(level pairs) of the previous two cells (newest first)
    uint32_t xa, xb;            // the same with cells before the chunk at level 0 (only used for t < 4)
    uint32_t A;                 // 4 * lowest threshold in the stack = lo of the top entry (J4: stack empty)
    uint32_t ts;                // start of the top entry's run (cell index inside the chunk)
    uint32_t top;               // shared-window address of the entry below the top (stk: the sentinel)
    uint32_t aprev;             // phase 1: 4 * max level of the 4 cells before this one (A lags until the drain)
    uint32_t qp;                // phase 1: shared-window address of the thread's next free queue slot
    uint32_t trel8;             // phase 1: (cells since the last drain) << 8
    // per-thread constants
    uint32_t lut, eps;          // shared-window addresses of the bucket table (biased, see level4) and the thresholds
    uint32_t agg;               // ... of the thread's column of histogram 1, level 0
    uint32_t sh;                // ... of the difference array D
    uint32_t stk;               // ... of the thread's stack column, depth 0 (the sentinel)
    uint32_t q0;                // ... of the thread's event queue, slot 0
    uint32_t ya_org;            // ... of the i-side window, index 0
    unsigned long long* grow;   // hist + b*K*n (rows indexed through rep)
    const int* rep;
    uint16_t* pre_out;
    float scale, dcap;
    uint32_t J4;
    int64_t n;

    __device__ __forceinline__ uint32_t level4(float d) const {
        uint32_t q = lds_u8(lut + bucket_bits(d, dcap, scale));   // lut is biased by -BUCKET_MAGIC_BITS
        float er = lds_f32(eps + q);
        uint32_t v4 = q + (d > er ? 4u : 0u);
        if (MULTI) {                                           // some bucket holds two or more thresholds
            while (d > lds_f32(eps + v4)) v4 += 4;
        }
        return v4;
    }

    // One run of `len` cells ended for the thresholds [lo4, hi4) / 4.  start == 0: it began at the chunk start.
    __device__ __forceinline__ void ended(uint32_t lo4, uint32_t hi4, uint32_t start, uint32_t len) {
        if (start != 0 && len < (uint32_t)LS) {
            const uint32_t col = sh + 4 * len;
            red_u32(col + lo4 * LS, 1u);
            red_u32(col + hi4 * LS, 0xffffffffu);
        } else if (start == 0) {
#pragma unroll 1
            for (uint32_t j4 = lo4; j4 < hi4; j4 += 4) pre_out[(j4 >> 2) * LW] = (uint16_t)len;
        } else {
#pragma unroll 1
            for (uint32_t j4 = lo4; j4 < hi4; j4 += 4) atomicAdd(&grow[(int64_t)rep[j4 >> 2] * n + len], 1ull);
        }
    }

    // The cell at position t has level v4 > A: the runs of the thresholds [A, v4) ended at the previous cell.
    __device__ __forceinline__ void pop_runs(uint32_t v4, uint32_t t) {
        uint32_t e = lds_u16(top);                             // the entry below the top (or the sentinel)
        uint32_t nlo = (e << 2) & 0xfcu;
        ended(A, min(nlo, v4), ts, t - ts);
        A = v4;                                                // the rest of the entry lives on ...
        if (nlo > v4) return;
#pragma unroll 1
        while (top != stk) {                                   // ... unless it ended entirely: next entry
            top -= SM::stk_row;
            ts = e >> 6;
            if (nlo == v4) return;
            const uint32_t lo = nlo;
            e = lds_u16(top);
            nlo = (e << 2) & 0xfcu;
            ended(lo, min(nlo, v4), ts, t - ts);
            if (nlo > v4) return;
        }
        A = J4;                                                // the sentinel is reached: everything ended
    }

    // A_new < A: the thresholds [A_new, A) have just completed 4 cells; their run started at t - 3.
    __device__ __forceinline__ void push_run(uint32_t a_new, uint32_t t) {
        if (A < J4) {
            top += SM::stk_row;
            sts_u16(top, (A >> 2) | (ts << 6));
        }
        A = a_new;
        ts = t - 3;
    }

    // One cell.  R = offset from the cursor = ring phase (static), t = position inside the chunk (t < 0: warm-up
    // cells before the chunk), cnt = this lane's number of cells.  PHASE 0: the first cells of the chunk (t < 4,
    // guarded), 1: the part of the chunk where every lane is inside (unguarded; t is not used), 2: the tail (guarded).
    template <int R, int PHASE>
    __device__ __forceinline__ void cell(int t, int cnt, int first_real) {
        constexpr bool GUARD = PHASE != 1;
        CD::template push<R>();
        if (GUARD && t < 0) {
            // cells before the start of the diagonal do not exist: not recurrent at any threshold
            uint32_t v4 = t < first_real ? J4 : level4(CD::template distance<R>());
            v2 = v1; v1 = v4;
            return;
        }
        if (GUARD && t >= cnt) return;
        const float d = CD::template distance<R>();
        const uint32_t v4 = level4(d);
        // aggregates: level, max of 2, max of 3 consecutive levels (thread-private columns)
        const uint32_t w2 = max(v4, v1), w3 = max(w2, v2);
        red_u32(agg + v4 * (SM::agg_row / 4), 1u);
        red_u32(agg + w2 * (SM::agg_row / 4), 1u << 10);
        red_u32(agg + w3 * (SM::agg_row / 4), 1u << 20);
        // runs of >= 4 cells: A_new = max level of the last 4 cells of the chunk.  The stack changes only when it
        // differs from the previous cell's.  Phase 1 does not touch the stack: the thread notes (cell, A_new) in its
        // queue and all lanes replay their queues together every QCELLS cells (drain), so that the divergent stack
        // code runs with most lanes busy instead of for one or two lanes per warp-cell.
        if (PHASE == 1) {
            const uint32_t a_new = max(w2, w2b);
            if (a_new != aprev) {
                sts_u16(qp, a_new + trel8 + ((uint32_t)R << 8));
                qp += SM::stk_row;
            }
            aprev = a_new;
        } else {
            uint32_t x2 = w2;
            if (PHASE == 0 && t == 0) x2 = v4;
            const uint32_t a_new = max(x2, PHASE == 0 ? xb : w2b);
            if (a_new != A) {
                if (v4 > A) pop_runs(v4, (uint32_t)t);
                else push_run(a_new, (uint32_t)t);
            }
            if (PHASE == 0) { xb = xa; xa = x2; }
        }
        v2 = v1; v1 = v4;
        w2b = w2a; w2a = w2;
    }

    // Replay the queued events of the window that started at cell win_t0 (call with the warp converged).
    __device__ __forceinline__ void drain(uint32_t win_t0) {
        const uint32_t nmax = __reduce_max_sync(FULL, qp - q0);
        uint32_t rp = q0;
#pragma unroll 1
        for (uint32_t k = 0; k < nmax; k += SM::stk_row) {
            if (rp < qp) {
                const uint32_t rec = lds_u16(rp);
                const uint32_t a_new = rec & 0xffu, t = win_t0 + (rec >> 8);
                if (a_new > A) pop_runs(a_new, t);            // a higher level: A_new is that level
                else push_run(a_new, t);
                rp += SM::stk_row;
            }
        }
        qp = q0;
        trel8 = 0;
    }

    template <int PHASE, int... R>
    __device__ __forceinline__ void superstep(int t, int cnt, int ds, std::integer_sequence<int, R...>) {
        (cell<R, PHASE>(t + R, cnt, ds), ...);
        CD::advance((int)sizeof...(R));
        if (PHASE == 1) trel8 += (uint32_t)sizeof...(R) << 8;
    }

    // End of the chunk (cnt > 0 cells): the prefix runs that never ended, and the run alive at the end for every
    // threshold (from the stack for j >= A/4, else 0..3 cells from the last levels).
    __device__ __forceinline__ void finish(uint32_t cnt, uint16_t* suf_out) {
        const uint32_t w3 = max(w2a, w2b);
#pragma unroll 1
        for (uint32_t j4 = 0; j4 < min(A, J4); j4 += 4)
            suf_out[(j4 >> 2) * LW] = (uint16_t)((v1 <= j4) + (w2a <= j4) + (w3 <= j4));
        uint32_t lo = A, st = ts;
#pragma unroll 1
        while (lo < J4) {
            const uint32_t e = lds_u16(top);
            const uint32_t nlo = (e << 2) & 0xfcu;
#pragma unroll 1
            for (uint32_t j4 = lo; j4 < nlo; j4 += 4) {
                suf_out[(j4 >> 2) * LW] = (uint16_t)(cnt - st);
                if (st == 0) pre_out[(j4 >> 2) * LW] = (uint16_t)cnt;
            }
            lo = nlo; st = e >> 6;
            if (top != stk) top -= SM::stk_row;
        }
    }
};

// The walk of one thread along its chunk.  Two instantiations (MULTI) so that the common case, every bucket of the
// level table holding at most one threshold, carries no refinement loop; a block executes only one of them.
template <int NORM, int M, int TAU, int NP, bool MULTI>
__device__ __forceinline__ void scan_chunk(Scanner<NORM, M, TAU, NP, MULTI>& sc, int cnt, int cnt_lo, int cnt_hi, int ds,
                                           uint32_t yb_org, uint16_t* suf_out) {
    using SC = Scanner<NORM, M, TAU, NP, MULTI>;
    constexpr int S = SC::S;
    constexpr int U = S == 3 ? 12 : (S > 3 ? S : 4);          // cells per super-step, a multiple of S
    static_assert(U + 2 <= WSLACK && U <= QCELLS, "window slack and queue capacity cover one super-step");
    using Seq = std::make_integer_sequence<int, U>;
    int t = -2;                                               // first cell is the warm-up cell t = -2
    sc.seek(sc.ya_org, yb_org, t);
    sc.prime();
    for (; t < 4; t += U) sc.template superstep<0>(t, cnt, ds, Seq{});   // warm-up cells and t < 4
    constexpr int SPW = QCELLS / U;                          // super-steps per drain window
    sc.aprev = sc.A;
    sc.qp = sc.q0;
    sc.trel8 = 0;
    while (t + U <= cnt_lo) {
        const int t0w = t;
#pragma unroll 1
        for (int w = 0; w < SPW && t + U <= cnt_lo; ++w, t += U) sc.template superstep<1>(t, cnt, ds, Seq{});
        sc.drain((uint32_t)t0w);
    }
    for (; t < cnt_hi; t += U) sc.template superstep<2>(t, cnt, ds, Seq{});
    if (cnt > 0) sc.finish((uint32_t)cnt, suf_out);
}

template <int NORM, int M, int TAU, int NP>
__global__ void __launch_bounds__(LW, (NP <= 10 ? 2 : 1)) line_scan_kernel(ScanArgs a) {
    using SM = ScanSmem<NP>;
    extern __shared__ __align__(16) char smem[];
    __shared__ int s_ob;
    __shared__ int s_rep[GK];

    const int tid = threadIdx.x;
    const int b = blockIdx.y;
    const uint32_t tile = blockIdx.x;
    const LineGroup& G = a.groups[(int64_t)b * a.NG + a.g];
    // which diagonal block / chunk is this tile
    find_diagonal_block(a.tile_start, a.n_ob, tile, &s_ob);
    // stage the group's table and thresholds, clear the histograms
    uint8_t* lut_s = (uint8_t*)(smem + SM::off_lut);
    float* eps_s = (float*)(smem + SM::off_eps);
    const int span = M > 0 ? (M - 1) * TAU : (a.m - 1) * a.tau;
    const int ps = M > 0 ? 1 : (int)a.v.ps;
    const int LA = window_la(a.L, span, 2, ps), LB = window_lb(a.L, span, 2, ps);
    float* ya_s = (float*)(smem + SM::off_ya);
    float* yb_s = ya_s + LA;
    uint32_t* agg_s = (uint32_t*)(smem + SM::off_agg);
    int32_t* sh_s = (int32_t*)(smem + SM::off_sh);
    uint16_t* stk_s = (uint16_t*)(smem + SM::off_stk);
    const int J = G.J;
    for (int q = tid; q < NB / 4; q += LW) ((uint32_t*)lut_s)[q] = ((const uint32_t*)G.lut)[q];
    if (tid <= GK) eps_s[tid] = G.epsd[tid];
    if (tid < GK) s_rep[tid] = G.rep_k[tid];
    for (int q = tid; q < SM::NLEV * LW; q += LW) agg_s[q] = 0;
    for (int q = tid; q < SM::NLEV * LS; q += LW) sh_s[q] = 0;
    stk_s[tid] = (uint16_t)J;                                  // the sentinel below every stack
    __syncthreads();
    const int ob = s_ob;
    const int c = (int)(tile - a.tile_start[ob]);
    const int L = a.L;
    const int64_t n = a.v.n;
    const int64_t o0 = a.v.w + (int64_t)LW * ob;            // w = 1, or the Theiler window
    const int64_t s = (int64_t)c * L;                       // chunk start along the diagonals
    // the two windows: the floats of the points s-2.. and s-2+o0..; the n points span (n-1)*ps + span + 1 floats
    const float* y = a.v.data + (int64_t)b * a.v.bs;
    const int64_t ny = (n - 1) * ps + span + 1;
    stage_windows(y, ny, (s - 2) * ps, (s - 2 + o0) * ps, ya_s, LA, yb_s, LB);
    __syncthreads();

    const int64_t o = o0 + tid;
    const int64_t len = n - o;                              // cells on this thread's diagonal (may be <= 0)
    int cnt = (int)max((int64_t)0, min((int64_t)L, len - s));
    const int cnt_hi = __shfl_sync(FULL, cnt, 0);           // the warp's longest lane (smallest o)
    const int cnt_lo = __shfl_sync(FULL, cnt, 31);
    unsigned long long* grow = a.hist + (int64_t)b * a.K * n;

    if (cnt_hi > 0) {
        const int64_t out_row = (((int64_t)b * a.tiles + tile) * (2 * NP)) * LW + tid;
        const uint32_t yb_org = pin(smem_addr(yb_s) + 4 * tid * ps);
        auto setup = [&](auto& sc) {
            sc.ya_org = smem_addr(ya_s);
            sc.lut = pin(smem_addr(lut_s) - BUCKET_MAGIC_BITS);   // indexed with bucket_bits()
            sc.eps = smem_addr(eps_s);
            sc.agg = pin(smem_addr(agg_s) + 4 * tid);
            sc.sh = smem_addr(sh_s);
            sc.stk = pin(smem_addr(stk_s) + 2 * tid);
            sc.q0 = pin(smem_addr(smem + SM::off_q) + 2 * tid);
            sc.grow = (unsigned long long*)pin64((unsigned long long)grow);   // kept in registers, not re-read per cell
            sc.rep = G.rep_k;                               // global copy: only read for lines of length >= LS
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
            sc.A = 0; sc.ts = 0; sc.top = sc.stk;           // every threshold: recurrent since the chunk start
        };
        const int first_real = -(int)min((int64_t)2, s);     // warm-up cells before it lie outside the plot
        if (G.multi) {
            Scanner<NORM, M, TAU, NP, true> sc;
            setup(sc);
            scan_chunk(sc, cnt, cnt_lo, cnt_hi, first_real, yb_org, a.suf + out_row);
        } else {
            Scanner<NORM, M, TAU, NP, false> sc;
            setup(sc);
            scan_chunk(sc, cnt, cnt_lo, cnt_hi, first_real, yb_org, a.suf + out_row);
        }
    }
    __syncthreads();
    // flush: aggregates (sum the 256 private columns of every level) and the short lines (prefix sums of D over j)
    {
        const int warp = tid >> 5, lane = tid & 31;
        unsigned long long* ag = a.agg + ((int64_t)b * a.NG + a.g) * 3 * (GK + 1);
        for (int lev = warp; lev <= J; lev += LW / 32) {
            const uint32_t* r = agg_s + lev * LW;
            uint32_t s1 = 0, s2 = 0, s3 = 0;
            for (int q = lane; q < LW; q += 32) { uint32_t w = r[q]; s1 += w & 0x3ffu; s2 += (w >> 10) & 0x3ffu; s3 += w >> 20; }
            for (int off = 16; off; off >>= 1) {
                s1 += __shfl_down_sync(FULL, s1, off);
                s2 += __shfl_down_sync(FULL, s2, off);
                s3 += __shfl_down_sync(FULL, s3, off);
            }
            if (lane == 0) {
                if (s1) atomicAdd(&ag[lev], (unsigned long long)s1);
                if (s2) atomicAdd(&ag[(GK + 1) + lev], (unsigned long long)s2);
                if (s3) atomicAdd(&ag[2 * (GK + 1) + lev], (unsigned long long)s3);
            }
        }
        for (int l = tid; l < LS; l += LW) {
            int32_t acc = 0;
            for (int j = 0; j < J; ++j) {
                acc += sh_s[j * LS + l];
                if (acc) atomicAdd(&grow[(int64_t)s_rep[j] * n + l], (unsigned long long)acc);
            }
        }
    }
}

// ---------------------------------------------------------------------------------------- stitching
// One thread per (diagonal, distinct threshold): join the (prefix, suffix) summaries of consecutive chunks and
// emit the lines of length >= 4 that touch a chunk border (including the two ends of the diagonal).
struct StitchArgs {
    int64_t n, w;
    int g, NG, K, L, n_ob, NP;
    const LineGroup* groups;
    const uint32_t* tile_start;
    unsigned long long* hist;
    const uint16_t* pre;
    const uint16_t* suf;
    uint32_t tiles;
};

__global__ void __launch_bounds__(LW) line_stitch_kernel(StitchArgs a) {
    const int ob = blockIdx.x, j = blockIdx.y, b = blockIdx.z;
    const LineGroup& G = a.groups[(int64_t)b * a.NG + a.g];
    if (j >= G.J) return;
    const int tid = threadIdx.x;
    const int64_t o = a.w + (int64_t)LW * ob + tid;
    const int64_t len = a.n - o;
    if (len <= 0) return;
    unsigned long long* row = a.hist + ((int64_t)b * a.K + G.rep_k[j]) * a.n;
    const uint32_t t0 = a.tile_start[ob];
    const int nc = (int)((len + a.L - 1) / a.L);
    uint32_t carry = 0;
    // the summaries of SB chunks are loaded together (independent loads), then joined in order
    constexpr int SB = 8;
    const int64_t stride = (int64_t)(2 * a.NP) * LW;
    const int64_t base = (((int64_t)b * a.tiles + t0) * (2 * a.NP) + j) * LW + tid;
    for (int c0 = 0; c0 < nc; c0 += SB) {
        uint32_t p[SB], sf[SB];
#pragma unroll
        for (int u = 0; u < SB; ++u) {
            const bool in = c0 + u < nc;
            p[u] = in ? a.pre[base + (int64_t)(c0 + u) * stride] : 0u;
            sf[u] = in ? a.suf[base + (int64_t)(c0 + u) * stride] : 0u;
        }
#pragma unroll
        for (int u = 0; u < SB; ++u) {
            if (c0 + u < nc) {
                const uint32_t cntc = (uint32_t)min((int64_t)a.L, len - (int64_t)(c0 + u) * a.L);
                if (p[u] == cntc) {
                    carry += cntc;
                } else {
                    const uint32_t tot = carry + p[u];
                    if (tot >= (uint32_t)LMIN_EXPLICIT) atomicAdd(&row[tot], 1ull);
                    carry = sf[u];
                }
            }
        }
    }
    if (carry >= (uint32_t)LMIN_EXPLICIT) atomicAdd(&row[carry], 1ull);
}

// ------------------------------------------------------------------------------------------ finalize
// One block per (distinct threshold, series): P(1), P(2), P(3) from the aggregates and the explicit lines
//   C  = sum_l l P(l),  Q2 = sum_{l>=2} (l-1) P(l),  Q3 = sum_{l>=3} (l-2) P(l)      (all exact integers)
// then the rows of caller thresholds that share this value are copied from the representative row.
__global__ void __launch_bounds__(1024) line_finalize_kernel(int64_t n, int g, int NG, int K,
                                                            const LineGroup* __restrict__ groups,
                                                            const unsigned long long* __restrict__ agg,
                                                            unsigned long long* __restrict__ hist, WsStatus* status) {
    const int j = blockIdx.x, b = blockIdx.y;
    const LineGroup& G = groups[(int64_t)b * NG + g];
    if (j >= G.J) return;
    unsigned long long* row = hist + ((int64_t)b * K + G.rep_k[j]) * n;
    unsigned long long e0 = 0, c4 = 0;
#pragma unroll 4
    for (int64_t l = LMIN_EXPLICIT + threadIdx.x; l < n; l += blockDim.x) {
        unsigned long long h = row[l];
        e0 += (unsigned long long)l * h;
        c4 += h;
    }
    __shared__ unsigned long long s_e0[32], s_c4[32];
    for (int off = 16; off; off >>= 1) {
        e0 += __shfl_down_sync(FULL, e0, off);
        c4 += __shfl_down_sync(FULL, c4, off);
    }
    if ((threadIdx.x & 31) == 0) { s_e0[threadIdx.x >> 5] = e0; s_c4[threadIdx.x >> 5] = c4; }
    __syncthreads();
    if (threadIdx.x == 0) {
        e0 = 0; c4 = 0;
        for (int q = 0; q < (int)(blockDim.x >> 5); ++q) { e0 += s_e0[q]; c4 += s_c4[q]; }
        const unsigned long long* ag = agg + ((int64_t)b * NG + g) * 3 * (GK + 1);
        unsigned long long C = 0, Q2 = 0, Q3 = 0;
        for (int u = 0; u <= j; ++u) { C += ag[u]; Q2 += ag[(GK + 1) + u]; Q3 += ag[2 * (GK + 1) + u]; }
        const long long P3 = (long long)Q3 - (long long)(e0 - 2 * c4);
        const long long P2 = (long long)Q2 - (long long)(e0 - c4) - 2 * P3;
        const long long P1 = (long long)C - (long long)e0 - 3 * P3 - 2 * P2;
        if (P1 < 0 || P2 < 0 || P3 < 0) atomicExch(&status->internal, 1);
        if (n > 1) row[1] = (unsigned long long)P1;
        if (n > 2) row[2] = (unsigned long long)P2;
        if (n > 3) row[3] = (unsigned long long)P3;
    }
}

__global__ void __launch_bounds__(256) line_copy_rows_kernel(int64_t n, int g, int NG, int K,
                                                             const LineGroup* __restrict__ groups,
                                                             unsigned long long* __restrict__ hist) {
    const int q = blockIdx.y, b = blockIdx.z;
    const LineGroup& G = groups[(int64_t)b * NG + g];
    if (q >= G.kcount) return;
    const int k = G.k_of[q], rep = G.rep_k[G.j_of[q]];
    if (k == rep) return;
    const unsigned long long* src = hist + ((int64_t)b * K + rep) * n;
    unsigned long long* dst = hist + ((int64_t)b * K + k) * n;
    for (int64_t l = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; l < n; l += (int64_t)gridDim.x * blockDim.x) dst[l] = src[l];
}

// ------------------------------------------------------------ general strided views (materialised X)
// One thread per diagonal, K run counters, global atomics.  Only used when the points are not a delay view of a
// series (point_stride != 1) or the embedding window does not fit the scan kernel's shared-memory windows.
template <int NORM>
__global__ void __launch_bounds__(128) line_strided_kernel(View v, const float* __restrict__ eps, int K,
                                                           unsigned long long* __restrict__ hist) {
    const int b = blockIdx.y;
    const int64_t o = v.w + (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
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

// ------------------------------------------------------------------------------------------ host side
struct LinePlan {
    bool scan;          // false: strided fallback
    int L, n_ob, NG, NP, span;
    uint32_t tiles;
    size_t smem;
};

int pairs_for(int kg) { return kg <= 10 ? 5 : (kg <= 20 ? 10 : 16); }

template <int NP>
size_t scan_smem_bytes(int L, int span, int ps) {
    return (size_t)ScanSmem<NP>::off_ya + 4 * ((size_t)window_la(L, span, 2, ps) + window_lb(L, span, 2, ps));
}
size_t scan_smem_bytes(int NP, int L, int span, int ps) {
    return NP == 5 ? scan_smem_bytes<5>(L, span, ps) : (NP == 10 ? scan_smem_bytes<10>(L, span, ps) : scan_smem_bytes<16>(L, span, ps));
}
constexpr size_t SMEM_PER_BLOCK_MAX = 227 * 1024 - 256;     // opt-in limit of sm_100a, minus the static part

LinePlan make_plan(const View& v, int K) {
    LinePlan p{};
    p.span = (int)std::min<int64_t>((int64_t)(v.m - 1) * v.cs, (int64_t)MAX_SPAN + 1);
    p.NG = (K + GK - 1) / GK;
    p.NP = pairs_for(std::min(K, GK));
    const int ps = (int)std::min<int64_t>(v.ps, 1 << 20);
    // tiled scan: delay views, and materialised points (point stride > 1) whose windows fit the shared memory
    p.scan = p.span <= MAX_SPAN && scan_smem_bytes(p.NP, 32, p.span, ps) <= SMEM_PER_BLOCK_MAX;
    // chunk length: aim at >= 8 waves of 3 blocks per SM over the whole batch, at most 1023 positions
    const double cells = (double)n_pairs(v) * (double)v.batch;
    int64_t L = (int64_t)std::ceil(cells / ((double)LW * 148.0 * 3.0 * 8.0));
    p.L = (int)std::max<int64_t>(32, std::min<int64_t>(LMAX, L));
    if (options().line_chunk > 0) p.L = (int)std::min<int64_t>(LMAX, options().line_chunk);
    // wide points: the two windows hold (2L + 512) points, so the chunk shrinks until they fit (one block per SM then)
    while (p.scan && p.L > 32 && scan_smem_bytes(p.NP, p.L, p.span, ps) > SMEM_PER_BLOCK_MAX) p.L = std::max(32, p.L / 2);
    const int64_t nd = n_diag(v);                              // the triangle of the counted diagonals w..n-1
    p.n_ob = (int)((nd - 1 + LW - 1) / LW);
    uint64_t tiles = 0;
    for (int ob = 0; ob < p.n_ob; ++ob) tiles += (uint64_t)((nd - 1 - (int64_t)LW * ob + p.L - 1) / p.L);
    p.tiles = (uint32_t)tiles;
    p.smem = scan_smem_bytes(p.NP, p.L, p.span, ps);
    return p;
}

template <int NORM, int M, int TAU, int NP>
rqa_status launch_scan(const ScanArgs& a, const LinePlan& p, int batch, cudaStream_t s) {
    auto kern = line_scan_kernel<NORM, M, TAU, NP>;
    RQA_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p.smem));
    kern<<<dim3(p.tiles, (unsigned)batch), LW, p.smem, s>>>(a);
    RQA_LAUNCH_CHECK();
    return RQA_OK;
}

template <int NORM, int NP>
rqa_status dispatch_embedding(const ScanArgs& a, const LinePlan& p, int batch, cudaStream_t s) {
    // the embeddings of BASELINE.json's large configs get a register ring; any other (m, tau) recomputes per cell
    const bool delay = a.v.ps == 1;
    if (delay && a.m == 3 && a.tau == 1) return launch_scan<NORM, 3, 1, NP>(a, p, batch, s);
    if (delay && a.m == 3 && a.tau == 3) return launch_scan<NORM, 3, 3, NP>(a, p, batch, s);
    if (delay && a.m == 5 && a.tau == 2) return launch_scan<NORM, 5, 2, NP>(a, p, batch, s);
    return launch_scan<NORM, 0, 0, NP>(a, p, batch, s);
}

template <int NORM>
rqa_status dispatch_pairs(const ScanArgs& a, const LinePlan& p, int batch, cudaStream_t s) {
    if (p.NP == 5) return dispatch_embedding<NORM, 5>(a, p, batch, s);
    if (p.NP == 10) return dispatch_embedding<NORM, 10>(a, p, batch, s);
    return dispatch_embedding<NORM, 16>(a, p, batch, s);
}

}  // namespace

rqa_status launch_tile_table(int64_t n, int L, int n_ob, uint32_t* tile_start, cudaStream_t s) {
    tile_table_kernel<<<1, 1024, 0, s>>>(n, L, n_ob, tile_start);
    RQA_LAUNCH_CHECK();
    return RQA_OK;
}

size_t line_workspace_bytes(const View& v, int K) {
    LinePlan p = make_plan(v, K);
    if (!p.scan) return 256;
    size_t bytes = 0;
    bytes += align_up(sizeof(LineGroup) * (size_t)v.batch * p.NG);
    bytes += align_up(sizeof(uint32_t) * ((size_t)p.n_ob + 1));
    bytes += align_up(sizeof(uint64_t) * (size_t)v.batch * p.NG * 3 * (GK + 1));
    bytes += align_up(sizeof(uint16_t) * (size_t)v.batch * p.tiles * 2 * p.NP * LW);
    bytes += align_up(sizeof(uint16_t) * (size_t)v.batch * p.tiles * 2 * p.NP * LW);
    return bytes;
}

rqa_status run_line_hist(const View& v, int norm, const float* d_eps, int K, uint64_t* d_hist, Arena& ws, cudaStream_t s) {
    WsStatus* status = (WsStatus*)ws.base;
    RQA_CUDA_TRY(cudaMemsetAsync(d_hist, 0, sizeof(uint64_t) * (size_t)v.batch * K * v.n, s));
    LinePlan p = make_plan(v, K);
    if (!p.scan) {
        dim3 grid((unsigned)((v.n - v.w + 127) / 128), (unsigned)v.batch);
        if (norm == RQA_NORM_MAX)
            line_strided_kernel<RQA_NORM_MAX><<<grid, 128, 0, s>>>(v, d_eps, K, (unsigned long long*)d_hist);
        else
            line_strided_kernel<RQA_NORM_EUCLID><<<grid, 128, 0, s>>>(v, d_eps, K, (unsigned long long*)d_hist);
        RQA_LAUNCH_CHECK();
        return RQA_OK;
    }
    LineGroup* groups = ws.take<LineGroup>((size_t)v.batch * p.NG);
    uint32_t* tile_start = ws.take<uint32_t>((size_t)p.n_ob + 1);
    unsigned long long* agg = (unsigned long long*)ws.take<uint64_t>((size_t)v.batch * p.NG * 3 * (GK + 1));
    uint16_t* pre = ws.take<uint16_t>((size_t)v.batch * p.tiles * 2 * p.NP * LW);
    uint16_t* suf = ws.take<uint16_t>((size_t)v.batch * p.tiles * 2 * p.NP * LW);
    if (!ws.ok()) { set_error("rqa_line_hist: workspace too small"); return RQA_ERR_WORKSPACE_TOO_SMALL; }
    RQA_CUDA_TRY(cudaMemsetAsync(agg, 0, sizeof(uint64_t) * (size_t)v.batch * p.NG * 3 * (GK + 1), s));
    line_groups_kernel<<<v.batch, 128, 0, s>>>(d_eps, K, p.NG, groups, status);
    RQA_LAUNCH_CHECK();
    {
        rqa_status st = launch_tile_table(n_diag(v), p.L, p.n_ob, tile_start, s);
        if (st != RQA_OK) return st;
    }
    for (int g = 0; g < p.NG; ++g) {
        ScanArgs a;
        a.v = v; a.g = g; a.NG = p.NG; a.K = K; a.L = p.L; a.n_ob = p.n_ob;
        a.groups = groups; a.tile_start = tile_start; a.hist = (unsigned long long*)d_hist; a.agg = agg;
        a.pre = pre; a.suf = suf; a.tiles = p.tiles; a.m = v.m; a.tau = (int)v.cs;
        rqa_status st = norm == RQA_NORM_MAX ? dispatch_pairs<RQA_NORM_MAX>(a, p, v.batch, s)
                                             : dispatch_pairs<RQA_NORM_EUCLID>(a, p, v.batch, s);
        if (st != RQA_OK) return st;
        StitchArgs sa;
        sa.n = v.n; sa.w = v.w; sa.g = g; sa.NG = p.NG; sa.K = K; sa.L = p.L; sa.n_ob = p.n_ob; sa.NP = p.NP;
        sa.groups = groups; sa.tile_start = tile_start; sa.hist = (unsigned long long*)d_hist; sa.pre = pre; sa.suf = suf;
        sa.tiles = p.tiles;
        line_stitch_kernel<<<dim3((unsigned)p.n_ob, (unsigned)(2 * p.NP), (unsigned)v.batch), LW, 0, s>>>(sa);
        RQA_LAUNCH_CHECK();
        line_finalize_kernel<<<dim3((unsigned)(2 * p.NP), (unsigned)v.batch), 1024, 0, s>>>(v.n, g, p.NG, K, groups, agg,
                                                                                         (unsigned long long*)d_hist, status);
        RQA_LAUNCH_CHECK();
        unsigned cb = (unsigned)std::min<int64_t>((v.n + 255) / 256, 64);
        line_copy_rows_kernel<<<dim3(cb, GK, (unsigned)v.batch), 256, 0, s>>>(v.n, g, p.NG, K, groups, (unsigned long long*)d_hist);
        RQA_LAUNCH_CHECK();
    }
    return RQA_OK;
}

}  // namespace rqa
