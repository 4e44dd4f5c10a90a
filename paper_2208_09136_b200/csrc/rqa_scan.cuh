// rqa_scan.cuh — the run-length machinery shared by the two line scans of librqa.so: the diagonal scan of
// rqa_line_hist (rqa_line.cu) and the column scan of rqa_vert_hist (rqa_vert.cu, reading
// S19).  A thread walks a sequence of cells (a diagonal, or a column of the plot), maps every distance to its LEVEL
// among the sorted thresholds and keeps the runs of all nested thresholds as a monotone stack; what differs between the
// two scans is only where the cells come from (the distance provider CDT) and how the plot is cut into work items.
// Internal to librqa.so; nothing here is shared with the oracle.
#pragma once

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


// ------------------------------------------------------------------------------------------ the scan
// Cell distances: CellDist (rqa_tiles.cuh) with two warm-up cells before the chunk.
// Shared-memory plan of the scan kernel (bytes); NP: the group has J <= 2*NP distinct thresholds.
// The series windows come last because their length depends on the run-time span (m-1)*tau and on the chunk length;
// there are one or two sets of them (double buffer).
template <int NP>
struct ScanSmem {
    static constexpr int NLEV = 2 * NP + 1;                   // levels 0..2NP
    static constexpr int off_lut = 0;
    static constexpr int off_eps = off_lut + NB;
    static constexpr int off_tot = off_eps + 4 * (GK + 4);    // uint32 tot[3][GK+1]: the block's aggregate totals of an item
    static constexpr int off_agg = off_tot + ((4 * 3 * (GK + 1) + 15) / 16) * 16;
    static constexpr int agg_row = 4 * LW;                    // one level: a word per thread = three 10-bit counters
    static constexpr int off_sh = off_agg + NLEV * agg_row;   // int32 D[NLEV][LS]: difference array over the thresholds
    static constexpr int stk_row = 2 * LW;                    // one stack depth: a 16-bit entry per thread
    static constexpr int off_stk = off_sh + 4 * NLEV * LS;    // uint16 stack[NLEV][LW]
    static constexpr int off_q = off_stk + NLEV * stk_row;    // uint16 queue[QCELLS][LW]: deferred stack events
    static constexpr int off_ya = off_q + QCELLS * stk_row;   // window sets, 16-byte aligned
    static_assert(off_agg % 16 == 0 && off_ya % 16 == 0, "bulk copies need 16-byte aligned shared addresses");
};
constexpr uint32_t CARRY_SEG = 0x80000000u;   // carry flag: the run has been alive since the start of the segment


// Run state of one diagonal.  Thresholds are nested, so after a cell of level v exactly the thresholds j >= v are
// inside a run, and the start of that run does not increase with j: the runs of all thresholds form a monotone stack.
// Only runs that matter for explicit emission are kept: thresholds j >= A = max(level of the last 4 cells) have a run
// of >= 4 cells (shorter lines come from the aggregates).  Entry = (lo, start) covers the thresholds [lo, lo of the
// entry below); the top entry (lo = A) lives in registers, the others in a per-thread shared-memory column as
// uint16 (start << 6 | lo), bottom-most a sentinel with lo = J.  Cells before the chunk count as level 0, so the
// initial entry (0, start 0) stands for "recurrent since the chunk start" (prefix runs; start 0 marks them).
// Per cell the state changes only when A changes: a higher level pops the entries it ends (one line length for a
// whole range of thresholds -> D[lo][len]++, D[hi][len]--), a lower A pushes one entry.  Cost independent of K.
// The (3,1) ring with more than 10 thresholds (one window set, plain staging) reads the i-side window four elements per load.
template <int M, int TAU, int NP>
__host__ __device__ constexpr bool scan_vec() { return M == 3 && TAU == 1 && NP > 5; }

// CDT supplies the cell distances along the walk (CellDist: a diagonal of the plot; ColDist in rqa_vert.cu: a column).
template <class CDT, int NP, bool MULTI>
struct ScannerT : CDT {
    using CD = CDT;
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
    uint32_t* carry;            // this thread's column of the block's carry buffer (index j * LW)
    uint32_t* pre_out;          // this thread's column of the segment's prefix summaries
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

    // One run of `len` cells ended for the thresholds [lo4, hi4) / 4.  start == 0: it began at the chunk start, i.e. it
    // continues the run that was alive at the end of the previous chunk (carry, per threshold).  A run that has been
    // alive since the segment start is the segment's prefix run: written for the stitch kernel, not counted here.
    __device__ __forceinline__ void ended(uint32_t lo4, uint32_t hi4, uint32_t start, uint32_t len) {
        if (start != 0 && len < (uint32_t)LS) {
            const uint32_t col = sh + 4 * len;
            red_u32(col + lo4 * LS, 1u);
            red_u32(col + hi4 * LS, 0xffffffffu);
        } else if (start == 0) {
#pragma unroll 1
            for (uint32_t j4 = lo4; j4 < hi4; j4 += 4) {
                const uint32_t c = carry[(j4 >> 2) * LW];
                const uint32_t tot = (c & ~CARRY_SEG) + len;
                if (c & CARRY_SEG) {
                    pre_out[(j4 >> 2) * LW] = tot;
                } else if (tot >= (uint32_t)LMIN_EXPLICIT) {
                    if (tot < (uint32_t)LS) {
                        const uint32_t col = sh + 4 * tot + j4 * LS;
                        red_u32(col, 1u);
                        red_u32(col + 4 * LS, 0xffffffffu);
                    } else {
                        atomicAdd(&grow[(int64_t)rep[j4 >> 2] * n + tot], 1ull);
                    }
                }
            }
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

    // Phase 1 walks the cells in GROUPS of up to four: first the loads and the level of every cell of the group
    // (independent dependency chains that the hardware overlaps: no atomic or store sits between their shared-memory
    // loads, which ptxas would otherwise have to keep in program order), then the aggregates and the event queue.
    template <int R>
    __device__ __forceinline__ uint32_t level_of_cell() {
        CD::template push<R>();
        return level4(CD::template distance<R>());
    }
    template <int R>
    __device__ __forceinline__ void account(uint32_t v4) {
        const uint32_t w2 = max(v4, v1), w3 = max(w2, v2);
        red_u32(agg + v4 * (SM::agg_row / 4), 1u);
        red_u32(agg + w2 * (SM::agg_row / 4), 1u << 10);
        red_u32(agg + w3 * (SM::agg_row / 4), 1u << 20);
        const uint32_t a_new = max(w2, w2b);
        if (a_new != aprev) {
            sts_u16(qp, a_new + trel8 + ((uint32_t)R << 8));
            qp += SM::stk_row;
        }
        aprev = a_new;
        v2 = v1; v1 = v4;
        w2b = w2a; w2a = w2;
    }
    template <int R0, int... Q>
    __device__ __forceinline__ void group(std::integer_sequence<int, Q...>) {
        const uint32_t v[sizeof...(Q)] = {level_of_cell<R0 + Q>()...};
        (account<R0 + Q>(v[Q]), ...);
    }
    template <int R0, int U>
    __device__ __forceinline__ void groups() {
        if constexpr (R0 < U) {
            constexpr int G = U - R0 >= 4 ? 4 : U - R0;
            group<R0>(std::make_integer_sequence<int, G>{});
            groups<R0 + G, U>();
        }
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
        if constexpr (PHASE == 1) groups<0, (int)sizeof...(R)>();
        else (cell<R, PHASE>(t + R, cnt, ds), ...);
        CD::advance((int)sizeof...(R));
        if (PHASE == 1) trel8 += (uint32_t)sizeof...(R) << 8;
    }

    // End of the chunk (cnt > 0 cells): the run alive at the end for every threshold becomes the carry of the next
    // chunk (from the stack for j >= A/4, else 0..3 cells from the last levels); a run that spans the whole chunk
    // extends the carry it started from (and keeps its segment flag).
    __device__ __forceinline__ void finish(uint32_t cnt) {
        const uint32_t w3 = max(w2a, w2b);
#pragma unroll 1
        for (uint32_t j4 = 0; j4 < min(A, J4); j4 += 4)
            carry[(j4 >> 2) * LW] = (v1 <= j4) + (w2a <= j4) + (w3 <= j4);
        uint32_t lo = A, st = ts;
#pragma unroll 1
        while (lo < J4) {
            const uint32_t e = lds_u16(top);
            const uint32_t nlo = (e << 2) & 0xfcu;
#pragma unroll 1
            for (uint32_t j4 = lo; j4 < nlo; j4 += 4) {
                if (st == 0) carry[(j4 >> 2) * LW] += cnt;
                else carry[(j4 >> 2) * LW] = cnt - st;
            }
            lo = nlo; st = e >> 6;
            if (top != stk) top -= SM::stk_row;
        }
    }
};

template <int NORM, int M, int TAU, int NP, bool MULTI>
using Scanner = ScannerT<CellDist<NORM, M, TAU, 2, scan_vec<M, TAU, NP>()>, NP, MULTI>;

// The walk of one thread along its chunk.  Two instantiations (MULTI) so that the common case, every bucket of the
// level table holding at most one threshold, carries no refinement loop; a block executes only one of them.
template <class SC>
__device__ __forceinline__ void scan_chunk(SC& sc, int cnt, int cnt_lo, int cnt_hi, int ds, uint32_t yb_org) {
    constexpr int S = SC::S;
    constexpr int U = S == 3 ? 12 : (S > 3 ? S : 4);          // cells per super-step, a multiple of S
    static_assert(U + 2 <= WSLACK && U <= QCELLS, "window slack and queue capacity cover one super-step");
    using Seq = std::make_integer_sequence<int, U>;
    int t = -2;                                               // first cell is the warm-up cell t = -2
    sc.seek(sc.ya_org, yb_org, t);
    sc.prime();
    for (; t < 4; t += U) sc.template superstep<0>(t, cnt, ds, Seq{});   // warm-up cells and t < 4
    // Drain on demand: a window of super-steps lasts until some lane's queue could overflow in the next super-step
    // (more than QCELLS - U entries) or the cell index inside the window would leave its 8 bits.  The replay loop runs
    // as long as the longest queue of the warp, so long windows keep more lanes busy in it: with a drain every 24
    // cells 7 of 32 lanes held an event per iteration (profiles/r2_scan_drain.md), white noise now fills about half.
    constexpr int WMAX = 240 / U;                            // super-steps per window at most
    constexpr uint32_t QHIGH = (uint32_t)(QCELLS - U) * (uint32_t)SC::SM::stk_row;
    sc.aprev = sc.A;
    sc.qp = sc.q0;
    sc.trel8 = 0;
    while (t + U <= cnt_lo) {
        const int t0w = t;
        int w = 0;
#pragma unroll 1
        do {
            sc.template superstep<1>(t, cnt, ds, Seq{});
            t += U;
            ++w;
        } while (w < WMAX && t + U <= cnt_lo && !__any_sync(FULL, sc.qp - sc.q0 > QHIGH));
        sc.drain((uint32_t)t0w);
    }
    for (; t < cnt_hi; t += U) sc.template superstep<2>(t, cnt, ds, Seq{});
    if (cnt > 0) sc.finish((uint32_t)cnt);
}


// The chunk's aggregates: sum the LW thread-private columns of every level into the block's totals and clear them
// (the counters are 10 bits wide: a chunk has at most 1023 cells).  Call with the whole block, between two barriers.
__device__ __forceinline__ void reduce_chunk_aggregates(uint32_t* agg_s, uint32_t* tot_s, int J) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int lev = warp; lev <= J; lev += LW / 32) {
        uint32_t* r = agg_s + lev * LW;
        uint32_t s1 = 0, s2 = 0, s3 = 0;
        for (int q = lane; q < LW; q += 32) {
            const uint32_t w = r[q];
            r[q] = 0;
            s1 += w & 0x3ffu; s2 += (w >> 10) & 0x3ffu; s3 += w >> 20;
        }
        for (int off = 16; off; off >>= 1) {
            s1 += __shfl_down_sync(FULL, s1, off);
            s2 += __shfl_down_sync(FULL, s2, off);
            s3 += __shfl_down_sync(FULL, s3, off);
        }
        if (lane == 0) { tot_s[lev] += s1; tot_s[(GK + 1) + lev] += s2; tot_s[2 * (GK + 1) + lev] += s3; }
    }
}

// End of a work item: the block's aggregate totals and its short lines (prefix sums of D over the thresholds) go to
// global memory; everything read is cleared for the next item.  ag = the series' aggregate block [3][GK+1], grow = its
// histogram rows, rep = distinct threshold -> caller row (shared copy).
__device__ __forceinline__ void flush_item(uint32_t* tot_s, int32_t* sh_s, int J, unsigned long long* ag,
                                           unsigned long long* grow, const int* rep, int64_t n) {
    const int tid = threadIdx.x;
    if (tid < 3 * (GK + 1) && tot_s[tid]) { atomicAdd(&ag[tid], (unsigned long long)tot_s[tid]); tot_s[tid] = 0; }
    for (int l = tid; l < LS; l += LW) {
        int32_t acc = 0;
        for (int j = 0; j <= J; ++j) {
            const int32_t dj = sh_s[j * LS + l];
            if (dj) sh_s[j * LS + l] = 0;
            acc += dj;
            if (acc && j < J) atomicAdd(&grow[(int64_t)rep[j] * n + l], (unsigned long long)acc);
        }
    }
}

}  // namespace

// Launchers of the small kernels both scans use (defined in rqa_line.cu).
//   groups    one block per series: sort the K thresholds, split them into groups of 32, build each group's level table
//   finalize  P(1..3) of every distinct threshold from the aggregates and the explicit lines, then the rows of duplicate
//             thresholds are copied from their representative row
rqa_status launch_line_groups(const float* d_eps, int K, int NG, int gs, int batch, void* groups, WsStatus* status, cudaStream_t s);
rqa_status launch_line_finalize(int64_t n, int NG, int NP, int K, int batch, const void* groups, const unsigned long long* agg,
                                unsigned long long* hist, WsStatus* status, cudaStream_t s);
int scan_pairs_for(int kg);          // NP of the scan instantiation for kg thresholds per group: 5, 10 or 16

}  // namespace rqa
