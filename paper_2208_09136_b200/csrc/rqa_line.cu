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
//            to global atomics (longer).
//   blocks : PERSISTENT.  The grid is (blocks per SM) x (SMs); a block draws work items from an atomic counter.  An
//            item is a SEGMENT = up to S consecutive chunks of one diagonal block of one series.  Inside a segment the
//            runs that cross a chunk border are carried in place (a per-thread, per-threshold length in an L2-resident
//            buffer owned by the block), so only segment borders are written as (prefix, suffix) summaries and joined
//            along each diagonal by the stitch kernel.  The two series windows of the next chunk are fetched by bulk
//            asynchronous copies (cp.async.bulk + mbarrier) into the other half of a double buffer while the current
//            chunk is scanned.

#include "rqa_scan.cuh"

namespace rqa {

namespace {

// One block per series: sort the K thresholds, split them into groups of 32, build each group's table.
__global__ void __launch_bounds__(128) line_groups_kernel(const float* __restrict__ eps, int K, int NG, int gs,
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
        const int base = g * gs;                              // gs <= GK thresholds per group
        const int kc = min(gs, K - base);
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

// tile_start[q] = number of tiles in the local diagonal blocks before q (q = 0..n_obl); local block q is the diagonal
// block ob = part + q * parts (this process' share of a split call; parts = 1: ob = q), its longest diagonal has
// nd - 1 - LW*ob cells, cut into tiles of T cells (T = L for the counting pass, S*L = one segment for the scan).
__global__ void __launch_bounds__(1024) tile_table_kernel(int64_t nd, int64_t T, int n_obl, int part, int parts,
                                                          uint32_t* __restrict__ tile_start) {
    __shared__ uint32_t s_part[1024];
    const int per = (n_obl + 1023) / 1024;
    const int lo = min(n_obl, (int)threadIdx.x * per), hi = min(n_obl, lo + per);
    uint32_t sum = 0;
    for (int q = lo; q < hi; ++q) sum += (uint32_t)((nd - 1 - (int64_t)LW * (part + (int64_t)q * parts) + T - 1) / T);
    s_part[threadIdx.x] = sum;
    __syncthreads();
    for (int off = 1; off < 1024; off <<= 1) {
        uint32_t t = threadIdx.x >= off ? s_part[threadIdx.x - off] : 0;
        __syncthreads();
        s_part[threadIdx.x] += t;
        __syncthreads();
    }
    uint32_t run = s_part[threadIdx.x] - sum;
    for (int q = lo; q < hi; ++q) {
        tile_start[q] = run;
        run += (uint32_t)((nd - 1 - (int64_t)LW * (part + (int64_t)q * parts) + T - 1) / T);
    }
    if (threadIdx.x == 1023) tile_start[n_obl] = s_part[1023];
}

struct ScanArgs {
    View v;
    int g, NG, K, L, S;         // threshold group, groups, thresholds, chunk length, chunks per segment
    int part, parts, n_obl;     // this process' diagonal blocks: ob = part + q*parts, q < n_obl
    int nbuf;                   // window sets in shared memory (2: bulk-copy double buffer)
    const LineGroup* groups;
    const uint32_t* seg_start;  // [n_obl+1] segments in the local diagonal blocks before q
    unsigned long long* hist;   // [batch][K][n]
    unsigned long long* agg;    // [batch][NG][3][GK+1]
    uint32_t* pre;              // [batch][segs][2*NP][LW]  prefix run of every threshold (recurrent since the segment start)
    uint32_t* suf;              // [batch][segs][2*NP][LW]  run alive at the segment end
    uint32_t* carry;            // [gridDim.x][2*NP][LW]    run alive at the end of the previous chunk of the segment
    unsigned int* counter;      // work-item counter (zeroed before the launch)
    uint32_t segs;              // segments per series (this part)
    int m, tau;                 // run-time embedding (used by the M == 0 variant)
};

template <int NORM, int M, int TAU, int NP>
__global__ void __launch_bounds__(LW, (NP <= 10 ? 2 : 1)) line_scan_kernel(ScanArgs a) {
    using SM = ScanSmem<NP>;
    constexpr bool VECK = scan_vec<M, TAU, NP>();              // vector loads of the i-side window: one set, plain staging
    extern __shared__ __align__(16) char smem[];
    __shared__ int s_q;
    __shared__ unsigned int s_item;
    __shared__ int s_rep[GK];
    __shared__ __align__(8) unsigned long long s_bar[2];

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    uint8_t* lut_s = (uint8_t*)(smem + SM::off_lut);
    float* eps_s = (float*)(smem + SM::off_eps);
    uint32_t* tot_s = (uint32_t*)(smem + SM::off_tot);
    uint32_t* agg_s = (uint32_t*)(smem + SM::off_agg);
    int32_t* sh_s = (int32_t*)(smem + SM::off_sh);
    uint16_t* stk_s = (uint16_t*)(smem + SM::off_stk);
    const int span = M > 0 ? (M - 1) * TAU : (a.m - 1) * a.tau;
    const int ps = M > 0 ? 1 : (int)a.v.ps;
    const int L = a.L;
    // one window set: i-side window, j-side window, each with 4 floats of slack for the 16-byte alignment of bulk copies
    const int LA = window_la(L, span, 2, ps) + 4, LB = window_lb(L, span, 2, ps) + 4;
    float* win_s = (float*)(smem + SM::off_ya);
    const int64_t n = a.v.n;
    const int64_t T = (int64_t)a.S * L;                         // cells per segment along the diagonals
    const int64_t ny = (n - 1) * ps + span + 1;                 // floats of one series
    const int64_t extent = (int64_t)(a.v.batch - 1) * a.v.bs + ny;   // floats of the whole batch: what bulk copies may touch
    const uint32_t bar0 = (uint32_t)__cvta_generic_to_shared(&s_bar[0]);
    uint32_t* carry_col = a.carry + ((size_t)blockIdx.x * (2 * NP)) * LW + tid;
    const unsigned int n_items = a.segs * (unsigned)a.v.batch;

    if (tid == 0) {
        mbar_init(bar0, 1);
        mbar_init(bar0 + 8, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    stk_s[tid] = 0;                                            // (the sentinel is set per series)
    // the aggregate columns, the difference array and the totals are cleared here once; every flush clears what it read
    for (int q = tid; q < SM::NLEV * LW; q += LW) agg_s[q] = 0;
    for (int q = tid; q < SM::NLEV * LS; q += LW) sh_s[q] = 0;
    if (tid < 3 * (GK + 1)) tot_s[tid] = 0;
    uint32_t parity = 0;                                       // bit u: phase of mbarrier u
    int cur_b = -1, J = 0;
    __syncthreads();

    // Bulk copy of chunk c's two windows into window set `u` (thread 0).  Returns false when the copy would touch
    // memory outside the batch's floats (the ends of the first and last series): the caller stages with plain loads.
    auto bulk_ok = [&](const float* y, int64_t sa, int64_t sb, int& sha, int& shb) -> bool {
        const int64_t ga = (y - a.v.data) + sa, gb = (y - a.v.data) + sb;      // float offsets from the batch base
        sha = (int)(((uintptr_t)(a.v.data + ga) >> 2) & 3);
        shb = (int)(((uintptr_t)(a.v.data + gb) >> 2) & 3);
        return !VECK && a.nbuf == 2 && ga - sha >= 0 && gb - shb >= 0 && ga - sha + LA <= extent && gb - shb + LB <= extent &&
               (((uintptr_t)a.v.data) & 3) == 0;
    };

    while (true) {
        if (tid == 0) s_item = atomicAdd(a.counter, 1u);
        __syncthreads();
        const unsigned int item = s_item;
        if (item >= n_items) break;
        const int b = (int)(item / a.segs);
        const uint32_t t_seg = item - (uint32_t)b * a.segs;
        find_diagonal_block(a.seg_start, a.n_obl, t_seg, &s_q);
        const LineGroup& G = a.groups[(int64_t)b * a.NG + a.g];
        if (b != cur_b) {                                     // another series: its table and thresholds
            J = G.J;
            for (int q = tid; q < NB / 4; q += LW) ((uint32_t*)lut_s)[q] = ((const uint32_t*)G.lut)[q];
            if (tid <= GK) eps_s[tid] = G.epsd[tid];
            if (tid < GK) s_rep[tid] = G.rep_k[tid];
            stk_s[tid] = (uint16_t)J;                          // the sentinel below every stack
            cur_b = b;
        }
        __syncthreads();
        const int q_ob = s_q;
        const int ob = a.part + q_ob * a.parts;
        const int seg = (int)(t_seg - a.seg_start[q_ob]);
        const int64_t o0 = a.v.w + (int64_t)LW * ob;          // w = 1, or the Theiler window
        const int64_t o = o0 + tid;
        const int64_t len = n - o;                            // cells on this thread's diagonal (may be <= 0)
        const int64_t seg_s = (int64_t)seg * T;               // segment start along the diagonals
        const int64_t len0 = n - o0;                          // the block's longest diagonal
        const int c_end = (int)min((int64_t)a.S, (len0 - seg_s + L - 1) / L);   // chunks of this segment
        const float* y = a.v.data + (int64_t)b * a.v.bs;
        unsigned long long* grow = a.hist + (int64_t)b * a.K * n;
        const size_t out_row = (((size_t)b * a.segs + t_seg) * (2 * NP)) * LW + tid;
        // every run is alive "since the segment start" until it ends: the segment's prefix runs go to the stitch kernel
        for (int j = 0; j < J; ++j) carry_col[j * LW] = CARRY_SEG;

        // windows of the first chunk
        int sha = 0, shb = 0;
        bool bulk = bulk_ok(y, (seg_s - 2) * ps, (seg_s - 2 + o0) * ps, sha, shb);
        if (bulk && tid == 0) {
            fence_proxy_async();
            mbar_expect_tx(bar0, 4u * (uint32_t)(LA + LB));
            bulk_g2s((uint32_t)__cvta_generic_to_shared(win_s), y + (seg_s - 2) * ps - sha, 4u * LA, bar0);
            bulk_g2s((uint32_t)__cvta_generic_to_shared(win_s + LA), y + (seg_s - 2 + o0) * ps - shb, 4u * LB, bar0);
        }
        for (int c = 0; c < c_end; ++c) {
            const int u = a.nbuf == 2 ? (c & 1) : 0;
            float* ya_s = win_s + (size_t)u * (LA + LB);
            float* yb_s = ya_s + LA;
            const int64_t s = seg_s + (int64_t)c * L;          // chunk start along the diagonals
            if (bulk) {
                mbar_wait(bar0 + 8 * u, (parity >> u) & 1u);
                parity ^= 1u << u;
            } else {
                // VECK: the element pushed by the first cell of a super-step (window index 12k + 2) is 16-byte aligned
                sha = VECK ? 2 : 0;
                shb = 0;
                stage_windows(y, ny, (s - 2) * ps, (s - 2 + o0) * ps, ya_s + sha, LA - 4, yb_s, LB);
                __syncthreads();
            }
            const int sha_c = sha, shb_c = shb;
            // the next chunk's windows, into the other set, while this chunk is scanned
            bool bulk_next = false;
            if (c + 1 < c_end) {
                bulk_next = bulk_ok(y, (s + L - 2) * ps, (s + L - 2 + o0) * ps, sha, shb);
                if (bulk_next && tid == 0) {
                    float* na = win_s + (size_t)(u ^ 1) * (LA + LB);
                    fence_proxy_async();
                    mbar_expect_tx(bar0 + 8 * (u ^ 1), 4u * (uint32_t)(LA + LB));
                    bulk_g2s((uint32_t)__cvta_generic_to_shared(na), y + (s + L - 2) * ps - sha, 4u * LA, bar0 + 8 * (u ^ 1));
                    bulk_g2s((uint32_t)__cvta_generic_to_shared(na + LA), y + (s + L - 2 + o0) * ps - shb, 4u * LB, bar0 + 8 * (u ^ 1));
                }
            }
            int cnt = (int)max((int64_t)0, min((int64_t)L, len - s));
            const int cnt_hi = __shfl_sync(FULL, cnt, 0);       // the warp's longest lane (smallest o)
            const int cnt_lo = __shfl_sync(FULL, cnt, 31);
            if (cnt_hi > 0) {
                const uint32_t yb_org = pin(smem_addr(yb_s) + 4 * (shb_c + tid * ps));
                auto setup = [&](auto& sc) {
                    sc.ya_org = smem_addr(ya_s) + 4 * sha_c;
                    sc.lut = pin(smem_addr(lut_s) - BUCKET_MAGIC_BITS);   // indexed with bucket_bits()
                    sc.eps = smem_addr(eps_s);
                    sc.agg = pin(smem_addr(agg_s) + 4 * tid);
                    sc.sh = smem_addr(sh_s);
                    sc.stk = pin(smem_addr(stk_s) + 2 * tid);
                    sc.q0 = pin(smem_addr(smem + SM::off_q) + 2 * tid);
                    sc.grow = (unsigned long long*)pin64((unsigned long long)grow);   // kept in registers, not re-read per cell
                    sc.rep = G.rep_k;                           // global copy: only read for lines of length >= LS
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
                    sc.A = 0; sc.ts = 0; sc.top = sc.stk;       // every threshold: recurrent since the chunk start
                };
                const int first_real = -(int)min((int64_t)2, s);   // warm-up cells before it lie outside the plot
                if (G.multi) {
                    Scanner<NORM, M, TAU, NP, true> sc;
                    setup(sc);
                    scan_chunk(sc, cnt, cnt_lo, cnt_hi, first_real, yb_org);
                } else {
                    Scanner<NORM, M, TAU, NP, false> sc;
                    setup(sc);
                    scan_chunk(sc, cnt, cnt_lo, cnt_hi, first_real, yb_org);
                }
            }
            bulk = bulk_next;
            __syncthreads();
            reduce_chunk_aggregates(agg_s, tot_s, J);
            __syncthreads();
        }
        // end of the segment: the runs still alive (and the prefix runs that never ended) for the stitch kernel
        if (len > seg_s) {
            for (int j = 0; j < J; ++j) {
                const uint32_t cj = carry_col[j * LW];
                if (cj & CARRY_SEG) a.pre[out_row + (size_t)j * LW] = cj & ~CARRY_SEG;
                a.suf[out_row + (size_t)j * LW] = cj & ~CARRY_SEG;
            }
        }
        flush_item(tot_s, sh_s, J, a.agg + ((int64_t)b * a.NG + a.g) * 3 * (GK + 1), grow, s_rep, n);
        __syncthreads();                                       // before s_item / the tables are overwritten
    }
}

// ---------------------------------------------------------------------------------------- stitching
// One thread per (diagonal, distinct threshold): join the (prefix, suffix) summaries of consecutive segments and
// emit the lines of length >= 4 that touch a segment border (including the two ends of the diagonal).
struct StitchArgs {
    int64_t n, w, T;            // T = cells per segment along the diagonals
    int g, NG, K, NP;
    int part, parts, n_obl;
    const LineGroup* groups;
    const uint32_t* seg_start;
    unsigned long long* hist;
    const uint32_t* pre;
    const uint32_t* suf;
    uint32_t segs;
};

__global__ void __launch_bounds__(LW) line_stitch_kernel(StitchArgs a) {
    const int q_ob = blockIdx.x, j = blockIdx.y, b = blockIdx.z;
    const LineGroup& G = a.groups[(int64_t)b * a.NG + a.g];
    if (j >= G.J) return;
    const int tid = threadIdx.x;
    const int64_t o = a.w + (int64_t)LW * (a.part + (int64_t)q_ob * a.parts) + tid;
    const int64_t len = a.n - o;
    if (len <= 0) return;
    unsigned long long* row = a.hist + ((int64_t)b * a.K + G.rep_k[j]) * a.n;
    const uint32_t t0 = a.seg_start[q_ob];
    const int nc = (int)((len + a.T - 1) / a.T);
    uint32_t carry = 0;
    // the summaries of SB segments are loaded together (independent loads), then joined in order
    constexpr int SB = 8;
    const int64_t stride = (int64_t)(2 * a.NP) * LW;
    const int64_t base = (((int64_t)b * a.segs + t0) * (2 * a.NP) + j) * LW + tid;
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
                const uint32_t cntc = (uint32_t)min(a.T, len - (int64_t)(c0 + u) * a.T);
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
                                                           unsigned long long* __restrict__ hist, int part, int parts) {
    const int b = blockIdx.y;
    if ((int)(blockIdx.x % (unsigned)parts) != part) return;   // a split call: blocks of diagonals are dealt round robin
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
    int L, S, NG, NP, gs, span, nbuf, blocks_per_sm;
    Tiling tl;          // segments (T = S*L cells) of this part's diagonal blocks
    unsigned grid;      // persistent blocks
    size_t smem;
};


template <int NP>
size_t scan_smem_bytes(int L, int span, int ps, int nbuf) {
    return (size_t)ScanSmem<NP>::off_ya + 4 * (size_t)nbuf * ((size_t)window_la(L, span, 2, ps) + window_lb(L, span, 2, ps) + 8);
}
size_t scan_smem_bytes(int NP, int L, int span, int ps, int nbuf) {
    return NP == 5 ? scan_smem_bytes<5>(L, span, ps, nbuf)
                   : (NP == 10 ? scan_smem_bytes<10>(L, span, ps, nbuf) : scan_smem_bytes<16>(L, span, ps, nbuf));
}
constexpr size_t SMEM_PER_BLOCK_MAX = 227 * 1024 - 256;     // opt-in limit of sm_100a, minus the static part
constexpr size_t SMEM_PER_SM = 228 * 1024, SMEM_BLOCK_RESERVED = 1024;

LinePlan make_plan(const View& v, int K, const Options& opt) {
    LinePlan p{};
    p.span = (int)std::min<int64_t>((int64_t)(v.m - 1) * v.cs, (int64_t)MAX_SPAN + 1);
    p.gs = group_size_for(K, opt);
    p.NG = (K + p.gs - 1) / p.gs;
    p.NP = scan_pairs_for(std::min(K, p.gs));
    p.blocks_per_sm = p.NP <= 10 ? 2 : 1;                      // the kernel's __launch_bounds__
    const int ps = (int)std::min<int64_t>(v.ps, 1 << 20);
    // tiled scan: delay views, and materialised points (point stride > 1) whose windows fit the shared memory
    p.scan = p.span <= MAX_SPAN && scan_smem_bytes(p.NP, 32, p.span, ps, 1) <= SMEM_PER_BLOCK_MAX;
    const int64_t nd = n_diag(v);                              // the triangle of the counted diagonals w..n-1
    const int sms = sm_count();
    const unsigned slots = (unsigned)(sms * p.blocks_per_sm);
    // chunk length: at most 1023 positions (10-bit counters and stack positions); short enough that every block
    // slot gets several chunks of a small problem
    const double cells = (double)n_pairs(v) * (double)v.batch / (double)opt.parts;
    int64_t L = (int64_t)std::ceil(cells / ((double)LW * slots * 4.0));
    p.L = (int)std::max<int64_t>(32, std::min<int64_t>(LMAX, L));
    if (opt.line_chunk > 0) p.L = (int)std::min<int64_t>(LMAX, opt.line_chunk);
    // window sets: two (bulk-copy double buffer) when they fit beside the per-thread state at this occupancy
    const size_t per_block = SMEM_PER_SM / p.blocks_per_sm - SMEM_BLOCK_RESERVED;
    const size_t budget = std::min(per_block, SMEM_PER_BLOCK_MAX);
    // (measured at config 4, profiles/r2_scan_knobs.md: with K = 20 the per-thread state leaves room for ONE window set of
    // a 1023-cell chunk at two blocks per SM; a second set would cost either the chunk length (L = 256: 44 ms per call)
    // or the second block (49 ms) against 34.5 ms with one set — the other block of the SM hides the staging)
    p.nbuf = p.scan && scan_smem_bytes(p.NP, p.L, p.span, ps, 2) <= budget ? 2 : 1;
    if (opt.line_buffers > 0) p.nbuf = opt.line_buffers;
    if (v.ps == 1 && v.m == 3 && v.cs == 1 && p.NP > 5) p.nbuf = 1;   // the instantiations with vector loads (scan_vec)
    // wide points: the two windows hold (2L + 512) points, so the chunk shrinks until they fit (one block per SM then)
    while (p.scan && scan_smem_bytes(p.NP, p.L, p.span, ps, p.nbuf) > SMEM_PER_BLOCK_MAX) {
        if (p.nbuf == 2) p.nbuf = 1;
        else if (p.L > 32) p.L = std::max(32, p.L / 2);
        else break;
    }
    // segment = S consecutive chunks walked by one block with the run state carried in place: long enough that the
    // summaries at segment borders are rare, short enough that the slowest block's last item is a small share of its
    // work (about 1/8)
    const Tiling chunks = make_tiling(nd, p.L, opt.part, opt.parts);
    const uint64_t all = chunks.tiles * (uint64_t)v.batch;
    int64_t S = (int64_t)(all / ((uint64_t)slots * 8));
    p.S = (int)std::max<int64_t>(1, std::min<int64_t>(8, S));
    if (opt.line_segment > 0) p.S = opt.line_segment;
    p.tl = make_tiling(nd, (int64_t)p.S * p.L, opt.part, opt.parts);
    p.grid = (unsigned)std::max<uint64_t>(1, std::min<uint64_t>(p.tl.tiles * (uint64_t)v.batch, slots));
    p.smem = scan_smem_bytes(p.NP, p.L, p.span, ps, p.nbuf);
    return p;
}

template <int NORM, int M, int TAU, int NP>
rqa_status launch_scan(const ScanArgs& a, const LinePlan& p, cudaStream_t s) {
    auto kern = line_scan_kernel<NORM, M, TAU, NP>;
    static thread_local size_t attr_set[8] = {0};             // per device: the largest size this thread has opted in to
    int dev = 0;
    RQA_CUDA_TRY(cudaGetDevice(&dev));
    if (dev >= 8 || attr_set[dev] < p.smem) {
        RQA_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_PER_BLOCK_MAX));
        if (dev < 8) attr_set[dev] = SMEM_PER_BLOCK_MAX;
    }
    kern<<<p.grid, LW, p.smem, s>>>(a);
    RQA_LAUNCH_CHECK();
    return RQA_OK;
}

template <int NORM, int NP>
rqa_status dispatch_embedding(const ScanArgs& a, const LinePlan& p, cudaStream_t s) {
    // the embeddings of BASELINE.json's large configs get a register ring; any other (m, tau) recomputes per cell
    const bool delay = a.v.ps == 1;
    if (delay && a.m == 1) return launch_scan<NORM, 1, 1, NP>(a, p, s);
    if (delay && a.m == 3 && a.tau == 1) return launch_scan<NORM, 3, 1, NP>(a, p, s);
    if (delay && a.m == 3 && a.tau == 3) return launch_scan<NORM, 3, 3, NP>(a, p, s);
    if (delay && a.m == 5 && a.tau == 2) return launch_scan<NORM, 5, 2, NP>(a, p, s);
    return launch_scan<NORM, 0, 0, NP>(a, p, s);
}

template <int NORM>
rqa_status dispatch_pairs(const ScanArgs& a, const LinePlan& p, cudaStream_t s) {
    if (p.NP == 5) return dispatch_embedding<NORM, 5>(a, p, s);
    if (p.NP == 10) return dispatch_embedding<NORM, 10>(a, p, s);
    return dispatch_embedding<NORM, 16>(a, p, s);
}

struct LineWs {
    LineGroup* groups;
    uint32_t* seg_start;
    unsigned long long* agg;
    unsigned int* counters;
    uint32_t *pre, *suf, *carry;
};
LineWs carve_line(Arena& ws, const View& v, const LinePlan& p) {
    LineWs w{};
    w.groups = ws.take<LineGroup>((size_t)v.batch * p.NG);
    w.seg_start = ws.take<uint32_t>((size_t)p.tl.n_obl + 1);
    w.agg = (unsigned long long*)ws.take<uint64_t>((size_t)v.batch * p.NG * 3 * (GK + 1));
    w.counters = ws.take<unsigned int>((size_t)p.NG);
    w.pre = ws.take<uint32_t>((size_t)v.batch * p.tl.tiles * 2 * p.NP * LW);
    w.suf = ws.take<uint32_t>((size_t)v.batch * p.tl.tiles * 2 * p.NP * LW);
    w.carry = ws.take<uint32_t>((size_t)p.grid * 2 * p.NP * LW);
    return w;
}

// a NaN, infinite or negative threshold is reported through the workspace status (the strided fallback's check; the
// tiled scan does it in line_groups_kernel)
__global__ void line_eps_check_kernel(const float* __restrict__ eps, int64_t count, WsStatus* status) {
    bool bad = false;
    for (int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; q < count; q += (int64_t)gridDim.x * blockDim.x) {
        const float x = eps[q];
        bad |= !(x >= 0.0f) || isinf(x);
    }
    if (bad) atomicExch(&status->bad_eps, 1);
}

}  // namespace

int scan_pairs_for(int kg) { return kg <= 10 ? 5 : (kg <= 20 ? 10 : 16); }

rqa_status launch_line_groups(const float* d_eps, int K, int NG, int gs, int batch, void* groups, WsStatus* status, cudaStream_t s) {
    line_groups_kernel<<<batch, 128, 0, s>>>(d_eps, K, NG, gs, (LineGroup*)groups, status);
    RQA_LAUNCH_CHECK();
    return RQA_OK;
}

rqa_status launch_line_finalize(int64_t n, int NG, int NP, int K, int batch, const void* groups, const unsigned long long* agg,
                                unsigned long long* hist, WsStatus* status, cudaStream_t s) {
    for (int g = 0; g < NG; ++g) {
        // one block per (distinct threshold, series) sums its histogram row: about 8 bins per thread
        const unsigned threads = (unsigned)std::max<int64_t>(64, std::min<int64_t>(1024, ((n / 8 + 31) / 32) * 32));
        line_finalize_kernel<<<dim3((unsigned)(2 * NP), (unsigned)batch), threads, 0, s>>>(n, g, NG, K, (const LineGroup*)groups, agg,
                                                                                          hist, status);
        RQA_LAUNCH_CHECK();
        unsigned cb = (unsigned)std::min<int64_t>((n + 255) / 256, 64);
        line_copy_rows_kernel<<<dim3(cb, GK, (unsigned)batch), 256, 0, s>>>(n, g, NG, K, (const LineGroup*)groups, hist);
        RQA_LAUNCH_CHECK();
    }
    return RQA_OK;
}

rqa_status launch_tile_table(const Tiling& t, uint32_t* tile_start, cudaStream_t s) {
    tile_table_kernel<<<1, 1024, 0, s>>>(t.nd, t.T, t.n_obl, t.part, t.parts, tile_start);
    RQA_LAUNCH_CHECK();
    return RQA_OK;
}

// The two one-block-per-series paths need no workspace beyond the status block.
static bool line_small_path(const View& v, int K, const Options& opt) {
    return opt.line_path == 0 && opt.line_chunk == 0 && opt.line_segment == 0 && opt.line_buffers == 0 && opt.parts == 1 &&
           small_line_fits(v, K);
}
static bool line_block_path(const View& v, int K, const Options& opt) {
    // (the tiled scan costs about batch x groups of 32 thresholds, the blocks one round per 2 x SMs series)
    const bool knobs = opt.line_chunk != 0 || opt.line_segment != 0 || opt.line_buffers != 0;
    return opt.parts == 1 && block_line_fits(v, K) &&
           (opt.line_path == 2 || (opt.line_path == 0 && !knobs && (int64_t)v.batch * ((K + GK - 1) / GK) >= 192));
}

size_t line_workspace_bytes(const View& v, int K, const Options& opt) {
    if (line_small_path(v, K, opt) || line_block_path(v, K, opt)) return 256;
    LinePlan p = make_plan(v, K, opt);
    if (!p.scan) return 256;
    Arena a(nullptr, ~(size_t)0);
    carve_line(a, v, p);
    return a.off;
}

rqa_status run_line_hist(const View& v, int norm, const float* d_eps, int K, uint64_t* d_hist, Arena& ws, cudaStream_t s,
                         const Options& opt) {
    WsStatus* status = (WsStatus*)ws.base;
    const size_t hist_words = (size_t)v.batch * K * v.n;
    // short series: one block per series, shared-memory distances and histogram (explicit scan knobs and split calls
    // keep the general machinery)
    if (line_small_path(v, K, opt)) return run_line_small(v, norm, d_eps, K, d_hist, status, s);
    // many series of moderate length: one block per series walks every diagonal once for all K thresholds (rqa_block.cu)
    if (line_block_path(v, K, opt)) return run_line_block(v, norm, d_eps, K, d_hist, status, s);
    RQA_CUDA_TRY(cudaMemsetAsync(d_hist, 0, sizeof(uint64_t) * hist_words, s));
    LinePlan p = make_plan(v, K, opt);
    if (!p.scan) {
        // thread-per-diagonal fallback: the diagonals are dealt to the parts block by block
        line_eps_check_kernel<<<1, 256, 0, s>>>(d_eps, (int64_t)v.batch * K, status);
        RQA_LAUNCH_CHECK();
        dim3 grid((unsigned)((v.n - v.w + 127) / 128), (unsigned)v.batch);
        if (norm == RQA_NORM_MAX)
            line_strided_kernel<RQA_NORM_MAX><<<grid, 128, 0, s>>>(v, d_eps, K, (unsigned long long*)d_hist, opt.part, opt.parts);
        else
            line_strided_kernel<RQA_NORM_EUCLID><<<grid, 128, 0, s>>>(v, d_eps, K, (unsigned long long*)d_hist, opt.part, opt.parts);
        RQA_LAUNCH_CHECK();
        return reduce_parts(opt, d_hist, hist_words, s);
    }
    LineWs w = carve_line(ws, v, p);
    if (!ws.ok()) { set_error("rqa_line_hist: workspace too small"); return RQA_ERR_WORKSPACE_TOO_SMALL; }
    const size_t agg_words = (size_t)v.batch * p.NG * 3 * (GK + 1);
    RQA_CUDA_TRY(cudaMemsetAsync(w.agg, 0, sizeof(uint64_t) * agg_words, s));
    RQA_CUDA_TRY(cudaMemsetAsync(w.counters, 0, sizeof(unsigned int) * (size_t)p.NG, s));
    {
        rqa_status st = launch_line_groups(d_eps, K, p.NG, p.gs, v.batch, w.groups, status, s);
        if (st != RQA_OK) return st;
    }
    if (p.tl.tiles > 0) {
        rqa_status st = launch_tile_table(p.tl, w.seg_start, s);
        if (st != RQA_OK) return st;
    }
    for (int g = 0; g < p.NG && p.tl.tiles > 0; ++g) {
        ScanArgs a;
        a.v = v; a.g = g; a.NG = p.NG; a.K = K; a.L = p.L; a.S = p.S;
        a.part = opt.part; a.parts = opt.parts; a.n_obl = p.tl.n_obl; a.nbuf = p.nbuf;
        a.groups = w.groups; a.seg_start = w.seg_start; a.hist = (unsigned long long*)d_hist; a.agg = w.agg;
        a.pre = w.pre; a.suf = w.suf; a.carry = w.carry; a.counter = w.counters + g; a.segs = (uint32_t)p.tl.tiles;
        a.m = v.m; a.tau = (int)v.cs;
        if (g == 0 && opt.ev_begin) RQA_CUDA_TRY(cudaEventRecord((cudaEvent_t)opt.ev_begin, s));
        rqa_status st = norm == RQA_NORM_MAX ? dispatch_pairs<RQA_NORM_MAX>(a, p, s) : dispatch_pairs<RQA_NORM_EUCLID>(a, p, s);
        if (st != RQA_OK) return st;
        if (g == 0 && opt.ev_end) RQA_CUDA_TRY(cudaEventRecord((cudaEvent_t)opt.ev_end, s));
        StitchArgs sa;
        sa.n = v.n; sa.w = v.w; sa.T = p.tl.T; sa.g = g; sa.NG = p.NG; sa.K = K; sa.NP = p.NP;
        sa.part = opt.part; sa.parts = opt.parts; sa.n_obl = p.tl.n_obl;
        sa.groups = w.groups; sa.seg_start = w.seg_start; sa.hist = (unsigned long long*)d_hist; sa.pre = w.pre; sa.suf = w.suf;
        sa.segs = (uint32_t)p.tl.tiles;
        line_stitch_kernel<<<dim3((unsigned)p.tl.n_obl, (unsigned)(2 * p.NP), (unsigned)v.batch), LW, 0, s>>>(sa);
        RQA_LAUNCH_CHECK();
    }
    // a split call: the explicit lines and the aggregates of all parts, summed, before P(1..3) are solved from them
    {
        rqa_status st = reduce_parts(opt, d_hist, hist_words, s);
        if (st != RQA_OK) return st;
        st = reduce_parts(opt, w.agg, agg_words, s);
        if (st != RQA_OK) return st;
    }
    {
        rqa_status st = launch_line_finalize(v.n, p.NG, p.NP, K, v.batch, w.groups, w.agg, (unsigned long long*)d_hist, status, s);
        if (st != RQA_OK) return st;
    }
    return RQA_OK;
}

}  // namespace rqa
