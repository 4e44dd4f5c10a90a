// rqa_select.cu — rqa_eps_for_rr: exact multi-target order statistics of the P = N'(N'-1)/2 pairwise
// distances ("preselect RR and use the corresponding eps"; readings S4-S6).
//
// The N'^2 distance matrix is never stored: distances are recomputed tile by tile.  Non-negative
// fp32 values order like their uint32 bit patterns, so every select below works on patterns.
//
// Three paths, all exact:
//   DIRECT   (P <= 2^22)  all P distances are written to a scratch buffer once and a 4-pass multi-target radix
//            select runs over the buffer.
//   BRACKET  (delay views, the headline path)  ONE full pass over the triangle:
//              1. a pseudo-random sample of S ~ 5.5 P^(2/3) pair distances is drawn and 2 sample order statistics
//                 per target (rank S*q -/+ 4.5 sigma) are found by the buffer select: a bracket (lo_k, hi_k] that
//                 holds the true eps_k with overwhelming probability;
//              2. the counting pass visits every cell once (tiles, sliding-window distance, level table as in the
//                 diagonal scan), counts the cells of every inter-boundary level exactly (thread-private
//                 shared-memory counters, no conflicts) and appends the few cells inside brackets to a candidate
//                 list.  Values with massive ties (a collapsed bracket, a bracket end the sample holds thousands of
//                 times) get a single-value level of their own: counted, never appended;
//              3. the exact counts locate each target's rank — this is a proof, not a guess: a single-value level
//                 gives eps_k and C_k at once, a bracket gives the rank among the candidates and the buffer select
//                 over them gives eps_k and C_k; if a rank falls outside every bracket (or the candidate list
//                 overflows) the series is flagged and handled by RADIX.
//   RADIX    (general strided views; fallback)  most-significant-digit radix select, 4 full passes of 8 bits, all K
//            targets resolved in each pass; targets that share a prefix share one 256-bin histogram.
#include <algorithm>
#include <cmath>
#include <type_traits>

#include "rqa_tiles.cuh"

namespace rqa {

namespace {

constexpr int BT = 64;                // targets per buffer-select call
constexpr int NCUT = 4 * GK + 4;       // boundary slots: 2 per bracket, 2 more when both ends carry massive ties
constexpr int NLEV_MAX = 4 * GK + 1;  // levels of the counting pass
constexpr int TIE_MASS = 2048;        // a bracket end seen this often in the sample gets a level of its own
constexpr int WCAP = 256;             // candidates a warp buffers in shared memory before flushing
constexpr int NBS = NB;               // buckets of the counting pass' level table (8 bytes each)
constexpr double BRACKET_SIGMAS = 4.5;
enum : uint8_t { LEVEL_OUT = 0, LEVEL_CAND = 1, LEVEL_POINT = 2 };

// ------------------------------------------------------------------------------------------ per-series state
struct SelState {
    int32_t fallback;                 // 1: the series is (re)done by the radix passes
    int32_t pad;
    unsigned long long ncand_local;   // candidates in THIS part's list (= ncand for an unsplit call)
    // the next SEL_REDUCE_WORDS words are summed over the parts of a split call after the counting pass
    unsigned long long ncand;         // candidates appended by the counting pass (may exceed the capacity)
    unsigned long long over;          // parts whose candidate list overflowed
    unsigned long long level_count[NLEV_MAX + 1];
    int32_t is_point[GK];             // target t of the group fell into a LEVEL_POINT level:
    float point_val[GK];              //   eps = that value,
    unsigned long long point_cnt[GK]; //   C = #{d <= eps}
};

constexpr size_t SEL_REDUCE_WORDS = 2 + NLEV_MAX + 1;

// state of one buffer select (<= BT targets) of one series
struct BufSel {
    int32_t G;                        // live groups (distinct prefixes)
    int32_t T;
    uint32_t gprefix[BT];             // distinct prefixes, ascending (determined high bits, low bits zero)
    int32_t group_of[BT];
    uint32_t prefix[BT];
    unsigned long long resid[BT];     // 1-based residual rank inside the prefix range
    unsigned long long below[BT];     // elements strictly below the prefix range
    unsigned long long base[BT];      // added to (below + ties) for the final count
    float out_val[BT];
    unsigned long long out_cnt[BT];   // #{x <= out_val} within the buffer
};

struct Ranks64 {
    unsigned long long r[BT];
};

// bracket boundaries of one group of <= GK targets of one series (the counting pass's level table)
struct SelTable {
    int32_t J;                        // boundaries in use, levels 0..J
    int32_t multi;                    // 1 if some bucket holds two or more boundaries (refine by a loop)
    int32_t heavy;                    // 1 if J > 2 * targets: counted by the second, wider launch of the counting pass
    int32_t pad;
    float scale, dcap;
    float beta[NCUT];           // ascending, beta[J..] = +inf
    uint8_t kind[NCUT];         // LEVEL_* of level q = (beta[q-1], beta[q]]
    uint2 lut[NBS];                   // bucket -> (bits of the first boundary not in a lower bucket, its index)
};

struct SampleRanks {                  // per target of the group: sample ranks of the bracket ends (0 = open end)
    unsigned long long lo[GK], hi[GK];
    unsigned long long rank[GK];      // the target's rank among all P distances
    int32_t kc;
};

// ------------------------------------------------------------------------------------------ small kernels
__global__ void sel_init_kernel(SelState* ss, int force_fallback) {
    SelState& s = ss[blockIdx.x];
    if (threadIdx.x == 0) { s.fallback = force_fallback; s.pad = 0; s.ncand = 0; s.over = 0; s.ncand_local = 0; }
    for (int q = threadIdx.x; q <= NLEV_MAX; q += blockDim.x) s.level_count[q] = 0;
}

__global__ void sel_group_reset_kernel(SelState* ss) {
    SelState& s = ss[blockIdx.x];
    if (threadIdx.x == 0) { s.ncand = 0; s.over = 0; s.ncand_local = 0; }
    for (int q = threadIdx.x; q <= NLEV_MAX; q += blockDim.x) s.level_count[q] = 0;
}

__device__ __forceinline__ uint64_t mix64(uint64_t z) {
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}

// S pseudo-random pairs i < j (uniform over the P pairs, with replacement) -> their distances.
template <int NORM>
__global__ void __launch_bounds__(256) sel_sample_kernel(View v, unsigned long long S, float* __restrict__ out) {
    const int b = blockIdx.y;
    const float* yb = v.data + (int64_t)b * v.bs;
    float* o = out + (int64_t)b * S;
    const uint32_t n = (uint32_t)v.n;
    for (unsigned long long s = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; s < S;
         s += (unsigned long long)gridDim.x * blockDim.x) {
        uint64_t h = mix64((s + 1) * 0x9E3779B97F4A7C15ull + (uint64_t)b * 0xD1B54A32D192ED03ull);
        uint32_t lo, hi;
        if (v.w <= 1) {
            uint32_t i = __umulhi((uint32_t)(h >> 32), n);
            uint32_t j = __umulhi((uint32_t)h, n - 1);
            if (j >= i) ++j;
            lo = min(i, j); hi = max(i, j);
        } else {
            // Theiler window: pair number r, uniform in [0, P_w), in the row-major order of sel_direct_kernel: row i
            // holds the D - i pairs (i, i+w..n-1), D = n - w rows, C(i) = i*D - i(i-1)/2 pairs before it
            const uint64_t D = (uint64_t)(v.n - v.w), Pw = D * (D + 1) / 2;
            const uint64_t r = __umul64hi(h, Pw);
            const double t = 2.0 * (double)D + 1.0;
            int64_t i = (int64_t)((t - sqrt(t * t - 8.0 * (double)r)) * 0.5);
            i = max((int64_t)0, min((int64_t)D - 1, i));
            while (i > 0 && (uint64_t)i * D - (uint64_t)i * (uint64_t)(i - 1) / 2 > r) --i;
            while ((uint64_t)(i + 1) * D - (uint64_t)(i + 1) * (uint64_t)i / 2 <= r) ++i;
            lo = (uint32_t)i;
            hi = (uint32_t)(i + v.w + (int64_t)(r - ((uint64_t)i * D - (uint64_t)i * (uint64_t)(i - 1) / 2)));
        }
        o[s] = point_distance<NORM>(yb, lo, hi, v.m, v.ps, v.cs);
    }
}

// All P distances, diagonal by diagonal (any strided view).
template <int NORM>
__global__ void __launch_bounds__(256) sel_direct_kernel(View v, unsigned long long P, float* __restrict__ out) {
    const int b = blockIdx.y;
    const float* yb = v.data + (int64_t)b * v.bs;
    float* o = out + (int64_t)b * P;
    const int64_t n = v.n, D = v.n - v.w;
    for (int64_t row = blockIdx.x; row < D; row += gridDim.x) {
        // row i: the D - i pairs (i, i+w..n-1) stored from offset i*D - i(i-1)/2
        const int64_t off = row * D - row * (row - 1) / 2 - (row + v.w);
        for (int64_t j = row + v.w + threadIdx.x; j < n; j += blockDim.x)
            o[off + j] = point_distance<NORM>(yb, row, j, v.m, v.ps, v.cs);
    }
}

// ---------------------------------------------------------------------------------------- buffer select
__device__ void bufsel_reset(BufSel& s, int T) {
    s.G = 1;
    s.T = T;
    s.gprefix[0] = 0;
}

__global__ void bufsel_init_kernel(BufSel* st, Ranks64 ranks, int T) {
    BufSel& s = st[blockIdx.x];
    const int t = threadIdx.x;
    if (t == 0) bufsel_reset(s, T);
    if (t < T) {
        s.group_of[t] = 0;
        s.prefix[t] = 0;
        s.resid[t] = ranks.r[t];
        s.below[t] = 0;
        s.base[t] = 0;
    }
}

// One 8-bit pass over the buffer of series b: n = n_ptr ? min(*n_ptr of the series, cap) : cap.
__global__ void __launch_bounds__(256) bufsel_pass_kernel(const float* __restrict__ buf, unsigned long long stride,
                                                         unsigned long long cap, const SelState* __restrict__ ss,
                                                         int use_ncand, int pass, const BufSel* __restrict__ st,
                                                         unsigned long long* __restrict__ bins) {
    extern __shared__ uint32_t sbins[];      // [G][256]
    __shared__ uint32_t s_gprefix[BT];
    const int b = blockIdx.y;
    if (use_ncand && ss[b].fallback) return;
    const BufSel& s = st[b];
    const int G = s.G;
    unsigned long long n = cap;
    if (use_ncand) n = min(cap, ss[b].ncand_local);
    for (int q = threadIdx.x; q < G * 256; q += blockDim.x) sbins[q] = 0;
    for (int q = threadIdx.x; q < G; q += blockDim.x) s_gprefix[q] = s.gprefix[q];
    __syncthreads();
    const uint32_t* x = (const uint32_t*)buf + (unsigned long long)b * stride;
    const int shift = 24 - 8 * pass;
    const uint32_t himask = pass == 0 ? 0u : (0xFFFFFFFFu << (32 - 8 * pass));
    auto count_key = [&](uint32_t key) {
        const uint32_t hi = key & himask;
        int lo = 0, hiq = G;                 // first group with gprefix >= hi
        while (lo < hiq) {
            int mid = (lo + hiq) >> 1;
            if (s_gprefix[mid] < hi) lo = mid + 1; else hiq = mid;
        }
        if (lo < G && s_gprefix[lo] == hi) atomicAdd(&sbins[lo * 256 + ((key >> shift) & 255u)], 1u);
    };
    // four keys per load where the series' buffer is 16-byte aligned (more bytes in flight per thread), then the tail
    const unsigned long long tid = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
    const unsigned long long nthreads = (unsigned long long)gridDim.x * blockDim.x;
    const unsigned long long nvec = (((uintptr_t)x & 15) == 0) ? n / 4 : 0;
    for (unsigned long long e = tid; e < nvec; e += nthreads) {
        const uint4 k4 = ((const uint4*)x)[e];
        count_key(k4.x); count_key(k4.y); count_key(k4.z); count_key(k4.w);
    }
    for (unsigned long long e = 4 * nvec + tid; e < n; e += nthreads) count_key(x[e]);
    __syncthreads();
    unsigned long long* gb = bins + (int64_t)b * BT * 256;
    for (int q = threadIdx.x; q < G * 256; q += blockDim.x) {
        uint32_t c = sbins[q];
        if (c) atomicAdd(&gb[q], (unsigned long long)c);
    }
}

// One block per series: every target picks its digit; then the groups are rebuilt and the bins cleared.
__global__ void __launch_bounds__(256) bufsel_resolve_kernel(BufSel* st, unsigned long long* bins, int pass,
                                                            const SelState* __restrict__ ss, int use_ncand) {
    const int b = blockIdx.x;
    if (use_ncand && ss[b].fallback) return;
    BufSel& s = st[b];
    const int T = s.T;
    unsigned long long* gb = bins + (int64_t)b * BT * 256;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nwarps = blockDim.x >> 5;
    const int shift = 24 - 8 * pass;
    __shared__ uint32_t s_prefix[BT];
    __shared__ int s_first[BT];
    for (int t = warp; t < T; t += nwarps) {
        const unsigned long long* h = gb + s.group_of[t] * 256;
        unsigned long long c[8], sum = 0;
        for (int q = 0; q < 8; ++q) { c[q] = h[lane * 8 + q]; sum += c[q]; }
        unsigned long long incl = sum;
        for (int off = 1; off < 32; off <<= 1) {
            unsigned long long u = __shfl_up_sync(FULL, incl, off);
            if (lane >= off) incl += u;
        }
        const unsigned long long resid = s.resid[t];
        unsigned ball = __ballot_sync(FULL, incl >= resid);
        int src = ball ? (__ffs(ball) - 1) : 31;      // ball == 0 only if the rank exceeds the buffer (flagged elsewhere)
        int digit = 255;
        unsigned long long e = incl - sum, ties = 0;
        if (lane == src) {
            for (int q = 0; q < 8; ++q) {
                if (e + c[q] >= resid) { digit = lane * 8 + q; ties = c[q]; break; }
                e += c[q];
            }
        }
        digit = __shfl_sync(FULL, digit, src);
        e = __shfl_sync(FULL, e, src);
        ties = __shfl_sync(FULL, ties, src);
        if (lane == 0) {
            uint32_t p = s.prefix[t] | ((uint32_t)digit << shift);
            s.prefix[t] = p;
            s_prefix[t] = p;
            unsigned long long below = s.below[t] + e;
            s.below[t] = below;
            s.resid[t] = resid - e;
            if (pass == 3) {
                s.out_val[t] = __uint_as_float(p);
                s.out_cnt[t] = below + ties;
            }
        }
    }
    __syncthreads();
    for (int t = threadIdx.x; t < T; t += blockDim.x) {
        int first = 1;
        for (int j = 0; j < t; ++j) first &= (s_prefix[j] != s_prefix[t]);
        s_first[t] = first;
    }
    __syncthreads();
    for (int t = threadIdx.x; t < T; t += blockDim.x) {
        int less = 0;
        for (int j = 0; j < T; ++j) less += (s_first[j] && s_prefix[j] < s_prefix[t]);
        s.group_of[t] = less;
        if (s_first[t]) s.gprefix[less] = s_prefix[t];
    }
    if (threadIdx.x == 0) {
        int G = 0;
        for (int j = 0; j < T; ++j) G += s_first[j];
        s.G = G;
    }
    for (int q = threadIdx.x; q < T * 256; q += blockDim.x) gb[q] = 0ull;
}

// ------------------------------------------------------------------------------- bracket table (per group)
// From the 2*kc sample order statistics: brackets (lo_k, hi_k].  A collapsed bracket (lo == hi = v: the sample sees
// massive ties at v) becomes the single-value interval (prev(v), v].  All bracket ends together are the ascending cut
// list beta[0..J); level q = (beta[q-1], beta[q]] has a kind:
//   LEVEL_CAND   inside a bracket: its cells are appended to the candidate list
//   LEVEL_POINT  a single fp32 value: counted only — a rank that falls into it has eps = beta[q] exactly
//   LEVEL_OUT    outside every bracket: counted only — a rank that falls into it is a miss (radix fallback)
// The bucket table entry of a bucket holds the first cut not in a lower bucket, its index, and in the two top bits
// whether that level and the next one are candidate levels (see Counter::cell).
__global__ void __launch_bounds__(512) sel_table_kernel(const BufSel* __restrict__ st, SampleRanks sr,
                                                       SelTable* __restrict__ tabs) {
    const int b = blockIdx.x;
    const BufSel& s = st[b];
    SelTable& T = tabs[b];
    __shared__ int s_J;
    __shared__ float s_scale, s_dcap;
    __shared__ float s_beta[NCUT];
    __shared__ uint8_t s_kind[NCUT];
    const float INF = __int_as_float(0x7f800000);
    if (threadIdx.x == 0) {
        float blo[GK], bhi[GK];
        int J = 0;
        for (int k = 0; k < sr.kc; ++k) {
            float lo = sr.lo[k] ? s.out_val[2 * k] : -1.0f;          // open lower end: below every distance
            float hi = sr.hi[k] ? s.out_val[2 * k + 1] : INF;        // open upper end
            const bool collapsed = lo == hi;
            if (collapsed) lo = nextafterf(hi, -INF);                // the single value hi (negative if hi == 0)
            blo[k] = lo; bhi[k] = hi;
            // an end that the sample holds TIE_MASS times or more is a value with massive ties: the cut just below
            // it makes it a level of its own (counted, never appended to the candidates)
            const bool mlo = !collapsed && sr.lo[k] && s.out_cnt[2 * k] - s.below[2 * k] >= (unsigned long long)TIE_MASS;
            const bool mhi = !collapsed && sr.hi[k] && s.out_cnt[2 * k + 1] - s.below[2 * k + 1] >= (unsigned long long)TIE_MASS;
            for (int e = 0; e < 4; ++e) {                            // insert the cuts, ascending, without duplicates
                if ((e == 2 && !mlo) || (e == 3 && !mhi)) continue;
                const float x = e == 0 ? lo : e == 1 ? hi : nextafterf(e == 2 ? lo : hi, -INF);
                int pos = 0;
                while (pos < J && s_beta[pos] < x) ++pos;
                if (pos < J && s_beta[pos] == x) continue;
                for (int q = J; q > pos; --q) s_beta[q] = s_beta[q - 1];
                s_beta[pos] = x;
                ++J;
            }
        }
        for (int q = J; q < NCUT; ++q) s_beta[q] = INF;
        for (int q = 0; q < NCUT; ++q) {
            uint8_t kind = LEVEL_OUT;
            if (q >= 1 && q < J) {
                const float c0 = s_beta[q - 1], c1 = s_beta[q];
                if (c1 < INF && (c0 == nextafterf(c1, -INF) || (c1 == 0.0f && c0 < 0.0f))) {   // distances are >= 0
                    kind = LEVEL_POINT;
                } else {
                    for (int k = 0; k < sr.kc; ++k)
                        if (blo[k] <= c0 && c1 <= bhi[k]) kind = LEVEL_CAND;
                }
            }
            s_kind[q] = kind;
        }
        float fmaxb = 0.0f;                                          // largest finite boundary
        for (int q = 0; q < J; ++q)
            if (s_beta[q] < INF) fmaxb = fmaxf(fmaxb, s_beta[q]);
        float dcap = fmaxb >= 3.0e38f ? 3.4028234e38f : nextafterf(fmaxb, INF);
        if (!(dcap > 0.0f)) dcap = 1.0e-30f;
        s_dcap = dcap;
        s_scale = bucket_scale(dcap, NBS);
        s_J = J;
        T.J = J; T.scale = s_scale; T.dcap = dcap; T.heavy = J > 2 * sr.kc; T.pad = 0;
    }
    __syncthreads();
    const int J = s_J;
    for (int q = threadIdx.x; q < NCUT; q += blockDim.x) { T.beta[q] = s_beta[q]; T.kind[q] = s_kind[q]; }
    int multi = 0;
    for (int q = threadIdx.x; q < NBS; q += blockDim.x) {
        int below = 0, inside = 0;
        for (int j = 0; j < J; ++j) {
            const float x = s_beta[j];
            // negative boundary: below every bucket; +inf: in the top bucket (never exceeded anyway)
            const bool neg = x < 0.0f;
            const uint32_t bj = neg ? 0u : bucket_of(x, s_dcap, s_scale);
            below += neg ? 1 : (bj < (uint32_t)q);
            inside += !neg && bj == (uint32_t)q;
        }
        const uint32_t f0 = s_kind[below] == LEVEL_CAND, f1 = s_kind[below + 1] == LEVEL_CAND;
        T.lut[q] = make_uint2(__float_as_uint(s_beta[below]), (uint32_t)below | ((2u * f0 + (f0 != f1)) << 30));
        multi |= inside > 1;
    }
    multi = __syncthreads_or(multi);
    if (threadIdx.x == 0) T.multi = multi;
}

// ------------------------------------------------------------------------------------------ counting pass
struct CountArgs {
    View v;
    int L, n_obl, part, parts;
    const uint32_t* tile_start;
    const SelTable* tabs;
    SelState* ss;
    float* cand;                      // [batch][cap]
    unsigned long long cap;
    int m, tau;
    unsigned long long* counter;      // work-item counter of this launch (zeroed before)
    uint32_t tiles;                   // tiles per series (this part)
};

struct CountSmem {
    static constexpr int off_lut = 0;                                   // uint2[NBS]
    static constexpr int off_beta = off_lut + 8 * NBS;                  // float[2*GK+4]
    static constexpr int off_kind = off_beta + 4 * (NCUT);        // uint8[2*GK+4]
    static constexpr int off_cand = off_kind + (NCUT);            // float[LW/32][WCAP]
    static constexpr int off_cols = off_cand + 4 * (LW / 32) * WCAP;    // uint32[nlev][LW/2]
    // per-thread level counters: `fields` threads share a word, 2 x 16 bits (chunks of <= 2047 cells) or, when the
    // group has many levels, 3 x 10 bits (chunks of <= 1023 cells)
    __host__ __device__ static constexpr int col_words(int fields) { return (LW + fields - 1) / fields; }
};

// The (3,1) ring reads the i-side window four elements per load (CellDist VEC).
template <int M, int TAU>
__host__ __device__ constexpr bool count_vec() { return M == 3 && TAU == 1; }

template <int NORM, int M, int TAU, bool MULTI>
struct Counter : CellDist<NORM, M, TAU, 0, count_vec<M, TAU>()> {
    using CD = CellDist<NORM, M, TAU, 0, count_vec<M, TAU>()>;
    uint32_t lut, beta, kind;         // shared-window addresses of the bucket table, the boundaries, the level kinds
    uint32_t cols;                    // ... of this thread's column, level 0
    uint32_t col_row;                 // bytes between the levels of a column
    float* wbuf;                      // this warp's candidate buffer
    float* gcand;                     // the series' candidate list
    unsigned long long* gncand;
    unsigned long long cap;
    float scale, dcap;
    uint32_t inc, wcount, lane_lt;

    __device__ __forceinline__ void flush_warp() {
        // all lanes hold the same wcount; lane 0 reserves space in the series' candidate list
        const int lane = threadIdx.x & 31;
        unsigned long long base = 0;
        if (lane == 0) base = atomicAdd(gncand, (unsigned long long)wcount);
        base = __shfl_sync(FULL, base, 0);
        __syncwarp();
        for (uint32_t q = lane; q < wcount; q += 32)
            if (base + q < cap) gcand[base + q] = wbuf[q];
        __syncwarp();
        wcount = 0;
    }

    template <int R, bool GUARD>
    __device__ __forceinline__ void cell(int t, int cnt) {
        CD::template push<R>();
        const bool live = !GUARD || t < cnt;
        const float d = CD::template distance<R>();
        float er;
        uint32_t q;
        lds_f32_u32(lut + 8 * bucket_bits(d, dcap, scale), er, q);   // one load: the boundary to compare with, its index
        // bits 30-31 of the entry say whether level q and level q+1 are candidate levels, encoded so that adding
        // 1 << 30 together with the level increment leaves the answer in bit 31; the level's byte offset below is
        // q * 2^10 modulo 2^32, which drops those bits.
        q += d > er ? 0x40000001u : 0u;
        bool cand = (int32_t)q < 0;
        if (MULTI) {                                          // some bucket holds two or more boundaries
            q &= 0xffffu;
            while (d > lds_f32(beta + 4 * q)) ++q;
            cand = lds_u8(kind + q) == LEVEL_CAND;
        }
        if (live) red_u32(cols + q * col_row, inc);         // col_row is a multiple of 4: bits 30-31 of q drop out
        const unsigned mc = __ballot_sync(FULL, live && cand);
        if (mc) {
            const uint32_t nc = __popc(mc);
            if (wcount + nc > (uint32_t)WCAP) flush_warp();
            if (live && cand) wbuf[wcount + __popc(mc & lane_lt)] = d;
            wcount += nc;
        }
    }
    // The unguarded bulk of a chunk walks the cells in GROUPS of up to four: first the loads and the level of every cell
    // of the group (independent dependency chains that the hardware overlaps: no atomic or store sits between their
    // shared-memory loads, which ptxas would otherwise have to keep in program order), then the counter increments, and
    // one vote per group decides whether any lane holds a candidate.
    template <int R>
    __device__ __forceinline__ uint32_t classify(float& d) {
        CD::template push<R>();
        d = CD::template distance<R>();
        float er;
        uint32_t q;
        lds_f32_u32(lut + 8 * bucket_bits(d, dcap, scale), er, q);
        q += d > er ? 0x40000001u : 0u;                       // bit 31: the cell's level is a candidate level (see cell())
        if (MULTI) {
            q &= 0xffffu;
            while (d > lds_f32(beta + 4 * q)) ++q;
            q |= lds_u8(kind + q) == LEVEL_CAND ? 0x80000000u : 0u;
        }
        return q;
    }
    __device__ __forceinline__ void append(float d, uint32_t q) {
        const bool cand = (int32_t)q < 0;
        const unsigned mc = __ballot_sync(FULL, cand);
        if (mc) {
            const uint32_t nc = __popc(mc);
            if (wcount + nc > (uint32_t)WCAP) flush_warp();
            if (cand) wbuf[wcount + __popc(mc & lane_lt)] = d;
            wcount += nc;
        }
    }
    template <int R0, int... Q>
    __device__ __forceinline__ void group(std::integer_sequence<int, Q...>) {
        float d[sizeof...(Q)];
        const uint32_t q[sizeof...(Q)] = {classify<R0 + Q>(d[Q])...};
        (red_u32(cols + q[Q] * col_row, inc), ...);          // col_row is a multiple of 4: bits 30-31 of q drop out
        if (__any_sync(FULL, (int32_t)(q[Q] | ...) < 0)) (append(d[Q], q[Q]), ...);
    }
    template <int R0, int U>
    __device__ __forceinline__ void groups() {
        if constexpr (R0 < U) {
            constexpr int G = U - R0 >= 4 ? 4 : U - R0;
            group<R0>(std::make_integer_sequence<int, G>{});
            groups<R0 + G, U>();
        }
    }
    template <bool GUARD, int... R>
    __device__ __forceinline__ void superstep(int t, int cnt, std::integer_sequence<int, R...>) {
        if constexpr (GUARD) (cell<R, GUARD>(t + R, cnt), ...);
        else groups<0, (int)sizeof...(R)>();
    }
};

template <int NORM, int M, int TAU>
__global__ void __launch_bounds__(LW, 2) sel_count_kernel(CountArgs a, int nlev, int fields, int heavy_pass) {
    // PERSISTENT: the grid is two blocks per SM; a block draws (series, tile) items from an atomic counter, series by series,
    // so that the level table is loaded once per series and block, not once per tile.
    extern __shared__ __align__(16) char smem[];
    __shared__ int s_ob;
    __shared__ unsigned long long s_item;
    const int tid = threadIdx.x;
    uint2* lut_s = (uint2*)(smem + CountSmem::off_lut);
    float* beta_s = (float*)(smem + CountSmem::off_beta);
    float* cand_s = (float*)(smem + CountSmem::off_cand);
    uint32_t* cols_s = (uint32_t*)(smem + CountSmem::off_cols);
    const int span = M > 0 ? (M - 1) * TAU : (a.m - 1) * a.tau;
    const int ps = M > 0 ? 1 : (int)a.v.ps;
    constexpr bool VECK = count_vec<M, TAU>();
    const int LA = window_la(a.L, span, 0, ps) + 4, LB = window_lb(a.L, span, 0, ps);   // 4 floats of slack: alignment
    const int col_words = CountSmem::col_words(fields), field_bits = fields == 2 ? 16 : 10;
    float* ya_s = (float*)(smem + ((CountSmem::off_cols + nlev * 4 * col_words + 15) & ~15));
    float* yb_s = ya_s + LA;
    // VECK: the element pushed by the first cell of a super-step (window index 12k + 2) is 16-byte aligned
    const int sha = VECK ? 2 : 0;
    for (int q = tid; q < nlev * col_words; q += LW) cols_s[q] = 0;
    const unsigned long long n_items = (unsigned long long)a.tiles * (unsigned long long)a.v.batch;
    int cur_b = -1;
    __syncthreads();
  while (true) {
    if (tid == 0) s_item = atomicAdd(a.counter, 1ull);
    __syncthreads();
    const unsigned long long item = s_item;
    if (item >= n_items) break;
    const int b = (int)(item / a.tiles);
    const uint32_t tile = (uint32_t)(item - (unsigned long long)b * a.tiles);
    const SelTable& T = a.tabs[b];
    // series given to the radix passes, and series of the other launch (extra tie levels: the wider second launch), are
    // skipped as a whole: the counter jumps to the next series
    if (a.ss[b].fallback || T.heavy != heavy_pass) {
        if (tid == 0) atomicMax(a.counter, (unsigned long long)(b + 1) * a.tiles);
        __syncthreads();
        continue;
    }
    find_diagonal_block(a.tile_start, a.n_obl, tile, &s_ob);
    if (b != cur_b) {
        for (int q = tid; q < NBS; q += LW) lut_s[q] = T.lut[q];
        if (tid < NCUT) { beta_s[tid] = T.beta[tid]; ((uint8_t*)(smem + CountSmem::off_kind))[tid] = T.kind[tid]; }
        cur_b = b;
    }
    __syncthreads();
    const int ob = a.part + s_ob * a.parts;                   // this part's diagonal blocks are interleaved
    const int c = (int)(tile - a.tile_start[s_ob]);
    const int L = a.L;
    const int64_t n = a.v.n;
    const int64_t o0 = a.v.w + (int64_t)LW * ob;
    const int64_t s = (int64_t)c * L;
    const float* y = a.v.data + (int64_t)b * a.v.bs;
    stage_windows(y, (n - 1) * ps + span + 1, s * ps, (s + o0) * ps, ya_s + sha, LA - 4, yb_s, LB);
    __syncthreads();

    const int64_t len = n - (o0 + tid);
    const int cnt = (int)max((int64_t)0, min((int64_t)L, len - s));
    const int cnt_hi = __shfl_sync(FULL, cnt, 0);
    const int cnt_lo = __shfl_sync(FULL, cnt, 31);

    if (cnt_hi > 0) {
        // two instantiations: the common case (no bucket with two boundaries) carries no refinement loop
        auto walk = [&](auto& ct) {
            using CT = std::remove_reference_t<decltype(ct)>;
            constexpr int S = CT::S;
            ct.m = a.m;
            ct.tau = a.tau;
            ct.ps = ps;
            ct.seek(smem_addr(ya_s) + 4 * sha, pin(smem_addr(yb_s) + 4 * tid * ps), 0);
            ct.lut = pin(smem_addr(lut_s) - 8u * BUCKET_MAGIC_BITS);   // indexed with 8 * bucket_bits()
            ct.beta = smem_addr(beta_s);
            ct.kind = smem_addr(smem + CountSmem::off_kind);
            ct.cols = pin(smem_addr(cols_s) + 4 * (tid % col_words));
            ct.col_row = pin(4u * (uint32_t)col_words);
            ct.wbuf = cand_s + (tid >> 5) * WCAP;
            ct.gcand = a.cand + (unsigned long long)b * a.cap;
            ct.gncand = &a.ss[b].ncand;
            ct.cap = a.cap;
            ct.scale = T.scale;
            ct.dcap = T.dcap;
            ct.inc = pin(1u << (field_bits * (tid / col_words)));
            ct.wcount = 0;
            ct.lane_lt = (1u << (tid & 31)) - 1u;
            ct.prime();
            constexpr int U = S == 3 ? 12 : (S > 3 ? S : 4);  // cells per super-step, a multiple of S (and of 4 with vector loads)
            using Seq = std::make_integer_sequence<int, U>;
            int t = 0;
            for (; t + U <= cnt_lo; t += U) { ct.template superstep<false>(t, cnt, Seq{}); ct.advance(U); }
            for (; t < cnt_hi; t += U) { ct.template superstep<true>(t, cnt, Seq{}); ct.advance(U); }
            if (ct.wcount) ct.flush_warp();
        };
        if (T.multi) {
            Counter<NORM, M, TAU, true> ct;
            walk(ct);
        } else {
            Counter<NORM, M, TAU, false> ct;
            walk(ct);
        }
    }
    __syncthreads();
    {
        const int warp = tid >> 5, lane = tid & 31;
        unsigned long long* lc = a.ss[b].level_count;
        for (int row = warp; row < nlev; row += LW / 32) {
            uint32_t* r = cols_s + row * col_words;
            uint32_t sum = 0;
            const uint32_t fmask = (1u << field_bits) - 1u;
            for (int q = lane; q < col_words; q += 32) {
                uint32_t w = r[q];
                r[q] = 0;                                      // cleared for the block's next tile
                sum += (w & fmask) + ((w >> field_bits) & fmask) + (fields == 3 ? w >> 20 : 0u);
            }
            for (int off = 16; off; off >>= 1) sum += __shfl_down_sync(FULL, sum, off);
            if (lane == 0 && sum) atomicAdd(&lc[row], (unsigned long long)sum);
        }
    }
    __syncthreads();                                          // before the next item overwrites s_item, s_ob and the windows
  }
}

// After the counting pass, before the parts of a split call are summed: this part's candidate count and whether its
// list overflowed.
__global__ void sel_local_kernel(SelState* ss, int batch, unsigned long long cap) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= batch) return;
    ss[b].ncand_local = ss[b].ncand;
    ss[b].over = ss[b].ncand > cap ? 1ull : 0ull;
}

// One block per series: exact level counts -> each target's level.  A candidate level: its rank among the candidates
// (the buffer select finishes it).  A single-value level: eps and C are known here.  Anything else: radix fallback.
__global__ void __launch_bounds__(64) sel_bracket_resolve_kernel(SelState* ss, const SelTable* __restrict__ tabs,
                                                               SampleRanks sr, BufSel* st) {
    const int b = blockIdx.x;
    SelState& s = ss[b];
    if (s.fallback) return;
    const SelTable& T = tabs[b];
    BufSel& bs = st[b];
    __shared__ unsigned long long s_cum[NLEV_MAX + 2], s_cnd[NLEV_MAX + 2];
    __shared__ int s_bad;
    if (threadIdx.x == 0) {
        unsigned long long cum = 0, cnd = 0;
        for (int v = 0; v <= T.J; ++v) {
            s_cum[v] = cum;                                   // cells in the levels below v
            s_cnd[v] = cnd;                                   // candidates in the levels below v
            cum += s.level_count[v];
            if (T.kind[v] == LEVEL_CAND) cnd += s.level_count[v];
        }
        s_cum[T.J + 1] = cum;
        s_bad = (cnd != s.ncand) || s.over != 0;
        bufsel_reset(bs, sr.kc);
    }
    __syncthreads();
    const int t = threadIdx.x;
    int bad = s_bad;
    if (t < sr.kc) {
        const unsigned long long r = sr.rank[t];
        int v = 0;
        while (v <= T.J && s_cum[v + 1] < r) ++v;             // first level whose cumulative count reaches r
        const int kind = v <= T.J ? T.kind[v] : LEVEL_OUT;
        const bool point = kind == LEVEL_POINT;
        if (kind == LEVEL_OUT) bad = 1;                       // the rank is not inside a bracket
        s.is_point[t] = point;
        if (point) {
            s.point_val[t] = T.beta[v];
            s.point_cnt[t] = s_cum[v + 1];
        }
        const bool sel = kind == LEVEL_CAND && !bad;          // otherwise the buffer select gets a harmless rank
        bs.group_of[t] = 0;
        bs.prefix[t] = 0;
        bs.below[t] = 0;
        bs.resid[t] = sel ? s_cnd[v] + (r - s_cum[v]) : 1;
        bs.base[t] = sel ? s_cum[v] - s_cnd[v] : 0;
    }
    if (__syncthreads_or(bad) && threadIdx.x == 0) s.fallback = 1;
}

struct TargetMap {
    int32_t k_of[BT];                 // target of this call -> caller's index
    int32_t T;
};

__global__ void sel_finish_kernel(const SelState* __restrict__ ss, const BufSel* __restrict__ st, TargetMap tm, int K,
                                  unsigned long long P, int use_flag, float* __restrict__ eps,
                                  unsigned long long* __restrict__ count, double* __restrict__ rr) {
    const int b = blockIdx.x, t = threadIdx.x;
    if (t >= tm.T || (use_flag && ss[b].fallback)) return;
    const BufSel& s = st[b];
    const int k = tm.k_of[t];
    const bool point = use_flag && ss[b].is_point[t];
    const unsigned long long c = point ? ss[b].point_cnt[t] : s.base[t] + s.out_cnt[t];
    eps[(int64_t)b * K + k] = point ? ss[b].point_val[t] : s.out_val[t];
    count[(int64_t)b * K + k] = c;
    rr[(int64_t)b * K + k] = (double)c / (double)P;
}

// ------------------------------------------------------------------------------------------ radix passes
struct SelBatch {
    int32_t G;
    int32_t pad;
    uint32_t gprefix[RQA_MAX_K];
    int32_t group_of[RQA_MAX_K];
    uint32_t prefix[RQA_MAX_K];
    uint64_t resid[RQA_MAX_K];
    uint64_t below[RQA_MAX_K];
};

struct Ranks {
    uint64_t r[RQA_MAX_K];
};

constexpr int SEL_W = 128;            // diagonals per tile (= threads)
constexpr int SEL_L = 512;            // positions per tile

__global__ void radix_init_kernel(SelBatch* st, Ranks ranks, int K) {
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

// One pass: digit histogram of the cells whose determined high bits match a live prefix.  Persistent blocks walk
// the tiles (128 diagonals x 512 positions) of the series that are flagged for the radix path.
template <int NORM>
__global__ void __launch_bounds__(SEL_W) radix_pass_kernel(View v, int pass, const SelBatch* __restrict__ st,
                                                           unsigned long long* __restrict__ bins, int K,
                                                           const SelState* __restrict__ ss, int part, int parts) {
    extern __shared__ uint32_t sbins[];      // [G][256]
    __shared__ uint32_t s_gprefix[RQA_MAX_K];
    const int b = blockIdx.y;
    if (!ss[b].fallback) return;
    const SelBatch& s = st[b];
    const int G = s.G;
    for (int q = threadIdx.x; q < G * 256; q += blockDim.x) sbins[q] = 0;
    for (int q = threadIdx.x; q < G; q += blockDim.x) s_gprefix[q] = s.gprefix[q];
    __syncthreads();
    const float* yb = v.data + (int64_t)b * v.bs;
    const int shift = 24 - 8 * pass;
    const uint32_t himask = pass == 0 ? 0u : (0xFFFFFFFFu << (32 - 8 * pass));
    const int64_t nx = (v.n - v.w + SEL_W - 1) / SEL_W, ny = (v.n - v.w + SEL_L - 1) / SEL_L;
    for (int64_t tile = (int64_t)blockIdx.x * parts + part; tile < nx * ny; tile += (int64_t)gridDim.x * parts) {
        const int64_t o = v.w + (tile % nx) * SEL_W + threadIdx.x;
        const int64_t i0 = (tile / nx) * SEL_L;
        if (o >= v.n) continue;
        const int64_t iend = min(i0 + (int64_t)SEL_L, v.n - o);
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

__global__ void __launch_bounds__(256) radix_resolve_kernel(SelBatch* st, unsigned long long* bins, int K, int pass,
                                                            unsigned long long P, const SelState* __restrict__ ss,
                                                            float* __restrict__ eps,
                                                            unsigned long long* __restrict__ count,
                                                            double* __restrict__ rr) {
    const int b = blockIdx.x;
    if (!ss[b].fallback) return;
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
            unsigned long long t = __shfl_up_sync(FULL, incl, off);
            if (lane >= off) incl += t;
        }
        const unsigned long long resid = s.resid[k];
        unsigned ball = __ballot_sync(FULL, incl >= resid);
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
        digit = __shfl_sync(FULL, digit, src);
        e = __shfl_sync(FULL, e, src);
        ties = __shfl_sync(FULL, ties, src);
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

// ------------------------------------------------------------------------------------------ host side
enum { PATH_AUTO = 0, PATH_DIRECT = 1, PATH_BRACKET = 2, PATH_RADIX = 3, PATH_BLOCK = 4 };

struct SelectPlan {
    int path;
    unsigned long long P, S, cap;     // pairs, sample size, candidate capacity per series
    int L;
    Tiling tl;                        // this part's tiles of the counting pass
    int span;
    int fields;                       // counting pass: threads per counter word (2 or 3)
    int gs;                           // targets per group (<= GK)
    int ps;                           // point stride in floats
};

size_t count_smem_bytes(int nlev, int fields, int L, int span, int ps) {
    return (((size_t)CountSmem::off_cols + (size_t)nlev * 4 * CountSmem::col_words(fields) + 15) & ~(size_t)15) +
           4 * ((size_t)window_la(L, span, 0, ps) + 4 + window_lb(L, span, 0, ps));
}
constexpr size_t SMEM_PER_BLOCK_MAX = 227 * 1024 - 256;     // opt-in limit of sm_100a, minus the static part

SelectPlan make_select_plan(const View& v, int K, const Options& opt) {
    SelectPlan p{};
    p.P = n_pairs(v);
    p.span = (int)std::min<int64_t>((int64_t)(v.m - 1) * v.cs, (int64_t)MAX_SPAN + 1);
    p.ps = (int)std::min<int64_t>(v.ps, 1 << 20);
    // more than 20 brackets per group: 10-bit counters (two blocks per SM still fit), so shorter chunks
    p.gs = group_size_for(K, opt);
    p.fields = std::min(K, p.gs) > 20 ? 3 : 2;
    // tiled counting pass: delay views, and materialised points whose windows fit beside the widest level table
    // (the heavy launch's, with the counter width this K uses)
    const int nlev_max = 2 * (2 * std::min(K, p.gs) + 1) - 1;
    const bool tiled_ok = p.span <= MAX_SPAN && count_smem_bytes(nlev_max, p.fields, 32, p.span, p.ps) <= SMEM_PER_BLOCK_MAX;
    p.path = opt.select_path;
    // one block per series (rqa_block.cu) where the batch can fill the GPU with such blocks; forced: any batch
    const bool block_ok = opt.parts == 1 && block_select_fits(v, K);
    if (p.path == PATH_BLOCK && !block_ok) p.path = PATH_AUTO;
    if (p.path == PATH_AUTO)
        p.path = p.P <= (1ull << 22) ? (block_ok && v.batch >= 12 ? PATH_BLOCK : PATH_DIRECT) : (tiled_ok ? PATH_BRACKET : PATH_RADIX);
    if (p.path == PATH_BRACKET && !tiled_ok) p.path = PATH_RADIX;
    if (p.path == PATH_DIRECT && p.P > (1ull << 28)) p.path = tiled_ok ? PATH_BRACKET : PATH_RADIX;
    if (p.path == PATH_BRACKET) {
        // Sample size: 5.5 * P^(2/3) balances the sample against the candidates for a few targets on a long series; a
        // group of kg targets has brackets that cover up to kg * (sigmas + 1) / sqrt(S) of the pairs (all of them near
        // the median), and a candidate list that cannot hold them sends the series to the radix passes (20 x slower):
        // with many targets on a series of moderate length S grows until the brackets cover at most 20 % (P <= 2^26)
        // or 10 % of the pairs.  (Measured: 100 series of 10^4 points at K = 99 261 -> 55 ms, 10 series of 2*10^4 points
        // at K = 99 105 -> 17 ms, config 5 46.7 -> 41 ms; config 4 unchanged.)
        const int kg = std::min(K, p.gs);
        const double cover = p.P <= (1ull << 26) ? 0.2 : 0.1;
        const double s_targets = std::pow(kg * (BRACKET_SIGMAS + 1.0) / cover, 2.0);
        double s = std::max(5.5 * std::pow((double)p.P, 2.0 / 3.0), s_targets);
        unsigned long long S = (unsigned long long)std::min(std::max(s, 65536.0), 268435456.0);
        if (opt.sample_size > 0) S = (unsigned long long)opt.sample_size;
        p.S = std::max<unsigned long long>(16, S);
        // capacity: 1.5 x the worst-case expected bracket content of one group (<= GK targets)
        // (a forced small sample on a long series is not allowed to claim more than 12 % of P)
        double frac = std::min(p.P <= (1ull << 28) ? 1.0 : 0.12, kg * (BRACKET_SIGMAS + 1.0) / std::sqrt((double)p.S));
        unsigned long long cap = (unsigned long long)(1.5 * frac * (double)p.P) + 4096;
        if (opt.cand_cap > 0) cap = (unsigned long long)opt.cand_cap;
        p.cap = std::min(cap, p.P);
        const double cells = (double)p.P * (double)v.batch / (double)opt.parts;
        int64_t L = (int64_t)std::ceil(cells / ((double)LW * sm_count() * 3.0 * 8.0));
        p.L = (int)std::max<int64_t>(32, std::min<int64_t>(p.fields == 3 ? 1023 : 2047, L));
        while (p.L > 32 && count_smem_bytes(nlev_max, p.fields, p.L, p.span, p.ps) > SMEM_PER_BLOCK_MAX) p.L = std::max(32, p.L / 2);
        p.tl = make_tiling(n_diag(v), p.L, opt.part, opt.parts);
    }
    return p;
}

template <int NORM, int M, int TAU>
rqa_status launch_count(const CountArgs& a, const SelectPlan& p, int nlev, int batch, cudaStream_t s) {
    auto kern = sel_count_kernel<NORM, M, TAU>;
    // second launch: only the series whose table carries extra single-value levels (massive ties); its blocks
    // of the other series return at once, and so do the first launch's blocks of those series
    const int nlev_heavy = 2 * nlev - 1;
    const size_t smem = count_smem_bytes(nlev, p.fields, p.L, p.span, p.ps), smem_heavy = count_smem_bytes(nlev_heavy, p.fields, p.L, p.span, p.ps);
    static thread_local bool attr_set[8] = {false};             // per device: opted in to the largest shared-memory size
    int dev = 0;
    RQA_CUDA_TRY(cudaGetDevice(&dev));
    if (dev >= 8 || !attr_set[dev]) {
        RQA_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_PER_BLOCK_MAX));
        if (dev < 8) attr_set[dev] = true;
    }
    if (smem_heavy > SMEM_PER_BLOCK_MAX) { set_error("rqa_eps_for_rr: counting pass needs %zu bytes of shared memory", smem_heavy); return RQA_ERR_UNSUPPORTED; }
    if (p.tl.tiles == 0) return RQA_OK;
    const unsigned grid = (unsigned)std::min<uint64_t>(p.tl.tiles * (uint64_t)batch, (uint64_t)(2 * sm_count()));
    CountArgs a0 = a, a1 = a;
    a0.tiles = a1.tiles = (uint32_t)p.tl.tiles;
    a1.counter = a.counter + 1;
    kern<<<grid, LW, smem, s>>>(a0, nlev, p.fields, 0);
    RQA_LAUNCH_CHECK();
    kern<<<grid, LW, smem_heavy, s>>>(a1, nlev_heavy, p.fields, 1);
    RQA_LAUNCH_CHECK();
    return RQA_OK;
}

template <int NORM>
rqa_status dispatch_count(const CountArgs& a, const SelectPlan& p, int nlev, int batch, cudaStream_t s) {
    const bool delay = p.ps == 1;
    if (delay && a.m == 1) return launch_count<NORM, 1, 1>(a, p, nlev, batch, s);
    if (delay && a.m == 3 && a.tau == 1) return launch_count<NORM, 3, 1>(a, p, nlev, batch, s);
    if (delay && a.m == 3 && a.tau == 3) return launch_count<NORM, 3, 3>(a, p, nlev, batch, s);
    if (delay && a.m == 5 && a.tau == 2) return launch_count<NORM, 5, 2>(a, p, nlev, batch, s);
    return launch_count<NORM, 0, 0>(a, p, nlev, batch, s);
}

// 4 radix passes over a buffer for the <= BT targets whose state is already initialised in `st`.
rqa_status run_bufsel(const float* buf, unsigned long long stride, unsigned long long cap, const SelState* ss,
                      int use_ncand, BufSel* st, unsigned long long* bins, int T, int batch, cudaStream_t s,
                      const Options* split = nullptr) {
    const size_t smem = (size_t)T * 256 * sizeof(uint32_t);
    static thread_local bool attr_set[8] = {false};
    int dev = 0;
    RQA_CUDA_TRY(cudaGetDevice(&dev));
    if (dev >= 8 || !attr_set[dev]) {
        RQA_CUDA_TRY(cudaFuncSetAttribute(bufsel_pass_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, BT * 256 * (int)sizeof(uint32_t)));
        if (dev < 8) attr_set[dev] = true;
    }
    unsigned blocks = (unsigned)std::max<unsigned long long>(1, std::min<unsigned long long>((cap + 2047) / 2048, 148 * 4));
    for (int pass = 0; pass < 4; ++pass) {
        bufsel_pass_kernel<<<dim3(blocks, (unsigned)batch), 256, smem, s>>>(buf, stride, cap, ss, use_ncand, pass, st, bins);
        RQA_LAUNCH_CHECK();
        if (split) {                                             // every part holds a share of the buffer: sum the digit bins
            rqa_status rs = reduce_parts(*split, bins, (size_t)batch * BT * 256, s);
            if (rs != RQA_OK) return rs;
        }
        bufsel_resolve_kernel<<<batch, 256, 0, s>>>(st, bins, pass, ss, use_ncand);
        RQA_LAUNCH_CHECK();
    }
    return RQA_OK;
}

struct SelectWs {
    SelState* ss;
    BufSel* st;
    unsigned long long* bins;         // [batch][BT][256]
    SelTable* tabs;
    uint32_t* tile_start;
    unsigned long long* counters;     // work-item counters of the two counting-pass launches
    float* sample;                    // [batch][S] (DIRECT: [batch][P])
    float* cand;                      // [batch][cap]
    SelBatch* rst;
    unsigned long long* rbins;        // [batch][K][256]
};

SelectWs carve(Arena& ws, const View& v, int K, const SelectPlan& p) {
    SelectWs w{};
    w.ss = ws.take<SelState>(v.batch);
    w.st = ws.take<BufSel>(v.batch);
    w.bins = (unsigned long long*)ws.take<uint64_t>((size_t)v.batch * BT * 256);
    w.rst = ws.take<SelBatch>(v.batch);
    w.rbins = (unsigned long long*)ws.take<uint64_t>((size_t)v.batch * K * 256);
    if (p.path == PATH_DIRECT) w.sample = ws.take<float>((size_t)v.batch * p.P);
    if (p.path == PATH_BRACKET) {
        w.tabs = ws.take<SelTable>(v.batch);
        w.tile_start = ws.take<uint32_t>((size_t)p.tl.n_obl + 1);
        w.counters = (unsigned long long*)ws.take<uint64_t>(2);
        w.sample = ws.take<float>((size_t)v.batch * p.S);
        w.cand = ws.take<float>((size_t)v.batch * p.cap);
    }
    return w;
}

}  // namespace

size_t select_workspace_bytes(const View& v, int K, const Options& opt) {
    SelectPlan p = make_select_plan(v, K, opt);
    Arena a(nullptr, ~(size_t)0);
    carve(a, v, K, p);
    return a.off;
}

rqa_status run_select(const View& v, int norm, const uint64_t* h_rank, int K, float* d_eps, uint64_t* d_count,
                      double* d_rr, Arena& ws, cudaStream_t s, const Options& opt) {
    // short series: one block sorts all distances of a series in shared memory (any explicit path choice, and a split
    // call, keep the general machinery)
    if (opt.select_path == PATH_AUTO && opt.parts == 1 && small_series(v))
        return run_select_small(v, norm, h_rank, K, d_eps, d_count, d_rr, s);
    const SelectPlan p = make_select_plan(v, K, opt);
    SelectWs w = carve(ws, v, K, p);
    if (!ws.ok()) { set_error("rqa_eps_for_rr: workspace too small"); return RQA_ERR_WORKSPACE_TOO_SMALL; }
    const unsigned long long P = p.P;
    unsigned long long* d_cnt = (unsigned long long*)d_count;

    sel_init_kernel<<<v.batch, 128, 0, s>>>(w.ss, p.path == PATH_RADIX ? 1 : 0);
    RQA_LAUNCH_CHECK();
    RQA_CUDA_TRY(cudaMemsetAsync(w.bins, 0, sizeof(uint64_t) * (size_t)v.batch * BT * 256, s));

    // targets sorted by rank (groups are contiguous in rank)
    int order[RQA_MAX_K];
    for (int k = 0; k < K; ++k) order[k] = k;
    std::stable_sort(order, order + K, [&](int a, int b) { return h_rank[a] < h_rank[b]; });

    if (p.path == PATH_BLOCK) {
        // every series in one block; a series with massive ties sets its fallback flag and is redone below
        rqa_status st = run_select_block(v, norm, h_rank, K, d_eps, d_count, d_rr, &w.ss[0].fallback, sizeof(SelState), s);
        if (st != RQA_OK) return st;
    }

    if (p.path == PATH_DIRECT) {
        unsigned blocks = (unsigned)std::min<int64_t>(v.n - v.w, 148 * 8);
        if (norm == RQA_NORM_MAX) sel_direct_kernel<RQA_NORM_MAX><<<dim3(blocks, v.batch), 256, 0, s>>>(v, P, w.sample);
        else sel_direct_kernel<RQA_NORM_EUCLID><<<dim3(blocks, v.batch), 256, 0, s>>>(v, P, w.sample);
        RQA_LAUNCH_CHECK();
        for (int base = 0; base < K; base += BT) {
            const int T = std::min(BT, K - base);
            Ranks64 rk{};
            TargetMap tm{};
            tm.T = T;
            for (int t = 0; t < T; ++t) { rk.r[t] = h_rank[order[base + t]]; tm.k_of[t] = order[base + t]; }
            bufsel_init_kernel<<<v.batch, BT, 0, s>>>(w.st, rk, T);
            RQA_LAUNCH_CHECK();
            rqa_status st = run_bufsel(w.sample, P, P, w.ss, 0, w.st, w.bins, T, v.batch, s);
            if (st != RQA_OK) return st;
            sel_finish_kernel<<<v.batch, BT, 0, s>>>(w.ss, w.st, tm, K, P, 0, d_eps, d_cnt, d_rr);
            RQA_LAUNCH_CHECK();
        }
        return RQA_OK;
    }

    if (p.path == PATH_BRACKET) {
        const unsigned long long S = p.S;
        {
            unsigned blocks = (unsigned)std::min<unsigned long long>((S + 255) / 256, 148 * 16);
            if (norm == RQA_NORM_MAX) sel_sample_kernel<RQA_NORM_MAX><<<dim3(blocks, v.batch), 256, 0, s>>>(v, S, w.sample);
            else sel_sample_kernel<RQA_NORM_EUCLID><<<dim3(blocks, v.batch), 256, 0, s>>>(v, S, w.sample);
            RQA_LAUNCH_CHECK();
        }
        rqa_status st = RQA_OK;
        if (p.tl.tiles > 0) st = launch_tile_table(p.tl, w.tile_start, s);
        if (st != RQA_OK) return st;
        for (int base = 0; base < K; base += p.gs) {
            const int kc = std::min(p.gs, K - base);
            SampleRanks sr{};
            Ranks64 rk{};
            TargetMap tm{};
            sr.kc = kc;
            tm.T = kc;
            for (int t = 0; t < kc; ++t) {
                const unsigned long long r = h_rank[order[base + t]];
                const double q = (double)r / (double)P;
                const double mean = q * (double)S, sd = std::sqrt((double)S * q * (1.0 - q));
                const double lo = std::floor(mean - BRACKET_SIGMAS * sd) - 1.0;
                const double hi = std::ceil(mean + BRACKET_SIGMAS * sd) + 1.0;
                sr.lo[t] = lo >= 1.0 ? (unsigned long long)lo : 0;
                sr.hi[t] = hi <= (double)S ? (unsigned long long)hi : 0;
                sr.rank[t] = r;
                rk.r[2 * t] = sr.lo[t] ? sr.lo[t] : 1;
                rk.r[2 * t + 1] = sr.hi[t] ? sr.hi[t] : S;
                tm.k_of[t] = order[base + t];
            }
            if (base > 0) {
                sel_group_reset_kernel<<<v.batch, 128, 0, s>>>(w.ss);
                RQA_LAUNCH_CHECK();
            }
            bufsel_init_kernel<<<v.batch, BT, 0, s>>>(w.st, rk, 2 * kc);
            RQA_LAUNCH_CHECK();
            st = run_bufsel(w.sample, S, S, w.ss, 0, w.st, w.bins, 2 * kc, v.batch, s);
            if (st != RQA_OK) return st;
            sel_table_kernel<<<v.batch, 512, 0, s>>>(w.st, sr, w.tabs);
            RQA_LAUNCH_CHECK();
            CountArgs a;
            a.v = v; a.L = p.L; a.n_obl = p.tl.n_obl; a.part = opt.part; a.parts = opt.parts;
            a.tile_start = w.tile_start; a.tabs = w.tabs; a.ss = w.ss;
            a.cand = w.cand; a.cap = p.cap; a.m = v.m; a.tau = (int)v.cs;
            a.counter = w.counters; a.tiles = (uint32_t)p.tl.tiles;
            RQA_CUDA_TRY(cudaMemsetAsync(w.counters, 0, 2 * sizeof(unsigned long long), s));
            const int nlev = 2 * kc + 1;
            if (base == 0 && opt.ev_begin) RQA_CUDA_TRY(cudaEventRecord((cudaEvent_t)opt.ev_begin, s));
            st = norm == RQA_NORM_MAX ? dispatch_count<RQA_NORM_MAX>(a, p, nlev, v.batch, s)
                                      : dispatch_count<RQA_NORM_EUCLID>(a, p, nlev, v.batch, s);
            if (st != RQA_OK) return st;
            if (base == 0 && opt.ev_end) RQA_CUDA_TRY(cudaEventRecord((cudaEvent_t)opt.ev_end, s));
            sel_local_kernel<<<(v.batch + 63) / 64, 64, 0, s>>>(w.ss, v.batch, p.cap);
            RQA_LAUNCH_CHECK();
            // a split call: the level counts (and candidate totals) of all parts, per series
            for (int b = 0; b < v.batch && opt.parts > 1; ++b) {
                st = reduce_parts(opt, &w.ss[b].ncand, SEL_REDUCE_WORDS, s);
                if (st != RQA_OK) return st;
            }
            sel_bracket_resolve_kernel<<<v.batch, 64, 0, s>>>(w.ss, w.tabs, sr, w.st);
            RQA_LAUNCH_CHECK();
            st = run_bufsel(w.cand, p.cap, p.cap, w.ss, 1, w.st, w.bins, kc, v.batch, s, opt.parts > 1 ? &opt : nullptr);
            if (st != RQA_OK) return st;
            sel_finish_kernel<<<v.batch, BT, 0, s>>>(w.ss, w.st, tm, K, P, 1, d_eps, d_cnt, d_rr);
            RQA_LAUNCH_CHECK();
        }
    }

    // radix passes: the whole job on the RADIX path, otherwise only the series the bracket path flagged (blocks of
    // other series return at once)
    Ranks ranks;
    for (int k = 0; k < K; ++k) ranks.r[k] = h_rank[k];
    RQA_CUDA_TRY(cudaMemsetAsync(w.rbins, 0, sizeof(uint64_t) * (size_t)v.batch * K * 256, s));
    radix_init_kernel<<<v.batch, RQA_MAX_K, 0, s>>>(w.rst, ranks, K);
    RQA_LAUNCH_CHECK();
    const size_t smem = (size_t)K * 256 * sizeof(uint32_t);
    auto kern = norm == RQA_NORM_MAX ? radix_pass_kernel<RQA_NORM_MAX> : radix_pass_kernel<RQA_NORM_EUCLID>;
    if (smem > 48 * 1024) RQA_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    const int64_t tiles = ((v.n - v.w + SEL_W - 1) / SEL_W) * ((v.n - v.w + SEL_L - 1) / SEL_L);
    dim3 grid((unsigned)std::min<int64_t>((tiles + opt.parts - 1) / opt.parts, 148 * 16), (unsigned)v.batch);
    for (int pass = 0; pass < 4; ++pass) {
        kern<<<grid, SEL_W, smem, s>>>(v, pass, w.rst, w.rbins, K, w.ss, opt.part, opt.parts);
        RQA_LAUNCH_CHECK();
        {
            rqa_status rs = reduce_parts(opt, w.rbins, (size_t)v.batch * K * 256, s);
            if (rs != RQA_OK) return rs;
        }
        radix_resolve_kernel<<<v.batch, 256, 0, s>>>(w.rst, w.rbins, K, pass, P, w.ss, d_eps, d_cnt, d_rr);
        RQA_LAUNCH_CHECK();
    }
    return RQA_OK;
}

}  // namespace rqa
