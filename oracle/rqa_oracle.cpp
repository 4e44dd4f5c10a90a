/*
 * rqa_oracle.cpp — plain, slow, single-file CPU ORACLE for the averaged-RQA hot path.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code, header, table or
 * helper with the CUDA library (paper_2208_09136_b200/csrc); neither side includes the other.
 *
 * What it computes is the plain definition, by brute force, in the paper's order:
 *
 *   embed        x_i[c] = y[i + c*tau]                      PAPER.md:115 (sec. 4.3, delay embedding;
 *                                                           forward indexing, reading S7)
 *   distance     d_ij = max_c |x_i[c] - x_j[c]|             PAPER.md:47-50 (sec. 2, Eq. 1, maximum norm)
 *                or sqrt(sum_c (x_i[c]-x_j[c])^2)           BASELINE.json configs[2] (Euclidean option,
 *                                                           fixed order c = 0..m-1, no FMA contraction)
 *   recurrence   R_ij = (d_ij <= eps)                       PAPER.md:47-55 (Eqs. 1-2) with reading S1 (<=)
 *   eps for RR   eps_k = the ceil(RR_k*P)-th smallest of    PAPER.md:78 (sec. 3, "preselect RR and use the
 *                the P = N'(N'-1)/2 distances (i<j)         corresponding eps") with readings S4-S6
 *   P_k(l)       number of maximal diagonal runs of         PAPER.md:69-72 (Eq. 4 and the sentence under
 *                length l in the upper triangle j>i         it), PAPER.md:125 (upper triangle only)
 *   DET_k, mean  Eq. 4 and Eq. 5
 *
 * Precision: fp32 series and distances (BASELINE.json), uint64 counts, fp64 ratios.
 * Build: g++ -O2 -ffp-contract=off [-fopenmp] (never -ffast-math: it switches on FTZ/DAZ).
 *
 * Pins (tests/test_oracle_pins.py, `-m "not gpu"`): hand-enumerated recurrence plots
 * (tests/golden/hand_cases.txt), closed forms for ramp / constant / exactly periodic series, numpy
 * order statistics, the counting certificate, sum_l l*P(l) = C, nesting, triangle symmetry, the i.i.d.
 * uniform-noise closed form DET ~ 1-(1-p)^2, exact-rational re-evaluation of the Euclidean chain; vertical lines:
 * hand-enumerated plots, numpy run-length brute force on the full matrix, sum_v v*P(v) = 2C, ramp closed form.
 * Nothing here is "parity unpinned".
 *
 * The only parallel construct is an optional OpenMP `parallel for` over diagonals / rows whose
 * iterations are independent and whose integer results are summed; it changes no arithmetic.
 */
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

enum { NORM_MAX = 0, NORM_EUCLID = 1 };

inline int64_t embedded_points(int64_t N, int m, int64_t tau) { return N - (int64_t)(m - 1) * tau; }

/* PAPER.md:47-50 (Eq. 1, maximum norm) / BASELINE.json configs[2] (Euclid, fixed order, no FMA). */
inline float distance(const float* y, int64_t i, int64_t j, int m, int64_t tau, int norm) {
    if (norm == NORM_MAX) {
        float d = 0.0f;
        for (int c = 0; c < m; ++c) {
            float t = std::fabs(y[i + c * tau] - y[j + c * tau]);
            d = std::fmax(d, t);
        }
        return d;
    }
    float t0 = y[i] - y[j];
    float s = t0 * t0;
    for (int c = 1; c < m; ++c) {
        float t = y[i + c * tau] - y[j + c * tau];
        float q = t * t;
        s = s + q;
    }
    return std::sqrt(s);
}

bool all_finite(const float* y, int64_t N) {
    for (int64_t n = 0; n < N; ++n)
        if (!std::isfinite(y[n])) return false;
    return true;
}

int pick_threads(int threads) {
#ifdef _OPENMP
    if (threads <= 0) return omp_get_max_threads();
    return threads;
#else
    (void)threads;
    return 1;
#endif
}

}  // namespace

extern "C" {

/* Status codes of the oracle (its own; not the library's). */
enum { ORACLE_OK = 0, ORACLE_BAD_ARG = 1, ORACLE_NONFINITE = 2 };

int rqa_oracle_max_threads(void) { return pick_threads(0); }

/* x_i[c] = y[i + c*tau], X row-major [N'][m].  PAPER.md:115. */
int rqa_oracle_embed(const float* y, int64_t N, int m, int64_t tau, float* X) {
    if (!y || !X || m < 1 || tau < 1) return ORACLE_BAD_ARG;
    int64_t Np = embedded_points(N, m, tau);
    if (Np < 1) return ORACLE_BAD_ARG;
    for (int64_t i = 0; i < Np; ++i)
        for (int c = 0; c < m; ++c) X[i * m + c] = y[i + c * tau];
    return ORACLE_OK;
}

/* Pairs counted with a Theiler window w >= 1 (w = 1: only the main diagonal is excluded, reading S9): the
 * pairs i<j with j - i >= w, P_w = (N'-w)(N'-w+1)/2 of them. */
static uint64_t pairs_with_window(int64_t Np, int64_t w) {
    return (uint64_t)(Np - w) * (uint64_t)(Np - w + 1) / 2;
}

/* All distances of the pairs i<j with j - i >= theiler, in row-major order of (i,j).  PAPER.md:47-50. */
static int distances_w(const float* y, int64_t N, int m, int64_t tau, int norm, int64_t theiler, float* out) {
    if (!y || !out || m < 1 || tau < 1 || theiler < 1) return ORACLE_BAD_ARG;
    int64_t Np = embedded_points(N, m, tau);
    if (Np < 2 || theiler > Np - 1) return ORACLE_BAD_ARG;
    int64_t p = 0;
    for (int64_t i = 0; i < Np; ++i)
        for (int64_t j = i + theiler; j < Np; ++j) out[p++] = distance(y, i, j, m, tau, norm);
    return ORACLE_OK;
}

/* All P = N'(N'-1)/2 distances of the pairs i<j, in row-major order of (i,j).  PAPER.md:47-50. */
int rqa_oracle_distances(const float* y, int64_t N, int m, int64_t tau, int norm, float* out) {
    return distances_w(y, N, m, tau, norm, 1, out);
}

/* Rank of the order statistic for a target recurrence rate: the literal fp64 expression
 * ceil(rr * (double)P), clamped to [1, P] (reading S5). */
uint64_t rqa_oracle_rank(double rr, uint64_t P) {
    double r = std::ceil(rr * (double)P);
    if (!(r >= 1.0)) return 1;
    if (r >= (double)P) return P;
    return (uint64_t)r;
}

/* eps_k = the r_k-th smallest distance (1-based), C_k = #{d <= eps_k}, realised RR_k = C_k / P.
 * Full enumeration + std::sort (4*P bytes).  PAPER.md:78 + readings S4-S6. */
int rqa_oracle_eps_for_rr(const float* y, int64_t N, int m, int64_t tau, int norm, const double* rr, int K,
                          float* eps, uint64_t* count, double* rr_realised, int64_t theiler) {
    if (!y || !rr || !eps || !count || !rr_realised || m < 1 || tau < 1 || K < 1 || theiler < 1) return ORACLE_BAD_ARG;
    int64_t Np = embedded_points(N, m, tau);
    if (Np < 2 || theiler > Np - 1) return ORACLE_BAD_ARG;
    if (!all_finite(y, N)) return ORACLE_NONFINITE;
    for (int k = 0; k < K; ++k)
        if (!(rr[k] > 0.0) || !(rr[k] <= 1.0)) return ORACLE_BAD_ARG;
    uint64_t P = pairs_with_window(Np, theiler);
    std::vector<float> d((size_t)P);
    int st = distances_w(y, N, m, tau, norm, theiler, d.data());
    if (st != ORACLE_OK) return st;
    std::sort(d.begin(), d.end());
    for (int k = 0; k < K; ++k) {
        uint64_t r = rqa_oracle_rank(rr[k], P);
        float e = d[(size_t)(r - 1)];
        eps[k] = e;
        uint64_t c = (uint64_t)(std::upper_bound(d.begin(), d.end(), e) - d.begin());
        count[k] = c;
        rr_realised[k] = (double)c / (double)P;
    }
    return ORACLE_OK;
}

/* The counting certificate: for every k, lt[k] = #{i<j : d_ij < eps_k}, le[k] = #{i<j : d_ij <= eps_k}, over the pairs
 * with j - i >= theiler.
 * eps is the r-th smallest distance iff lt < r <= le.  O(1) extra memory, no sort.  Used where the
 * 4*P-byte sorted array does not fit (N = 1e5) and as an independent check of the sort-based path. */
int rqa_oracle_count_lt_le(const float* y, int64_t N, int m, int64_t tau, int norm, const float* eps, int K,
                           uint64_t* lt, uint64_t* le, int threads, int64_t theiler) {
    if (!y || !eps || !lt || !le || m < 1 || tau < 1 || K < 1 || theiler < 1) return ORACLE_BAD_ARG;
    int64_t Np = embedded_points(N, m, tau);
    if (Np < 2 || theiler > Np - 1) return ORACLE_BAD_ARG;
    int nt = pick_threads(threads);
    std::vector<uint64_t> acc_lt((size_t)nt * K, 0), acc_le((size_t)nt * K, 0);
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 16) num_threads(nt)
#endif
    for (int64_t i = 0; i < Np; ++i) {
#ifdef _OPENMP
        int t = omp_get_thread_num();
#else
        int t = 0;
#endif
        uint64_t* a = &acc_lt[(size_t)t * K];
        uint64_t* b = &acc_le[(size_t)t * K];
        for (int64_t j = i + theiler; j < Np; ++j) {           /* theiler = 1: every pair i < j (reading S9) */
            float d = distance(y, i, j, m, tau, norm);
            for (int k = 0; k < K; ++k) {
                a[k] += (d < eps[k]) ? 1u : 0u;
                b[k] += (d <= eps[k]) ? 1u : 0u;
            }
        }
    }
    for (int k = 0; k < K; ++k) {
        lt[k] = 0;
        le[k] = 0;
        for (int t = 0; t < nt; ++t) {
            lt[k] += acc_lt[(size_t)t * K + k];
            le[k] += acc_le[(size_t)t * K + k];
        }
    }
    return ORACLE_OK;
}

/* Diagonal-line histogram.  hist is [K][N'] uint64, hist[k][l] = number of maximal runs of length l of
 * recurrent cells (d <= eps_k) along the diagonals o = 1..N'-1 of the upper triangle (cells (i, i+o),
 * i = 0..N'-1-o).  Runs touching either end of a diagonal count with their truncated length (reading
 * S8); the main diagonal is excluded (S2).  hist[k][0] = 0.
 *   lower != 0 scans the lower triangle instead (cells (i+o, i)); by the symmetry of R
 *   the result must be identical — used only as a pin.
 *   theiler = w > 1 scans the diagonals o = w..N'-1 only (a Theiler window; the paper uses none).
 *   threads: 1 = the literal serial loop; >1 (or 0 = all) splits the diagonals over OpenMP threads with
 *   private histograms that are summed.  PAPER.md:69-72, 125. */
int rqa_oracle_line_hist(const float* y, int64_t N, int m, int64_t tau, int norm, const float* eps, int K,
                         uint64_t* hist, int lower, int threads, int64_t theiler) {
    if (!y || !eps || !hist || m < 1 || tau < 1 || K < 1 || theiler < 1) return ORACLE_BAD_ARG;
    int64_t Np = embedded_points(N, m, tau);
    if (Np < 2 || theiler > Np - 1) return ORACLE_BAD_ARG;
    int nt = pick_threads(threads);
    std::memset(hist, 0, sizeof(uint64_t) * (size_t)K * (size_t)Np);
    std::vector<uint64_t> priv;
    if (nt > 1) priv.assign((size_t)nt * (size_t)K * (size_t)Np, 0);
    for (int k = 0; k < K; ++k) {
        const float e = eps[k];
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 8) num_threads(nt) if (nt > 1)
#endif
        for (int64_t o = theiler; o < Np; ++o) {              /* theiler = 1: every diagonal but the main one */
            uint64_t* h = hist + (size_t)k * Np;
#ifdef _OPENMP
            if (nt > 1) h = priv.data() + ((size_t)omp_get_thread_num() * K + k) * (size_t)Np;
#endif
            int64_t run = 0;
            for (int64_t i = 0; i + o < Np; ++i) {
                float d = lower ? distance(y, i + o, i, m, tau, norm) : distance(y, i, i + o, m, tau, norm);
                if (d <= e) {
                    ++run;
                } else {
                    if (run > 0) h[run] += 1;
                    run = 0;
                }
            }
            if (run > 0) h[run] += 1;
        }
    }
    if (nt > 1)
        for (int t = 0; t < nt; ++t)
            for (size_t q = 0; q < (size_t)K * (size_t)Np; ++q) hist[q] += priv[(size_t)t * K * Np + q];
    return ORACLE_OK;
}

/* Vertical-line histogram ("other RQA measures"; the paper defines no vertical-line measure itself —
 * DESIGN.md reading S19 fixes the convention).  The FULL symmetric N' x N' recurrence matrix is walked
 * column by column: in column j the cell (i, j) is recurrent iff |i - j| >= theiler (theiler = 1: only the main
 * diagonal is excluded, readings S2/S9) and d(x_i, x_j) <= eps_k.  vhist[k][v] = number of maximal runs of exactly v
 * recurrent cells along i; the excluded band splits a column in two; runs touching the border of the plot or the band
 * count with their truncated length (as S8).  vhist is [K][N'] uint64, vhist[k][0] = 0.  Every recurrent cell of the
 * upper triangle is visited twice (as (i,j) and as (j,i)), so sum_v v*vhist[k][v] = 2*C_k.
 *   threads: 1 = the literal serial loop; >1 (0 = all) splits the columns over OpenMP threads (private histograms). */
int rqa_oracle_vert_hist(const float* y, int64_t N, int m, int64_t tau, int norm, const float* eps, int K,
                         uint64_t* vhist, int threads, int64_t theiler) {
    if (!y || !eps || !vhist || m < 1 || tau < 1 || K < 1 || theiler < 1) return ORACLE_BAD_ARG;
    int64_t Np = embedded_points(N, m, tau);
    if (Np < 2 || theiler > Np - 1) return ORACLE_BAD_ARG;
    int nt = pick_threads(threads);
    std::memset(vhist, 0, sizeof(uint64_t) * (size_t)K * (size_t)Np);
    std::vector<uint64_t> priv;
    if (nt > 1) priv.assign((size_t)nt * (size_t)K * (size_t)Np, 0);
    for (int k = 0; k < K; ++k) {
        const float e = eps[k];
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 8) num_threads(nt) if (nt > 1)
#endif
        for (int64_t j = 0; j < Np; ++j) {                     /* column j */
            uint64_t* h = vhist + (size_t)k * Np;
#ifdef _OPENMP
            if (nt > 1) h = priv.data() + ((size_t)omp_get_thread_num() * K + k) * (size_t)Np;
#endif
            int64_t run = 0;
            for (int64_t i = 0; i < Np; ++i) {                 /* down the column */
                const int64_t gap = i > j ? i - j : j - i;
                const bool rec = gap >= theiler && distance(y, i, j, m, tau, norm) <= e;
                if (rec) {
                    ++run;
                } else {
                    if (run > 0) h[run] += 1;
                    run = 0;
                }
            }
            if (run > 0) h[run] += 1;
        }
    }
    if (nt > 1)
        for (int t = 0; t < nt; ++t)
            for (size_t q = 0; q < (size_t)K * (size_t)Np; ++q) vhist[q] += priv[(size_t)t * K * Np + q];
    return ORACLE_OK;
}

/* Laminarity and trapping time from the vertical-line histogram (textbook definitions, Marwan et al. 2007 — the
 * paper's ref. [2], which PAPER.md:86 points to; not written out in the paper):
 *   LAM_k = sum_{v>=v_min} v*P_k(v) / sum_{v>=1} v*P_k(v),   TT_k = sum_{v>=v_min} v*P_k(v) / sum_{v>=v_min} P_k(v)
 * (0 where the denominator is empty).  Integer sums exact in uint64, one fp64 divide each. */
int rqa_oracle_lam_tt(const uint64_t* vhist, int K, int64_t n_points, int64_t v_min, double* lam, double* tt) {
    if (!vhist || !lam || !tt || K < 1 || n_points < 2 || v_min < 1) return ORACLE_BAD_ARG;
    for (int k = 0; k < K; ++k) {
        uint64_t all = 0, num = 0, lines = 0;
        for (int64_t v = 1; v < n_points; ++v) {
            const uint64_t h = vhist[(size_t)k * n_points + v];
            all += (uint64_t)v * h;
            if (v >= v_min) { num += (uint64_t)v * h; lines += h; }
        }
        lam[k] = all ? (double)num / (double)all : 0.0;
        tt[k] = lines ? (double)num / (double)lines : 0.0;
    }
    return ORACLE_OK;
}

/* DET_k = sum_{l>=l_min} l*P_k(l) / sum_{l>=1} l*P_k(l)  (Eq. 4, with readings S2/D3);
 * mean = (1/K) sum_k DET_k, summed k = 0..K-1 left to right (Eq. 5, reading S11).
 * Integer sums are exact in uint64; one fp64 divide per k.  An empty denominator gives DET = 0. */
int rqa_oracle_det_avg(const uint64_t* hist, int K, int64_t n_points, int64_t l_min, double* det,
                       double* det_mean) {
    if (!hist || !det || !det_mean || K < 1 || n_points < 2 || l_min < 1) return ORACLE_BAD_ARG;
    double sum = 0.0;
    for (int k = 0; k < K; ++k) {
        uint64_t num = 0, den = 0;
        for (int64_t l = 1; l < n_points; ++l) {
            uint64_t w = (uint64_t)l * hist[(size_t)k * n_points + l];
            den += w;
            if (l >= l_min) num += w;
        }
        det[k] = den ? (double)num / (double)den : 0.0;
        sum += det[k];
    }
    *det_mean = sum / (double)K;
    return ORACLE_OK;
}

/* Eq. 5 for every cut-off RR* (the paper evaluates RR* = 1..99): prefix[k] = (1/(k+1)) sum_{i<=k} DET_i,
 * summed left to right, in the order the rates were given.  prefix[0] = DET_0. */
int rqa_oracle_det_prefix_avg(const double* det, int K, double* prefix) {
    if (!det || !prefix || K < 1) return ORACLE_BAD_ARG;
    double sum = 0.0;
    for (int k = 0; k < K; ++k) {
        sum += det[k];
        prefix[k] = sum / (double)(k + 1);
    }
    return ORACLE_OK;
}

/* The other measures read off the histogram ("DET, L, L_max and RR"): average diagonal line length
 * L_k = sum_{l>=l_min} l*P_k(l) / sum_{l>=l_min} P_k(l) (0 without lines), longest line L_max, and the recurrence rate
 * sum_{l>=1} l*P_k(l) / P with P = N'(N'-1)/2 (reading S2: upper triangle, main diagonal excluded); and the Shannon
 * entropy of the line-length distribution, ENTR_k = -sum_{l>=l_min} p(l) ln p(l), p(l) = P_k(l) / sum_{l>=l_min} P_k(l)
 * (one of the "other RQA measures" of PAPER.md:86; the paper does not define it, this is the textbook definition). */
int rqa_oracle_line_measures(const uint64_t* hist, int K, int64_t n_points, int64_t l_min, double* L, uint64_t* Lmax,
                             double* rr_hist, double* entr, int64_t theiler) {
    if (!hist || !L || !Lmax || !rr_hist || !entr || K < 1 || n_points < 2 || l_min < 1 || theiler < 1 ||
        theiler > n_points - 1)
        return ORACLE_BAD_ARG;
    const double P = (double)pairs_with_window(n_points, theiler);
    for (int k = 0; k < K; ++k) {
        uint64_t pts = 0, lpts = 0, lines = 0, lmax = 0;
        for (int64_t l = 1; l < n_points; ++l) {
            const uint64_t h = hist[(size_t)k * n_points + l];
            pts += (uint64_t)l * h;
            if (l >= l_min) { lpts += (uint64_t)l * h; lines += h; }
            if (h) lmax = (uint64_t)l;
        }
        L[k] = lines ? (double)lpts / (double)lines : 0.0;
        Lmax[k] = lmax;
        rr_hist[k] = (double)pts / P;
        /* entropy of the line-length distribution, the definition written out: -sum p(l) ln p(l), l ascending */
        double e = 0.0;
        for (int64_t l = l_min; l < n_points && lines; ++l) {
            const uint64_t h = hist[(size_t)k * n_points + l];
            if (h) { const double pl = (double)h / (double)lines; e -= pl * std::log(pl); }
        }
        entr[k] = e;
    }
    return ORACLE_OK;
}

/* Sorting rate S (Eq. 6).  measure[i][j]: the measure of series j (series given in their natural
 * order, y = [1..n]) in realisation i.  x_j = place of series j when the n values are ordered ascending (equal values
 * keep their given order), z = y reversed.  S = (sum_i sum_j |z_j-y_j| - sum_i sum_j |x_j-y_j|) / sum_i sum_j |z_j-y_j|. */
int rqa_oracle_sorting_rate(const double* measure, int R, int n, double* S) {
    if (!measure || !S || R < 1 || n < 2) return ORACLE_BAD_ARG;
    std::vector<int> order(n), x(n);
    long long worst = 0, dep = 0;
    for (int i = 0; i < R; ++i) {
        const double* m = measure + (size_t)i * n;
        for (int j = 0; j < n; ++j) order[j] = j;
        std::stable_sort(order.begin(), order.end(), [m](int a, int b) { return m[a] < m[b]; });
        for (int place = 0; place < n; ++place) x[order[place]] = place + 1;
        for (int j = 0; j < n; ++j) {
            const int y = j + 1, z = n - j;
            worst += std::llabs((long long)z - y);
            dep += std::llabs((long long)x[j] - y);
        }
    }
    *S = (double)(worst - dep) / (double)worst;
    return ORACLE_OK;
}

}  // extern "C"
