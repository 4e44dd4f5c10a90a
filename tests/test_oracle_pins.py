"""Pins for the CPU oracle (oracle/rqa_oracle.cpp): everything here checks the oracle against something
other than itself — hand-enumerated recurrence plots, closed forms, library order statistics, invariants,
exact rational arithmetic, a statistical closed form.  CPU only (`-m "not gpu"`).

Citations are PAPER.md lines (= /root/reference/PAPER.md) and DESIGN.md readings S1..S18.
"""
import math
from fractions import Fraction
from pathlib import Path

import numpy as np
import pytest

from paper_2208_09136_b200 import workloads as wl

GOLDEN = Path(__file__).resolve().parent / "golden" / "hand_cases.txt"
NORMS = {"max": 0, "euclid": 1}


# ------------------------------------------------------------------------------------ hand enumeration
def _hand_cases():
    cases = []
    for line in GOLDEN.read_text().splitlines():
        if not line.strip() or line.startswith("#"):
            continue
        name, y, m, tau, norm, rr, eps, C, hist, det = [f.strip() for f in line.split("|")]
        e = np.float32(np.sqrt(np.float32(5.0))) if eps == "sqrt5" else np.float32(float(eps))
        h = {int(a): int(b) for a, b in (t.split(":") for t in hist.split(","))}
        num, den = det.split("/")
        cases.append(pytest.param(np.array(y.split(), dtype=np.float32), int(m), int(tau), NORMS[norm], float(rr),
                                  e, int(C), h, Fraction(int(num), int(den)), id=name))
    return cases


@pytest.mark.parametrize("y,m,tau,norm,rr,eps,C,hist,det", _hand_cases())
def test_hand_enumerated(oracle, y, m, tau, norm, rr, eps, C, hist, det):
    r = oracle.sweep(y, m, tau, [rr], norm, l_min=2)
    P = oracle.n_pairs(len(y), m, tau)
    assert r["eps"][0] == eps
    assert int(r["count"][0]) == C
    assert r["rr"][0] == C / P
    got = {int(l): int(c) for l, c in enumerate(r["hist"][0]) if c}
    assert got == hist
    assert abs(r["det"][0] - float(det)) <= 1e-15
    assert r["det_mean"] == r["det"][0]          # the average of one value is the value itself


# ------------------------------------------------------------------------------------------ rank (S5)
def test_rank_literal_fp64(oracle):
    assert oracle.rank(0.07, 100) == 8      # 0.07*100 = 7.000000000000001 -> ceil = 8 (wart kept, reading S5)
    assert oracle.rank(0.3, 10) == 3
    assert oracle.rank(0.1, 3) == 1
    assert oracle.rank(1e-12, 1000) == 1    # clamp below
    assert oracle.rank(1.0, 4753) == 4753   # clamp above
    P = 4999750003
    for rr in wl.rr_log(20, 0.001, 0.2):
        assert oracle.rank(rr, P) == math.ceil(rr * float(P))


# ------------------------------------------------------------------------------- embedding
@pytest.mark.parametrize("m,tau", [(1, 1), (3, 1), (4, 6), (5, 2)])
def test_embed_is_delay_view(oracle, m, tau):
    y = wl.gaussian(11, 64).astype(np.float32)
    X = oracle.embed(y, m, tau)
    ref = np.stack([y[c * tau: c * tau + len(y) - (m - 1) * tau] for c in range(m)], axis=1)
    assert X.shape == ref.shape and np.array_equal(X, ref)


# -------------------------------------------------------------- eps against a library order statistic
def _numpy_condensed(y, m, tau, norm):
    n = len(y) - (m - 1) * tau
    X = np.stack([y[c * tau: c * tau + n] for c in range(m)], axis=1).astype(np.float32)
    diff = X[:, None, :] - X[None, :, :]                       # fp32 subtraction, one rounding each
    if norm == 0:
        D = np.abs(diff).max(axis=2)
    else:
        sq = diff * diff
        s = sq[:, :, 0]
        for c in range(1, m):
            s = s + sq[:, :, c]                                 # fixed order c = 0..m-1, fp32 each step
        D = np.sqrt(s)
    iu = np.triu_indices(n, 1)
    return D[iu].astype(np.float32)


@pytest.mark.parametrize("norm", [0, 1])
@pytest.mark.parametrize("m,tau,N,seed", [(1, 1, 40, 1), (3, 1, 97, 2), (4, 6, 150, 3), (5, 2, 120, 4)])
def test_eps_matches_numpy_partition(oracle, m, tau, N, seed, norm):
    y = wl.gaussian(seed, N).astype(np.float32)
    rr = np.array([0.003, 0.01, 0.05, 0.1, 0.25, 0.5, 0.99, 1.0])
    eps, cnt, rrr = oracle.eps_for_rr(y, m, tau, rr, norm)
    d = _numpy_condensed(y, m, tau, norm)
    assert np.array_equal(np.sort(d), np.sort(oracle.distances(y, m, tau, norm)))
    P = len(d)
    for k, r_ in enumerate(rr):
        r = min(max(math.ceil(r_ * float(P)), 1), P)
        e = np.partition(d, r - 1)[r - 1]
        assert eps[k] == e
        assert int(cnt[k]) == int((d <= e).sum())
        assert rrr[k] == int(cnt[k]) / P


def test_eps_ties_and_duplicates(oracle):
    # quantised series -> massive ties; several targets share one eps (reading S6)
    y = (np.floor(wl.uniform01(5, 80) * 4)).astype(np.float32)
    rr = np.array([0.05, 0.2, 0.21, 0.5, 0.9])
    eps, cnt, _ = oracle.eps_for_rr(y, 2, 1, rr, 0)
    d = _numpy_condensed(y, 2, 1, 0)
    for k in range(len(rr)):
        r = math.ceil(rr[k] * len(d))
        assert eps[k] == np.sort(d)[r - 1]
        assert int(cnt[k]) == int((d <= eps[k]).sum()) >= r
    assert len(set(eps.tolist())) < len(rr)


# ------------------------------------------------------------------------------ counting certificate
@pytest.mark.parametrize("norm", [0, 1])
def test_certificate_brackets_rank(oracle, norm):
    y = wl.add_noise(wl.logistic_signal(300, 9), 1.0, 9)
    rr = wl.rr_log(12, 0.001, 0.3)
    eps, cnt, _ = oracle.eps_for_rr(y, 3, 1, rr, norm)
    P = oracle.n_pairs(len(y), 3, 1)
    lt, le = oracle.count_lt_le(y, 3, 1, eps, norm, threads=2)
    for k in range(len(rr)):
        r = oracle.rank(rr[k], P)
        assert int(lt[k]) < r <= int(le[k])
        assert int(le[k]) == int(cnt[k])
    # a value that is not the order statistic must fail the certificate
    lt2, le2 = oracle.count_lt_le(y, 3, 1, np.nextafter(eps, np.float32(np.inf)), norm, threads=1)
    assert all(int(lt2[k]) >= oracle.rank(rr[k], P) for k in range(len(rr)))


# ------------------------------------------------------------------------------------- closed forms
@pytest.mark.parametrize("m,tau,N", [(1, 1, 50), (3, 2, 61), (4, 6, 120)])
def test_ramp_closed_form(oracle, m, tau, N):
    """y_i = i: d_ij = j - i for any (m, tau) under the max norm, so the sorted distances are (N'-1) ones,
    (N'-2) twos, ...; eps_k = smallest o* with sum_{o<=o*}(N'-o) >= r_k; P_k(l) = 1 for l = N'-o*..N'-1."""
    y = np.arange(N, dtype=np.float32)
    n = N - (m - 1) * tau
    P = n * (n - 1) // 2
    rr = np.array([0.01, 0.1, 0.33, 0.5, 0.77, 1.0])
    r = oracle.sweep(y, m, tau, rr, 0)
    for k, q in enumerate(rr):
        rank = min(max(math.ceil(q * float(P)), 1), P)
        cum, ostar = 0, 0
        while cum < rank:
            ostar += 1
            cum += n - ostar
        assert r["eps"][k] == np.float32(ostar)
        assert int(r["count"][k]) == cum
        exp = np.zeros(n, dtype=np.uint64)
        exp[n - ostar: n] = 1
        assert np.array_equal(r["hist"][k], exp)


def test_constant_series(oracle):
    y = np.full(30, 2.5, dtype=np.float32)
    r = oracle.sweep(y, 2, 3, [0.001, 0.5, 1.0], 0)
    n = 27
    assert np.all(r["eps"] == 0) and np.all(r["count"] == n * (n - 1) // 2)
    exp = np.ones(n, dtype=np.uint64)
    exp[0] = 0
    for k in range(3):
        assert np.array_equal(r["hist"][k], exp)      # one line per diagonal, lengths 1..N'-1


def test_exactly_periodic_series(oracle):
    """y_n = T[n mod q] with distinct table values: at eps = 0 a cell recurs iff o = 0 (mod q), so every
    diagonal is all-or-nothing and P(N' - q t) = 1.  (The config-2 SNR=inf structure.)"""
    T = np.array([0.0, 3.0, 1.0, 7.0, 4.0, 9.0, 2.0], dtype=np.float32)
    q, N, m, tau = len(T), 100, 3, 2
    y = T[np.arange(N) % q]
    n = N - (m - 1) * tau
    P = n * (n - 1) // 2
    c0 = sum(n - q * t for t in range(1, n) if q * t < n)
    rr_in = (c0 - 0.5) / P            # rank <= c0 -> eps = 0
    rr_out = (c0 + 0.5) / P           # first rank beyond the zeros -> eps > 0
    r = oracle.sweep(y, m, tau, [rr_in, rr_out], 0)
    assert r["eps"][0] == 0 and int(r["count"][0]) == c0
    exp = np.zeros(n, dtype=np.uint64)
    for t in range(1, n):
        if q * t < n:
            exp[n - q * t] = 1
    assert np.array_equal(r["hist"][0], exp)
    assert r["det"][0] == 1.0
    assert r["eps"][1] > 0


def test_config2_sine_snr_inf_closed_form(oracle):
    """SURVEY.md sec. 8(d), config 2 at SNR = inf: 39 fully recurrent diagonals o = 25..975, 18 798 zero
    distances; targets 0.01-0.03 give eps = 0, C = 18 798, DET = 1; 0.04 is the first with eps > 0."""
    w = wl.config2()
    y = w.series[0]
    r = oracle.sweep(y, w.m, w.tau, w.rr, w.norm)
    assert w.n_points == 982 and w.n_pairs == 481671
    for k in range(3):
        assert r["eps"][k] == 0 and int(r["count"][k]) == 18798 and r["det"][k] == 1.0
        nz = np.nonzero(r["hist"][k])[0]
        assert sorted(nz.tolist()) == sorted(982 - 25 * t for t in range(1, 40))
        assert np.all(r["hist"][k][nz] == 1)
    assert r["eps"][3] > 0 and oracle.rank(w.rr[3], w.n_pairs) == 19267


# ---------------------------------------------------------------------------------------- invariants
@pytest.mark.parametrize("norm", [0, 1])
@pytest.mark.parametrize("maker", ["noise", "logistic", "sine"])
def test_invariants_sum_nesting_symmetry(oracle, maker, norm):
    N, m, tau = 260, 3, 2
    if maker == "noise":
        y = wl.gaussian(21, N).astype(np.float32)
    elif maker == "logistic":
        y = wl.add_noise(wl.logistic_signal(N, 22), 3.0, 22)
    else:
        y = wl.add_noise(wl.sine_signal(N), 1.0, 23)
    rr = wl.rr_log(9, 0.002, 0.4)
    r = oracle.sweep(y, m, tau, rr, norm)
    n = N - (m - 1) * tau
    l = np.arange(n, dtype=np.uint64)
    hist = r["hist"]
    # sum_l l P_k(l) = C_k  ("RR can also be calculated from the histogram")
    assert np.array_equal((hist * l).sum(axis=1), r["count"])
    assert np.all(hist[:, 0] == 0)
    # nesting: eps ascending -> C_k non-decreasing, sum_{l>=L} l P_k(l) non-decreasing in k for every L
    assert np.all(np.diff(r["eps"]) >= 0) and np.all(np.diff(r["count"].astype(np.int64)) >= 0)
    tail = np.cumsum((hist * l)[:, ::-1], axis=1)[:, ::-1].astype(np.int64)
    assert np.all(np.diff(tail, axis=0) >= 0)
    # symmetry: the lower triangle gives the identical histogram
    assert np.array_equal(oracle.line_hist(y, m, tau, r["eps"], norm, lower=True), hist)
    # the OpenMP split over diagonals changes nothing
    assert np.array_equal(oracle.line_hist(y, m, tau, r["eps"], norm, threads=3), hist)


def test_line_hist_brute_force_tiny(oracle):
    """Independent run count on the explicit 0/1 matrix built with numpy (np.diagonal + split on zeros)."""
    for seed in range(6):
        N, m, tau = 24 + seed, 2, 1 + seed % 3
        y = np.round(wl.gaussian(100 + seed, N) * 2).astype(np.float32)
        n = N - (m - 1) * tau
        eps = np.array([0.0, 1.0, 2.5], dtype=np.float32)
        X = np.stack([y[c * tau: c * tau + n] for c in range(m)], axis=1)
        D = np.abs(X[:, None, :] - X[None, :, :]).max(axis=2)
        hist = oracle.line_hist(y, m, tau, eps, 0)
        for k, e in enumerate(eps):
            R = (D <= e).astype(np.int8)
            exp = np.zeros(n, dtype=np.uint64)
            for o in range(1, n):
                s = "".join(map(str, np.diagonal(R, o)))
                for run in s.split("0"):
                    if run:
                        exp[len(run)] += 1
            assert np.array_equal(hist[k], exp)


# ----------------------------------------------------------------------- statistical closed form (m = 1)
def test_iid_uniform_det_closed_form(oracle):
    """i.i.d. U(0,1), m = 1, max norm: a cell recurs with p = 2 eps - eps^2 and neighbouring cells on a
    diagonal are independent, so a recurrent cell is isolated with probability (1-p)^2 and
    DET (l_min = 2) ~ 1 - (1-p)^2.  Band: 3*(2 sigma_b) + 2/N', sigma_b binomial."""
    N = 2000
    for seed in (31, 32):
        y = wl.uniform01(seed, N).astype(np.float32)
        rr = np.array([0.05, 0.1, 0.2])
        r = oracle.sweep(y, 1, 1, rr, 0)
        for k in range(3):
            e = float(r["eps"][k])
            p = 2 * e - e * e
            assert abs(p - rr[k]) < 0.01                 # eps really is the rr-quantile of |U1-U2|
            q = (1 - p) ** 2
            sigma_b = math.sqrt(q * (1 - q) / float(r["count"][k]))
            assert abs(r["det"][k] - (1 - q)) <= 3 * (2 * sigma_b) + 2.0 / N


# ------------------------------------------------------------------- Euclid: exact rational re-evaluation
def _round_f32(x: Fraction) -> Fraction:
    """Round an exact rational to the nearest binary32 value (ties to even), subnormals included."""
    if x == 0:
        return Fraction(0)
    s = -1 if x < 0 else 1
    a = abs(x)
    e = math.floor(math.log2(a)) if a >= 1 else -math.ceil(math.log2(1 / a))
    while Fraction(2) ** e > a:
        e -= 1
    while Fraction(2) ** (e + 1) <= a:
        e += 1
    q = max(e - 23, -149)                                  # exponent of the last place
    scaled = a / (Fraction(2) ** q)
    n = scaled.numerator // scaled.denominator
    rem = scaled - n
    if rem > Fraction(1, 2) or (rem == Fraction(1, 2) and n % 2 == 1):
        n += 1
    return s * n * (Fraction(2) ** q)


def test_euclid_chain_is_exactly_rounded_fp32(oracle):
    rng_vals = wl.gaussian(77, 400)
    scales = [1.0, 1e-3, 1e-19, 3e-23, 1e10]               # 1e-19..3e-23: squares fall into the subnormals
    m, tau = 3, 2
    for sc in scales:
        y = (rng_vals[:40] * sc).astype(np.float32)
        got = oracle.distances(y, m, tau, 1)
        n = len(y) - (m - 1) * tau
        p = 0
        for i in range(n):
            for j in range(i + 1, n):
                s = None
                for c in range(m):
                    t = _round_f32(Fraction(float(y[i + c * tau])) - Fraction(float(y[j + c * tau])))
                    sq = _round_f32(t * t)
                    s = sq if s is None else _round_f32(s + sq)
                # correctly rounded sqrt of an fp32 value: fp64 sqrt then one rounding is safe (53 >= 2*24+2)
                exp = np.float32(math.sqrt(float(s)))
                assert got[p] == exp, (sc, i, j)
                p += 1


def test_max_norm_is_exact(oracle):
    y = (wl.gaussian(78, 60) * 1e-20).astype(np.float32)
    got = oracle.distances(y, 2, 3, 0)
    n = len(y) - 3
    p = 0
    for i in range(n):
        for j in range(i + 1, n):
            e = max(_round_f32(abs(Fraction(float(y[i + c * 3])) - Fraction(float(y[j + c * 3])))) for c in range(2))
            assert Fraction(float(got[p])) == e
            p += 1


# ------------------------------------------------------------------------------------- DET and mean
def test_det_avg_integer_recompute(oracle):
    y = wl.add_noise(wl.lorenz_signal(400), 1.0, 41)
    rr = wl.rr_log(7, 0.005, 0.3)
    r = oracle.sweep(y, 3, 3, rr, 0)
    hist = r["hist"]
    n = hist.shape[1]
    for l_min in (1, 2, 3, 10, n - 1, n, n + 5):
        det, mean = oracle.det_avg(hist, l_min)
        acc = 0.0
        for k in range(len(rr)):
            num = sum(l * int(hist[k, l]) for l in range(max(l_min, 1), n))
            den = sum(l * int(hist[k, l]) for l in range(1, n))
            assert abs(det[k] - float(Fraction(num, den))) <= 1e-15
            acc += det[k]
        assert abs(mean - acc / len(rr)) <= 1e-15
        if l_min == 1:
            assert np.all(det == 1.0)
        if l_min >= n:
            assert np.all(det == 0.0)                      # reading S12


def test_det_avg_empty_denominator(oracle):
    hist = np.zeros((2, 10), dtype=np.uint64)
    hist[1, 3] = 2
    det, mean = oracle.det_avg(hist, 2)
    assert det[0] == 0.0 and det[1] == 1.0 and mean == 0.5


# ----------------------------------------------------------------------------------------- workloads
def test_workloads_are_seeded_and_shaped():
    a, b = wl.config1(), wl.config1()
    assert np.array_equal(a.series, b.series) and a.series.dtype == np.float32
    assert (a.batch, a.N, a.n_points, a.n_pairs, a.K) == (4, 100, 98, 4753, 10)
    c2 = wl.config2()
    assert (c2.batch, c2.N, c2.n_points, c2.n_pairs) == (5, 1000, 982, 481671)
    assert np.allclose(wl.rr_log(20, 0.001, 0.2)[[0, -1]], [0.001, 0.2])
    assert wl.rr_linear(10)[6] == 0.07
    g = wl.gaussian(1, 200001)
    assert abs(g.mean()) < 0.01 and abs(g.std() - 1) < 0.01
    assert np.array_equal(wl.splitmix64(3, 5, offset=2), wl.splitmix64(3, 7)[2:])
    y = wl.logistic_signal(500, 7)
    assert y.min() > 0 and y.max() < 1
    assert wl.fnv1a64(np.zeros(0, dtype=np.uint8)) == 0xCBF29CE484222325


# ---------------------------------------------------------------- rows f1/f2: Eq. 5 curve, L / L_max / RR, Eq. 6
def test_det_prefix_avg_pins(oracle):
    """Eq. 5 for every cut-off: the average of one value is the value itself, a hand
    example, the last entry is the plain mean, and exact rational arithmetic on random input."""
    assert oracle.det_prefix_avg([0.625]).tolist() == [0.625]
    assert oracle.det_prefix_avg([0.5, 1.0, 0.0]).tolist() == [0.5, 0.75, 0.5]
    rng = np.random.default_rng(5)
    det = rng.random(99)
    got = oracle.det_prefix_avg(det)
    acc = Fraction(0)
    for k in range(99):
        acc += Fraction(float(det[k]))
        assert abs(Fraction(float(got[k])) - acc / (k + 1)) < Fraction(1, 10**13)
    hist = np.zeros((3, 12), dtype=np.uint64)
    hist[0, 1], hist[0, 3] = 4, 1
    hist[1, 2], hist[1, 5] = 2, 1
    hist[2, 1] = 7
    d, mean = oracle.det_avg(hist, 2)
    assert oracle.det_prefix_avg(d)[-1] == pytest.approx(mean, abs=1e-15)


def test_line_measures_hand_cases(oracle):
    """L, L_max and RR from the histogram on two hand-enumerated recurrence plots of SURVEY.md 8c:
    A (y=0,1,0,1,0,1, m=1, rr=0.4): P(2)=P(4)=1 -> L=3, L_max=4, RR=6/15.
    E (y=0,2,1,4,0,2,1,4,3, m=2, tau=2, rr=0.5): P(1)=5,P(2)=2,P(3)=1,P(5)=1 -> L=(4+3+5)/4=3, L_max=5, RR=17/21."""
    r = oracle.sweep(np.array([0, 1, 0, 1, 0, 1], dtype=np.float32), 1, 1, [0.4], oracle.NORM_MAX, 2)
    L, Lmax, rr, entr = oracle.line_measures(r["hist"], 2)
    assert (L[0], int(Lmax[0]), rr[0]) == (3.0, 4, 6 / 15)
    assert entr[0] == pytest.approx(math.log(2.0), abs=1e-15)          # two lines of different length: p = 1/2, 1/2
    r = oracle.sweep(np.array([0, 2, 1, 4, 0, 2, 1, 4, 3], dtype=np.float32), 2, 2, [0.5], oracle.NORM_MAX, 2)
    L, Lmax, rr, entr = oracle.line_measures(r["hist"], 2)
    assert (L[0], int(Lmax[0]), rr[0]) == (3.0, 5, 17 / 21)
    assert entr[0] == pytest.approx(1.5 * math.log(2.0), abs=1e-15)    # p = 1/2, 1/4, 1/4
    assert rr[0] == r["rr"][0]                       # "RR can also be calculated from the histogram"
    L1, _, _, e1 = oracle.line_measures(r["hist"], 1)    # l_min = 1: all 9 lines, 17 points
    assert L1[0] == 17 / 9
    p = np.array([5, 2, 1, 1]) / 9.0
    assert e1[0] == pytest.approx(float(-(p * np.log(p)).sum()), abs=1e-15)
    empty = np.zeros((1, 7), dtype=np.uint64)
    L, Lmax, rr, entr = oracle.line_measures(empty, 2)
    assert (L[0], int(Lmax[0]), rr[0], entr[0]) == (0.0, 0, 0.0, 0.0)
    single = np.zeros((1, 7), dtype=np.uint64)
    single[0, 3] = 11                                 # one line length only: no uncertainty
    assert oracle.line_measures(single, 2)[3][0] == 0.0


def test_sorting_rate_pins(oracle):
    """Eq. 6: the worst case sums to 500 for 10 series x 10 realisations, so the
    reversed order gives S = 0 and the natural order S = 1; one adjacent swap per realisation costs 2 of 50; and an
    independent rank computation (numpy argsort) on every permutation of 4 series."""
    import itertools
    up = np.tile(np.arange(10, dtype=np.float64), (10, 1))
    assert oracle.sorting_rate(up) == 1.0
    assert oracle.sorting_rate(up[:, ::-1]) == 0.0
    assert sum(abs(11 - 2 * j) for j in range(1, 11)) * 10 == 500
    sw = up.copy()
    sw[:, [0, 1]] = sw[:, [1, 0]]
    assert oracle.sorting_rate(sw) == pytest.approx((500 - 20) / 500, abs=1e-15)
    half = up.copy()
    half[5:] = half[5:, ::-1]                        # five realisations sorted, five reversed
    assert oracle.sorting_rate(half) == 0.5
    for perm in itertools.permutations(range(4)):
        m = np.array([perm], dtype=np.float64)
        x = np.empty(4, dtype=int)
        x[np.argsort(m[0], kind="stable")] = np.arange(1, 5)
        dep = int(np.abs(x - np.arange(1, 5)).sum())
        assert oracle.sorting_rate(m) == pytest.approx((8 - dep) / 8, abs=1e-15)
    ties = np.array([[1.0, 1.0, 1.0]])               # equal values keep their given order: perfectly "sorted"
    assert oracle.sorting_rate(ties) == 1.0


@pytest.mark.parametrize("w", [1, 2, 7, 58])
def test_theiler_window_brute_force(oracle, w):
    """Theiler window (row f3; the paper uses none, reading S9): only pairs with j - i >= w.  An independent numpy
    brute force on the full distance matrix: the order statistic over the selected pairs, and the run lengths along
    the diagonals w..N'-1.  w = 1 is the default path; w = N'-1 leaves the single pair (0, N'-1)."""
    y = wl.add_noise(wl.sine_signal(64, 9), 1.5, 31)
    m, tau = 2, 3
    n = len(y) - (m - 1) * tau
    if w == 58:
        w = n - 1
    X = np.stack([y[c * tau:c * tau + n] for c in range(m)], axis=1)
    D = np.abs(X[:, None, :] - X[None, :, :]).max(axis=2).astype(np.float32)
    sel = np.sort(np.concatenate([np.diagonal(D, o) for o in range(w, n)]))
    P = len(sel)
    assert P == (n - w) * (n - w + 1) // 2
    rr = np.array([0.05, 0.3, 1.0])
    eps, cnt, rrr = oracle.eps_for_rr(y, m, tau, rr, oracle.NORM_MAX, theiler=w)
    for k in range(3):
        r = min(P, max(1, math.ceil(rr[k] * P)))
        assert eps[k] == sel[r - 1] and cnt[k] == int((sel <= eps[k]).sum()) and rrr[k] == cnt[k] / P
    hist = oracle.line_hist(y, m, tau, eps, oracle.NORM_MAX, theiler=w)
    want = np.zeros_like(hist)
    for k in range(3):
        for o in range(w, n):
            run = 0
            for v in np.append(np.diagonal(D, o) <= eps[k], False):
                if v:
                    run += 1
                elif run:
                    want[k, run] += 1
                    run = 0
    assert np.array_equal(hist, want)
    assert np.array_equal((hist * np.arange(n, dtype=np.uint64)).sum(axis=1), cnt)
    assert np.array_equal(oracle.line_measures(hist, 2, theiler=w)[2], rrr)      # RR from the histogram, over P_w
    if w == 1:
        assert np.array_equal(hist, oracle.line_hist(y, m, tau, eps, oracle.NORM_MAX))


def test_certificate_with_theiler_window(oracle):
    """count_lt_le over the pairs with j - i >= w brackets the rank of the windowed order statistic, and agrees with a
    numpy count on the full distance matrix."""
    y = np.round(wl.gaussian(321, 150) * 5).astype(np.float32) / 5
    for w in (1, 2, 9, 140):
        rr = [0.05, 0.3, 0.9]
        eps, cnt, _ = oracle.eps_for_rr(y, 2, 3, rr, 0, theiler=w)
        lt, le = oracle.count_lt_le(y, 2, 3, eps, 0, threads=2, theiler=w)
        n = len(y) - 3
        Pw = (n - w) * (n - w + 1) // 2
        D = _numpy_condensed_full(y, 2, 3, 0)
        i, j = np.indices(D.shape)
        sel = (j - i) >= w
        for k in range(3):
            r = oracle.rank(rr[k], Pw)
            assert lt[k] < r <= le[k] and le[k] == cnt[k]
            assert lt[k] == int((D[sel] < eps[k]).sum()) and le[k] == int((D[sel] <= eps[k]).sum())


# ------------------------------------------------------------------ vertical lines (reading S19; LAM, TT)
VGOLDEN = Path(__file__).resolve().parent / "golden" / "hand_cases_vertical.txt"


def _vertical_cases():
    cases = []
    for line in VGOLDEN.read_text().splitlines():
        if not line.strip() or line.startswith("#"):
            continue
        name, y, m, tau, norm, eps, w, hist, lam, tt = [f.strip() for f in line.split("|")]
        h = {int(a): int(b) for a, b in (t.split(":") for t in hist.split(","))}
        cases.append(pytest.param(np.array(y.split(), dtype=np.float32), int(m), int(tau), NORMS[norm], np.float32(float(eps)),
                                  int(w), h, Fraction(*map(int, lam.split("/"))), Fraction(*map(int, tt.split("/"))), id=name))
    return cases


@pytest.mark.parametrize("y,m,tau,norm,eps,w,hist,lam,tt", _vertical_cases())
def test_vertical_hand_enumerated(oracle, y, m, tau, norm, eps, w, hist, lam, tt):
    vh = oracle.vert_hist(y, m, tau, [eps], norm, theiler=w)
    got = {int(v): int(c) for v, c in enumerate(vh[0]) if c}
    assert got == hist
    L, T = oracle.lam_tt(vh, 2)
    assert abs(L[0] - float(lam)) <= 1e-15 and abs(T[0] - float(tt)) <= 1e-15


def _numpy_vertical(y, m, tau, norm, eps, w):
    """Independent run count on the FULL matrix: every column as a string of 0/1 split at the zeros."""
    D = _numpy_condensed_full(y, m, tau, norm)
    n = D.shape[0]
    i, j = np.indices((n, n))
    R = (D <= eps) & (np.abs(i - j) >= w)
    h = np.zeros(n, dtype=np.uint64)
    for col in range(n):
        for run in "".join("1" if x else "0" for x in R[:, col]).split("0"):
            if run:
                h[len(run)] += 1
    return h


def _numpy_condensed_full(y, m, tau, norm):
    n = len(y) - (m - 1) * tau
    X = np.stack([y[c * tau: c * tau + n] for c in range(m)], axis=1).astype(np.float32)
    diff = X[:, None, :] - X[None, :, :]
    if norm == 0:
        return np.abs(diff).max(axis=2)
    sq = diff * diff
    s = sq[:, :, 0]
    for c in range(1, m):
        s = s + sq[:, :, c]
    return np.sqrt(s)


@pytest.mark.parametrize("m,tau,N,w,norm", [(1, 1, 60, 1, 0), (3, 1, 90, 1, 0), (2, 3, 77, 4, 0), (3, 2, 64, 1, 1), (4, 1, 50, 46, 0)])
def test_vertical_brute_force_full_matrix(oracle, m, tau, N, w, norm):
    y = np.round(wl.gaussian(500 + N, N) * 4).astype(np.float32) / 4       # quantised: ties and long runs
    eps = np.array([0.0, 0.5, 1.25, 3.0], dtype=np.float32)
    vh = oracle.vert_hist(y, m, tau, eps, norm, theiler=w)
    for k, e in enumerate(eps):
        assert np.array_equal(vh[k], _numpy_vertical(y, m, tau, norm, e, w))
    # threads change nothing
    assert np.array_equal(vh, oracle.vert_hist(y, m, tau, eps, norm, threads=0, theiler=w))


def test_vertical_sum_is_twice_the_pair_count_and_ramp_closed_form(oracle):
    # every recurrent pair (i<j) is one cell of column j and one of column i: sum_v v*P(v) = 2*C  (symmetry)
    y = wl.logistic_signal(400, seed=77).astype(np.float32)
    r = oracle.sweep(y, 3, 1, wl.rr_linear(10), 0, 2)
    vh = oracle.vert_hist(y, 3, 1, r["eps"], 0)
    v = np.arange(vh.shape[1], dtype=np.uint64)
    assert np.array_equal((vh * v).sum(axis=1), 2 * r["count"])
    # ramp y_i = i, max norm, eps = q: column j has a run of min(j, q) cells above the diagonal and min(n-1-j, q) below
    n, q = 57, 5
    ramp = np.arange(n, dtype=np.float32)
    vh = oracle.vert_hist(ramp, 1, 1, np.array([q], dtype=np.float32), 0)[0]
    expect = np.zeros(n, dtype=np.uint64)
    for j in range(n):
        for run in (min(j, q), min(n - 1 - j, q)):
            if run:
                expect[run] += 1
    assert np.array_equal(vh, expect)
