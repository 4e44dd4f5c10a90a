"""Seeded synthetic workloads shaped like the paper's (sec. 4) and BASELINE.json's configs.

This module holds NONE of the method's arithmetic (no distances, thresholds, histograms): it only
produces input series and recurrence-rate lists.  It is the one module that both the CUDA path's callers
(tests, bench.py) and the oracle's callers use, so both sides see bit-identical fp32 inputs and the same
fp64 RR array (reading S5: the RR list is generated once, here).

No public dataset or benchmark suite is involved: every series is generated from the formulas below.

Random numbers: a counter-based SplitMix64 stream (value i of stream `seed` depends only on (seed, i)),
uniform = ((x >> 11) + 0.5) * 2**-53, Gaussian = Box-Muller written out (both outputs used).

Seeds: seed = 220809136 + 100000*config + 1000*signal + 10*snr_index + realisation,
signal: 0 sine, 1 logistic, 2 Lorenz, 3 white noise.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from functools import lru_cache

import numpy as np

SEED_BASE = 220809136
SIG_SINE, SIG_LOGISTIC, SIG_LORENZ, SIG_NOISE = 0, 1, 2, 3
SIGNAL_NAMES = {SIG_SINE: "sine", SIG_LOGISTIC: "logistic", SIG_LORENZ: "lorenz", SIG_NOISE: "noise"}
NORM_MAX, NORM_EUCLID = 0, 1

_M64 = (1 << 64) - 1


def make_seed(config: int, signal: int, snr_index: int, realisation: int = 0) -> int:
    return SEED_BASE + 100000 * config + 1000 * signal + 10 * snr_index + realisation


# ----------------------------------------------------------------------------------------------- RNG
def splitmix64(seed: int, n: int, offset: int = 0) -> np.ndarray:
    """n outputs of the counter-based SplitMix64 stream `seed`, starting at counter `offset`."""
    idx = np.arange(offset + 1, offset + n + 1, dtype=np.uint64)
    with np.errstate(over="ignore"):
        z = np.uint64(seed & _M64) + idx * np.uint64(0x9E3779B97F4A7C15)
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        z = z ^ (z >> np.uint64(31))
    return z


def uniform01(seed: int, n: int, offset: int = 0) -> np.ndarray:
    """n uniforms in the open interval (0, 1), fp64."""
    z = splitmix64(seed, n, offset)
    return ((z >> np.uint64(11)).astype(np.float64) + 0.5) * (2.0 ** -53)


def gaussian(seed: int, n: int) -> np.ndarray:
    """n standard normal deviates (Box-Muller, both outputs used), fp64."""
    h = (n + 1) // 2
    u = uniform01(seed, 2 * h)
    r = np.sqrt(-2.0 * np.log(u[0::2]))
    a = 2.0 * math.pi * u[1::2]
    out = np.empty(2 * h, dtype=np.float64)
    out[0::2] = r * np.cos(a)
    out[1::2] = r * np.sin(a)
    return out[:n]


# ------------------------------------------------------------------------------------- clean signals
def sine_signal(N: int, period: int = 25) -> np.ndarray:
    """sin(2*pi*(n mod period)/period): exactly `period`-periodic (PAPER.md:103-105 shape; BASELINE config 2)."""
    n = np.arange(N, dtype=np.int64) % period
    return np.sin(2.0 * math.pi * n.astype(np.float64) / period)


def logistic_signal(N: int, seed: int, r: float = 4.0, transient: int = 1000) -> np.ndarray:
    """x <- r x (1-x), x0 = 0.1 + 0.8 u(seed), `transient` steps dropped (r=4 per BASELINE)."""
    x = 0.1 + 0.8 * float(uniform01(seed ^ 0x5851F42D4C957F2D, 1)[0])
    for _ in range(transient):
        x = r * x * (1.0 - x)
    out = np.empty(N, dtype=np.float64)
    for n in range(N):
        out[n] = x
        x = r * x * (1.0 - x)
    return out


@lru_cache(maxsize=16)
def _lorenz_x(N: int, start: tuple, transient: int, every: int, dt: float) -> np.ndarray:
    s, rho, b = 10.0, 28.0, 8.0 / 3.0
    x, y, z = start
    out = np.empty(N, dtype=np.float64)
    h2, h6 = 0.5 * dt, dt / 6.0
    total = transient + N * every
    k = 0
    for step in range(total):
        if step >= transient and (step - transient) % every == 0:
            out[k] = x
            k += 1
        ax, ay, az = s * (y - x), x * (rho - z) - y, x * y - b * z
        x2, y2, z2 = x + h2 * ax, y + h2 * ay, z + h2 * az
        bx, by, bz = s * (y2 - x2), x2 * (rho - z2) - y2, x2 * y2 - b * z2
        x3, y3, z3 = x + h2 * bx, y + h2 * by, z + h2 * bz
        cx, cy, cz = s * (y3 - x3), x3 * (rho - z3) - y3, x3 * y3 - b * z3
        x4, y4, z4 = x + dt * cx, y + dt * cy, z + dt * cz
        dx, dy, dz = s * (y4 - x4), x4 * (rho - z4) - y4, x4 * y4 - b * z4
        x += h6 * (ax + 2.0 * bx + 2.0 * cx + dx)
        y += h6 * (ay + 2.0 * by + 2.0 * cy + dy)
        z += h6 * (az + 2.0 * bz + 2.0 * cz + dz)
    out.setflags(write=False)
    return out


def lorenz_signal(N: int, start=(1.0, 1.0, 1.0), transient: int = 10000, every: int = 5, dt: float = 0.01,
                  zscore: bool = True) -> np.ndarray:
    """Lorenz (sigma=10, rho=28, beta=8/3), classical RK4, x-component every `every`-th step after
    `transient` steps, z-scored (BASELINE config 3)."""
    x = np.array(_lorenz_x(int(N), tuple(float(v) for v in start), int(transient), int(every), float(dt)))
    if zscore:
        x = (x - x.mean()) / x.std()
    return x


def add_noise(clean: np.ndarray, snr: float, seed: int) -> np.ndarray:
    """clean + N(0, (sigma_signal/SNR)^2), sigma_signal = population std of the clean fp64 series; cast to
    fp32 once.  snr = inf adds nothing.  (BASELINE config 1 states sigma_noise = sigma_signal / SNR.)"""
    if math.isinf(snr):
        return clean.astype(np.float32)
    sigma = float(np.std(clean)) / snr
    return (clean + sigma * gaussian(seed, len(clean))).astype(np.float32)


# -------------------------------------------------------------------------------------------- RR lists
def rr_linear(K: int = 10, step: float = 0.01) -> np.ndarray:
    """k/100.0 for k = 1..K when step = 0.01 (fp64)."""
    return np.array([k / round(1.0 / step) for k in range(1, K + 1)], dtype=np.float64)


def rr_log(K: int, lo: float, hi: float) -> np.ndarray:
    """lo * (hi/lo)**(k/(K-1)), k = 0..K-1 (fp64)."""
    return np.array([lo * math.pow(hi / lo, k / (K - 1.0)) for k in range(K)], dtype=np.float64)


# --------------------------------------------------------------------------------------------- configs
@dataclass
class Workload:
    """One call of the hot path: a batch of equally long series sharing (m, tau, norm, rr, l_min)."""
    name: str
    series: np.ndarray            # float32 [batch][N]
    m: int
    tau: int
    norm: int
    rr: np.ndarray                # float64 [K]
    l_min: tuple = (2,)
    labels: list = field(default_factory=list)   # one dict per series: signal, snr, seed

    @property
    def batch(self) -> int:
        return self.series.shape[0]

    @property
    def N(self) -> int:
        return self.series.shape[1]

    @property
    def n_points(self) -> int:
        return self.N - (self.m - 1) * self.tau

    @property
    def n_pairs(self) -> int:
        n = self.n_points
        return n * (n - 1) // 2

    @property
    def K(self) -> int:
        return len(self.rr)

    @property
    def units(self) -> int:
        """recurrence cells x thresholds over the whole batch (BASELINE.json metric's numerator)."""
        return self.batch * self.n_pairs * self.K


def _label(signal, snr, seed):
    return {"signal": SIGNAL_NAMES[signal], "snr": snr, "seed": seed}


def config1(N: int = 100) -> Workload:
    """Logistic r=4, N=100, SNR in {inf, 10, 1, 0.1}; m=3, tau=1, max; K=10 linear."""
    snrs = [math.inf, 10.0, 1.0, 0.1]
    rows, labels = [], []
    for si, snr in enumerate(snrs):
        seed = make_seed(1, SIG_LOGISTIC, si)
        rows.append(add_noise(logistic_signal(N, seed), snr, seed))
        labels.append(_label(SIG_LOGISTIC, snr, seed))
    return Workload("config1_logistic_N100", np.stack(rows), 3, 1, NORM_MAX, rr_linear(10), (2,), labels)


def config2(N: int = 1000) -> Workload:
    """sin(2 pi n/25), N=1000, SNR in {inf, 3, 1, 0.3, 0.1}; m=4, tau=6, max; K=10 linear; batch of 5."""
    snrs = [math.inf, 3.0, 1.0, 0.3, 0.1]
    rows, labels = [], []
    clean = sine_signal(N)
    for si, snr in enumerate(snrs):
        seed = make_seed(2, SIG_SINE, si)
        rows.append(add_noise(clean, snr, seed))
        labels.append(_label(SIG_SINE, snr, seed))
    return Workload("config2_sine_N1000", np.stack(rows), 4, 6, NORM_MAX, rr_linear(10), (2,), labels)


def config3(norm: int = NORM_MAX, N: int = 10000) -> Workload:
    """Lorenz x, N=1e4, z-scored, SNR in {inf, 3, 1, 0.3, 0.1, 0.03}; m=3, tau=3; max or Euclid; K=20 log."""
    snrs = [math.inf, 3.0, 1.0, 0.3, 0.1, 0.03]
    rows, labels = [], []
    clean = lorenz_signal(N)
    for si, snr in enumerate(snrs):
        seed = make_seed(3, SIG_LORENZ, si)
        rows.append(add_noise(clean, snr, seed))
        labels.append(_label(SIG_LORENZ, snr, seed))
    nm = "max" if norm == NORM_MAX else "euclid"
    return Workload(f"config3_lorenz_N{N}_{nm}", np.stack(rows), 3, 3, norm, rr_log(20, 0.001, 0.2), (2,), labels)


def config4(N: int = 100000, which=None, realisation: int = 0) -> Workload:
    """Headline: N=1e5 logistic and Lorenz x at SNR in {1, 0.1}, plus white noise; m=3, tau=1, max; K=20 log.
    `which` selects a subset of the five series by index (0 logistic/1, 1 logistic/0.1, 2 lorenz/1,
    3 lorenz/0.1, 4 white noise); `realisation` picks the noise/initial-condition seeds (bench.py gives every
    rank its own)."""
    specs = [(SIG_LOGISTIC, 1.0, 0), (SIG_LOGISTIC, 0.1, 1), (SIG_LORENZ, 1.0, 0), (SIG_LORENZ, 0.1, 1),
             (SIG_NOISE, 0.0, 0)]
    if which is not None:
        specs = [specs[i] for i in which]
    rows, labels = [], []
    for sig, snr, si in specs:
        seed = make_seed(4, sig, si, realisation)
        if sig == SIG_LOGISTIC:
            rows.append(add_noise(logistic_signal(N, seed), snr, seed))
        elif sig == SIG_LORENZ:
            rows.append(add_noise(lorenz_signal(N), snr, seed))
        else:
            rows.append(gaussian(seed, N).astype(np.float32))
        labels.append(_label(sig, snr, seed))
    return Workload(f"config4_long_N{N}", np.stack(rows), 3, 1, NORM_MAX, rr_log(20, 0.001, 0.2), (2,), labels)


def config5(N: int = 20000, n_snr: int = 8, n_seeds: int = 4) -> Workload:
    """Batch sweep: {sine, logistic, Lorenz} x 8 SNRs 10^(1-3i/7) x 4 seeds = 96 series of N=2e4; m=5, tau=2,
    max; K=32 log 0.0005..0.3; l_min in {2, 3}."""
    rows, labels = [], []
    for sig in (SIG_SINE, SIG_LOGISTIC, SIG_LORENZ):
        for si in range(n_snr):
            snr = 10.0 ** (1.0 - 3.0 * si / 7.0)
            for real in range(n_seeds):
                seed = make_seed(5, sig, si, real)
                cseed = make_seed(5, sig, 0, real)       # the clean signal depends on the realisation only
                if sig == SIG_SINE:
                    clean = sine_signal(N)
                elif sig == SIG_LOGISTIC:
                    clean = logistic_signal(N, cseed)
                else:
                    u = uniform01(cseed ^ 0x2545F4914F6CDD1D, 3)
                    clean = lorenz_signal(N, start=(1.0 + u[0], 1.0 + u[1], 1.0 + u[2]))
                rows.append(add_noise(clean, snr, seed))
                labels.append(_label(sig, snr, seed))
    return Workload(f"config5_batch_N{N}", np.stack(rows), 5, 2, NORM_MAX, rr_log(32, 0.0005, 0.3), (2, 3), labels)


def paper_group(signal: str, level: float, N: int, n_real: int = 10, K: int = 99) -> Workload:
    """One cell of the paper's 3 x 3 x 4 grid: one dynamics at one SNR level and one length, i.e. the
    10 SNRs level*{0.1, 0.2, .., 1.0} ("SNR L. level") x n_real realisations of the noise = 10*n_real series, row
    index = realisation*10 + snr_index, ascending SNR.  Here SNR is the paper's VARIANCE ratio:
    sigma_noise = sigma_signal / sqrt(SNR).  Dynamics as in PAPER.md:103-115: sine with 25 cycles over the series,
    logistic map at r = 3.679 (band merging, frequent laminar states), Lorenz x (RK4, dt = 0.01) embedded with m = 3,
    tau = 3; the other two are not embedded (m = 1).  RR_k = k/100, k = 1..K (RR* in 1..99 percent).
    The clean series is the same for the whole group; only the noise differs between rows."""
    sig = {"sine": SIG_SINE, "logistic": SIG_LOGISTIC, "lorenz": SIG_LORENZ}[signal]
    base = make_seed(6, sig, 0, 0) + 7919 * int(round(math.log10(N))) + 104729 * int(round(10 * math.log10(level) + 20))
    if sig == SIG_SINE:
        clean = np.sin(2.0 * math.pi * 25.0 * np.arange(N, dtype=np.float64) / N)
        m, tau = 1, 1
    elif sig == SIG_LOGISTIC:
        clean = logistic_signal(N, base, r=3.679)
        m, tau = 1, 1
    else:
        clean = lorenz_signal(N, every=1)
        m, tau = 3, 3
    rows, labels = [], []
    for real in range(n_real):
        for si in range(10):
            snr = level * (si + 1) / 10.0
            seed = base + 1000003 * (real + 1) + 10 * si
            rows.append(add_noise(clean, math.sqrt(snr), seed))
            labels.append(_label(sig, snr, seed))
    return Workload(f"paper_group_{signal}_snrL{level:g}_N{N}_x{10 * n_real}", np.stack(rows), m, tau, NORM_MAX,
                    rr_linear(K), (2,), labels)


def fnv1a64(a: np.ndarray) -> int:
    """FNV-1a-64 checksum of an array's bytes (logged with results so runs can be matched)."""
    h = 0xCBF29CE484222325
    for b in np.ascontiguousarray(a).tobytes():
        h = ((h ^ b) * 0x100000001B3) & _M64
    return h
