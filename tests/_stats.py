"""Statistical comparison helpers for the chaotic-ensemble parity tests (reading R14/R16):
two-proportion 99 % intervals, a seeded bootstrap on the difference of means, and the collision-count
histogram in the bins {0, 1, 2, 3-4, 5-8, ...}.  Test code only."""
import numpy as np

Z99 = 2.5758293035489004  # two-sided 99 % normal quantile


def two_proportion_ok(k1: int, n1: int, k2: int, n2: int, z: float = Z99):
    """True when p1 - p2 lies inside the z-interval of the pooled two-proportion test.
    Returns (ok, difference, half-width)."""
    p1, p2 = k1 / n1, k2 / n2
    p = (k1 + k2) / (n1 + n2)
    half = z * np.sqrt(max(p * (1.0 - p), 1.0 / (n1 + n2)) * (1.0 / n1 + 1.0 / n2))
    return abs(p1 - p2) <= half, p1 - p2, half


def bootstrap_mean_diff_ok(a: np.ndarray, b: np.ndarray, B: int = 2000, seed: int = 12345, level: float = 0.99):
    """True when 0 lies inside the `level` bootstrap interval of mean(a) - mean(b).
    Returns (ok, observed difference, (lo, hi))."""
    rng = np.random.default_rng(seed)
    a, b = np.asarray(a, dtype=np.float64), np.asarray(b, dtype=np.float64)
    ia = rng.integers(0, len(a), (B, len(a)))
    ib = rng.integers(0, len(b), (B, len(b)))
    d = a[ia].mean(axis=1) - b[ib].mean(axis=1)
    lo, hi = np.quantile(d, [(1 - level) / 2, 1 - (1 - level) / 2])
    return lo <= 0.0 <= hi, a.mean() - b.mean(), (lo, hi)


def ncoll_bins(n_coll: np.ndarray, nbins: int = 32) -> np.ndarray:
    """bin 0: n_coll = 0; bin b >= 1: 2^(b-1) <= n_coll < 2^b  (the layout of ia_summary.hist_ncoll)."""
    n_coll = np.asarray(n_coll, dtype=np.uint64)
    b = np.zeros(len(n_coll), dtype=np.int64)
    nz = n_coll > 0
    b[nz] = np.floor(np.log2(n_coll[nz].astype(np.float64))).astype(np.int64) + 1
    return np.bincount(np.minimum(b, nbins - 1), minlength=nbins)


def histogram_ok(h1: np.ndarray, h2: np.ndarray, z: float = Z99):
    """Per-bin two-proportion test; returns (all ok, list of failing bins)."""
    n1, n2 = int(h1.sum()), int(h2.sum())
    bad = []
    for b, (k1, k2) in enumerate(zip(h1, h2)):
        if k1 + k2 == 0:
            continue
        ok, d, half = two_proportion_ok(int(k1), n1, int(k2), n2, z)
        if not ok:
            bad.append((b, int(k1), int(k2), d, half))
    return not bad, bad
