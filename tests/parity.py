"""Parity rules GPU vs oracle (BASELINE.json north_star).  Test infrastructure only."""
import numpy as np


def unpack(flags, T):
    b = np.unpackbits(np.ascontiguousarray(flags).view(np.uint8), axis=-1, bitorder="little")
    return b[..., :T]


def compare_flags(gpu_flags, ora_flags, margin, T, max_window):
    """Returns dict(n_mismatch, n_explained, n_unexplained).  A mismatch is explained when an oracle
    margin bit (window sum within 1e-5 relative of its threshold) lies within 2*max_window of it along
    either axis: a flipped borderline decision cascades through substitution inside the cone."""
    g = unpack(gpu_flags, T)
    o = unpack(ora_flags, T)
    diff = g != o
    idx = np.argwhere(diff)
    n_exp = 0
    R = 2 * max_window
    for s, c, t in idx:
        m = margin[s, max(0, c - R):c + R + 1, max(0, t - R):t + R + 1]
        n_exp += bool(m.any())
    return dict(n_mismatch=int(len(idx)), n_explained=int(n_exp), n_unexplained=int(len(idx) - n_exp),
                n_samples=int(g.size))


def assert_flags(gpu_flags, ora, T, max_window, exact=False):
    r = compare_flags(gpu_flags, ora["flags"], ora["margin"], T, max_window)
    if exact:
        assert r["n_mismatch"] == 0, r
    assert r["n_unexplained"] == 0, r
    # north_star: near-threshold mismatches must total <= 1e-6 of samples (at least one allowed slot
    # is not granted: for small blocks this means zero)
    assert r["n_explained"] <= 1e-6 * r["n_samples"], r
    return r


def assert_stats(gpu_stats, ora_stats, rel=1e-6):
    ok = ora_stats["n_nonfinite"] == 0
    assert np.array_equal(gpu_stats["n_nonfinite"], ora_stats["n_nonfinite"])
    g, o = gpu_stats[ok], ora_stats[ok]
    # median: bit-exact
    assert np.array_equal(g["median"].view(np.uint32), o["median"].view(np.uint32)), \
        (g["median"][:4], o["median"][:4])
    for f in ("mean", "stddev"):
        scale = np.maximum(np.abs(o[f]), np.finfo(np.float64).tiny)
        err = np.abs(g[f] - o[f]) / scale
        err = np.where(o[f] == g[f], 0.0, err)
        assert err.max(initial=0.0) <= rel, (f, err.max(), g[f][:4], o[f][:4])
