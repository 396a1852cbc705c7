"""GPU parity at the sizes BASELINE.json states for configs 3, 4 and 5 (north_star: "on all 5 configs"), in the
launch configuration bench.py times.  The oracle computes streams one by one, so flags are compared on a
stated random sample of whole streams (>= 64); the statistics of EVERY stream are compared (the oracle's
lofo_statistics per stream), and so are properties that hold at any size."""
import numpy as np
import pytest
from concurrent.futures import ThreadPoolExecutor

from parity import assert_flags, assert_stats

pytestmark = pytest.mark.gpu
N_SAMPLE = 64


@pytest.fixture(scope="module")
def lof():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1701_08197_b200 import build, lof as m
    build.build_lib()
    return m


@pytest.fixture(scope="module")
def wl():
    from paper_1701_08197_b200 import workloads
    return workloads


def _oracle_stats_all(lofo, power_of, S):
    """lofo_statistics of every stream (power_of(s) returns float32 [C][T])."""
    out = np.zeros(S, lofo.STATS_DTYPE)

    def work(s):
        out[s] = lofo.statistics(power_of(s))
    with ThreadPoolExecutor(16) as ex:
        list(ex.map(work, range(S)))
    return out


def _pick(S, seed):
    rng = np.random.default_rng(seed)
    return np.unique(np.concatenate([[0, S - 1], rng.choice(S, size=min(S, N_SAMPLE), replace=False)]))


def _popcount_rows(flags):
    return np.unpackbits(flags.view(np.uint8), axis=-1).reshape(flags.shape[0], -1).sum(axis=1).astype(np.uint64)


def test_config3_full(lof, lofo, wl):
    import torch
    w = wl.config3(0, want_truth=False)                    # 7564 streams x 16 x 768
    S, C, T = w.power.shape
    assert (S, C, T) == (7564, 16, 768)
    f = lof.Flagger(S, C, T, max_window=64)
    flags, stats = f.flag_block(torch.from_numpy(w.power).cuda())
    torch.cuda.synchronize()
    assert f.path_used() == lof.PATH_FUSED
    g, st = lof.flags_to_numpy(flags), lof.stats_to_numpy(stats)
    f.close()
    st_o = _oracle_stats_all(lofo, lambda s: w.power[s], S)
    g_cmp = st.copy(); g_cmp["n_flagged"] = 0
    assert_stats(g_cmp, st_o)
    pick = _pick(S, 3)
    prm = lofo.make_params(len(pick), C, T, max_window=64)
    ora = lofo.flag_block_threads(prm, w.power[pick], 16, want_margin=True)
    r = assert_flags(g[pick], ora, T, 64)
    assert r["n_mismatch"] > 0 or np.array_equal(st["n_flagged"][pick], ora["stats"]["n_flagged"])
    assert np.array_equal(_popcount_rows(g), st["n_flagged"])
    print("cfg3 full", r)


def test_config4_full_ci16(lof, lofo, wl):
    """96 streams x 32 subbands x 195 312 complex int16 (2.4 GB): four groups of 26 streams (s0 > 0),
    cooperative time tiles, frequency run across subbands."""
    import torch
    w = wl.config4(0)                                      # full size
    S, C, T = w.S, w.C, w.T
    assert (S, C, T) == (96, 32, 195312)
    f = lof.Flagger(S, C, T, max_window=256)
    xd = torch.from_numpy(w.volt).cuda()
    flags, stats = f.flag_block(xd)
    torch.cuda.synchronize()
    assert f.path_used() == lof.PATH_LONGROW_COOP
    g, st = lof.flags_to_numpy(flags), lof.stats_to_numpy(stats)
    rs, rc = f.row_sums()
    rs, rc = rs.cpu().numpy(), rc.cpu().numpy().view(np.uint32)
    f.close()
    del xd
    st_o = _oracle_stats_all(lofo, lambda s: lofo.power_from_ci16(w.volt[s]), S)
    g_cmp = st.copy(); g_cmp["n_flagged"] = 0
    assert_stats(g_cmp, st_o)
    pick = _pick(S, 4)                                     # 64 + of the 96 streams, from every group
    assert len(pick) >= 64
    prm = lofo.make_params(len(pick), C, T, max_window=256)
    power = lofo.power_from_ci16(w.volt[pick])
    ora = lofo.flag_block_threads(prm, power, 16, want_margin=True)
    r = assert_flags(g[pick], ora, T, 256)
    if r["n_mismatch"] == 0:
        assert np.array_equal(st["n_flagged"][pick], ora["stats"]["n_flagged"])
        assert np.array_equal(rc[pick], ora["rowcnt"])
        np.testing.assert_allclose(rs[pick], ora["rowsum"], rtol=1e-6, atol=0)
    assert np.array_equal(_popcount_rows(g), st["n_flagged"])
    assert (g[..., -1] >> np.uint32(T % 32)).max() == 0    # padding bits of the last word
    print("cfg4 full", r)


def test_config5_full_history_300(lof, lofo, wl):
    """488 subbands x 16 x 12 208, 10 consecutive blocks, history flagger with the paper's H = 300.
    Flags, row decisions and ring contents of 64 sampled subbands against the oracle, every block."""
    import torch
    S, C, T, H = 488, 16, 12208, 300
    gen = wl.Config5Stream(0, want_truth=False)
    kw = dict(max_window=64, history_length=H, history_min_fill=2)
    f = lof.Flagger(S, C, T, **kw)
    pick = _pick(S, 5)
    prm = lofo.make_params(len(pick), C, T, **kw)
    hist = lofo.History(prm)
    n_row_flagged = 0
    for k in range(10):
        w = gen.next_block()
        flags, stats = f.flag_block(torch.from_numpy(w.power).cuda())
        torch.cuda.synchronize()
        assert f.path_used() == lof.PATH_LONGROW_SEG
        g, st = lof.flags_to_numpy(flags), lof.stats_to_numpy(stats)
        ora = lofo.flag_block_threads(prm, w.power[pick], 16, want_margin=True)
        assert_stats(st[pick], ora["stats"])
        r = assert_flags(g[pick], ora, T, 64)
        assert r["n_mismatch"] == 0                        # so that the row means below are comparable
        assert np.array_equal(_popcount_rows(g), st["n_flagged"])
        oflags = ora["flags"].copy()
        rf_o, near = hist.update(ora["rowsum"], ora["rowcnt"], oflags)
        rf_g = f.history_update(flags)
        torch.cuda.synchronize()
        rf_g = rf_g.cpu().numpy()[pick]
        differ = rf_g != rf_o
        assert not (differ & (near == 0)).any()          # decisions may differ only at near-ties (|cur-thr| <= 1e-5 |thr|)
        if differ.any():                                   # from here on the two rings hold different entries
            break
        assert np.array_equal(lof.flags_to_numpy(flags)[pick], oflags)
        ring_g, head_g, cnt_g = [a.cpu().numpy() for a in f.history_export()]
        ring_o, head_o, cnt_o = hist.export()
        assert np.array_equal(head_g.view(np.uint32)[pick], head_o)
        assert np.array_equal(cnt_g.view(np.uint32)[pick], cnt_o)
        np.testing.assert_allclose(ring_g[pick], ring_o, rtol=1e-6)
        n_row_flagged += int(rf_o.sum())
    assert cnt_o.max() == 10 and n_row_flagged > 0         # the ring never fills in 10 blocks (H = 300)
    f.close()
