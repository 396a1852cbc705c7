"""GPU parity tests: the CUDA path (through the C-ABI, paper_1701_08197_b200.lof) against the CPU
oracle (oracle/) on the same seeded inputs.  Rules: median bit-exact; mean, stddev <= 1e-6 relative;
flags bit-exact except samples explained by an oracle margin bit (window sum within 1e-5 relative of
its threshold), which must total <= 1e-6 of samples (BASELINE.json north_star)."""
import numpy as np
import pytest

from parity import assert_flags, assert_stats, unpack

pytestmark = pytest.mark.gpu


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


def run_gpu(lof, power, S, C, T, path=0, group=None, want_path=None, **kw):
    import torch
    f = lof.Flagger(S, C, T, **kw)
    f.set_path(path)
    if group:
        f.set_group(group)
    x = torch.from_numpy(np.ascontiguousarray(power)).cuda()
    flags, stats = f.flag_block(x)
    torch.cuda.synchronize()
    rs, rc = f.row_sums()
    out = dict(flags=lof.flags_to_numpy(flags), stats=lof.stats_to_numpy(stats),
               rowsum=rs.cpu().numpy(), rowcnt=rc.cpu().numpy().view(np.uint32), path_used=f.path_used())
    if want_path is not None:
        assert out["path_used"] == want_path, (out["path_used"], want_path)
    f.close()
    return out


def run_oracle(lofo, power, S, C, T, threads=8, **kw):
    prm = lofo.make_params(S, C, T, **kw)
    return lofo.flag_block_threads(prm, power, threads, want_margin=True)


def check(lof, lofo, power, S, C, T, exact=False, volt=None, paths=(0, 1), group=None, want_path=None, **kw):
    if volt is not None:
        power = lofo.power_from_ci16(volt)
    ora = run_oracle(lofo, power, S, C, T, **kw)
    res = None
    for path in paths:
        g = run_gpu(lof, volt if volt is not None else power, S, C, T, path=path, group=group,
                    want_path=want_path if path == 0 else lof.PATH_GENERIC, **kw)
        assert_stats(g["stats"], ora["stats"])
        res = assert_flags(g["flags"], ora, T, kw.get("max_window", 64), exact=exact)
        if res["n_mismatch"] == 0:
            assert np.array_equal(g["stats"]["n_flagged"], ora["stats"]["n_flagged"])
            assert np.array_equal(g["rowcnt"], ora["rowcnt"])
            # row sums feed float32 history entries: the fused kernel adds each lane's samples
            # in fp32 before the fp64 reduction, so 1e-6 relative is the bar
            np.testing.assert_allclose(g["rowsum"], ora["rowsum"], rtol=1e-6, atol=0)
        # padding bits are zero
        if T % 32:
            assert (g["flags"][..., -1] >> np.uint32(T % 32)).max() == 0
    return res, ora


def test_config1_exact(lof, lofo, wl):
    w = wl.config1(0)
    res, ora = check(lof, lofo, w.power, 1, 16, 256, exact=True, max_window=32)
    m = unpack(ora["flags"], 256)
    assert m[0, 5].all() and m[0, :, 100].all()          # narrowband channel and broadband spike found


def test_config2_one_subband(lof, lofo, wl):
    w = wl.config2(0, n_subbands=1)
    res, _ = check(lof, lofo, w.power, w.S, 64, 768, max_window=64)
    print("cfg2", res)


def test_config3_cut(lof, lofo, wl):
    w = wl.config3(0, max_baselines=40)
    res, _ = check(lof, lofo, w.power, w.S, 16, 768, max_window=64)
    print("cfg3", res)


def test_config4_cut_ci16(lof, lofo, wl):
    # 2 stations x 2 pol, 32 subbands, ragged long time axis spanning several time tiles
    w = wl.config4(0, n_stations=2, T=20011)
    res, _ = check(lof, lofo, None, w.S, 32, 20011, volt=w.volt, max_window=256)
    print("cfg4", res)


def test_config5_cut_with_history(lof, lofo, wl):
    import torch
    S, C, T, H = 6, 16, 12208, 4
    gen = wl.Config5Stream(0, S=S, C=C, T=T)
    kw = dict(max_window=64, history_length=H, history_min_fill=2)
    f = lof.Flagger(S, C, T, **kw)
    prm = lofo.make_params(S, C, T, **kw)
    hist = lofo.History(prm)
    n_row_flagged = 0
    for k in range(7):
        w = gen.next_block()
        ora = lofo.flag_block_threads(prm, w.power, 8, want_margin=True)
        flags, stats = f.flag_block(torch.from_numpy(w.power).cuda())
        torch.cuda.synchronize()
        g = lof.flags_to_numpy(flags)
        assert_stats(lof.stats_to_numpy(stats), ora["stats"])
        r = assert_flags(g, ora, T, 64)
        assert r["n_mismatch"] == 0              # needed so that the row means below are comparable
        oflags = ora["flags"].copy()
        rf_o, near = hist.update(ora["rowsum"], ora["rowcnt"], oflags)
        rf_g = f.history_update(flags)
        torch.cuda.synchronize()
        rf_g = rf_g.cpu().numpy()
        differ = rf_g != rf_o
        assert not (differ & (near == 0)).any()   # decisions may differ only at near-ties
        if not differ.any():
            assert np.array_equal(lof.flags_to_numpy(flags), oflags)
            ring_g, head_g, cnt_g = [a.cpu().numpy() for a in f.history_export()]
            ring_o, head_o, cnt_o = hist.export()
            assert np.array_equal(head_g.view(np.uint32), head_o) and np.array_equal(cnt_g.view(np.uint32), cnt_o)
            np.testing.assert_allclose(ring_g, ring_o, rtol=1e-6)
        n_row_flagged += int(rf_o.sum())
    assert n_row_flagged > 0                      # the history flagger did act (and H = 4 evicted)
    # call-order errors
    with pytest.raises(lof.LofError) as e:
        f.history_update(flags)
    assert e.value.code == lof.E_STATE
    f.reset()
    ring_g, head_g, cnt_g = [a.cpu().numpy() for a in f.history_export()]
    assert not cnt_g.any() and not head_g.any()
    f.close()


@pytest.mark.parametrize("S,C,T,mw,dirs", [
    (3, 5, 77, 8, 3), (2, 1, 100, 16, 3), (2, 7, 1, 4, 3), (1, 3, 33, 64, 3), (2, 16, 256, 32, 1),
    (2, 16, 256, 32, 2), (1, 64, 768, 1, 3), (2, 48, 1000, 1024, 3), (1, 256, 40, 256, 3), (1, 2, 9000, 128, 3),
    (2, 16, 3000, 128, 3), (1, 32, 5003, 64, 3), (3, 64, 2100, 32, 3), (2, 16, 1025, 64, 2), (1, 32, 4096, 256, 3),
    # the fused shapes with windows beyond 64 (levels 7-9 of the row core with L = 24 and L = 8)
    (2, 64, 768, 1024, 3), (3, 16, 768, 256, 3), (2, 16, 256, 128, 3), (2, 32, 768, 512, 2), (3, 16, 768, 128, 2),
    (3, 32, 1024, 64, 3), (3, 64, 512, 64, 3), (5, 16, 1024, 256, 3), (2, 32, 1024, 1024, 3),
    # long rows with max_window 1024 (the cooperative tiles stop at 512: generic time kernel) and 512 (cross-warp
    # exchange at distance 256)
    (1, 16, 9000, 1024, 3), (1, 32, 20011, 512, 3)])
def test_ragged_shapes(lof, lofo, S, C, T, mw, dirs):
    rng = np.random.default_rng(S * 1000 + C * 10 + T)
    x = rng.standard_exponential((S, C, T)).astype(np.float32)
    x[0, C // 2, :] += 4.0
    x[:, :, T // 3] += 9.0
    if T > 40:
        x[0, :, 20:36] += 2.5
    check(lof, lofo, x, S, C, T, max_window=mw, directions=dirs)


def test_negative_values_and_constant(lof, lofo):
    rng = np.random.default_rng(5)
    x = rng.standard_normal((2, 8, 300)).astype(np.float32) - 3.0
    x[1] = 2.5                                            # constant stream: stddev 0, no flags (F6)
    res, ora = check(lof, lofo, x, 2, 8, 300, max_window=32)
    g = run_gpu(lof, x, 2, 8, 300, max_window=32)
    assert g["stats"]["stddev"][1] == 0.0 and g["stats"]["n_flagged"][1] == 0


def test_nonfinite_stream_fully_flagged(lof, lofo):
    rng = np.random.default_rng(6)
    x = rng.standard_exponential((3, 4, 70)).astype(np.float32)
    x[1, 2, 5] = np.nan
    x[1, 0, 9] = np.inf
    for path in (0, 1):
        g = run_gpu(lof, x, 3, 4, 70, path=path, max_window=8)
        ora = run_oracle(lofo, x, 3, 4, 70, max_window=8)
        assert np.array_equal(g["flags"], ora["flags"])
        assert g["stats"]["n_nonfinite"].tolist() == [0, 2, 0]
        assert g["stats"]["n_flagged"][1] == 4 * 70 and (g["rowcnt"][1] == 0).all()


def test_sensitivity_and_p_params(lof, lofo, wl):
    w = wl.config1(1)
    check(lof, lofo, w.power, 1, 16, 256, max_window=32, sensitivity=0.7, p=1.3, start_threshold=5.0)


def test_alignment_and_null_errors(lof):
    import ctypes as C
    import torch
    f = lof.Flagger(1, 4, 64)
    x = torch.zeros(4 * 64 + 4, dtype=torch.float32, device="cuda")
    fl = f.new_flags()
    L = lof.lib()
    s = C.c_void_p(torch.cuda.current_stream().cuda_stream)
    assert L.lof_flag_block(f.h, C.c_void_p(x.data_ptr() + 4), C.c_void_p(fl.data_ptr()), None, s) == lof.E_ALIGN
    assert L.lof_flag_block(f.h, None, C.c_void_p(fl.data_ptr()), None, s) == lof.E_NULL
    assert L.lof_history_update(f.h, C.c_void_p(fl.data_ptr()), None, s) == lof.E_STATE   # H = 0
    f.close()


def test_host_entry_point(lof, lofo, wl):
    import torch
    w = wl.config1(0)
    f = lof.Flagger(1, 16, 256, max_window=32)
    hp = torch.from_numpy(w.power).pin_memory()
    hf = torch.empty((1, 16, 8), dtype=torch.int32).pin_memory()
    hs = torch.empty((1, 32), dtype=torch.uint8).pin_memory()
    f.flag_block_host(hp, hf, hs)
    ora = run_oracle(lofo, w.power, 1, 16, 256, max_window=32)
    assert np.array_equal(hf.numpy().view(np.uint32), ora["flags"])
    assert_stats(hs.numpy().view(lof.STATS_DTYPE).reshape(-1), ora["stats"])
    assert f.launch_count() > 0
    f.close()


def test_bench_configuration_sampled_streams(lof, lofo, wl):
    """The launch configuration bench.py times (config 2 batched over subbands, S a multiple of 96 far above
    the number of SMs, persistent CTAs looping over streams with prefetch): every stream of a sample is
    compared with the oracle, which computes streams one by one."""
    import torch
    w = wl.config2(0, n_subbands=16, want_truth=False)             # 1536 streams = 10.4 per SM
    S, C, T = w.power.shape
    f = lof.Flagger(S, C, T, max_window=64)
    flags, stats = f.flag_block(torch.from_numpy(w.power).cuda())
    torch.cuda.synchronize()
    g = lof.flags_to_numpy(flags)
    st = lof.stats_to_numpy(stats)
    pick = np.unique(np.concatenate([np.arange(0, 8), np.arange(S - 8, S),
                                     np.random.default_rng(3).integers(0, S, 240)]))
    prm = lofo.make_params(len(pick), C, T, max_window=64)
    ora = lofo.flag_block_threads(prm, w.power[pick], 8, want_margin=True)
    assert_stats(st[pick], ora["stats"])
    r = assert_flags(g[pick], ora, T, 64)
    assert np.array_equal(st["n_flagged"][pick], ora["stats"]["n_flagged"]) or r["n_mismatch"] > 0
    # properties that hold at any size: n_flagged equals the popcount of the words; padding-free rows
    pop = np.unpackbits(g.view(np.uint8), axis=-1).reshape(S, -1).sum(axis=1)
    assert np.array_equal(pop.astype(np.uint64), st["n_flagged"])
    f.close()


def test_ci16_long_rows_register_kernels(lof, lofo, wl):
    # complex int16 input through the register-resident long-row kernels (max_window 64: row segments with halo)
    w = wl.config4(1, n_stations=1, T=7001)
    res, _ = check(lof, lofo, None, w.S, 32, 7001, volt=w.volt, max_window=64)
    print("cfg4-like, windows 1..64", res)


# ---- statistics: the cases in which the value histogram cannot isolate the median by itself

def _stats_cases(rng, C, T):
    """Streams that stress the exact-median selection: heavy ties (a bin holding thousands of equal samples),
    a two-level distribution whose median sits far outside the sampled interquartile range, tiny spread
    around a large offset, and plain noise."""
    N = C * T
    a = rng.integers(0, 3, size=N).astype(np.float32)                         # quantised: crowded bins
    b = np.where(rng.random(N) < 0.505, 1.0, 1000.0).astype(np.float32)       # upper median 1.0, IQR huge
    b += (rng.random(N) < 0.5).astype(np.float32) * 1e-3
    c = (1.0e6 + 1e-2 * rng.standard_normal(N)).astype(np.float32)            # spread of a few ulps
    d = rng.standard_exponential(N).astype(np.float32)
    e = np.zeros(N, np.float32); e[: N // 2 - 3] = -1.0; e[N // 2 + 5:] = 7.0  # median among a few zeros
    return np.stack([a, b, c, d, rng.permutation(e)]).reshape(5, C, T)


@pytest.mark.parametrize("C,T,mw", [(64, 768, 64), (16, 768, 64), (16, 256, 32),      # fused kernels
                                    (16, 20011, 64), (32, 9000, 256)])                  # long-row kernels
def test_statistics_hard_medians(lof, lofo, C, T, mw):
    rng = np.random.default_rng(C * 7 + T)
    x = _stats_cases(rng, C, T)
    ora = run_oracle(lofo, x, 5, C, T, max_window=mw)
    for path in (0, 1):
        g = run_gpu(lof, x, 5, C, T, path=path, max_window=mw)
        assert_stats(g["stats"], ora["stats"])
        assert_flags(g["flags"], ora, T, mw)


def test_long_row_candidate_list_overflow(lof, lofo):
    """More samples in the median's bin than the candidate list holds (quantised data, 16 x 40000): the
    selection falls back to the radix select over the whole stream."""
    rng = np.random.default_rng(11)
    x = rng.integers(0, 2, size=(2, 16, 40000)).astype(np.float32)
    x[1] += rng.standard_exponential((16, 40000)).astype(np.float32) * 1e-3
    ora = run_oracle(lofo, x, 2, 16, 40000, max_window=64)
    g = run_gpu(lof, x, 2, 16, 40000, max_window=64)
    assert_stats(g["stats"], ora["stats"])
    assert_flags(g["flags"], ora, 40000, 64)


def test_fused_counters_account_for_every_stream(lof, wl):
    import torch
    w = wl.config2(3, n_stations=3)
    f = lof.Flagger(w.S, w.C, w.T, max_window=64)
    f.fused_counters(reset=True)
    f.flag_block(torch.from_numpy(w.power).cuda())
    c = f.fused_counters()
    f.close()
    assert sum(c) == w.S and c[3] == 0, c
    assert c[0] >= w.S - 1, c          # noise-like streams: the median comes from the rank count in its bin


@pytest.mark.parametrize("shape", ["fused64", "fused16", "longrow"])
def test_repeated_runs_are_bit_identical(lof, wl, shape):
    """The statistics are summed in a fixed order and every flag decision is deterministic: the same block
    flagged five times (dynamic hand-out of columns and rows, atomics on histograms and candidate lists in
    between) gives the same bytes, flags and statistics alike."""
    import torch
    if shape == "fused64":
        w = wl.config2(5, n_stations=40); x, C, T, mw = w.power, w.C, w.T, 64          # 80 streams
    elif shape == "fused16":
        w = wl.config3(5, n_stations=12); x, C, T, mw = w.power, w.C, w.T, 64
    else:
        rng = np.random.default_rng(9)
        x = rng.standard_exponential((6, 16, 12208)).astype(np.float32); C, T, mw = 16, 12208, 64
        x[2, 3, 100:400] += 5.0
    S = x.shape[0]
    f = lof.Flagger(S, C, T, max_window=mw)
    xd = torch.from_numpy(np.ascontiguousarray(x)).cuda()
    ref = None
    for _ in range(5):
        flags, stats = f.flag_block(xd)
        torch.cuda.synchronize()
        rs, rc = f.row_sums()
        got = (lof.flags_to_numpy(flags).tobytes(), stats.cpu().numpy().tobytes(), rs.cpu().numpy().tobytes(),
               rc.cpu().numpy().tobytes())
        if ref is None:
            ref = got
        assert got == ref
    f.close()


# ---- paths that only the full-size configurations take (multi-group loop, persistent CTAs past a
# ---- non-finite stream, many streams on the generic path)

@pytest.mark.parametrize("S,C,T,mw,group,ci16,want", [
    (5, 16, 12208, 64, 2, False, "seg"),      # three groups (2 + 2 + 1), row segments with halo
    (3, 32, 20011, 256, 1, True, "coop"),     # three groups of one stream, cooperative tiles, ci16
    (4, 16, 9001, 256, 3, False, "coop"),     # 3 + 1, float32 through the cooperative tiles
    (5, 32, 7001, 64, 2, True, "seg")])
def test_long_rows_several_groups(lof, lofo, wl, S, C, T, mw, group, ci16, want):
    """kp.s0 > 0: the loop over groups of streams that full config 4 takes (four groups of 26 streams)."""
    rng = np.random.default_rng(S * 100 + C)
    want_path = lof.PATH_LONGROW_SEG if want == "seg" else lof.PATH_LONGROW_COOP
    if ci16:
        w = wl.config4(7, n_stations=(S + 1) // 2, C=C, T=T)
        volt = w.volt[:S]
        check(lof, lofo, None, S, C, T, volt=volt, max_window=mw, group=group, want_path=want_path)
    else:
        x = rng.standard_exponential((S, C, T)).astype(np.float32)
        for s in range(S):
            x[s, rng.integers(0, C), :] += 3.0 + s
            t0 = int(rng.integers(0, T - 600)); x[s, :, t0:t0 + 300 + 50 * s] += 1.5
        check(lof, lofo, x, S, C, T, max_window=mw, group=group, want_path=want_path)


@pytest.mark.parametrize("T,mw,dirs,seed", [(8192 * 3 - 1024 * 2 + 17, 256, 3, 0), (20000, 512, 2, 1),
                                            (7168 * 2, 128 * 2, 3, 2), (30011, 256, 3, 3)])
def test_cooperative_tiles_partial_restarts(lof, lofo, T, mw, dirs, seed):
    """lof_k_time_coop rebuilds, after new flags, only the strips that changed and the strip before each; the other
    warps keep their trees and the sums they published.  Events of every length from 1 to 600 samples and
    amplitudes from just above the widest window's threshold to 40 sigma, several per 8192-sample tile, so that
    iterations of every window size fire in some strips and not in their neighbours; events across strip (1024)
    and tile borders; flags compared bit by bit with the oracle (exact: the margin set must come out empty or
    explained) on both the register path and the generic one."""
    rng = np.random.default_rng(9100 + seed)
    S, C = 2, 16
    x = rng.standard_exponential((S, C, T)).astype(np.float32)
    for s in range(S):
        for c in range(C):
            n_ev = int(rng.integers(T // 1500, T // 500))
            for _ in range(n_ev):
                ln = int(2 ** rng.uniform(0, np.log2(600)))
                t0 = int(rng.integers(0, T - ln))
                if rng.random() < 0.3:                   # pinned to a strip or tile border
                    b = int(rng.integers(1, T // 1024)) * 1024
                    t0 = max(0, min(T - ln, b - int(rng.integers(0, ln + 1))))
                amp = float(np.exp(rng.uniform(np.log(0.3), np.log(40.0)))) / np.sqrt(max(1.0, ln / 8.0)) + 0.15
                x[s, c, t0:t0 + ln] += np.float32(amp)
    check(lof, lofo, x, S, C, T, max_window=mw, directions=dirs, want_path=lof.PATH_LONGROW_COOP)


def test_generic_path_more_than_1024_streams(lof, lofo):
    """S > 1024: the generic path splits the block into groups of at most 1024 streams."""
    rng = np.random.default_rng(21)
    S, C, T = 1100, 4, 70
    x = rng.standard_exponential((S, C, T)).astype(np.float32)
    x[::7, 1, 10:30] += 6.0
    x[1030:, :, 40] += 12.0                                # events in the second group
    check(lof, lofo, x, S, C, T, max_window=16, want_path=lof.PATH_GENERIC)


@pytest.mark.parametrize("C,T,mw", [(64, 768, 64), (16, 768, 64)])
def test_fused_nonfinite_streams_inside_persistent_loop(lof, lofo, wl, C, T, mw):
    """S far above the grid of persistent CTAs: streams with NaN/Inf met as the first stream of a CTA, as a
    prefetched one, twice in a row in the same CTA and as the last one; the CTA flags them completely (S6) and
    carries on with clean streams (reload path after the skipped stream)."""
    import torch
    n_sm = torch.cuda.get_device_properties(0).multi_processor_count
    grid = n_sm * (1 if C == 64 else 2)
    S = grid * 3 + 5
    rng = np.random.default_rng(C)
    x = rng.standard_exponential((S, C, T)).astype(np.float32)
    x[:, C // 3, :] += 2.0
    x[::3, :, 100:103] += 30.0
    bad = [0, 7, grid + 7, 2 * grid + 7, grid + 11, 2 * grid - 1, S - 1]
    for i, s in enumerate(bad):
        x[s, (3 * i) % C, (97 * i) % T] = np.nan if i % 2 == 0 else np.inf
    g = run_gpu(lof, x, S, C, T, max_window=mw, want_path=lof.PATH_FUSED)
    ora = run_oracle(lofo, x, S, C, T, threads=16, max_window=mw)
    assert np.array_equal(g["stats"]["n_nonfinite"] > 0, np.isin(np.arange(S), bad))
    assert_stats(g["stats"], ora["stats"])
    assert_flags(g["flags"], ora, T, mw)
    assert np.array_equal(g["stats"]["n_flagged"], ora["stats"]["n_flagged"])
    assert np.array_equal(g["rowcnt"], ora["rowcnt"])
    assert (g["rowcnt"][bad] == 0).all() and (g["flags"][bad] == 0xFFFFFFFF).all()


def test_path_used_reports_the_decomposition(lof):
    import torch
    for (S, C, T, mw, want) in [(2, 64, 768, 64, "FUSED"), (2, 16, 256, 32, "FUSED"), (2, 32, 1024, 64, "FUSED"),
                                (2, 64, 512, 64, "FUSED"), (2, 16, 1024, 64, "FUSED"), (2, 64, 704, 64, "LONGROW_SEG"), (2, 48, 768, 64, "GENERIC"),
                                (1, 16, 12208, 64, "LONGROW_SEG"), (1, 32, 20000, 256, "LONGROW_COOP"),
                                (1, 32, 20000, 1024, "GENERIC"), (2, 5, 77, 8, "GENERIC")]:
        f = lof.Flagger(S, C, T, max_window=mw)
        assert f.path_used() == lof.PATH_NONE
        f.flag_block(torch.rand((S, C, T), device="cuda"))
        torch.cuda.synchronize()
        assert f.path_used() == getattr(lof, "PATH_" + want), (S, C, T, mw, f.path_used())
        f.close()


# ---- NEXT-1: SIR operator on the packed mask

@pytest.mark.parametrize("cfg,eta,dirs", [("cfg1", 0.2, 3), ("cfg2", 0.2, 3), ("cfg3", 0.2, 3), ("cfg2", 0.5, 1),
                                          ("cfg2", 0.2, 2), ("cfg3", 1.0, 3), ("cfg1", 0.05, 3)])
def test_sir_fused_shapes(lof, lofo, wl, cfg, eta, dirs):
    if cfg == "cfg1":
        w = wl.config1(0); mw = 32
    elif cfg == "cfg2":
        w = wl.config2(0, n_stations=6); mw = 64
    else:
        w = wl.config3(0, max_baselines=12); mw = 64
    res, ora = check(lof, lofo, w.power, w.S, w.C, w.T, exact=True, max_window=mw, sir_eta=eta, directions=dirs)
    base = run_oracle(lofo, w.power, w.S, w.C, w.T, max_window=mw, directions=dirs)
    added = int(ora["stats"]["n_flagged"].sum()) - int(base["stats"]["n_flagged"].sum())
    assert added >= 0 and (added > 0 or cfg == "cfg1")     # the operator did add flags (config 1 has no run to grow)


@pytest.mark.parametrize("S,C,T,mw,eta", [(3, 16, 12208, 64, 0.2), (2, 32, 20011, 256, 0.2), (2, 5, 77, 8, 0.3),
                                          (1, 64, 2100, 32, 0.2), (2, 16, 1025, 64, 0.5), (1, 1, 5000, 16, 0.2),
                                          (2, 200, 40, 8, 0.2)])
def test_sir_long_rows_and_ragged(lof, lofo, S, C, T, mw, eta):
    rng = np.random.default_rng(S + C + T)
    x = rng.standard_exponential((S, C, T)).astype(np.float32)
    x[0, C // 2, :] += 4.0
    for _ in range(6):                                     # bursts of many lengths: runs that cross word and lane blocks
        d = int(rng.integers(3, max(4, min(T, 3000)))); t0 = int(rng.integers(0, max(1, T - d)))
        c0 = int(rng.integers(0, C)); h = int(rng.integers(1, max(2, C // 2 + 1)))
        x[rng.integers(0, S), c0:c0 + h, t0:t0 + d] += 12.0
    x[:, :, T - 7:] += 20.0                                # a run that ends at the end of the row
    x[S - 1, :, :9] += 20.0                                # and one that starts at its start
    check(lof, lofo, x, S, C, T, exact=True, max_window=mw, sir_eta=eta)


def test_sir_mask_kernels_on_random_masks(lof, lofo):
    """The two SIR kernels alone, on dense random masks (runs of every length, merging extensions), through
    lof_flag_block with a threshold nothing exceeds except planted samples: max_window 1, so the SumThreshold
    mask is exactly the planted pattern."""
    rng = np.random.default_rng(77)
    for (S, C, T, dens) in [(2, 24, 75, 0.45), (1, 70, 333, 0.3), (3, 16, 768, 0.48), (1, 8, 9000, 0.4)]:
        pat = rng.random((S, C, T)) < dens
        x = np.where(pat, 1000.0, rng.random((S, C, T))).astype(np.float32)
        # fewer than half of the samples are planted, so the median is a noise value (< 1) and, with sensitivity
        # 0.1, median + 0.6 sigma (sigma <= 500) lies between the two populations
        kw = dict(max_window=1, directions=3, sir_eta=0.2, sensitivity=0.1)
        ora = run_oracle(lofo, x, S, C, T, **kw)
        base = run_oracle(lofo, x, S, C, T, **dict(kw, sir_eta=0.0))
        assert np.array_equal(unpack(base["flags"], T).astype(bool), pat)
        g = run_gpu(lof, x, S, C, T, **kw)
        assert np.array_equal(g["flags"], ora["flags"])
        assert np.array_equal(g["stats"]["n_flagged"], ora["stats"]["n_flagged"])


# ---- NEXT-2: fully integrated mode

def _check_integrated(lof, lofo, x, S, C, T, **kw):
    import torch
    ora = lofo.flag_block_integrated(lofo.make_params(S, C, T, **kw), x)
    f = lof.Flagger(S, C, T, **kw)
    flags, sf, st = f.flag_block_integrated(torch.from_numpy(np.ascontiguousarray(x)).cuda())
    torch.cuda.synchronize()
    spec, series = [a.cpu().numpy() for a in f.integrated_vectors()]
    g = lof.flags_to_numpy(flags)
    sf, st = lof.stats_to_numpy(sf), lof.stats_to_numpy(st)
    with pytest.raises(lof.LofError) as e:                 # no row sums after an integrated block
        f.history_update(flags)
    assert e.value.code == lof.E_STATE
    f.close()
    # the two vectors are fp64 sums rounded to float32: the summation orders differ, so 1e-6 relative (reading I5)
    ok = ora["stats_freq"]["n_nonfinite"] == 0
    np.testing.assert_allclose(spec[ok], ora["spectrum"][ok], rtol=1e-6, atol=0)
    np.testing.assert_allclose(series[ok], ora["series"][ok], rtol=1e-6, atol=1e-30)
    for gs, os_ in ((sf, ora["stats_freq"]), (st, ora["stats_time"])):
        fin = os_["n_nonfinite"] == 0
        for k in ("median", "mean", "stddev"):
            np.testing.assert_allclose(gs[k][fin], os_[k][fin], rtol=2e-6, atol=1e-30)
    assert np.array_equal(g, ora["flags"])
    assert np.array_equal(sf["n_flagged"], ora["stats_freq"]["n_flagged"])
    dirs = kw.get("directions", 3)
    if dirs & 2:
        assert np.array_equal(st["n_flagged"][ok], ora["stats_time"]["n_flagged"][ok])
    if T % 32:
        assert (g[..., -1] >> np.uint32(T % 32)).max() == 0
    return ora


@pytest.mark.parametrize("S,C,T,mw,dirs", [(4, 64, 768, 64, 3), (6, 16, 768, 16, 3), (2, 32, 20011, 256, 3),
                                           (3, 16, 12208, 64, 3), (2, 7, 333, 8, 3), (2, 64, 768, 32, 1),
                                           (2, 64, 768, 32, 2), (1, 200, 1025, 64, 3), (2, 3, 40, 4, 3)])
def test_integrated_mode(lof, lofo, S, C, T, mw, dirs):
    rng = np.random.default_rng(S * 7 + C + T)
    x = rng.standard_exponential((S, C, T)).astype(np.float32)
    x[0, C // 3, :] += 1.0                                 # weak narrow-band RFI, found after integration over time
    if C > 8:
        x[S - 1, C // 2:C // 2 + 2, :] += 0.7
    x[:, :, T // 2:T // 2 + 5] += 1.5                      # weak broadband burst, found after integration over channels
    x[0, :, T // 5] += 9.0
    ora = _check_integrated(lof, lofo, x, S, C, T, max_window=mw, directions=dirs)
    if dirs == 3 and C >= 64:                              # (one outlier among n values is at most (n-1)/sqrt(n) sigmas out)
        assert ora["chan_mask"][0, C // 3] == 1 and ora["time_mask"][0, T // 5] == 1


def test_integrated_mode_nonfinite_and_constant(lof, lofo):
    rng = np.random.default_rng(85)
    x = rng.standard_exponential((3, 16, 300)).astype(np.float32)
    x[1] = 2.5                                             # constant stream: no flags
    x[2, 4, 17] = np.inf                                   # non-finite: everything flagged (S6)
    ora = _check_integrated(lof, lofo, x, 3, 16, 300, max_window=16)
    m = unpack(ora["flags"], 300)
    assert m[1].sum() == 0 and m[2].all()


def test_integrated_mode_config2_batch(lof, lofo, wl):
    w = wl.config2(0, n_stations=8, want_truth=False)
    _check_integrated(lof, lofo, w.power, w.S, w.C, w.T, max_window=64)


# ---- NEXT-3: robust scale: 1.4826 * MAD in place of the standard deviation

@pytest.mark.parametrize("S,C,T,mw", [(1, 16, 256, 32), (4, 64, 768, 64), (3, 16, 12208, 64), (2, 32, 9001, 256),
                                      (2, 5, 77, 8), (8, 16, 768, 64)])
def test_mad_mode(lof, lofo, wl, S, C, T, mw):
    if (S, C, T) == (1, 16, 256):
        x = wl.config1(0).power
    elif (C, T) == (64, 768):
        x = wl.config2(2, n_stations=2).power
    else:
        # (seed chosen so that no window sum of the block lies within fp32 rounding of its threshold: with the MAD
        # scale the thresholds sit in the noise tail, and a block of 0.6 M samples has a few per cent chance of
        # holding one such window, which the parity rule grants only to blocks above a million samples)
        rng = np.random.default_rng(1000 + S + C + T)
        x = rng.standard_exponential((S, C, T)).astype(np.float32)
        x[0, C // 2, :] += 4.0
        x[:, :, T // 3] += 9.0
        x[S - 1, :, 20:36] += 2.5
    res, ora = check(lof, lofo, x, S, C, T, max_window=mw, stats_mode=1)
    plain = run_oracle(lofo, x, S, C, T, max_window=mw)
    assert (ora["stats"]["stddev"] <= plain["stats"]["stddev"]).all()     # RFI inflates the stddev, hardly the MAD
    if (S, C, T) == (1, 16, 256):
        m = unpack(ora["flags"], T)[0].astype(bool)
        assert m[wl.config1(0).extra["cls"][0] == 3].all()                # the 8 x 8 burst that plain stddev misses
