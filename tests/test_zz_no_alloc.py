"""lof_sir_noalloc (include/lof.h): the SIR operator on a packed mask through the entry point that allocates
nothing (its intermediate mask is a static device array), against the existing path: lof_flag_block with
sir_eta > 0, which runs the same operator with a context's cudaMalloc'ed buffer.  Integer work: bit-exact flags,
equal n_flagged, every other stats field untouched.  Named test_zz_* so that pytest collects it last."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def lof():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1701_08197_b200 import build, lof as m
    build.build_lib()
    return m


def _block(seed, S, C, T):
    """Noise with a loud channel, bursts of many lengths and a run that ends at the row's end: runs of flags
    along both axes for the operator to grow."""
    rng = np.random.default_rng(seed)
    x = rng.standard_exponential((S, C, T)).astype(np.float32)
    x[0, C // 2, :] += 4.0
    for _ in range(8):
        d = int(rng.integers(3, max(4, min(T, 2000)))); t0 = int(rng.integers(0, max(1, T - d)))
        c0 = int(rng.integers(0, C)); h = int(rng.integers(1, max(2, C // 2 + 1)))
        x[rng.integers(0, S), c0:c0 + h, t0:t0 + d] += 12.0
    x[:, :, max(0, T - 7):] += 20.0
    return x


def _existing_path(lof, x, S, C, T, mw, eta, dirs):
    """(mask before the operator, its stats, mask after, its stats) from lof_flag_block without / with sir_eta."""
    import torch
    xd = torch.from_numpy(x).cuda()
    out = []
    for e in (0.0, eta):
        f = lof.Flagger(S, C, T, max_window=mw, directions=dirs, sir_eta=e)
        flags, stats = f.flag_block(xd)
        torch.cuda.synchronize()
        out += [flags.clone(), stats.clone()]
        f.close()
    return out


CASES = [  # S, C, T, max_window, eta, directions
    (6, 64, 768, 64, 0.2, 3),        # 64-channel register column kernel, time rows of 24 words
    (3, 16, 12208, 64, 0.2, 3),      # long rows: 32 lanes per row, staged
    (2, 5, 77, 8, 0.3, 3),           # any-C column kernel, ragged last word, one lane per row
    (2, 32, 20011, 256, 0.5, 3),     # rows too long for the staged time kernel
    (4, 16, 1025, 64, 0.2, 2),       # time only: one pass, copied back from the static array
    (4, 64, 768, 64, 1.0, 1),        # frequency only, eta = 1
]


def _run_case(lof, case, seed):
    import torch
    S, C, T, mw, eta, dirs = case
    x = _block(seed, S, C, T)
    f0, s0, f1, s1 = _existing_path(lof, x, S, C, T, mw, eta, dirs)
    return dict(case=case, before=(f0, s0), want=(f1, s1))


def _compare(lof, got_f, got_s, r):
    want_f, want_s = r["want"]
    gf, wf = lof.flags_to_numpy(got_f), lof.flags_to_numpy(want_f)
    assert np.array_equal(gf, wf), (r["case"], int((gf != wf).sum()))
    gs, ws = lof.stats_to_numpy(got_s), lof.stats_to_numpy(want_s)
    assert np.array_equal(gs["n_flagged"], ws["n_flagged"]), r["case"]
    assert got_s.cpu().numpy().tobytes() == want_s.cpu().numpy().tobytes(), r["case"]   # nothing else touched


def test_no_alloc_matches_existing_path_two_calls_in_a_row(lof):
    """Every pair of consecutive cases: two calls back to back on one stream, no synchronisation between them
    (different shapes, so the second call finds the first one's mask in the shared array), then the same two
    again; each against lof_flag_block(sir_eta)."""
    import torch
    runs = [_run_case(lof, c, 100 + i) for i, c in enumerate(CASES)]
    grew = 0
    for a, b in zip(runs, runs[1:] + runs[:1]):
        for _ in range(2):
            outs = []
            for r in (a, b):
                S, C, T, mw, eta, dirs = r["case"]
                f, s = r["before"][0].clone(), r["before"][1].clone()
                lof.sir_noalloc(f, s, T, eta, dirs)
                outs.append((f, s))
            torch.cuda.synchronize()
            for (f, s), r in zip(outs, (a, b)):
                _compare(lof, f, s, r)
        grew += int((lof.flags_to_numpy(a["want"][0]) != lof.flags_to_numpy(a["before"][0])).sum())
    assert grew > 0                                        # the operator did something in these cases


def test_no_alloc_same_call_twice_is_identical_and_eta_zero_is_identity(lof):
    import torch
    r = _run_case(lof, CASES[0], 7)
    S, C, T, mw, eta, dirs = r["case"]
    res = []
    for _ in range(2):
        f, s = r["before"][0].clone(), r["before"][1].clone()
        lof.sir_noalloc(f, s, T, eta, dirs)
        torch.cuda.synchronize()
        res.append((f.cpu().numpy().tobytes(), s.cpu().numpy().tobytes()))
        _compare(lof, f, s, r)
    assert res[0] == res[1]
    f, s = r["before"][0].clone(), r["before"][1].clone()
    lof.sir_noalloc(f, s, T, 0.0, dirs)
    torch.cuda.synchronize()
    assert torch.equal(f, r["before"][0]) and torch.equal(s, r["before"][1])


def test_no_alloc_rejects_what_it_cannot_hold(lof):
    """Beyond LOF_NOALLOC_MAX_WORDS mask words: LOF_E_SIZE and the mask is untouched; bad arguments: LOF_E_PARAM /
    LOF_E_NULL / LOF_E_ALIGN.  A mask of exactly the maximum is accepted."""
    import ctypes as C_
    import torch
    L = lof.lib()
    W, T = 32, 1024                                         # 2048 words per stream: 1024 streams fill the array
    S = lof.NOALLOC_MAX_WORDS // (64 * W) + 1               # one stream too many
    flags = torch.zeros((S, 64, W), dtype=torch.int32, device="cuda")
    flags[:, 3, 2] = 0x00FFFF00
    stats = torch.zeros((S, 32), dtype=torch.uint8, device="cuda")
    keep = flags.clone()
    with pytest.raises(lof.LofError) as e:
        lof.sir_noalloc(flags, stats, T, 0.2)
    assert e.value.code == lof.E_SIZE and "static scratch" in str(e.value)
    torch.cuda.synchronize()
    assert torch.equal(flags, keep) and int(stats.sum()) == 0

    def call(fp, sp, S_, C_n, T_, eta, dirs, dev=0):
        return L.lof_sir_noalloc(C_.c_void_p(fp), C_.c_void_p(sp), C_.c_uint32(S_), C_.c_uint32(C_n), C_.c_uint32(T_),
                                 C_.c_float(eta), C_.c_uint32(dirs), C_.c_int(dev), C_.c_void_p(0))
    fp, sp = flags.data_ptr(), stats.data_ptr()
    assert call(0, sp, 2, 64, 768, 0.2, 3) == lof.E_NULL
    assert call(fp, 0, 2, 64, 768, 0.2, 3) == lof.E_NULL
    assert call(fp + 4, sp, 2, 64, 768, 0.2, 3) == lof.E_ALIGN
    for bad in [(0, 64, 768, 0.2, 3), (2, 0, 768, 0.2, 3), (2, 64, 0, 0.2, 3), (2, 300, 768, 0.2, 3),
                (2, 64, 768, -0.1, 3), (2, 64, 768, 1.5, 3), (2, 64, 768, float("nan"), 3), (2, 64, 768, 0.2, 0),
                (2, 64, 768, 0.2, 4)]:
        assert call(fp, sp, *bad) == lof.E_PARAM, bad
    assert call(fp, sp, 2, 64, 768, 0.2, 3, dev=64) == lof.E_PARAM
    # exactly the maximum: accepted, and a run of 16 samples grows by 3 on each side along time
    S_ok = lof.NOALLOC_MAX_WORDS // (64 * W)
    assert S_ok * 64 * W == lof.NOALLOC_MAX_WORDS
    sub_f, sub_s = flags[:S_ok], stats[:S_ok]
    lof.sir_noalloc(sub_f, sub_s, T, 0.2, 2)
    torch.cuda.synchronize()
    got = lof.flags_to_numpy(sub_f)
    assert (got[:, 3, 2] == 0x07FFFFE0).all() and int((got != 0).sum()) == S_ok
    assert (lof.stats_to_numpy(sub_s)["n_flagged"] == 6).all()
