"""ctypes loader for the ORACLE (oracle/lof_oracle.cpp) — test infrastructure, not the product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It imports nothing from the CUDA package.  numpy arrays in, numpy out.
"""
import ctypes as C
import os
import subprocess
from concurrent.futures import ThreadPoolExecutor

import numpy as np

_DIR = os.path.dirname(os.path.abspath(__file__))
# LOFO_SANITIZE=1: a second build with -fsanitize=address,undefined (tests/test_oracle_sanitizers.py runs the
# pins against it in a subprocess that preloads libasan)
_SAN = bool(os.environ.get("LOFO_SANITIZE"))
_SO = os.path.join(_DIR, "liblof_oracle_san.so" if _SAN else "liblof_oracle.so")
_SRC = [os.path.join(_DIR, "lof_oracle.cpp"), os.path.join(_DIR, "lof_oracle.h")]
MARGIN_REL = 1e-5     # north_star: "window sum lies within 1e-5 relative of its threshold"


def build(force=False):
    """g++ -O2 build of the oracle shared library (building the checker is not using it)."""
    if force or not os.path.exists(_SO) or any(os.path.getmtime(s) > os.path.getmtime(_SO) for s in _SRC):
        san = ["-O1", "-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined"] if _SAN else ["-O2"]
        subprocess.check_call(["g++"] + san + ["-std=c++17", "-fPIC", "-shared", "-Wall", "-o", _SO, _SRC[0]])
    return _SO


class Params(C.Structure):
    _fields_ = [("n_streams", C.c_uint32), ("n_channels", C.c_uint32), ("n_time", C.c_uint32),
                ("p", C.c_double), ("sensitivity", C.c_double), ("start_threshold", C.c_double),
                ("max_window", C.c_uint32), ("directions", C.c_uint32),
                ("history_length", C.c_uint32), ("history_min_fill", C.c_uint32),
                ("history_sensitivity", C.c_double), ("sir_eta", C.c_double), ("stats_mode", C.c_uint32)]


STATS_DTYPE = np.dtype([("median", np.float32), ("n_nonfinite", np.uint32), ("mean", np.float64),
                        ("stddev", np.float64), ("n_flagged", np.uint64)], align=True)
assert STATS_DTYPE.itemsize == 32

_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.lofo_flag_block.restype = C.c_int
        _lib.lofo_history_create.restype = C.c_void_p
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def make_params(S, Cn, T, p=1.5, sensitivity=1.0, start_threshold=6.0, max_window=64, directions=3,
                history_length=0, history_min_fill=2, history_sensitivity=0.0, sir_eta=0.0, stats_mode=0):
    return Params(S, Cn, T, p, sensitivity, start_threshold, max_window, directions,
                  history_length, history_min_fill, history_sensitivity, float(np.float32(sir_eta)), stats_mode)


def factor_table(n, start_threshold=6.0, p=1.5):
    out = np.zeros(n, np.float64)
    lib().lofo_factor_table(C.c_double(start_threshold), C.c_double(p), C.c_uint32(n), _p(out))
    return out


def threshold_table(median, stddev, n, start_threshold=6.0, p=1.5, sensitivity=1.0):
    out = np.zeros(n, np.float64)
    lib().lofo_threshold_table(C.c_double(median), C.c_double(stddev), C.c_double(start_threshold),
                               C.c_double(p), C.c_double(sensitivity), C.c_uint32(n), _p(out))
    return out


def statistics(x):
    x = np.ascontiguousarray(x, np.float32).ravel()
    st = np.zeros(1, STATS_DTYPE)
    lib().lofo_statistics(_p(x), C.c_uint64(x.size), _p(st))
    return st[0]


def mad(x, median):
    x = np.ascontiguousarray(x, np.float32).ravel()
    lib().lofo_mad.restype = C.c_float
    return float(lib().lofo_mad(_p(x), C.c_uint64(x.size), C.c_float(median)))


def sumthreshold_1d(x, thresholds, mask=None, literal=False, margin_rel=MARGIN_REL):
    """One SumThreshold run on a 1-D line.  Returns (mask uint8[n], margin uint8[n])."""
    x = np.ascontiguousarray(x, np.float32)
    n = x.size
    m = np.zeros(n, np.uint8) if mask is None else np.ascontiguousarray(mask, np.uint8).copy()
    mg = np.zeros(n, np.uint8)
    thr = np.ascontiguousarray(thresholds, np.float64)
    f = lib().lofo_sumthreshold_1d_literal if literal else lib().lofo_sumthreshold_1d_fast
    f(_p(x), C.c_uint64(n), C.c_int64(1), _p(m), C.c_int64(1), _p(thr), C.c_uint32(thr.size),
      _p(mg), C.c_double(margin_rel))
    return m, mg


def flag_block(prm, power, want_mask_freq=False, want_margin=False, literal=False,
               margin_rel=MARGIN_REL):
    """power float32[S][C][T] -> dict(flags, stats, rowsum, rowcnt[, mask_freq][, margin])."""
    S, Cn, T = prm.n_streams, prm.n_channels, prm.n_time
    power = np.ascontiguousarray(power, np.float32).reshape(S, Cn, T)
    W = (T + 31) // 32
    out = dict(flags=np.zeros((S, Cn, W), np.uint32), stats=np.zeros(S, STATS_DTYPE),
               rowsum=np.zeros((S, Cn), np.float64), rowcnt=np.zeros((S, Cn), np.uint32))
    mf = np.zeros((S, Cn, T), np.uint8) if want_mask_freq else None
    mg = np.zeros((S, Cn, T), np.uint8) if want_margin else None
    rc = lib().lofo_flag_block(C.byref(prm), _p(power), _p(out["flags"]), _p(out["stats"]),
                               _p(out["rowsum"]), _p(out["rowcnt"]), _p(mf), _p(mg),
                               C.c_double(margin_rel), C.c_int(1 if literal else 0))
    if rc != 0:
        raise ValueError("lofo_flag_block: bad parameters")
    if want_mask_freq:
        out["mask_freq"] = mf
    if want_margin:
        out["margin"] = mg
    return out


def flag_block_threads(prm, power, n_threads, **kw):
    """The paper's CPU decomposition (one thread per subband): whole streams per
    thread, each thread running the single-threaded oracle.  ctypes releases the GIL."""
    S = prm.n_streams
    power = np.ascontiguousarray(power, np.float32).reshape(S, prm.n_channels, prm.n_time)
    bounds = np.linspace(0, S, min(n_threads, S) + 1).astype(int)
    parts = [(a, b) for a, b in zip(bounds[:-1], bounds[1:]) if b > a]

    def work(ab):
        a, b = ab
        q = Params.from_buffer_copy(prm)
        q.n_streams = b - a
        return flag_block(q, power[a:b], **kw)

    with ThreadPoolExecutor(len(parts)) as ex:
        outs = list(ex.map(work, parts))
    return {k: np.concatenate([o[k] for o in outs], axis=0) for k in outs[0]}


def sir_1d(mask, eta):
    """SIR operator on one line (uint8 0/1).  Returns the extended mask."""
    m = np.ascontiguousarray(mask, np.uint8).copy()
    lib().lofo_sir_1d(_p(m), C.c_uint64(m.size), C.c_int64(1), C.c_double(float(np.float32(eta))))
    return m


def sir_block(flags, T, eta, directions=3):
    """SIR operator on packed flags uint32[S][C][ceil(T/32)] (frequency, then time).  Returns a new array."""
    f = np.ascontiguousarray(flags, np.uint32).copy()
    S, Cn, W = f.shape
    assert W == (T + 31) // 32
    lib().lofo_sir_block(_p(f), C.c_uint64(S), C.c_uint64(Cn), C.c_uint64(T), C.c_double(float(np.float32(eta))),
                         C.c_uint32(directions))
    return f


def flag_block_integrated(prm, power):
    """Fully integrated mode.  Returns dict(flags, spectrum, series, chan_mask, time_mask,
    stats_freq, stats_time)."""
    S, Cn, T = prm.n_streams, prm.n_channels, prm.n_time
    power = np.ascontiguousarray(power, np.float32).reshape(S, Cn, T)
    W = (T + 31) // 32
    out = dict(flags=np.zeros((S, Cn, W), np.uint32), spectrum=np.zeros((S, Cn), np.float32),
               series=np.zeros((S, T), np.float32), chan_mask=np.zeros((S, Cn), np.uint8),
               time_mask=np.zeros((S, T), np.uint8), stats_freq=np.zeros(S, STATS_DTYPE),
               stats_time=np.zeros(S, STATS_DTYPE))
    lib().lofo_flag_block_integrated.restype = C.c_int
    rc = lib().lofo_flag_block_integrated(C.byref(prm), _p(power), _p(out["flags"]), _p(out["spectrum"]),
                                          _p(out["series"]), _p(out["chan_mask"]), _p(out["time_mask"]),
                                          _p(out["stats_freq"]), _p(out["stats_time"]))
    if rc != 0:
        raise ValueError("lofo_flag_block_integrated: bad parameters")
    return out


def power_from_ci16(volt):
    volt = np.ascontiguousarray(volt, np.int16)
    n = volt.size // 2
    out = np.zeros(volt.shape[:-1], np.float32)
    lib().lofo_power_from_ci16(_p(volt), C.c_uint64(n), _p(out))
    return out


class History:
    """Oracle history flagger state."""

    def __init__(self, prm):
        self.prm = Params.from_buffer_copy(prm)
        self.h = C.c_void_p(lib().lofo_history_create(C.byref(self.prm)))

    def __del__(self):
        if getattr(self, "h", None):
            lib().lofo_history_destroy(self.h)
            self.h = None

    def reset(self):
        lib().lofo_history_reset(self.h)

    def update(self, rowsum, rowcnt, flags, near_rel=MARGIN_REL):
        """flags is modified in place.  Returns (row_flagged uint8[S][C], near uint8[S][C])."""
        S, Cn = self.prm.n_streams, self.prm.n_channels
        rowsum = np.ascontiguousarray(rowsum, np.float64)
        rowcnt = np.ascontiguousarray(rowcnt, np.uint32)
        assert flags.flags["C_CONTIGUOUS"] and flags.dtype == np.uint32
        rf = np.zeros((S, Cn), np.uint8)
        near = np.zeros((S, Cn), np.uint8)
        lib().lofo_history_update(self.h, _p(rowsum), _p(rowcnt), _p(flags), _p(rf), _p(near),
                                  C.c_double(near_rel))
        return rf, near

    def export(self):
        S, Cn, H = self.prm.n_streams, self.prm.n_channels, self.prm.history_length
        ring = np.zeros((S, Cn, H), np.float32)
        head = np.zeros((S, Cn), np.uint32)
        count = np.zeros((S, Cn), np.uint32)
        lib().lofo_history_export(self.h, _p(ring), _p(head), _p(count))
        return ring, head, count


def unpack_flags(flags, T):
    """uint32[..., ceil(T/32)] -> uint8[..., T], LSB first."""
    b = np.unpackbits(flags.view(np.uint8), axis=-1, bitorder="little")
    return b[..., :T]
