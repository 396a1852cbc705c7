"""Thin ctypes binding of include/lof.h — argument marshalling only; every step of the path runs in
the CUDA kernels of csrc/.  PyTorch supplies device memory and streams, nothing else.

There is no CPU fallback: if liblof.so is missing or no CUDA device is usable, calls raise.
"""
import ctypes as C
import os

import numpy as np

_DIR = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("LOF_LIB_PATH") or os.path.join(_DIR, "liblof.so")   # override: kernel experiments

DIR_FREQ, DIR_TIME = 1, 2
STATS_PLAIN, STATS_MAD = 0, 1
MAX_LEVELS = 11
E_NULL, E_PARAM, E_ALIGN, E_STATE, E_CUDA, E_SIZE = -1, -2, -3, -4, -5, -6
NOALLOC_MAX_WORDS = 2 * 1024 * 1024      # include/lof.h LOF_NOALLOC_MAX_WORDS
PATH_NONE, PATH_FUSED, PATH_LONGROW_SEG, PATH_LONGROW_COOP, PATH_GENERIC = 0, 1, 2, 3, 4

EXPORTS = ["lof_create", "lof_destroy", "lof_flag_block", "lof_flag_block_ci16", "lof_flag_block_integrated",
           "lof_integrated_vectors", "lof_history_update",
           "lof_reset", "lof_row_sums", "lof_history_export", "lof_flag_block_host", "lof_factor_table",
           "lof_launch_count", "lof_set_path", "lof_path_used", "lof_set_group", "lof_fused_counters", "lof_fused_cycles", "lof_sir_noalloc", "lof_strerror", "lof_last_cuda_error"]


class Params(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("device", C.c_int32),
                ("n_streams", C.c_uint32), ("n_channels", C.c_uint32), ("n_time", C.c_uint32),
                ("p", C.c_float), ("sensitivity", C.c_float), ("start_threshold", C.c_float),
                ("max_window", C.c_uint32), ("directions", C.c_uint32),
                ("history_length", C.c_uint32), ("history_min_fill", C.c_uint32),
                ("history_sensitivity", C.c_float), ("sir_eta", C.c_float), ("stats_mode", C.c_uint32)]


STATS_DTYPE = np.dtype([("median", np.float32), ("n_nonfinite", np.uint32), ("mean", np.float64),
                        ("stddev", np.float64), ("n_flagged", np.uint64)], align=True)
assert STATS_DTYPE.itemsize == 32


class LofError(RuntimeError):
    def __init__(self, code, what):
        self.code = code
        super().__init__(what)


_lib = None


def lib():
    """Loads liblof.so (built by paper_1701_08197_b200.build).  Fails loudly if it is absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise LofError(E_CUDA, f"{LIB_PATH} not built: run python -m paper_1701_08197_b200.build")
        L = C.CDLL(LIB_PATH)
        L.lof_strerror.restype = C.c_char_p
        L.lof_last_cuda_error.restype = C.c_char_p
        L.lof_launch_count.restype = C.c_uint64
        L.lof_launch_count.argtypes = [C.c_void_p]
        for name in ("lof_create", "lof_destroy", "lof_flag_block", "lof_flag_block_ci16",
                     "lof_flag_block_integrated", "lof_integrated_vectors",
                     "lof_history_update", "lof_reset", "lof_row_sums", "lof_history_export",
                     "lof_flag_block_host", "lof_factor_table", "lof_set_path", "lof_path_used", "lof_set_group",
                     "lof_fused_counters", "lof_fused_cycles", "lof_sir_noalloc"):
            getattr(L, name).restype = C.c_int
        _lib = L
    return _lib


def _check(rc):
    if rc != 0:
        L = lib()
        msg = L.lof_strerror(rc).decode()
        if rc == E_CUDA:
            msg += ": " + L.lof_last_cuda_error().decode()
        raise LofError(rc, msg)


def make_params(S, Cn, T, p=1.5, sensitivity=1.0, start_threshold=6.0, max_window=64, directions=3,
                history_length=0, history_min_fill=2, history_sensitivity=0.0, sir_eta=0.0, stats_mode=0, device=0):
    return Params(C.sizeof(Params), device, S, Cn, T, p, sensitivity, start_threshold, max_window,
                  directions, history_length, history_min_fill, history_sensitivity, sir_eta, stats_mode)


def factor_table(n, start_threshold=6.0, p=1.5):
    prm = make_params(1, 1, 1, p=p, start_threshold=start_threshold)
    out = (C.c_double * n)()
    _check(lib().lof_factor_table(C.byref(prm), out, C.c_uint32(n)))
    return np.array(out[:], np.float64)


def _ptr(t):
    return C.c_void_p(0 if t is None else t.data_ptr())


def _stream(stream):
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


class Flagger:
    """One lof_ctx.  Tensors are torch CUDA tensors; the flagger allocates outputs when not given."""

    def __init__(self, S, Cn, T, **kw):
        import torch
        self.torch = torch
        self.prm = make_params(S, Cn, T, **kw)
        self.S, self.Cn, self.T, self.W = S, Cn, T, (T + 31) // 32
        self.dev = torch.device("cuda", self.prm.device)
        h = C.c_void_p()
        _check(lib().lof_create(C.byref(self.prm), C.byref(h)))
        self.h = h

    def close(self):
        if getattr(self, "h", None):
            lib().lof_destroy(self.h)
            self.h = None

    __del__ = close

    def new_flags(self):
        return self.torch.empty((self.S, self.Cn, self.W), dtype=self.torch.int32, device=self.dev)

    def new_stats(self):
        return self.torch.empty((self.S, 32), dtype=self.torch.uint8, device=self.dev)

    def flag_block(self, power, flags=None, stats=None, stream=None):
        """power: float32 [S][C][T] (lof_flag_block) or int16 [S][C][T][2] (lof_flag_block_ci16)."""
        t = self.torch
        flags = self.new_flags() if flags is None else flags
        stats = self.new_stats() if stats is None else stats
        assert power.is_cuda and power.is_contiguous() and flags.is_contiguous()
        if power.dtype == t.float32:
            assert power.numel() == self.S * self.Cn * self.T
            fn = lib().lof_flag_block
        elif power.dtype == t.int16:
            assert power.numel() == self.S * self.Cn * self.T * 2
            fn = lib().lof_flag_block_ci16
        else:
            raise TypeError("power must be float32 or int16 (complex pairs)")
        _check(fn(self.h, _ptr(power), _ptr(flags), _ptr(stats), _stream(stream)))
        return flags, stats

    def flag_block_integrated(self, power, flags=None, stats_freq=None, stats_time=None, stream=None):
        """Fully integrated mode: returns (flags, stats of the spectrum, stats of the series)."""
        flags = self.new_flags() if flags is None else flags
        stats_freq = self.new_stats() if stats_freq is None else stats_freq
        stats_time = self.new_stats() if stats_time is None else stats_time
        assert power.is_cuda and power.is_contiguous() and power.dtype == self.torch.float32
        assert power.numel() == self.S * self.Cn * self.T
        _check(lib().lof_flag_block_integrated(self.h, _ptr(power), _ptr(flags), _ptr(stats_freq), _ptr(stats_time),
                                               _stream(stream)))
        return flags, stats_freq, stats_time

    def integrated_vectors(self, stream=None):
        t = self.torch
        spec = t.empty((self.S, self.Cn), dtype=t.float32, device=self.dev)
        series = t.empty((self.S, self.T), dtype=t.float32, device=self.dev)
        _check(lib().lof_integrated_vectors(self.h, _ptr(spec), _ptr(series), _stream(stream)))
        return spec, series

    def history_update(self, flags, row_flagged=None, stream=None):
        t = self.torch
        if row_flagged is None:
            row_flagged = t.empty((self.S, self.Cn), dtype=t.uint8, device=self.dev)
        _check(lib().lof_history_update(self.h, _ptr(flags), _ptr(row_flagged), _stream(stream)))
        return row_flagged

    def reset(self, stream=None):
        _check(lib().lof_reset(self.h, _stream(stream)))

    def row_sums(self, stream=None):
        """rowsum [S][C] float64 and rowcnt [S][C] (uint32 bit patterns in an int32 tensor)."""
        t = self.torch
        rs = t.empty((self.S, self.Cn), dtype=t.float64, device=self.dev)
        rc = t.empty((self.S, self.Cn), dtype=t.int32, device=self.dev)
        _check(lib().lof_row_sums(self.h, _ptr(rs), _ptr(rc), _stream(stream)))
        return rs, rc

    def history_export(self, stream=None):
        t = self.torch
        H = self.prm.history_length
        ring = t.empty((self.S, self.Cn, H), dtype=t.float32, device=self.dev)
        head = t.empty((self.S, self.Cn), dtype=t.int32, device=self.dev)
        count = t.empty((self.S, self.Cn), dtype=t.int32, device=self.dev)
        _check(lib().lof_history_export(self.h, _ptr(ring), _ptr(head), _ptr(count), _stream(stream)))
        return ring, head, count

    def flag_block_host(self, h_input, h_flags, h_stats=None):
        """End to end with HOST tensors/arrays (pinned torch tensors or numpy arrays)."""
        def hp(a):
            if a is None:
                return C.c_void_p(0)
            return C.c_void_p(a.data_ptr() if hasattr(a, "data_ptr") else a.ctypes.data)
        is_ci16 = 1 if str(h_input.dtype).endswith("int16") else 0
        _check(lib().lof_flag_block_host(self.h, hp(h_input), C.c_int(is_ci16), hp(h_flags), hp(h_stats)))

    def launch_count(self):
        return int(lib().lof_launch_count(self.h))

    def set_path(self, path):
        _check(lib().lof_set_path(self.h, C.c_int(path)))

    def path_used(self):
        return int(lib().lof_path_used(self.h))

    def set_group(self, max_streams):
        _check(lib().lof_set_group(self.h, C.c_uint32(max_streams)))

    def fused_cycles(self):
        out = (C.c_uint64 * 8)()
        _check(lib().lof_fused_cycles(self.h, out))
        return [int(v) for v in out]

    def fused_counters(self, reset=False):
        out = (C.c_uint64 * 4)()
        _check(lib().lof_fused_counters(self.h, out, C.c_int(1 if reset else 0)))
        return [int(v) for v in out]


def sir_noalloc(flags, stats, n_time, eta, directions=3, stream=None):
    """lof_sir_noalloc (include/lof.h): the SIR operator in place on a packed mask, no context, no allocation.
    flags: int32/uint32 [S][C][W] CUDA tensor; stats: uint8 [S][32] CUDA tensor (n_flagged grows)."""
    S, Cn, W = flags.shape
    assert W == (n_time + 31) // 32 and flags.is_contiguous() and stats.is_contiguous()
    _check(lib().lof_sir_noalloc(_ptr(flags), _ptr(stats), C.c_uint32(S), C.c_uint32(Cn), C.c_uint32(n_time),
                                 C.c_float(eta), C.c_uint32(directions), C.c_int(flags.device.index),
                                 _stream(stream)))


def stats_to_numpy(stats):
    """uint8 [S][32] device tensor -> numpy structured array (lof_stream_stats)."""
    return stats.cpu().numpy().view(STATS_DTYPE).reshape(-1)


def flags_to_numpy(flags):
    return flags.cpu().numpy().view(np.uint32)
