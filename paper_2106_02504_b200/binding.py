"""ctypes binding of librlxpp.so (include/rlxpp.h) -- argument marshalling only.

Every function below has the name of the C entry point it calls and does nothing but
turn torch tensors / numpy arrays into raw pointers and check the return code; every
step of the hot path runs in the CUDA kernels of csrc/rlxpp.cu.  PyTorch supplies
device memory and the CUDA stream, nothing else.  There is no CPU fallback: if the
shared library is missing or a call fails, RlxppError is raised.
"""
import ctypes
import os

import numpy as np

from . import build as _build

RLXPP_STREAM_MAJOR = 0
RLXPP_INTERLEAVED = 1
RLXPP_AOS = 0
RLXPP_SOA = 1
RLXPP_ENGINE_UMMA = 0
RLXPP_ENGINE_IMAD = 1
RLXPP_STATIC_MAX_STREAMS = 65536
RLXPP_STATIC_SCRATCH_BYTES = 5255168

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "librlxpp.so")


class RlxppError(RuntimeError):
    pass


_lib = None

_SIGNATURES = {
    "rlxpp_create": (ctypes.c_int, [ctypes.POINTER(ctypes.c_void_p), ctypes.c_uint64, ctypes.c_uint64, ctypes.c_uint32,
                                    ctypes.c_void_p]),
    "rlxpp_destroy": (ctypes.c_int, [ctypes.c_void_p]),
    "rlxpp_skip": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_uint64]),
    "rlxpp_skip_each": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p]),
    "rlxpp_advance_states": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_uint64, ctypes.c_uint32, ctypes.c_uint32,
                                            ctypes.c_int, ctypes.c_void_p]),
    "rlxpp_generate_doubles": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_uint64, ctypes.c_int]),
    "rlxpp_generate_reduce": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_uint64]),
    "rlxpp_generate_doubles_host": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_uint64, ctypes.c_int]),
    "rlxpp_generate_reduce_host": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_uint64]),
    "rlxpp_get_state": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p,
                                       ctypes.c_void_p]),
    "rlxpp_set_state": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]),
    "rlxpp_set_state_ranlux": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]),
    "rlxpp_multiplier": (ctypes.c_int, [ctypes.c_uint32, ctypes.c_void_p]),
    "rlxpp_seed_state": (ctypes.c_int, [ctypes.c_uint64, ctypes.c_uint32, ctypes.c_void_p]),
    "rlxpp_umma_matrix": (ctypes.c_int, [ctypes.c_uint32, ctypes.c_void_p]),
    "rlxpp_set_engine": (ctypes.c_int, [ctypes.c_int]),
    "rlxpp_get_engine": (ctypes.c_int, []),
    "rlxpp_set_chunks": (ctypes.c_int, [ctypes.c_int]),
    "rlxpp_generate_u48": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_uint64, ctypes.c_int]),
    "rlxpp_generate_floats": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_uint64, ctypes.c_int]),
    "rlxpp_generate_normal": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_uint64, ctypes.c_int]),
    "rlxpp_generate_doubles_static": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_uint64, ctypes.c_uint32, ctypes.c_void_p,
                                                     ctypes.c_uint64, ctypes.c_int, ctypes.c_void_p]),
    "rlxpp_host_generate": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_uint32, ctypes.c_uint64,
                                           ctypes.c_uint64, ctypes.c_void_p]),
    "rlxpp_device_view": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p]),
    "rlxpp_generate_ragged": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_uint64,
                                             ctypes.c_int]),
    "rlxpp_generate_ragged_reduce": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p,
                                                    ctypes.c_int]),
    "rlxpp_rare_counts": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_int]),
    "rlxpp_n_streams": (ctypes.c_uint64, [ctypes.c_void_p]),
    "rlxpp_has_fixed_multiplier": (ctypes.c_int, [ctypes.c_uint32]),
    "rlxpp_launch_count": (ctypes.c_uint64, []),
    "rlxpp_measure_imad_peak": (ctypes.c_int, [ctypes.c_int, ctypes.POINTER(ctypes.c_double), ctypes.c_void_p]),
    "rlxpp_measure_hbm_write_peak": (ctypes.c_int, [ctypes.c_uint64, ctypes.c_int, ctypes.POINTER(ctypes.c_double),
                                                    ctypes.c_void_p]),
    "rlxpp_measure_hbm_write_pieces": (ctypes.c_int, [ctypes.c_uint64, ctypes.c_uint64, ctypes.c_uint32, ctypes.c_int,
                                                      ctypes.POINTER(ctypes.c_double), ctypes.c_void_p]),
    "rlxpp_last_error": (ctypes.c_char_p, []),
    "rlxpp_version": (ctypes.c_char_p, []),
}
#: every symbol include/rlxpp.h declares (tests check the header against this and the .so)
EXPORTS = tuple(_SIGNATURES)


def load(build_if_missing: bool = True):
    """Loads librlxpp.so (building it in-tree with nvcc first if it is absent or stale)."""
    global _lib
    if _lib is not None:
        return _lib
    path = LIB_PATH
    if build_if_missing:
        try:
            path = _build.build()
        except Exception as e:  # nvcc missing on the box: fall back to the shipped .so, else fail loudly
            if not os.path.exists(LIB_PATH):
                raise RlxppError(f"librlxpp.so is missing and could not be built: {e}") from e
            path = LIB_PATH
    if not os.path.exists(path):
        raise RlxppError(f"{path} not found: run `python -m paper_2106_02504_b200.build`")
    lib = ctypes.CDLL(path)
    for name, (res, args) in _SIGNATURES.items():
        fn = getattr(lib, name)  # AttributeError if the library lacks a declared symbol
        fn.restype = res
        fn.argtypes = args
    _lib = lib
    return lib


def _check(rc: int, what: str):
    if rc != 0:
        msg = load().rlxpp_last_error()
        raise RlxppError(f"{what} failed ({rc}): {msg.decode() if msg else ''}")


def _ptr(t):
    """Raw address of a torch tensor (device or host), numpy array, int or None."""
    if t is None:
        return None
    if isinstance(t, int):
        return t
    if isinstance(t, np.ndarray):
        if not t.flags["C_CONTIGUOUS"]:
            raise RlxppError("numpy buffer must be C-contiguous")
        return t.ctypes.data
    if not t.is_contiguous():
        raise RlxppError("tensor must be contiguous")
    return t.data_ptr()


def _current_stream():
    import torch
    return torch.cuda.current_stream().cuda_stream


class Handle:
    """Owns an rlxpp_t*; destroyed on close() / garbage collection."""

    def __init__(self, ptr, n_streams, p):
        self.ptr = ptr
        self.n_streams = n_streams
        self.p = p

    def close(self):
        if self.ptr:
            load().rlxpp_destroy(self.ptr)
            self.ptr = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def rlxpp_create(n_streams: int, seed: int, p: int, cuda_stream=None) -> Handle:
    h = ctypes.c_void_p()
    s = _current_stream() if cuda_stream is None else cuda_stream
    _check(load().rlxpp_create(ctypes.byref(h), n_streams, seed & (2**64 - 1), p, s), "rlxpp_create")
    return Handle(h, n_streams, p)


def rlxpp_destroy(h: Handle):
    h.close()


def rlxpp_skip(h: Handle, n: int):
    _check(load().rlxpp_skip(h.ptr, n), "rlxpp_skip")


def rlxpp_skip_each(h: Handle, n_dev):
    _check(load().rlxpp_skip_each(h.ptr, _ptr(n_dev)), "rlxpp_skip_each")


def rlxpp_advance_states(states_dev, n_states: int, p: int, reps: int, layout: int = RLXPP_AOS, cuda_stream=None):
    s = _current_stream() if cuda_stream is None else cuda_stream
    _check(load().rlxpp_advance_states(_ptr(states_dev), n_states, p, reps, layout, s), "rlxpp_advance_states")


def rlxpp_generate_doubles(h: Handle, out_dev, n_per_stream: int, layout: int = RLXPP_STREAM_MAJOR):
    _check(load().rlxpp_generate_doubles(h.ptr, _ptr(out_dev), n_per_stream, layout), "rlxpp_generate_doubles")


def rlxpp_generate_reduce(h: Handle, sum_dev, sumsq_dev, n_per_stream: int):
    _check(load().rlxpp_generate_reduce(h.ptr, _ptr(sum_dev), _ptr(sumsq_dev), n_per_stream), "rlxpp_generate_reduce")


def rlxpp_generate_u48(h: Handle, out_dev, n_per_stream: int, layout: int = RLXPP_STREAM_MAJOR):
    _check(load().rlxpp_generate_u48(h.ptr, _ptr(out_dev), n_per_stream, layout), "rlxpp_generate_u48")


def rlxpp_generate_floats(h: Handle, out_dev, n_per_stream: int, layout: int = RLXPP_STREAM_MAJOR):
    _check(load().rlxpp_generate_floats(h.ptr, _ptr(out_dev), n_per_stream, layout), "rlxpp_generate_floats")


def rlxpp_generate_normal(h: Handle, out_dev, n_per_stream: int, layout: int = RLXPP_STREAM_MAJOR):
    _check(load().rlxpp_generate_normal(h.ptr, _ptr(out_dev), n_per_stream, layout), "rlxpp_generate_normal")


def rlxpp_generate_doubles_static(lcg_dev, n_streams: int, p: int, out_dev, n_per_stream: int,
                                  layout: int = RLXPP_STREAM_MAJOR, cuda_stream=None):
    """The generator for callers that must not allocate device memory (include/rlxpp.h): states in, doubles and
    advanced states out, scratch in the library's own fixed device array (at most RLXPP_STATIC_MAX_STREAMS streams)."""
    s = _current_stream() if cuda_stream is None else cuda_stream
    _check(load().rlxpp_generate_doubles_static(_ptr(lcg_dev), n_streams, p, _ptr(out_dev), n_per_stream, layout, s),
           "rlxpp_generate_doubles_static")


def rlxpp_host_generate(lcg: np.ndarray, pos: int, p: int, skip: int, n: int):
    """-> (doubles[n], new lcg uint64[9], new cursor); host only."""
    state = np.ascontiguousarray(lcg, dtype=np.uint64).copy()
    cur = ctypes.c_uint32(pos)
    out = np.empty(max(n, 1), np.float64)
    _check(load().rlxpp_host_generate(state.ctypes.data, ctypes.addressof(cur), p, skip & (2**64 - 1), n, out.ctypes.data),
           "rlxpp_host_generate")
    return out[:n], state, int(cur.value)


class RlxppView(ctypes.Structure):
    """rlxpp_view_t of include/rlxpp_device.cuh: what a kernel using the device API takes."""
    _fields_ = [("st", ctypes.c_void_p), ("n", ctypes.c_uint64), ("A", ctypes.c_void_p), ("bmat", ctypes.c_void_p)]


def rlxpp_device_view(h: Handle) -> RlxppView:
    v = RlxppView()
    _check(load().rlxpp_device_view(h.ptr, ctypes.addressof(v)), "rlxpp_device_view")
    return v


def rlxpp_generate_ragged(h: Handle, counts_dev, out_dev, ld: int, cooperative=True):
    _check(load().rlxpp_generate_ragged(h.ptr, _ptr(counts_dev), _ptr(out_dev), ld, int(cooperative)),
           "rlxpp_generate_ragged")


def rlxpp_generate_ragged_reduce(h: Handle, counts_dev, sum_dev, sumsq_dev, cooperative=True):
    _check(load().rlxpp_generate_ragged_reduce(h.ptr, _ptr(counts_dev), _ptr(sum_dev), _ptr(sumsq_dev), int(cooperative)),
           "rlxpp_generate_ragged_reduce")


def rlxpp_generate_doubles_host(h: Handle, out_host, n_per_stream: int, layout: int = RLXPP_STREAM_MAJOR):
    _check(load().rlxpp_generate_doubles_host(h.ptr, _ptr(out_host), n_per_stream, layout),
           "rlxpp_generate_doubles_host")


def rlxpp_generate_reduce_host(h: Handle, sum_host, sumsq_host, n_per_stream: int):
    _check(load().rlxpp_generate_reduce_host(h.ptr, _ptr(sum_host), _ptr(sumsq_host), n_per_stream),
           "rlxpp_generate_reduce_host")


def rlxpp_get_state(h: Handle, ranlux_dev=None, carry_dev=None, pos_dev=None, lcg_dev=None):
    _check(load().rlxpp_get_state(h.ptr, _ptr(ranlux_dev), _ptr(carry_dev), _ptr(pos_dev), _ptr(lcg_dev)),
           "rlxpp_get_state")


def rlxpp_set_state(h: Handle, lcg_dev, pos_dev=None):
    _check(load().rlxpp_set_state(h.ptr, _ptr(lcg_dev), _ptr(pos_dev)), "rlxpp_set_state")


def rlxpp_set_state_ranlux(h: Handle, ranlux_dev, carry_dev=None, pos_dev=None):
    _check(load().rlxpp_set_state_ranlux(h.ptr, _ptr(ranlux_dev), _ptr(carry_dev), _ptr(pos_dev)), "rlxpp_set_state_ranlux")


def rlxpp_multiplier(p: int) -> np.ndarray:
    out = np.zeros(9, np.uint64)
    _check(load().rlxpp_multiplier(p, out.ctypes.data), "rlxpp_multiplier")
    return out


def rlxpp_seed_state(seed: int, p: int) -> np.ndarray:
    out = np.zeros(9, np.uint64)
    _check(load().rlxpp_seed_state(seed & (2**64 - 1), p, out.ctypes.data), "rlxpp_seed_state")
    return out


def rlxpp_umma_matrix(p: int) -> np.ndarray:
    out = np.zeros((72, 72), np.uint8)
    _check(load().rlxpp_umma_matrix(p, out.ctypes.data), "rlxpp_umma_matrix")
    return out


def rlxpp_set_engine(engine: int):
    _check(load().rlxpp_set_engine(engine), "rlxpp_set_engine")


def rlxpp_set_chunks(n_chunks: int):
    _check(load().rlxpp_set_chunks(n_chunks), "rlxpp_set_chunks")


def rlxpp_get_engine() -> int:
    return int(load().rlxpp_get_engine())


RLXPP_RARE_KINDS = 8
RLXPP_RARE_NAMES = ("fold_borrow", "fold_carry", "fold_top", "ranlux_carry", "ranlux_near", "ranlux_umax", "ranlux_v0",
                    "ranlux_third")


def rlxpp_rare_counts(reset: bool = False) -> np.ndarray:
    out = np.zeros(RLXPP_RARE_KINDS, np.uint64)
    _check(load().rlxpp_rare_counts(out.ctypes.data, int(reset)), "rlxpp_rare_counts")
    return out


def rlxpp_n_streams(h: Handle) -> int:
    return int(load().rlxpp_n_streams(h.ptr))


def rlxpp_has_fixed_multiplier(p: int) -> bool:
    return bool(load().rlxpp_has_fixed_multiplier(p))


def rlxpp_launch_count() -> int:
    return int(load().rlxpp_launch_count())


def rlxpp_measure_imad_peak(iters: int = 5, cuda_stream=None) -> float:
    out = ctypes.c_double(0.0)
    s = _current_stream() if cuda_stream is None else cuda_stream
    _check(load().rlxpp_measure_imad_peak(iters, ctypes.byref(out), s), "rlxpp_measure_imad_peak")
    return out.value


def rlxpp_measure_hbm_write_peak(nbytes: int, iters: int = 5, cuda_stream=None) -> float:
    out = ctypes.c_double(0.0)
    s = _current_stream() if cuda_stream is None else cuda_stream
    _check(load().rlxpp_measure_hbm_write_peak(nbytes, iters, ctypes.byref(out), s), "rlxpp_measure_hbm_write_peak")
    return out.value


def rlxpp_measure_hbm_write_pieces(rows: int, pitch_bytes: int, piece_bytes: int, iters: int = 3, cuda_stream=None) -> float:
    out = ctypes.c_double(0.0)
    s = _current_stream() if cuda_stream is None else cuda_stream
    _check(load().rlxpp_measure_hbm_write_pieces(rows, pitch_bytes, piece_bytes, iters, ctypes.byref(out), s),
           "rlxpp_measure_hbm_write_pieces")
    return out.value


def rlxpp_last_error() -> str:
    return load().rlxpp_last_error().decode()


def rlxpp_version() -> str:
    return load().rlxpp_version().decode()
