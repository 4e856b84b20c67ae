"""ctypes binding of the C++ oracle (oracle/rlxpp_oracle.cpp).  TEST INFRASTRUCTURE ONLY.

Every function here only marshals numpy arrays into the C calls; all the
arithmetic is in the C++ file, which cites the paper passage each step follows.
Big integers cross the boundary as little-endian uint64[9] / uint64[18].
"""
import ctypes
import os

import numpy as np

from . import build as _build

_lib = ctypes.CDLL(_build.build())

_u64p = ctypes.POINTER(ctypes.c_uint64)
_u32p = ctypes.POINTER(ctypes.c_uint32)
_u8p = ctypes.POINTER(ctypes.c_uint8)
_f64p = ctypes.POINTER(ctypes.c_double)


def _p(a, t):
    return None if a is None else a.ctypes.data_as(t)


def int_to_limbs(x: int, n: int = 9) -> np.ndarray:
    return np.array([(x >> (64 * i)) & (2**64 - 1) for i in range(n)], dtype=np.uint64)


def limbs_to_int(a) -> int:
    return sum(int(v) << (64 * i) for i, v in enumerate(np.asarray(a).reshape(-1)))


def modulus() -> int:
    out = np.zeros(9, np.uint64)
    _lib.orc_modulus(_p(out, _u64p))
    return limbs_to_int(out)


def multiply9x9(a: int, b: int) -> int:
    out = np.zeros(18, np.uint64)
    _lib.orc_multiply9x9(_p(int_to_limbs(a), _u64p), _p(int_to_limbs(b), _u64p), _p(out, _u64p))
    return limbs_to_int(out)


def mod_m(z: int) -> int:
    out = np.zeros(9, np.uint64)
    _lib.orc_mod_m(_p(int_to_limbs(z, 18), _u64p), _p(out, _u64p))
    return limbs_to_int(out)


def mod_m_longdiv(z: int) -> int:
    out = np.zeros(9, np.uint64)
    _lib.orc_mod_m_longdiv(_p(int_to_limbs(z, 18), _u64p), _p(out, _u64p))
    return limbs_to_int(out)


def mulmod(a: int, b: int) -> int:
    out = np.zeros(9, np.uint64)
    _lib.orc_mulmod(_p(int_to_limbs(a), _u64p), _p(int_to_limbs(b), _u64p), _p(out, _u64p))
    return limbs_to_int(out)


def powmod(base: int, e: int) -> int:
    ne = max(1, (e.bit_length() + 63) // 64)
    out = np.zeros(9, np.uint64)
    _lib.orc_powmod(_p(int_to_limbs(base), _u64p), _p(int_to_limbs(e, ne), _u64p), ctypes.c_int(ne), _p(out, _u64p))
    return limbs_to_int(out)


def multiplier(p: int) -> int:
    out = np.zeros(9, np.uint64)
    _lib.orc_multiplier(ctypes.c_uint32(p), _p(out, _u64p))
    return limbs_to_int(out)


def swb_steps(V: int, c: int, nsteps: int):
    v = int_to_limbs(V)
    cc = ctypes.c_uint(c)
    _lib.orc_swb_steps(_p(v, _u64p), ctypes.byref(cc), ctypes.c_uint64(nsteps))
    return limbs_to_int(v), int(cc.value)


def to_lcg(V: int, c: int) -> int:
    out = np.zeros(9, np.uint64)
    _lib.orc_to_lcg(_p(int_to_limbs(V), _u64p), ctypes.c_uint(c), _p(out, _u64p))
    return limbs_to_int(out)


def to_ranlux(X: int):
    out = np.zeros(9, np.uint64)
    cc = ctypes.c_uint(0)
    _lib.orc_to_ranlux(_p(int_to_limbs(X), _u64p), _p(out, _u64p), ctypes.byref(cc))
    return limbs_to_int(out), int(cc.value)


def to_ranlux_def(X: int):
    out = np.zeros(9, np.uint64)
    cc = ctypes.c_uint(0)
    _lib.orc_to_ranlux_def(_p(int_to_limbs(X), _u64p), _p(out, _u64p), ctypes.byref(cc))
    return limbs_to_int(out), int(cc.value)


def seed_state(seed: int, p: int) -> int:
    out = np.zeros(9, np.uint64)
    _lib.orc_seed_state(ctypes.c_uint64(seed), ctypes.c_uint32(p), _p(out, _u64p))
    return limbs_to_int(out)


def seed_state_exp(seed: int, p: int, log2e: int) -> int:
    out = np.zeros(9, np.uint64)
    _lib.orc_seed_state_exp(ctypes.c_uint64(seed), ctypes.c_uint32(p), ctypes.c_int(log2e), _p(out, _u64p))
    return limbs_to_int(out)


def hardware_threads() -> int:
    return int(_lib.orc_hardware_threads())


def advance_states(states: np.ndarray, p: int, reps: int, nthreads: int = 1) -> np.ndarray:
    """states: [n][9] uint64 (AoS).  Returns a new array: A^reps x mod m, canonical."""
    out = np.ascontiguousarray(states, dtype=np.uint64).copy()
    assert out.ndim == 2 and out.shape[1] == 9
    _lib.orc_advance_states(_p(out, _u64p), ctypes.c_uint64(out.shape[0]), ctypes.c_uint32(p),
                            ctypes.c_uint32(reps), ctypes.c_int(nthreads))
    return out


def streams(seeds, p: int, n_per_stream: int, skips=None, want=("doubles",), nthreads: int = 1) -> dict:
    """Generates stream-major outputs for the given seeds.  want: any of
    'ints', 'doubles', 'sums', 'state'."""
    seeds = np.ascontiguousarray(seeds, dtype=np.uint64)
    n = seeds.shape[0]
    sk = None if skips is None else np.ascontiguousarray(skips, dtype=np.uint64)
    res = {}
    out48 = np.zeros((n, n_per_stream), np.uint64) if "ints" in want else None
    outd = np.zeros((n, n_per_stream), np.float64) if "doubles" in want else None
    s = np.zeros(n, np.float64) if "sums" in want else None
    q = np.zeros(n, np.float64) if "sums" in want else None
    st = "state" in want
    X = np.zeros((n, 9), np.uint64) if st else None
    V = np.zeros((n, 9), np.uint64) if st else None
    c = np.zeros(n, np.uint32) if st else None
    pos = np.zeros(n, np.uint32) if st else None
    _lib.orc_streams(_p(seeds, _u64p), _p(sk, _u64p), ctypes.c_uint64(n), ctypes.c_uint32(p),
                     ctypes.c_uint64(n_per_stream), _p(out48, _u64p), _p(outd, _f64p), _p(s, _f64p), _p(q, _f64p),
                     _p(X, _u64p), _p(V, _u64p), _p(c, _u32p), _p(pos, _u32p), ctypes.c_int(nthreads))
    if out48 is not None:
        res["ints"] = out48
    if outd is not None:
        res["doubles"] = outd
    if s is not None:
        res["sum"], res["sumsq"] = s, q
    if st:
        res["X"], res["V"], res["c"], res["pos"] = X, V, c, pos
    return res


def engine_run(X: int, pos: int, p: int, ops):
    """ops: list of ('draw', n) / ('skip', n).  Returns (X, pos, [48-bit ints drawn])."""
    x = int_to_limbs(X)
    pp = ctypes.c_uint(pos)
    is_skip = np.array([1 if o[0] == "skip" else 0 for o in ops], np.uint8)
    amount = np.array([o[1] for o in ops], np.uint64)
    ndraw = int(sum(o[1] for o in ops if o[0] == "draw"))
    out = np.zeros(max(ndraw, 1), np.uint64)
    _lib.orc_engine_run(_p(x, _u64p), ctypes.byref(pp), ctypes.c_uint32(p), _p(is_skip, _u8p), _p(amount, _u64p),
                        ctypes.c_int(len(ops)), _p(out, _u64p))
    return limbs_to_int(x), int(pp.value), [int(v) for v in out[:ndraw]]


def normals(k48) -> np.ndarray:
    """Box-Muller normals of consecutive PAIRS of 48-bit draws along the last axis (even length)."""
    k = np.ascontiguousarray(k48, dtype=np.uint64)
    assert k.shape[-1] % 2 == 0
    z = np.zeros(k.shape, np.float64)
    _lib.orc_normals(_p(k, _u64p), ctypes.c_uint64(k.size // 2), _p(z, _f64p))
    return z
