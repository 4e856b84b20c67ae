"""CPU tests of the C-ABI library itself: it loads, exports every symbol include/rlxpp.h declares,
and its HOST logic (multiplier, seed state, the byte matrix of the UMMA engine) is right, checked
against Python big integers -- not against the oracle, which shares no code with the library.
No kernel is launched here; on a box without a GPU every compute entry point must fail loudly."""
import ctypes
import os
import re

import numpy as np
import pytest

import paper_2106_02504_b200 as rlx

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
M = (1 << 576) - (1 << 240) + 1
A1 = M - (M - 1) // (1 << 24)    # D2: a = b^-1 mod m


def to_int(limbs):
    return sum(int(v) << (64 * i) for i, v in enumerate(limbs))


def test_library_exports_every_declared_symbol():
    header = open(os.path.join(ROOT, "include", "rlxpp.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\b(rlxpp_[a-z0-9_]+)\s*\(", header))
    assert declared, "no declarations found in include/rlxpp.h"
    assert declared == set(rlx.EXPORTS), declared ^ set(rlx.EXPORTS)
    lib = rlx.load()
    raw = ctypes.CDLL(rlx.LIB_PATH)
    for name in declared:
        assert hasattr(raw, name), name
    assert lib.rlxpp_version().decode().startswith("rlxpp")


@pytest.mark.parametrize("p", [1, 24, 389, 1024, 2048, 100])
def test_host_multiplier_is_a_pow_p(p):
    assert (A1 << 24) % M == 1
    assert to_int(rlx.rlxpp_multiplier(p)) == pow(A1, p, M)


def test_host_seed_state_is_power_of_the_multiplier():
    for seed in (0, 1, 2, 1024, 2**64 - 1):
        assert to_int(rlx.rlxpp_seed_state(seed, 2048)) == pow(A1, 2048 * (1 << 96) * seed, M)


@pytest.mark.parametrize("p", [24, 389, 2048, 7])
def test_umma_byte_matrix_reproduces_the_modular_product(p):
    """sum_n (sum_k xb_k B[n][k]) 2^(8n) == A x (mod m), every column sum < 2^23 (so the s32
    accumulators of tcgen05.mma kind::i8 are exact) and the total < 2^591 (one 15-bit fold)."""
    B = rlx.rlxpp_umma_matrix(p).astype(object)
    A = pow(A1, p, M)
    for k in range(72):  # column k of the matrix is A 2^(8k) mod m, canonical
        Rk = sum(int(B[n][k]) << (8 * n) for n in range(72))
        assert Rk == (A << (8 * k)) % M
    rng = np.random.default_rng(20210602 + p)
    xs = [int.from_bytes(rng.bytes(72), "little") for _ in range(40)]
    xs += [0, 1, M - 1, M, (1 << 576) - 1, M - (1 << 240), int.from_bytes(b"\xff" * 72, "little")]
    for x in xs:
        xb = np.array(list(x.to_bytes(72, "little")), dtype=object)
        acc = [int(sum(int(B[n][k]) * int(xb[k]) for k in range(72))) for n in range(72)]
        assert max(acc) < 1 << 23
        z = sum(a << (8 * n) for n, a in enumerate(acc))
        assert z < 1 << 591
        assert z % M == A * x % M


def test_engine_selection_and_errors_without_gpu():
    assert rlx.rlxpp_get_engine() == rlx.RLXPP_ENGINE_UMMA
    rlx.rlxpp_set_engine(rlx.RLXPP_ENGINE_IMAD)
    assert rlx.rlxpp_get_engine() == rlx.RLXPP_ENGINE_IMAD
    rlx.rlxpp_set_engine(rlx.RLXPP_ENGINE_UMMA)
    with pytest.raises(rlx.RlxppError, match="unknown engine"):
        rlx.rlxpp_set_engine(7)
    with pytest.raises(rlx.RlxppError):
        rlx.rlxpp_multiplier(0)
    import torch
    if not torch.cuda.is_available():  # no CPU fallback: creation must fail, not compute on the host
        with pytest.raises(rlx.RlxppError):
            rlx.rlxpp_create(16, 1, 2048, cuda_stream=0)


# ---------------------------------------------------------------- host engine
def _py_stream(X, pos, A, n):
    """Python big-integer model of D4 / D6 / D8, written here (closed form V = floor(2^576 X / m))."""
    out = []
    for _ in range(n):
        if pos == 12:
            X, pos = A * X % M, 0
        V = (X << 576) // M
        out.append((V >> (48 * pos)) & ((1 << 48) - 1))
        pos += 1
    return out, X, pos


def _limbs(x):
    return np.array([(x >> (64 * i)) & (2**64 - 1) for i in range(9)], dtype=np.uint64)


@pytest.mark.parametrize("p", [2048, 24, 389])
def test_host_engine_matches_big_integer_model(p):
    A = pow(A1, p, M)
    X0 = pow(A, (1 << 96) * 1, M)  # seed 1 (reading c-7)
    d, st, pos = rlx.rlxpp_host_generate(_limbs(X0), 12, p, 0, 40)
    want, Xe, pe = _py_stream(X0, 12, A, 40)
    assert [int(v * 2.0**48) for v in d] == want and to_int(st) == Xe and pos == pe
    if p == 2048:  # survey vectors: first three draws of seed 1
        assert want[:3] == [0x2e3ae8639566, 0x2508dc725c8a, 0xa279f7cf2ea3]
    # continue from the returned state with a skip: one sequence
    for skip in (0, 1, 11, 12, 13, 2**40 + 7, 2**64 - 1):
        d2, st2, pos2 = rlx.rlxpp_host_generate(st, pos, p, skip, 15)
        k = (pe + skip - 1) // 12 if skip else 0
        Xs = pow(A, k, M) * Xe % M
        ps = pe + skip - 12 * k
        want2, X2, p2 = _py_stream(Xs, ps, A, 15)
        assert [int(v * 2.0**48) for v in d2] == want2 and to_int(st2) == X2 and pos2 == p2
    # non-canonical input (>= m) is reduced; the zero state is a fixed point with all draws 0.0
    d3, st3, _ = rlx.rlxpp_host_generate(_limbs(M + 5), 12, p, 0, 3)
    assert [int(v * 2.0**48) for v in d3] == _py_stream(5, 12, A, 3)[0]
    d4, st4, _ = rlx.rlxpp_host_generate(_limbs(0), 3, p, 0, 20)
    assert not d4.any() and to_int(st4) == 0
    with pytest.raises(rlx.RlxppError):
        rlx.rlxpp_host_generate(_limbs(1), 13, p, 0, 1)


@pytest.mark.parametrize("example", ["device_api_example.cu", "tile_api_example.cu", "fixed_api_example.cu"])
def test_public_device_header_is_self_contained(tmp_path, example):
    """include/rlxpp_device.cuh (per-thread generator) and include/rlxpp_tile.cuh (block-cooperative tensor-core
    advance) alone are enough to write a kernel: nvcc compiles a user kernel that includes nothing else
    (cross-compilation for sm_100a, no GPU needed)."""
    import shutil
    import subprocess
    nvcc = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(nvcc):
        pytest.skip("nvcc not found")
    src = os.path.join(ROOT, "tests", "data", example)
    res = subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-std=c++17", "-I", os.path.join(ROOT, "include"),
                          "-c", src, "-o", str(tmp_path / "example.o")], capture_output=True, text=True)
    assert res.returncode == 0, res.stdout + res.stderr


def test_fixed_multiplier_rows_header_is_what_its_generator_writes(tmp_path):
    """include/rlxpp_rows.cuh (the IMAD engine's 4 x 324 immediates) is committed although build() regenerates it;
    it must be exactly csrc/gen_rows.py's output, and its immediates must be the limbs of A 2^(32 i) mod m."""
    import importlib.util
    import re
    here = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "paper_2106_02504_b200", "csrc")
    spec = importlib.util.spec_from_file_location("gen_rows", os.path.join(here, "gen_rows.py"))
    gen = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(gen)
    tracked = open(os.path.join(ROOT, "include", "rlxpp_rows.cuh")).read()
    body = "\n\n".join(gen.emit_level(p) for p in gen.LEVELS)
    assert body in tracked, "include/rlxpp_rows.cuh is stale: run python -m paper_2106_02504_b200.build"
    # the immediates themselves, against Python: row i of level p = limbs of a^p 2^(32 i) mod m (324 per level)
    for p, block in zip(gen.LEVELS, re.split(r"// ---- p = \d+:", tracked)[1:]):
        A = pow(A1, p, M)
        kA = [int(v, 16) for v in re.findall(r"0x([0-9a-f]{8})u", block.split("kA[18]")[1].split(";")[0])]
        assert sum(v << (32 * i) for i, v in enumerate(kA)) == A
        row0 = [int(v, 16) for v in re.findall(r"x\[0\] \* 0x([0-9a-f]{8})u", block)]
        assert len(row0) == 18
        rows = {0: [row0[2 * (k // 2) + (k % 2)] for k in range(18)]}  # E[k], O[k] pairs are columns 2k, 2k + 1
        for i, asm in enumerate(re.findall(r"// row (\d+)\n(.*?)\"}\"", block, re.S)):
            imm = [int(v, 16) for v in re.findall(r"%20, 0x([0-9a-f]{8});", asm[1])]
            assert len(imm) == 18 and int(asm[0]) == i + 1
            rows[i + 1] = [imm[k // 2] if k % 2 == 0 else imm[9 + k // 2] for k in range(18)]  # even chain, then odd chain
        assert len(rows) == 18
        for i in range(18):
            assert sum(v << (32 * k) for k, v in enumerate(rows[i])) == (A << (32 * i)) % M, (p, i)


def test_normal_coefficients_header_is_what_its_generator_writes():
    """csrc/normal_coeffs.cuh (polynomials of rlxpp_generate_normal) is committed; it must be the output of
    csrc/gen_normal_coeffs.py (mpmath near-minimax fits), and the fits must be as good as the header says."""
    mp = pytest.importorskip("mpmath")
    import importlib.util
    here = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "paper_2106_02504_b200", "csrc")
    spec = importlib.util.spec_from_file_location("gen_normal_coeffs", os.path.join(here, "gen_normal_coeffs.py"))
    gen = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(gen)
    text = gen.render()
    assert text == open(os.path.join(here, "normal_coeffs.cuh")).read()
    # independent of chebyfit's own error estimate: sin(pi r), cos(pi r) and ln(m) rebuilt in exact arithmetic from the
    # printed fp64 coefficients (their rounding included): within 2^-54 = a quarter ulp
    import re
    polys = {}
    for name, body in re.findall(r"void poly_(\w+)\(.*?\{(.*?)\n\}", text, re.S):
        polys[name] = [mp.mpf(float.fromhex(c)) for c in re.findall(r"(-?0x[0-9a-f.]+p[+-]\d+)\)?;", body)]
    assert {k: len(v) for k, v in polys.items()} == {"sinpi": 7, "cospi": 7, "atanh": 8}
    horner = lambda cs, z: mp.polyval(cs, z)
    for t in range(0, 101):
        r = mp.mpf(t) / 400  # |r| <= 1/4
        z = r * r
        s = r * (mp.pi + z * horner(polys["sinpi"], z))
        c = 1 + z * horner(polys["cospi"], z)
        assert abs(s - mp.sin(mp.pi * r)) <= mp.mpf(2) ** -54 * max(mp.sin(mp.pi * r), mp.mpf(10) ** -30)
        assert abs(c - mp.cos(mp.pi * r)) <= mp.mpf(2) ** -54
        m = mp.sqrt(mp.mpf(1) / 2) + (mp.sqrt(2) - mp.sqrt(mp.mpf(1) / 2)) * t / 100
        sv = (m - 1) / (m + 1)
        zz = sv * sv
        ln = 2 * sv + sv * zz * horner(polys["atanh"], zz)
        assert abs(ln - mp.log(m)) <= mp.mpf(2) ** -54 * max(abs(mp.log(m)), mp.mpf(10) ** -30)
