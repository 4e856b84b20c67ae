"""Out-of-bounds writes, checked by the library's own means: every device buffer a kernel family writes is carved out of a
larger allocation whose margins hold a sentinel, and the margins must come back untouched.

compute-sanitizer cannot be run on the GPU pool this project is measured on (profiles/sanitizer_r03.md), so this is the
memcheck stand-in for stores: it covers each output path of each entry point -- direct stores, the shared-memory stages
feeding TMA boxes (whole-block rows, rings for shifted rows, the warp's row stage for odd pitches, float row boxes), the
fused sums, the ragged device-API kernels, the raw advance in both layouts, state export and the static-scratch entry
point -- on a stream count with a ragged last tile, with one common cursor, an odd common cursor and per-stream cursors,
and with the work cut into chunks.  What the buffers must CONTAIN is the parity tests' business (tests/test_gpu_parity.py);
here only: nothing is written outside them, and every element inside is written (no sentinel left), where the call
defines all of them.
"""
import numpy as np
import pytest

from paper_2106_02504_b200 import inputs

pytestmark = pytest.mark.gpu

SENTINEL = np.array([0xA5A5A5A5A5A5A5A5], np.uint64).view(np.int64)[0]  # as a double: -1.6e-129, never a draw
GUARD = 4096  # 8-byte words on each side (32 KB: wider than any box or row piece the kernels store)


@pytest.fixture(scope="module")
def torch():
    import torch as _torch
    if not _torch.cuda.is_available():
        pytest.fail("the gpu-marked tests need a CUDA device (there is no CPU fallback)")
    return _torch


@pytest.fixture(scope="module")
def rlx(torch):
    import paper_2106_02504_b200 as _rlx
    _rlx.load()
    _rlx.rlxpp_set_engine(_rlx.RLXPP_ENGINE_UMMA)
    yield _rlx
    _rlx.rlxpp_set_chunks(0)
    _rlx.rlxpp_set_engine(_rlx.RLXPP_ENGINE_UMMA)


class Guarded:
    """`words` 8-byte words between two sentinel margins; .t is the interior as int64 (16-byte aligned)."""

    def __init__(self, torch, words):
        self.torch = torch
        self.buf = torch.full((GUARD + words + GUARD,), int(SENTINEL), dtype=torch.int64, device="cuda")
        self.t = self.buf[GUARD:GUARD + words]
        assert self.t.data_ptr() % 16 == 0

    def check(self, what, full=True):
        self.torch.cuda.synchronize()
        lo, hi = self.buf[:GUARD], self.buf[GUARD + self.t.numel():]
        assert bool((lo == int(SENTINEL)).all()), f"{what}: wrote below the buffer"
        assert bool((hi == int(SENTINEL)).all()), f"{what}: wrote past the buffer"
        if full:
            assert not bool((self.t == int(SENTINEL)).any()), f"{what}: left elements of the buffer unwritten"


def cursors(rlx, torch, h, kind):
    if kind == "odd":
        rlx.rlxpp_skip(h, 3)
    elif kind == "even":
        rlx.rlxpp_skip(h, 2)
    elif kind == "each":
        rlx.rlxpp_skip_each(h, torch.from_numpy(inputs.cfg5_skip_distances(h.n_streams).view(np.int64)).cuda())


@pytest.mark.parametrize("chunks", [0, 3])
@pytest.mark.parametrize("kind", ["aligned", "even", "odd", "each"])
def test_generate_calls_stay_inside_their_buffers(rlx, torch, kind, chunks):
    n = 300  # two whole tiles of 128 and a ragged one
    rlx.rlxpp_set_chunks(chunks)
    for layout in (rlx.RLXPP_STREAM_MAJOR, rlx.RLXPP_INTERLEAVED):
        for per in (96, 38, 200, 1536 if kind == "aligned" else 122):
            h = rlx.rlxpp_create(n, 1, 2048)
            cursors(rlx, torch, h, kind)
            what = f"{kind} cursors, layout {layout}, {per} per stream, chunks {chunks}"
            g = Guarded(torch, n * per)
            rlx.rlxpp_generate_doubles(h, g.t.view(torch.float64), per, layout)
            g.check("doubles: " + what)
            g = Guarded(torch, n * per)
            rlx.rlxpp_generate_u48(h, g.t, per, layout)
            g.check("u48: " + what)
            g = Guarded(torch, n * per // 2)
            rlx.rlxpp_generate_floats(h, g.t.view(torch.float32), per, layout)
            g.check("floats: " + what)
            g = Guarded(torch, n * per)
            rlx.rlxpp_generate_normal(h, g.t.view(torch.float64), per, layout)
            g.check("normal: " + what)
            S, Q = Guarded(torch, n), Guarded(torch, n)
            rlx.rlxpp_generate_reduce(h, S.t.view(torch.float64), Q.t.view(torch.float64), per)
            S.check("sum: " + what)
            Q.check("sumsq: " + what)
            rlx.rlxpp_destroy(h)
    rlx.rlxpp_set_chunks(0)


def test_short_calls_in_time_parallel_lanes_stay_inside_their_buffers(rlx, torch):
    n = 300
    for layout in (rlx.RLXPP_STREAM_MAJOR, rlx.RLXPP_INTERLEAVED):
        h = rlx.rlxpp_create(n, 1, 2048)
        for per in (384, 96, 48):  # K = 32, 8, 4 lanes per tile
            g = Guarded(torch, n * per)
            rlx.rlxpp_generate_doubles(h, g.t.view(torch.float64), per, layout)
            g.check(f"lanes, layout {layout}, {per} per stream")
            g = Guarded(torch, n * per // 2)
            rlx.rlxpp_generate_floats(h, g.t.view(torch.float32), per, layout)
            g.check(f"lanes floats, layout {layout}, {per} per stream")
        rlx.rlxpp_destroy(h)


@pytest.mark.parametrize("mode", [0, 1, 2, 3])
def test_device_api_kernels_stay_inside_their_buffers(rlx, torch, mode):
    n, ld = 300, 40
    h = rlx.rlxpp_create(n, 1, 2048)
    cursors(rlx, torch, h, "each")
    cnt = torch.from_numpy((inputs.splitmix64(7, n) % np.uint64(ld + 1)).astype(np.uint32).view(np.int32)).cuda()
    g = Guarded(torch, n * ld)
    rlx.rlxpp_generate_ragged(h, cnt, g.t.view(torch.float64), ld, mode)
    g.check(f"ragged mode {mode}", full=False)  # entries beyond a stream's count stay untouched by contract
    S, Q = Guarded(torch, n), Guarded(torch, n)
    rlx.rlxpp_generate_ragged_reduce(h, cnt, S.t.view(torch.float64), Q.t.view(torch.float64), mode)
    S.check(f"ragged sum mode {mode}")
    Q.check(f"ragged sumsq mode {mode}")
    rlx.rlxpp_destroy(h)


@pytest.mark.parametrize("engine", ["umma", "imad"])
def test_raw_advance_and_state_export_stay_inside_their_buffers(rlx, torch, engine):
    rlx.rlxpp_set_engine(rlx.RLXPP_ENGINE_UMMA if engine == "umma" else rlx.RLXPP_ENGINE_IMAD)
    try:
        n = 1001  # odd: the last pair of tiles is half empty and ragged
        src = torch.from_numpy(inputs.cfg2_states(n - 64).view(np.int64)).cuda().reshape(n, 9)
        for layout, data in ((rlx.RLXPP_AOS, src), (rlx.RLXPP_SOA, src.t().contiguous())):
            for p in (2048, 777):
                g = Guarded(torch, 9 * n)
                g.t.copy_(data.reshape(-1))
                rlx.rlxpp_advance_states(g.t, n, p, 3, layout)
                g.check(f"advance_states {engine} layout {layout} p {p}", full=False)
        h = rlx.rlxpp_create(300, 9, 389)
        V, X, c, pos = Guarded(torch, 2700), Guarded(torch, 2700), Guarded(torch, 150), Guarded(torch, 150)
        rlx.rlxpp_get_state(h, V.t, c.t.view(torch.int32), pos.t.view(torch.int32), X.t)
        for g, name in ((V, "ranlux"), (X, "lcg"), (c, "carry"), (pos, "cursor")):
            g.check(f"get_state {name}", full=False)
        # arrays that are only 8-byte aligned take the per-thread path of the export / import kernels instead of the
        # shared-memory stage: same contents, same bounds, and a handle loaded from them exports the same states
        V8, X8 = Guarded(torch, 2701), Guarded(torch, 2701)
        rlx.rlxpp_get_state(h, V8.t[1:], None, None, X8.t[1:])
        V8.check("get_state ranlux, 8-byte aligned", full=False)
        X8.check("get_state lcg, 8-byte aligned", full=False)
        assert int(V8.t[0]) == int(SENTINEL) and int(X8.t[0]) == int(SENTINEL)
        assert torch.equal(V8.t[1:], V.t) and torch.equal(X8.t[1:], X.t)
        for src in (X.t, X8.t[1:]):
            h2 = rlx.rlxpp_create(300, 1, 389)
            rlx.rlxpp_set_state(h2, src, pos.t.view(torch.int32)[:300])
            back = Guarded(torch, 2700)
            rlx.rlxpp_get_state(h2, None, None, None, back.t)
            back.check("set_state / get_state round trip", full=False)
            assert torch.equal(back.t, X.t)
            rlx.rlxpp_destroy(h2)
        rlx.rlxpp_destroy(h)
    finally:
        rlx.rlxpp_set_engine(rlx.RLXPP_ENGINE_UMMA)


def test_static_scratch_entry_point_stays_inside_its_buffers(rlx, torch):
    n = 300
    for layout in (rlx.RLXPP_STREAM_MAJOR, rlx.RLXPP_INTERLEAVED):
        for per in (96, 204):
            X = Guarded(torch, 9 * n)
            X.t.copy_(torch.from_numpy(inputs.cfg2_states(n - 64).view(np.int64)).cuda().reshape(-1))
            g = Guarded(torch, n * per)
            rlx.rlxpp_generate_doubles_static(X.t, n, 2048, g.t.view(torch.float64), per, layout)
            g.check(f"static, layout {layout}, {per} per stream")
            X.check("static: states", full=False)
