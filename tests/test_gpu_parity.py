"""GPU parity: the CUDA path (through the C ABI, via the ctypes binding) against the CPU oracle,
element by element, tolerance 0 -- every step of RANLUX++ is exact integer arithmetic or exactly
representable fp64, and the fused sums are evaluated in the same order
with the same single-rounding fma on both sides (reading c-14).

Small cases span several 128-thread blocks and a ragged tail and are compared in full; the
BASELINE.json full sizes run in bench.py's launch configuration and are compared on sampled
streams (the oracle computes any stream on its own) plus size-independent properties.
"""
from fractions import Fraction

import numpy as np
import pytest

from paper_2106_02504_b200 import inputs

pytestmark = pytest.mark.gpu

M = (1 << 576) - (1 << 240) + 1


@pytest.fixture(scope="module")
def torch():
    import torch as _torch
    if not _torch.cuda.is_available():
        pytest.fail("the gpu-marked tests need a CUDA device (there is no CPU fallback)")
    return _torch


@pytest.fixture(scope="module", params=["umma", "imad"])
def rlx(torch, request):
    """Every parity test runs once per engine of the LCG advance (include/rlxpp.h): the tensor-core
    path (default) and the IMAD path; both must match the oracle bit for bit."""
    import paper_2106_02504_b200 as _rlx
    _rlx.load()
    _rlx.rlxpp_set_engine(_rlx.RLXPP_ENGINE_UMMA if request.param == "umma" else _rlx.RLXPP_ENGINE_IMAD)
    yield _rlx
    _rlx.rlxpp_set_engine(_rlx.RLXPP_ENGINE_UMMA)


@pytest.fixture(scope="module")
def nthreads(oracle):
    return max(1, oracle.hardware_threads())


def bits(a):
    return np.ascontiguousarray(a).view(np.uint64)


def assert_bits_equal(got, want, what):
    g, w = bits(got), bits(want)
    assert g.shape == w.shape, (what, g.shape, w.shape)
    bad = np.nonzero(g != w)
    assert bad[0].size == 0, f"{what}: {bad[0].size} mismatches, first at {[int(b[0]) for b in bad]}: " \
                             f"got {g[tuple(b[0] for b in bad)]:#x} want {w[tuple(b[0] for b in bad)]:#x}"


def gpu_state(rlx, torch, h):
    n = h.n_streams
    V = torch.empty((n, 9), dtype=torch.int64, device="cuda")
    X = torch.empty((n, 9), dtype=torch.int64, device="cuda")
    c = torch.empty(n, dtype=torch.int32, device="cuda")
    pos = torch.empty(n, dtype=torch.int32, device="cuda")
    rlx.rlxpp_get_state(h, V, c, pos, X)
    torch.cuda.synchronize()
    return (V.cpu().numpy().view(np.uint64), c.cpu().numpy().view(np.uint32), pos.cpu().numpy().view(np.uint32),
            X.cpu().numpy().view(np.uint64))


def check_state(rlx, torch, h, ref, what):
    V, c, pos, X = gpu_state(rlx, torch, h)
    assert_bits_equal(X, ref["X"], what + " LCG state")
    assert_bits_equal(V, ref["V"], what + " RANLUX numbers")
    assert np.array_equal(c, ref["c"]), what + " carry"
    assert np.array_equal(pos, ref["pos"]), what + " cursor"


# ------------------------------------------------------------------------------------- host helpers
def test_host_multiplier_and_seed_state_match_oracle(rlx, oracle):
    for p in (1, 24, 389, 1024, 2048, 777):
        assert inputs.limbs_to_int(rlx.rlxpp_multiplier(p)) == oracle.multiplier(p)
    for seed, p in ((0, 2048), (1, 2048), (2**64 - 1, 2048), (12345, 24), (7, 389)):
        assert inputs.limbs_to_int(rlx.rlxpp_seed_state(seed, p)) == oracle.seed_state(seed, p)


# ------------------------------------------------------------------------------------- config 1
def test_cfg1_smallest_instance_full_compare(rlx, torch, oracle, nthreads):
    """BASELINE.json configs[0]: 1,024 streams, seeds 1..1024, p = 2048, 32 advances = 384 doubles per
    stream, stream-major, all 393,216 doubles and the final states bit-exact."""
    n, per = 1024, 384
    h = rlx.rlxpp_create(n, 1, 2048)
    out = torch.empty((n, per), dtype=torch.float64, device="cuda")
    rlx.rlxpp_generate_doubles(h, out, per, rlx.RLXPP_STREAM_MAJOR)
    torch.cuda.synchronize()
    ref = oracle.streams(inputs.seeds(n), 2048, per, want=("doubles", "state"), nthreads=nthreads)
    assert_bits_equal(out.cpu().numpy(), ref["doubles"], "cfg1 doubles")
    check_state(rlx, torch, h, ref, "cfg1")
    got = out.cpu().numpy()
    assert got.min() >= 0.0 and got.max() < 1.0
    assert np.array_equal(got * 2.0**48, np.floor(got * 2.0**48))  # the 2^-48 lattice
    rlx.rlxpp_destroy(h)


# ------------------------------------------------------------------------------------- config 2
@pytest.mark.parametrize("layout", ["aos", "soa"])
@pytest.mark.parametrize("p", [2048, 24, 100])
def test_cfg2_advance_states_small(rlx, torch, oracle, nthreads, layout, p):
    """Raw LCG advance: random states in [0, m), the 64 edge states (0, 1, m-1, m-2^240, [m, 2^576),
    top limb all ones), 16 repetitions in place; n = 5,000 + 64 is not a multiple of the block size.
    p = 100 takes the generic-multiplier kernel."""
    states = inputs.cfg2_states(5000)
    n = states.shape[0]
    want = oracle.advance_states(states, p, 16, nthreads)
    if layout == "aos":
        dev = torch.from_numpy(states.view(np.int64)).cuda()
        rlx.rlxpp_advance_states(dev, n, p, 16, rlx.RLXPP_AOS)
        got = dev.cpu().numpy().view(np.uint64)
    else:
        dev = torch.from_numpy(np.ascontiguousarray(states.T).view(np.int64)).cuda()
        rlx.rlxpp_advance_states(dev, n, p, 16, rlx.RLXPP_SOA)
        got = np.ascontiguousarray(dev.cpu().numpy().view(np.uint64).T)
    assert_bits_equal(got, want, f"cfg2 {layout} p={p}")
    assert all(inputs.limbs_to_int(r) < M for r in got[-64:])


def test_cfg2_reps_zero_canonicalises_and_empty_is_noop(rlx, torch, oracle):
    states = inputs.cfg2_edge_states()
    dev = torch.from_numpy(states.view(np.int64)).cuda()
    rlx.rlxpp_advance_states(dev, 64, 2048, 0, rlx.RLXPP_AOS)
    got = dev.cpu().numpy().view(np.uint64)
    for g, s in zip(got, states):
        assert inputs.limbs_to_int(g) == inputs.limbs_to_int(s) % M
    rlx.rlxpp_advance_states(dev, 0, 2048, 16, rlx.RLXPP_AOS)  # n == 0
    assert np.array_equal(dev.cpu().numpy().view(np.uint64), got)
    one = torch.from_numpy(states[:1].copy().view(np.int64)).cuda()  # a single state (9 words: odd tail)
    rlx.rlxpp_advance_states(one, 1, 2048, 3, rlx.RLXPP_AOS)
    assert_bits_equal(one.cpu().numpy(), oracle.advance_states(states[:1], 2048, 3), "single state")


def test_cfg2_full_size(rlx, torch, oracle, nthreads):
    """BASELINE.json configs[1] at full size: 2^20 + 64 states x 16 advances, every state compared."""
    states = inputs.cfg2_states(1 << 20)
    n = states.shape[0]
    dev = torch.from_numpy(states.view(np.int64)).cuda()
    rlx.rlxpp_advance_states(dev, n, 2048, 16, rlx.RLXPP_AOS)
    got = dev.cpu().numpy().view(np.uint64)
    want = oracle.advance_states(states, 2048, 16, nthreads)
    assert_bits_equal(got, want, "cfg2 full")


# ------------------------------------------------------------------------------------- config 3
def test_cfg3_interleaved_small(rlx, torch, oracle, nthreads):
    n, per = 1000, 1536  # 7 full blocks + a ragged one; 128 advances per stream
    h = rlx.rlxpp_create(n, 1, 2048)
    out = torch.empty((per, n), dtype=torch.float64, device="cuda")
    rlx.rlxpp_generate_doubles(h, out, per, rlx.RLXPP_INTERLEAVED)
    torch.cuda.synchronize()
    ref = oracle.streams(inputs.seeds(n), 2048, per, want=("doubles", "state"), nthreads=nthreads)
    assert_bits_equal(out.cpu().numpy().T, ref["doubles"], "cfg3 small")
    check_state(rlx, torch, h, ref, "cfg3 small")


_CFG3_CHECKSUMS = {}


def cfg3_oracle_checksums(oracle, nthreads, n, per, p=2048):
    """Per draw index k, over ALL n streams: the wrapping sum of the 48-bit integers and the wrapping sum weighted
    with 2 i + 1 (i = stream), from the oracle alone (chunks of 2^16 streams; computed once per session)."""
    key = (n, per, p)
    if key not in _CFG3_CHECKSUMS:
        s1 = np.zeros(per, np.uint64)
        s2 = np.zeros(per, np.uint64)
        step = 1 << 16
        with np.errstate(over="ignore"):
            for lo in range(0, n, step):
                cnt = min(step, n - lo)
                k = oracle.streams(inputs.seeds(n)[lo:lo + cnt], p, per, want=("ints",), nthreads=nthreads)["ints"]
                w = (np.arange(lo, lo + cnt, dtype=np.uint64) * np.uint64(2) + np.uint64(1))[:, None]
                s1 += k.sum(axis=0, dtype=np.uint64)
                s2 += (k * w).sum(axis=0, dtype=np.uint64)
        _CFG3_CHECKSUMS[key] = (s1, s2)
    return _CFG3_CHECKSUMS[key]


def gpu_checksums_interleaved(torch, out, n, per):
    s1 = torch.zeros(per, dtype=torch.int64, device="cuda")
    s2 = torch.zeros(per, dtype=torch.int64, device="cuda")
    w_all = torch.arange(n, dtype=torch.int64, device="cuda") * 2 + 1
    for lo in range(0, per, 64):
        k = (out[lo:lo + 64] * 2.0**48).to(torch.int64)  # exact: 48-bit integers
        s1[lo:lo + 64] = k.sum(dim=1)
        s2[lo:lo + 64] = (k * w_all[None, :]).sum(dim=1)
    return s1.cpu().numpy().view(np.uint64), s2.cpu().numpy().view(np.uint64)


@pytest.mark.parametrize("layout", ["interleaved", "stream_major"])
def test_cfg3_full_size_sampled(rlx, torch, oracle, nthreads, layout):
    """BASELINE.json configs[2] in bench.py's launch configuration: 2^20 streams x 1,536 doubles,
    12.9 GB, interleaved (the config's layout) and stream-major (bench.py --layout stream_major).  Sampled
    streams (first and last blocks, a stride through the rest) are compared in full; the whole array is
    checked for range and lattice on the device, and through two 64-bit checksums per draw index against the
    oracle's checksums of all 2^20 streams."""
    n, per = 1 << 20, 1536
    h = rlx.rlxpp_create(n, 1, 2048)
    il = layout == "interleaved"
    out = torch.empty((per, n) if il else (n, per), dtype=torch.float64, device="cuda")
    rlx.rlxpp_generate_doubles(h, out, per, rlx.RLXPP_INTERLEAVED if il else rlx.RLXPP_STREAM_MAJOR)
    torch.cuda.synchronize()
    idx = np.unique(np.concatenate([np.arange(0, 130), np.arange(n - 130, n), np.arange(0, n, 4099)]))
    tidx = torch.from_numpy(idx).cuda()
    got = out[:, tidx].cpu().numpy().T if il else out[tidx].cpu().numpy()
    ref = oracle.streams(inputs.seeds(n)[idx], 2048, per, want=("doubles", "state"), nthreads=nthreads)
    assert_bits_equal(got, ref["doubles"], f"cfg3 full, {layout} (sampled streams)")
    flat = out.view(-1)
    step = 128 * n
    for lo in range(0, per * n, step):  # properties at any size, chunked to bound temporaries
        blk = flat[lo:lo + step]
        assert bool((blk >= 0).all()) and bool((blk < 1).all())
        sc = blk * 2.0**48
        assert bool((sc == sc.floor()).all())
    # every one of the 1.6 G doubles: two 64-bit checksums per draw index against the oracle's
    s1 = torch.zeros(per, dtype=torch.int64, device="cuda")
    s2 = torch.zeros(per, dtype=torch.int64, device="cuda")
    w_all = torch.arange(n, dtype=torch.int64, device="cuda") * 2 + 1
    if il:
        for lo in range(0, per, 64):
            k = (out[lo:lo + 64] * 2.0**48).to(torch.int64)  # exact: 48-bit integers
            s1[lo:lo + 64] = k.sum(dim=1)
            s2[lo:lo + 64] = (k * w_all[None, :]).sum(dim=1)
    else:
        for lo in range(0, n, 1 << 15):
            k = (out[lo:lo + (1 << 15)] * 2.0**48).to(torch.int64)
            s1 += k.sum(dim=0)
            s2 += (k * w_all[lo:lo + (1 << 15), None]).sum(dim=0)
    o1, o2 = cfg3_oracle_checksums(oracle, nthreads, n, per)
    assert np.array_equal(s1.cpu().numpy().view(np.uint64), o1), f"cfg3 full, {layout}: sum checksum"
    assert np.array_equal(s2.cpu().numpy().view(np.uint64), o2), f"cfg3 full, {layout}: weighted checksum"
    V, c, pos, X = gpu_state(rlx, torch, h)
    assert_bits_equal(X[idx], ref["X"], "cfg3 full state")
    assert np.all(pos == 12)
    del out


# ------------------------------------------------------------------------------------- config 4
@pytest.mark.parametrize("p", [24, 389, 1024, 2048])
def test_cfg4_luxury_sweep_small(rlx, torch, oracle, nthreads, p):
    n, per = 700, 6144
    h = rlx.rlxpp_create(n, 1, p)
    out = torch.empty((per, n), dtype=torch.float64, device="cuda")
    rlx.rlxpp_generate_doubles(h, out, per, rlx.RLXPP_INTERLEAVED)
    torch.cuda.synchronize()
    ref = oracle.streams(inputs.seeds(n), p, per, want=("doubles", "state"), nthreads=nthreads)
    assert_bits_equal(out.cpu().numpy().T, ref["doubles"], f"cfg4 p={p}")
    check_state(rlx, torch, h, ref, f"cfg4 p={p}")


def test_cfg4_p24_is_direct_subtract_with_borrow(rlx, torch, oracle):
    """p = 24 skips nothing: the GPU stream must be the raw RANLUX (SWB) sequence started from the
    seeded state (reading c-13), here produced by the oracle's direct SWB stepper."""
    n, per = 64, 120
    h = rlx.rlxpp_create(n, 1, 24)
    out = torch.empty((n, per), dtype=torch.float64, device="cuda")
    rlx.rlxpp_generate_doubles(h, out, per, rlx.RLXPP_STREAM_MAJOR)
    got = (out.cpu().numpy() * 2.0**48).astype(np.uint64)
    for i in (0, 1, 63):
        V, c = oracle.to_ranlux(oracle.seed_state(1 + i, 24))
        want = []
        for _ in range(per // 12):
            V, c = oracle.swb_steps(V, c, 24)
            want += [(V >> (48 * j)) & (2**48 - 1) for j in range(12)]
        assert [int(v) for v in got[i]] == want


@pytest.mark.parametrize("p", [24, 389, 1024, 2048])
def test_cfg4_full_size_sampled(rlx, torch, oracle, nthreads, p):
    n, per = 1 << 18, 6144
    h = rlx.rlxpp_create(n, 1, p)
    out = torch.empty((per, n), dtype=torch.float64, device="cuda")
    rlx.rlxpp_generate_doubles(h, out, per, rlx.RLXPP_INTERLEAVED)
    torch.cuda.synchronize()
    idx = np.unique(np.concatenate([np.arange(0, 40), np.arange(n - 40, n), np.arange(0, n, 2731)]))
    got = out[:, torch.from_numpy(idx).cuda()].cpu().numpy().T
    ref = oracle.streams(inputs.seeds(n)[idx], p, per, want=("doubles",), nthreads=nthreads)
    assert_bits_equal(got, ref["doubles"], f"cfg4 full p={p}")
    g1, g2 = gpu_checksums_interleaved(torch, out, n, per)  # all 1.6 G doubles, as in the cfg3 test
    o1, o2 = cfg3_oracle_checksums(oracle, nthreads, n, per, p)
    assert np.array_equal(g1, o1) and np.array_equal(g2, o2), f"cfg4 full p={p}: checksums over all streams"
    del out


# ------------------------------------------------------------------------------------- config 5
def test_cfg5_skip_and_fused_reduce_small(rlx, torch, oracle, nthreads):
    n, per = 3000, 49152 // 8
    dist = inputs.cfg5_skip_distances(n)
    h = rlx.rlxpp_create(n, 1, 2048)
    rlx.rlxpp_skip_each(h, torch.from_numpy(dist.view(np.int64)).cuda())
    s = torch.empty(n, dtype=torch.float64, device="cuda")
    q = torch.empty(n, dtype=torch.float64, device="cuda")
    rlx.rlxpp_generate_reduce(h, s, q, per)
    torch.cuda.synchronize()
    ref = oracle.streams(inputs.seeds(n), 2048, per, skips=dist, want=("sums", "state"), nthreads=nthreads)
    assert_bits_equal(s.cpu().numpy(), ref["sum"], "cfg5 sum")
    assert_bits_equal(q.cpu().numpy(), ref["sumsq"], "cfg5 sum of squares")
    check_state(rlx, torch, h, ref, "cfg5 small")


_CFG5_ORACLE = {}


def test_cfg5_full_size_all_streams(rlx, torch, oracle, nthreads):
    """BASELINE.json configs[4] in bench.py's launch configuration: 2^18 streams, random 64-bit skips, 49,152
    doubles each reduced in registers.  ALL 2 x 2^18 sums, states and cursors are compared bit for bit: the oracle
    runs the whole config (1.07 G advances, about half a minute on the host cores; once per session)."""
    n, per = 1 << 18, 49152
    dist = inputs.cfg5_skip_distances(n)
    h = rlx.rlxpp_create(n, 1, 2048)
    rlx.rlxpp_skip_each(h, torch.from_numpy(dist.view(np.int64)).cuda())
    s = torch.empty(n, dtype=torch.float64, device="cuda")
    q = torch.empty(n, dtype=torch.float64, device="cuda")
    rlx.rlxpp_generate_reduce(h, s, q, per)
    torch.cuda.synchronize()
    if "ref" not in _CFG5_ORACLE:
        _CFG5_ORACLE["ref"] = oracle.streams(inputs.seeds(n), 2048, per, skips=dist, want=("sums", "state"), nthreads=nthreads)
    ref = _CFG5_ORACLE["ref"]
    assert_bits_equal(s.cpu().numpy(), ref["sum"], "cfg5 full sum")
    assert_bits_equal(q.cpu().numpy(), ref["sumsq"], "cfg5 full sumsq")
    check_state(rlx, torch, h, ref, "cfg5 full")
    rlx.rlxpp_destroy(h)


# ------------------------------------------------------------------------------------- other outputs (8f-2)
def _floats_of(ints):
    """The two 24-bit RANLUX numbers of every 48-bit draw as floats x 2^-24 (exact), low number first."""
    lo = (ints & np.uint64(0xFFFFFF)).astype(np.float32) * np.float32(2.0**-24)
    hi = (ints >> np.uint64(24)).astype(np.float32) * np.float32(2.0**-24)
    return np.stack([lo, hi], axis=-1).reshape(ints.shape[0], -1)


@pytest.mark.parametrize("aligned", [True, False])
def test_u48_and_float_outputs_are_the_same_draws(rlx, torch, oracle, nthreads, aligned):
    """rlxpp_generate_u48 / rlxpp_generate_floats give the 48-bit integers and the 24-bit numbers of the
    SAME sequence as the doubles, in both layouts, interleaved with double draws on one cursor."""
    n, p = 700, 2048
    nd = 48 if aligned else 41          # draws per call
    h = rlx.rlxpp_create(n, 8, p)
    dist = None
    if not aligned:
        dist = inputs.splitmix64(31337, n) % np.uint64(50)
        rlx.rlxpp_skip_each(h, torch.from_numpy(dist.view(np.int64)).cuda())
    u_sm = torch.zeros((n, nd), dtype=torch.int64, device="cuda")
    rlx.rlxpp_generate_u48(h, u_sm, nd, rlx.RLXPP_STREAM_MAJOR)
    u_il = torch.zeros((nd, n), dtype=torch.int64, device="cuda")
    rlx.rlxpp_generate_u48(h, u_il, nd, rlx.RLXPP_INTERLEAVED)
    f_sm = torch.zeros((n, 2 * nd), dtype=torch.float32, device="cuda")
    rlx.rlxpp_generate_floats(h, f_sm, 2 * nd, rlx.RLXPP_STREAM_MAJOR)
    f_il = torch.zeros((2 * nd, n), dtype=torch.float32, device="cuda")
    rlx.rlxpp_generate_floats(h, f_il, 2 * nd, rlx.RLXPP_INTERLEAVED)
    d = torch.zeros((n, nd), dtype=torch.float64, device="cuda")
    rlx.rlxpp_generate_doubles(h, d, nd, rlx.RLXPP_STREAM_MAJOR)
    torch.cuda.synchronize()
    ref = oracle.streams(inputs.seeds(n, 8), p, 5 * nd, skips=dist, want=("ints", "doubles", "state"), nthreads=nthreads)
    ints = ref["ints"]
    assert np.array_equal(u_sm.cpu().numpy().view(np.uint64), ints[:, :nd])
    assert np.array_equal(u_il.cpu().numpy().view(np.uint64).T, ints[:, nd:2 * nd])
    assert np.array_equal(f_sm.cpu().numpy().view(np.uint32), _floats_of(ints[:, 2 * nd:3 * nd]).view(np.uint32))
    assert np.array_equal(f_il.cpu().numpy().T.copy().view(np.uint32), _floats_of(ints[:, 3 * nd:4 * nd]).view(np.uint32))
    assert_bits_equal(d.cpu().numpy(), ref["doubles"][:, 4 * nd:], "doubles after the other output forms")
    check_state(rlx, torch, h, ref, "after u48 / floats")
    fl = f_sm.cpu().numpy()
    assert fl.min() >= 0.0 and fl.max() < 1.0 and np.all(fl * 2.0**24 == np.floor(fl * 2.0**24))  # 2^-24 lattice
    with pytest.raises(rlx.RlxppError, match="even"):
        rlx.rlxpp_generate_floats(h, f_sm, 7, rlx.RLXPP_STREAM_MAJOR)
    rlx.rlxpp_destroy(h)


NORMAL_ULPS = 6  # log <= 1 ulp (halved by the sqrt), sqrt and product 0.5 each, sincospi <= 2, oracle 0.5


def assert_within_ulps(got, want, ulps, what):
    got, want = np.asarray(got), np.asarray(want)
    assert got.shape == want.shape, (what, got.shape, want.shape)
    bad = np.nonzero(~(np.abs(got - want) <= ulps * np.spacing(np.abs(want))))
    assert bad[0].size == 0, f"{what}: {bad[0].size} values off by more than {ulps} ulp, first at " \
                             f"{[int(b[0]) for b in bad]}: got {got[tuple(b[0] for b in bad)]!r} " \
                             f"want {want[tuple(b[0] for b in bad)]!r}"


@pytest.mark.parametrize("layout", ["stream_major", "interleaved"])
def test_normal_deviates_are_box_muller_of_the_draw_pairs(rlx, torch, oracle, nthreads, layout):
    """rlxpp_generate_normal (DESIGN reading N-1) against oracle.normals of the oracle's own 48-bit
    draws.  One deviate per draw position: an aligned call (TMA boxes + directly stored tail when stream-major),
    a call that ends inside a pair, one that starts inside a pair, and one after per-stream skips of random
    parity; the cursor and state must be those of the same number of plain draws."""
    n = 3 * 128 + 45
    sm = layout == "stream_major"
    lay = rlx.RLXPP_STREAM_MAJOR if sm else rlx.RLXPP_INTERLEAVED
    dist = inputs.splitmix64(99, n) % np.uint64(1000)
    counts = [12 * 19, 37, 41]
    total = 12 * 19 + 37 + 41 + 1000 + 100
    total += total % 2
    k = oracle.streams(inputs.seeds(n, 5), 2048, total, want=("ints",), nthreads=nthreads)["ints"]
    z = oracle.normals(k)  # pairs (2i, 2i + 1) counted from each stream's first draw
    h = rlx.rlxpp_create(n, 5, 2048)

    def call(per):
        out = torch.full((n, per) if sm else (per, n), np.nan, dtype=torch.float64, device="cuda")
        rlx.rlxpp_generate_normal(h, out, per, lay)
        torch.cuda.synchronize()
        return out.cpu().numpy() if sm else out.cpu().numpy().T

    at = 0
    for per in counts:
        assert_within_ulps(call(per), z[:, at:at + per], NORMAL_ULPS, f"normals {layout}, draws {at}..{at + per}")
        at += per
    rlx.rlxpp_skip_each(h, torch.from_numpy(dist.view(np.int64)).cuda())
    got = call(100)
    want = np.stack([z[i, at + int(dist[i]):at + int(dist[i]) + 100] for i in range(n)])
    assert_within_ulps(got, want, NORMAL_ULPS, f"normals {layout} after per-stream skips")
    ref = oracle.streams(inputs.seeds(n, 5), 2048, 100, skips=dist + np.uint64(at), want=("state",), nthreads=nthreads)
    check_state(rlx, torch, h, ref, "after normals")
    # uniform doubles continue where the normals stopped
    d = torch.empty((n, 24), dtype=torch.float64, device="cuda")
    rlx.rlxpp_generate_doubles(h, d, 24, rlx.RLXPP_STREAM_MAJOR)
    ref = oracle.streams(inputs.seeds(n, 5), 2048, 24, skips=dist + np.uint64(at + 100), want=("doubles",), nthreads=nthreads)
    assert_bits_equal(d.cpu().numpy(), ref["doubles"], "doubles after normals")
    rlx.rlxpp_destroy(h)


def test_normal_deviates_accuracy_sweep(rlx, torch, oracle, nthreads):
    """3.9 M deviates (8,192 streams x 480, the TMA path and its directly stored tail of a row) against the long-double
    oracle: none beyond the 6 ulp bar, the mean well under one ulp (measured on B200: max 3 ulp, mean 0.42,
    99.9 % within 2)."""
    n, per = 8192, 480
    h = rlx.rlxpp_create(n, 3, 2048)
    out = torch.empty((n, per), dtype=torch.float64, device="cuda")
    rlx.rlxpp_generate_normal(h, out, per, rlx.RLXPP_STREAM_MAJOR)
    torch.cuda.synchronize()
    got = out.cpu().numpy()
    z = oracle.normals(oracle.streams(inputs.seeds(n, 3), 2048, per, want=("ints",), nthreads=nthreads)["ints"])
    assert_within_ulps(got, z, NORMAL_ULPS, "normals sweep")
    err = np.abs(got - z) / np.spacing(np.abs(z))
    assert float(err.mean()) < 1.0
    assert abs(float(got.mean())) < 5.0 / np.sqrt(got.size) and abs(float(got.var()) - 1.0) < 5.0 * np.sqrt(2.0 / got.size)
    rlx.rlxpp_destroy(h)


def test_p24_floats_are_the_raw_ranlux_numbers(rlx, torch, oracle):
    """p = 24: the floats are the subtract-with-borrow numbers themselves (x 2^-24), one by one, from
    the oracle's direct SWB stepper (reading c-13)."""
    n, per = 40, 240
    h = rlx.rlxpp_create(n, 1, 24)
    out = torch.empty((n, per), dtype=torch.float32, device="cuda")
    rlx.rlxpp_generate_floats(h, out, per, rlx.RLXPP_STREAM_MAJOR)
    got = (out.cpu().numpy().astype(np.float64) * 2.0**24).astype(np.uint64)
    for i in (0, 7, 39):
        V, c = oracle.to_ranlux(oracle.seed_state(1 + i, 24))
        want = []
        for _ in range(per // 24):
            V, c = oracle.swb_steps(V, c, 24)
            want += [(V >> (24 * j)) & (2**24 - 1) for j in range(24)]
        assert [int(v) for v in got[i]] == want
    rlx.rlxpp_destroy(h)


# ------------------------------------------------------------------------------------- device API (8f-1)
@pytest.mark.parametrize("p", [2048, 100])
@pytest.mark.parametrize("coop", [True, False, 2, 3])
def test_device_api_ragged_draws_match_the_stream(rlx, torch, oracle, nthreads, coop, p):
    """include/rlxpp_device.cuh through rlxpp_generate_ragged: every stream draws its own number of
    doubles (0 .. 70, so lanes of a warp run out of their blocks at different calls), from per-stream
    cursors, twice in a row, then the library's bulk kernel continues the same streams.  Everything
    must be the one sequence the oracle gives for that stream; cooperative and per-thread advance agree,
    and so does a kernel that alternates draw_coop() and draw() on the same Stream (coop = 2: a spare block
    made by draw_coop() must be entered, not recomputed past, by draw()); coop = 3 is include/rlxpp_tile.cuh's
    rlxpp_dev::TileStream, the block-cooperative tensor-core advance (ragged counts: threads ask for passes at different
    calls, some threads of a CTA are done long before others, the last CTA is ragged).  p = 2048 takes the per-thread
    generator with the rows baked in (rlxpp_dev::StreamT<2048>, include/rlxpp_rows.cuh), p = 100 the run-time multiplier."""
    n, ld = 1000, 72
    dist = inputs.splitmix64(77, n) % np.uint64(30)
    c1 = (inputs.splitmix64(78, n) % np.uint64(71)).astype(np.uint32)
    c2 = (inputs.splitmix64(79, n) % np.uint64(71)).astype(np.uint32)
    c1[:4] = (0, 1, 12, 70)
    h = rlx.rlxpp_create(n, 3, p)
    rlx.rlxpp_skip_each(h, torch.from_numpy(dist.view(np.int64)).cuda())
    o1 = torch.full((n, ld), -1.0, dtype=torch.float64, device="cuda")
    o2 = torch.full((n, ld), -1.0, dtype=torch.float64, device="cuda")
    rlx.rlxpp_generate_ragged(h, torch.from_numpy(c1.view(np.int32)).cuda(), o1, ld, coop)
    rlx.rlxpp_generate_ragged(h, torch.from_numpy(c2.view(np.int32)).cuda(), o2, ld, coop)
    tail = 25
    o3 = torch.empty((n, tail), dtype=torch.float64, device="cuda")
    rlx.rlxpp_generate_doubles(h, o3, tail, rlx.RLXPP_STREAM_MAJOR)
    torch.cuda.synchronize()
    ref = oracle.streams(inputs.seeds(n, 3), p, 2 * 70 + tail, skips=dist, want=("doubles",), nthreads=nthreads)["doubles"]
    g1, g2, g3 = o1.cpu().numpy(), o2.cpu().numpy(), o3.cpu().numpy()
    for i in range(n):
        a, b = int(c1[i]), int(c2[i])
        assert_bits_equal(g1[i, :a], ref[i, :a], f"ragged first call, stream {i}")
        assert_bits_equal(g2[i, :b], ref[i, a:a + b], f"ragged second call, stream {i}")
        assert_bits_equal(g3[i], ref[i, a + b:a + b + tail], f"bulk kernel after the device API, stream {i}")
        assert np.all(g1[i, a:] == -1.0) and np.all(g2[i, b:] == -1.0)  # nothing written past a stream's count
    rlx.rlxpp_destroy(h)


@pytest.mark.parametrize("coop", [True, False, 2, 3])
def test_device_api_ragged_reduce(rlx, torch, oracle, nthreads, coop):
    n, p = 700, 389
    cnt = (inputs.splitmix64(5150, n) % np.uint64(200)).astype(np.uint32)
    h = rlx.rlxpp_create(n, 1, p)
    rlx.rlxpp_skip(h, 7)
    s = torch.empty(n, dtype=torch.float64, device="cuda")
    q = torch.empty(n, dtype=torch.float64, device="cuda")
    rlx.rlxpp_generate_ragged_reduce(h, torch.from_numpy(cnt.view(np.int32)).cuda(), s, q, coop)
    torch.cuda.synchronize()
    ref = oracle.streams(inputs.seeds(n), p, 7 + 200, want=("doubles",), nthreads=nthreads)["doubles"][:, 7:]
    S, Q = np.zeros(n), np.zeros(n)
    from fractions import Fraction
    for i in range(n):
        a = b = 0.0
        for t in range(int(cnt[i])):
            d = float(ref[i, t])
            a = a + d
            b = float(Fraction(d) * Fraction(d) + Fraction(b))  # fma: one correctly rounded result (c-14)
        S[i], Q[i] = a, b
    assert_bits_equal(s.cpu().numpy(), S, "ragged sum")
    assert_bits_equal(q.cpu().numpy(), Q, "ragged sum of squares")
    V, c, pos, X = gpu_state(rlx, torch, h)
    for i in (0, 1, 31, 32, 699):
        Xe, pe, _ = oracle.engine_run(oracle.seed_state(1 + i, p), 12, p, [("skip", 7), ("draw", int(cnt[i]))])
        assert inputs.limbs_to_int(X[i]) == Xe and int(pos[i]) == pe
    rlx.rlxpp_destroy(h)


def test_host_engine_hands_over_with_the_device(rlx, torch, oracle):
    """a stream moves device -> host -> device mid-block and
    stays one sequence: get_state, rlxpp_host_generate on the host, set_state, generate on the device."""
    n, p = 130, 2048
    h = rlx.rlxpp_create(n, 21, p)
    a = torch.empty((n, 17), dtype=torch.float64, device="cuda")
    rlx.rlxpp_generate_doubles(h, a, 17, rlx.RLXPP_STREAM_MAJOR)  # cursor 5 in the second block
    V, c, pos, X = gpu_state(rlx, torch, h)
    host_draws = np.empty((n, 20))
    Xn, posn = X.copy(), pos.copy()
    for i in range(n):
        host_draws[i], Xn[i], posn[i] = rlx.rlxpp_host_generate(X[i], int(pos[i]), p, 3, 20)  # skip 3, draw 20
    rlx.rlxpp_set_state(h, torch.from_numpy(Xn.view(np.int64)).cuda(), torch.from_numpy(posn.astype(np.int32)).cuda())
    b = torch.empty((n, 30), dtype=torch.float64, device="cuda")
    rlx.rlxpp_generate_doubles(h, b, 30, rlx.RLXPP_STREAM_MAJOR)
    torch.cuda.synchronize()
    ref = oracle.streams(inputs.seeds(n, 21), p, 17 + 3 + 20 + 30, want=("doubles",))["doubles"]
    assert_bits_equal(a.cpu().numpy(), ref[:, :17], "device part 1")
    assert_bits_equal(host_draws, ref[:, 20:40], "host part")
    assert_bits_equal(b.cpu().numpy(), ref[:, 40:], "device part 2")
    rlx.rlxpp_destroy(h)


# ------------------------------------------------------------------------------------- cursor logic
def test_unaligned_draw_counts_and_uniform_skip(rlx, torch, oracle, nthreads):
    """Draw counts that are not multiples of 12, interleaved with uniform skips (D8): the
    concatenation must equal the oracle's engine driven with the same operations."""
    n = 300
    h = rlx.rlxpp_create(n, 77, 2048)
    ops = [("draw", 7), ("draw", 5), ("skip", 1), ("draw", 13), ("skip", 12), ("draw", 1), ("skip", 2**40 + 5),
           ("draw", 30), ("draw", 0), ("skip", 0), ("draw", 12), ("draw", 24), ("skip", 2**64 - 1), ("draw", 3)]
    chunks = []
    for kind, k in ops:
        if kind == "skip":
            rlx.rlxpp_skip(h, k)
        else:
            out = torch.full((n, max(k, 1)), -1.0, dtype=torch.float64, device="cuda")
            rlx.rlxpp_generate_doubles(h, out, k, rlx.RLXPP_STREAM_MAJOR)
            if k:
                chunks.append(out.cpu().numpy())
            else:
                assert bool((out == -1.0).all())
    got = (np.concatenate(chunks, axis=1) * 2.0**48).astype(np.uint64)
    V, c, pos, X = gpu_state(rlx, torch, h)
    for i in (0, 1, 127, 128, 299):
        X0 = oracle.seed_state(77 + i, 2048)
        Xe, pe, draws = oracle.engine_run(X0, 12, 2048, ops)
        assert [int(v) for v in got[i]] == draws
        assert inputs.limbs_to_int(X[i]) == Xe and int(pos[i]) == pe


def test_unaligned_interleaved_and_reduce_after_per_stream_skips(rlx, torch, oracle, nthreads):
    n, per = 515, 100
    dist = inputs.splitmix64(99, n) % np.uint64(40)  # small distances: every cursor value occurs
    h = rlx.rlxpp_create(n, 5, 389)
    rlx.rlxpp_skip_each(h, torch.from_numpy(dist.view(np.int64)).cuda())
    out = torch.empty((per, n), dtype=torch.float64, device="cuda")
    rlx.rlxpp_generate_doubles(h, out, per, rlx.RLXPP_INTERLEAVED)
    ref = oracle.streams(inputs.seeds(n, 5), 389, per, skips=dist, want=("doubles", "state"), nthreads=nthreads)
    assert_bits_equal(out.cpu().numpy().T, ref["doubles"], "unaligned interleaved")
    check_state(rlx, torch, h, ref, "unaligned interleaved")
    s = torch.empty(n, dtype=torch.float64, device="cuda")
    rlx.rlxpp_generate_reduce(h, s, None, 31)  # sumsq omitted
    ref2 = oracle.streams(inputs.seeds(n, 5), 389, per + 31, skips=dist, want=("doubles",), nthreads=nthreads)
    want = np.zeros(n)
    for t in range(per, per + 31):
        want = want + ref2["doubles"][:, t]
    assert_bits_equal(s.cpu().numpy(), want, "reduce after unaligned draws")


@pytest.mark.parametrize("n_chunks", [2, 3, 7])
def test_chunked_work_items_give_the_same_results(rlx, torch, oracle, nthreads, n_chunks):
    """UMMA engine: the persistent kernel cuts a tile's draws into chunks handed to different CTAs
    (rlxpp_set_chunks forces it at a small size; cfg4 / cfg5 full size use it by default).  State,
    cursor and partial sums travel through global memory between chunks: results must not change.
    More tiles (41) than fit a chunk-major order by accident, ragged last tile, ragged last chunk."""
    n, per = 41 * 128 - 29, 12 * 50
    dist = inputs.splitmix64(4242, n) % np.uint64(1000)
    rlx.rlxpp_set_chunks(n_chunks)
    try:
        # aligned cursors, both store layouts
        h = rlx.rlxpp_create(n, 9, 2048)
        a = torch.empty((n, per), dtype=torch.float64, device="cuda")
        rlx.rlxpp_generate_doubles(h, a, per, rlx.RLXPP_STREAM_MAJOR)
        b = torch.empty((per, n), dtype=torch.float64, device="cuda")
        rlx.rlxpp_generate_doubles(h, b, per, rlx.RLXPP_INTERLEAVED)
        ref = oracle.streams(inputs.seeds(n, 9), 2048, 2 * per, want=("doubles", "state"), nthreads=nthreads)
        assert_bits_equal(a.cpu().numpy(), ref["doubles"][:, :per], "chunked stream-major")
        assert_bits_equal(b.cpu().numpy().T, ref["doubles"][:, per:], "chunked interleaved")
        check_state(rlx, torch, h, ref, "chunked aligned")
        rlx.rlxpp_destroy(h)
        # per-stream cursors, draw count not a multiple of 12, fused sums carried across chunks
        per2 = per + 5
        h = rlx.rlxpp_create(n, 9, 2048)
        rlx.rlxpp_skip_each(h, torch.from_numpy(dist.view(np.int64)).cuda())
        s = torch.empty(n, dtype=torch.float64, device="cuda")
        q = torch.empty(n, dtype=torch.float64, device="cuda")
        rlx.rlxpp_generate_reduce(h, s, q, per2)
        c = torch.empty((per2, n), dtype=torch.float64, device="cuda")
        rlx.rlxpp_generate_doubles(h, c, per2, rlx.RLXPP_INTERLEAVED)
        s2 = torch.empty(n, dtype=torch.float64, device="cuda")
        rlx.rlxpp_generate_reduce(h, s2, None, per2)  # no sum of squares: library scratch carries it
        torch.cuda.synchronize()
        ref = oracle.streams(inputs.seeds(n, 9), 2048, per2, skips=dist, want=("sums",), nthreads=nthreads)
        assert_bits_equal(s.cpu().numpy(), ref["sum"], "chunked sum")
        assert_bits_equal(q.cpu().numpy(), ref["sumsq"], "chunked sum of squares")
        ref = oracle.streams(inputs.seeds(n, 9), 2048, 3 * per2, skips=dist, want=("doubles", "state"), nthreads=nthreads)
        assert_bits_equal(c.cpu().numpy().T, ref["doubles"][:, per2:2 * per2], "chunked unaligned interleaved")
        want = np.zeros(n)
        for t in range(2 * per2, 3 * per2):
            want = want + ref["doubles"][:, t]
        assert_bits_equal(s2.cpu().numpy(), want, "chunked sum without sumsq")
        check_state(rlx, torch, h, ref, "chunked unaligned")
        rlx.rlxpp_destroy(h)
    finally:
        rlx.rlxpp_set_chunks(0)


@pytest.mark.parametrize("blocks", [1, 7, 8, 9, 15, 16, 21, 43])
def test_stream_major_rows_of_any_length(rlx, torch, oracle, nthreads, blocks):
    """Stream-major output, aligned cursors (UMMA engine: 256-byte boxes through the TMA for whole cycles of
    8 blocks, direct stores for the rest of a row; csrc/stages.cuh StreamMajorStage).  Row lengths on both sides of
    the cycle, rows that are not 128- or 256-byte multiples, a ragged last warp and tile (rows the tensor
    map must clip), and a guard band behind the buffer that must stay untouched.  Two calls in a row: the
    second continues the streams."""
    n, per = 3 * 128 + 45, 12 * blocks
    guard = 4096
    h = rlx.rlxpp_create(n, 77, 2048)
    ref = oracle.streams(inputs.seeds(n, 77), 2048, 2 * per, want=("doubles", "state"), nthreads=nthreads)
    for call in range(2):
        buf = torch.full((n * per + guard,), -1.0, dtype=torch.float64, device="cuda")
        rlx.rlxpp_generate_doubles(h, buf, per, rlx.RLXPP_STREAM_MAJOR)
        torch.cuda.synchronize()
        got = buf.cpu().numpy()
        assert_bits_equal(got[:n * per].reshape(n, per), ref["doubles"][:, call * per:(call + 1) * per],
                          f"stream-major rows of {blocks} blocks, call {call}")
        assert np.all(got[n * per:] == -1.0), "wrote behind the output buffer"
    check_state(rlx, torch, h, ref, "stream-major rows")
    rlx.rlxpp_destroy(h)


@pytest.mark.parametrize("case", [0, 1, 2, 3, 4, 5])
def test_random_call_sequences_against_the_oracle(rlx, torch, oracle, nthreads, case):
    """Differential test of the whole C ABI on one handle: a seeded random sequence of skips (uniform and per
    stream), and generate calls of every output form, layout and count (multiples of 12, of 96, odd counts, 1),
    each compared with the oracle at the streams' absolute draw positions; the state at the end.  Catches
    anything that depends on what the previous call left behind (cursor bookkeeping, the aligned fast paths,
    chunk plans, staging buffers)."""
    rng = np.random.default_rng(1000 + case)
    n = int(rng.choice([1, 31, 128, 3 * 128 + 77, 1000]))
    p = int(rng.choice([2048, 2048, 389, 24]))
    seed0 = int(rng.integers(1, 1 << 40))
    seeds = inputs.seeds(n, seed0)
    g = np.zeros(n, dtype=np.uint64)  # draws consumed so far, per stream
    h = rlx.rlxpp_create(n, seed0, p)
    for step in range(14):
        op = rng.choice(["doubles", "u48", "floats", "normal", "reduce", "skip", "skip_each"])
        what = f"case {case} step {step} {op} (n = {n}, p = {p})"
        if op == "skip":
            d = int(rng.choice([0, 1, 11, 12, 13, 1000, (1 << 40) + 5]))
            rlx.rlxpp_skip(h, d)
            g += np.uint64(d)
            continue
        if op == "skip_each":
            d = inputs.splitmix64(int(rng.integers(1 << 30)), n) % np.uint64(rng.choice([2, 12, 5000]))
            rlx.rlxpp_skip_each(h, torch.from_numpy(d.view(np.int64)).cuda())
            g += d
            continue
        per = int(rng.choice([1, 5, 12, 24, 96, 97, 108, 12 * 23, 12 * 16, 250]))
        sm = bool(rng.integers(0, 2))
        lay = rlx.RLXPP_STREAM_MAJOR if sm else rlx.RLXPP_INTERLEAVED
        shape = (lambda k: (n, k) if sm else (k, n))
        rows = (lambda t: t.cpu().numpy() if sm else t.cpu().numpy().T)
        if op == "reduce":
            S = torch.empty(n, dtype=torch.float64, device="cuda")
            Q = torch.empty(n, dtype=torch.float64, device="cuda")
            rlx.rlxpp_generate_reduce(h, S, Q, per)
            ref = oracle.streams(seeds, p, per, skips=g, want=("sums",), nthreads=nthreads)
            assert_bits_equal(S.cpu().numpy(), ref["sum"], what + " sum")
            assert_bits_equal(Q.cpu().numpy(), ref["sumsq"], what + " sumsq")
        elif op == "normal":
            out = torch.empty(shape(per), dtype=torch.float64, device="cuda")
            rlx.rlxpp_generate_normal(h, out, per, lay)
            odd = (g & np.uint64(1)).astype(np.int64)
            k = oracle.streams(seeds, p, per + 2 + (per & 1), skips=g - odd.astype(np.uint64), want=("ints",), nthreads=nthreads)["ints"]
            z = oracle.normals(k)
            want = np.stack([z[i, odd[i]:odd[i] + per] for i in range(n)])
            assert_within_ulps(rows(out), want, NORMAL_ULPS, what)
        else:
            ref = oracle.streams(seeds, p, per, skips=g, want=("ints", "doubles"), nthreads=nthreads)
            if op == "doubles":
                out = torch.empty(shape(per), dtype=torch.float64, device="cuda")
                rlx.rlxpp_generate_doubles(h, out, per, lay)
                assert_bits_equal(rows(out), ref["doubles"], what)
            elif op == "u48":
                out = torch.empty(shape(per), dtype=torch.int64, device="cuda")
                rlx.rlxpp_generate_u48(h, out, per, lay)
                assert np.array_equal(rows(out).view(np.uint64), ref["ints"]), what
            else:
                out = torch.empty(shape(2 * per), dtype=torch.float32, device="cuda")
                rlx.rlxpp_generate_floats(h, out, 2 * per, lay)
                lo = (ref["ints"] & np.uint64(0xFFFFFF)).astype(np.float32) * np.float32(2.0**-24)
                hi = (ref["ints"] >> np.uint64(24)).astype(np.float32) * np.float32(2.0**-24)
                want = np.stack([lo, hi], axis=-1).reshape(n, 2 * per)
                assert np.array_equal(rows(out).view(np.uint32), want.view(np.uint32)), what
        g += np.uint64(per)
    ref = oracle.streams(seeds, p, 0, skips=g, want=("state",), nthreads=nthreads)
    check_state(rlx, torch, h, ref, f"case {case} final")
    rlx.rlxpp_destroy(h)


@pytest.mark.parametrize("skip, counts", [(0, [250, 1000, 12 * 9 + 2]), (4, [500, 130]), (5, [500]), (0, [251, 300]),
                                          (8, [640, 384]), (4, [1536])])
def test_stream_major_calls_that_are_not_whole_blocks(rlx, torch, oracle, nthreads, skip, counts):
    """Stream-major with one common cursor that is inside a block, or a draw count that is not a multiple of 12
    (rlxpp.cu launch_stream_major_split: head + whole blocks through the aligned path with the row pitch of the
    whole call + tail; odd cursors / odd counts take the general path whole).  All output forms; ragged tile; the
    guard band behind the buffer stays untouched."""
    n = 2 * 128 + 77
    h = rlx.rlxpp_create(n, 8, 2048)
    if skip:
        rlx.rlxpp_skip(h, skip)
    at = skip
    for per in counts:
        for form in ("doubles", "u48", "normal"):
            buf = torch.full((n * per + 512,), -1.0, dtype=torch.float64, device="cuda")
            if form == "doubles":
                rlx.rlxpp_generate_doubles(h, buf, per, rlx.RLXPP_STREAM_MAJOR)
            elif form == "u48":
                rlx.rlxpp_generate_u48(h, buf.view(torch.int64), per, rlx.RLXPP_STREAM_MAJOR)
            else:
                rlx.rlxpp_generate_normal(h, buf, per, rlx.RLXPP_STREAM_MAJOR)
            torch.cuda.synchronize()
            raw = buf.cpu().numpy()
            got = raw[:n * per].reshape(n, per)
            assert np.all(raw[n * per:] == -1.0), "wrote behind the output buffer"
            what = f"skip {skip}, draws {at}..{at + per}, {form}"
            if form == "normal":
                lo = at - (at & 1)
                k = oracle.streams(inputs.seeds(n, 8), 2048, per + 2 + (per & 1), skips=np.full(n, lo, np.uint64),
                                   want=("ints",), nthreads=nthreads)["ints"]
                assert_within_ulps(got, oracle.normals(k)[:, at - lo:at - lo + per], NORMAL_ULPS, what)
            else:
                ref = oracle.streams(inputs.seeds(n, 8), 2048, per, skips=np.full(n, at, np.uint64),
                                     want=("ints", "doubles"), nthreads=nthreads)
                if form == "doubles":
                    assert_bits_equal(got, ref["doubles"], what)
                else:
                    assert np.array_equal(got.view(np.uint64), ref["ints"]), what
            at += per
    ref = oracle.streams(inputs.seeds(n, 8), 2048, 0, skips=np.full(n, at, np.uint64), want=("state",), nthreads=nthreads)
    check_state(rlx, torch, h, ref, "after split calls")
    rlx.rlxpp_destroy(h)


def test_generic_multiplier_streams(rlx, torch, oracle, nthreads):
    """A luxury level without baked-in rows (p = 100) runs the full multiply9x9 + mod_m kernels."""
    assert not rlx.rlxpp_has_fixed_multiplier(100)
    n, per = 260, 60
    h = rlx.rlxpp_create(n, 2**64 - 3, 100)  # seeds wrap mod 2^64
    out = torch.empty((n, per), dtype=torch.float64, device="cuda")
    rlx.rlxpp_generate_doubles(h, out, per, rlx.RLXPP_STREAM_MAJOR)
    ref = oracle.streams(inputs.seeds(n, 2**64 - 3), 100, per, want=("doubles", "state"), nthreads=nthreads)
    assert_bits_equal(out.cpu().numpy(), ref["doubles"], "generic p=100")
    check_state(rlx, torch, h, ref, "generic p=100")


# ------------------------------------------------------------------------------------- state I/O
def test_set_state_edge_states_and_roundtrip(rlx, torch, oracle):
    """Import crafted LCG states (incl. 0, m-1, values >= m and the to_ranlux boundary cases), export
    them in the paper's stored form and draw one block from each."""
    edge = [0, 1, 2, M - 1, M - 2, M, M + 5, 2**576 - 1, M - (1 << 240), 1 << 240, (1 << 336) - 1, 1 << 336,
            (1 << 336) + 1, (1 << 575), ((1 << 240) - 1) << 336, (((1 << 240) - 1) << 336) + (1 << 336) - 1]
    rng = np.random.default_rng(3)
    for _ in range(200):  # Xl + Xh near 2^336 and D near 0 (reading D4 / c-4)
        xh = int.from_bytes(rng.bytes(30), "little")
        edge.append(((xh << 336) + ((1 << 336) - xh + int(rng.integers(-2, 3)))) % 2**576)
        edge.append(((xh << 336) + (xh << 96) + int(rng.integers(0, 2**20))) % 2**576)
    n = len(edge)
    states = np.stack([inputs.int_to_limbs(x) for x in edge])
    h = rlx.rlxpp_create(n, 1, 2048)
    rlx.rlxpp_set_state(h, torch.from_numpy(states.view(np.int64)).cuda(), None)
    V, c, pos, X = gpu_state(rlx, torch, h)
    for i, x in enumerate(edge):
        xc = x % M
        assert inputs.limbs_to_int(X[i]) == xc
        Vo, co = oracle.to_ranlux(xc)
        assert inputs.limbs_to_int(V[i]) == Vo and int(c[i]) == co, f"to_ranlux edge {i}"
    out = torch.empty((n, 12), dtype=torch.float64, device="cuda")
    rlx.rlxpp_generate_doubles(h, out, 12, rlx.RLXPP_STREAM_MAJOR)
    got = (out.cpu().numpy() * 2.0**48).astype(np.uint64)
    A = oracle.multiplier(2048)
    for i, x in enumerate(edge):
        Vo, _ = oracle.to_ranlux(oracle.mulmod(A, x % M))
        assert [int(v) for v in got[i]] == [(Vo >> (48 * j)) & (2**48 - 1) for j in range(12)]


# ------------------------------------------------------------------------------------- host variants
def test_set_state_from_the_papers_stored_form(rlx, torch, oracle, nthreads):
    """SURVEY 8a-2 / reading D3: rlxpp_set_state_ranlux runs `to_lcg` (X = V - (V >> 336) + c) on the device.
    (a) arbitrary packed numbers and both carries -- random, all zero, all ones (c = 1 reaches m -> 0), top ten
    numbers all ones, only old / only new numbers -- against the oracle's to_lcg; (b) a generator moved through
    get_state -> set_state_ranlux mid-block continues bit for bit."""
    rng = np.random.default_rng(11)
    full = (1 << 576) - 1
    Vs = [0, 1, full, full, full - 1, full >> 240, (full >> 336) << 336, 1 << 336, (1 << 336) - 1, 1 << 575]
    cs = [0, 1, 0, 1, 1, 1, 1, 0, 1, 0]
    for _ in range(246):
        Vs.append(int.from_bytes(rng.bytes(72), "little"))
        cs.append(int(rng.integers(0, 2)))
    n = len(Vs)
    h = rlx.rlxpp_create(n, 1, 2048)
    Vd = torch.from_numpy(np.stack([inputs.int_to_limbs(v) for v in Vs]).view(np.int64)).cuda()
    cd = torch.from_numpy(np.array(cs, dtype=np.int32)).cuda()
    rlx.rlxpp_set_state_ranlux(h, Vd, cd, None)
    _, _, pos, X = gpu_state(rlx, torch, h)
    for i in range(n):
        assert inputs.limbs_to_int(X[i]) == oracle.to_lcg(Vs[i], cs[i]) % M, f"to_lcg case {i}"
    assert np.all(pos == 12)
    rlx.rlxpp_destroy(h)
    # (b) hand-over in the stored form, cursors inside a block
    n, first, rest = 300, 17, 43
    a = rlx.rlxpp_create(n, 31, 2048)
    d1 = torch.empty((n, first), dtype=torch.float64, device="cuda")
    rlx.rlxpp_generate_doubles(a, d1, first, rlx.RLXPP_STREAM_MAJOR)
    V = torch.empty((n, 9), dtype=torch.int64, device="cuda")
    c = torch.empty(n, dtype=torch.int32, device="cuda")
    pos = torch.empty(n, dtype=torch.int32, device="cuda")
    rlx.rlxpp_get_state(a, V, c, pos, None)
    b = rlx.rlxpp_create(n, 999, 2048)
    rlx.rlxpp_set_state_ranlux(b, V, c, pos)
    d2 = torch.empty((n, rest), dtype=torch.float64, device="cuda")
    rlx.rlxpp_generate_doubles(b, d2, rest, rlx.RLXPP_STREAM_MAJOR)
    ref = oracle.streams(inputs.seeds(n, 31), 2048, first + rest, want=("doubles", "state"), nthreads=nthreads)
    assert_bits_equal(d2.cpu().numpy(), ref["doubles"][:, first:], "continued from the stored form")
    check_state(rlx, torch, b, ref, "continued from the stored form")
    rlx.rlxpp_destroy(a)
    rlx.rlxpp_destroy(b)


def test_host_destination_variants(rlx, torch, oracle, nthreads):
    n, per = 2100, 48
    ref = oracle.streams(inputs.seeds(n), 2048, per, want=("doubles", "sums"), nthreads=nthreads)
    for layout in (rlx.RLXPP_STREAM_MAJOR, rlx.RLXPP_INTERLEAVED):
        h = rlx.rlxpp_create(n, 1, 2048)
        shape = (n, per) if layout == rlx.RLXPP_STREAM_MAJOR else (per, n)
        out = torch.empty(shape, dtype=torch.float64).pin_memory()
        rlx.rlxpp_generate_doubles_host(h, out, per, layout)
        got = out.numpy() if layout == rlx.RLXPP_STREAM_MAJOR else out.numpy().T
        assert_bits_equal(got, ref["doubles"], f"host variant layout {layout}")
    h = rlx.rlxpp_create(n, 1, 2048)
    s = np.zeros(n)
    q = np.zeros(n)
    rlx.rlxpp_generate_reduce_host(h, s, q, per)
    assert_bits_equal(s, ref["sum"], "host reduce sum")
    assert_bits_equal(q, ref["sumsq"], "host reduce sumsq")


def test_errors_are_reported_not_swallowed(rlx, torch):
    with pytest.raises(rlx.RlxppError):
        rlx.rlxpp_create(0, 1, 2048)
    with pytest.raises(rlx.RlxppError):
        rlx.rlxpp_create(10, 1, 0)
    h = rlx.rlxpp_create(10, 1, 2048)
    with pytest.raises(rlx.RlxppError):
        rlx.rlxpp_generate_doubles(h, None, 12, rlx.RLXPP_STREAM_MAJOR)
    with pytest.raises(rlx.RlxppError):
        rlx.rlxpp_generate_doubles(h, torch.empty(120, dtype=torch.float64, device="cuda"), 12, 7)
    assert "layout" in rlx.rlxpp_last_error()
    before = rlx.rlxpp_launch_count()
    rlx.rlxpp_generate_doubles(h, torch.empty(120, dtype=torch.float64, device="cuda"), 12, rlx.RLXPP_STREAM_MAJOR)
    assert rlx.rlxpp_launch_count() == before + 1


def test_errors_of_the_widened_calls_and_the_store_probe(rlx, torch):
    h = rlx.rlxpp_create(64, 1, 2048)
    with pytest.raises(rlx.RlxppError):
        rlx.rlxpp_generate_normal(h, None, 12, rlx.RLXPP_STREAM_MAJOR)
    with pytest.raises(rlx.RlxppError):
        rlx.rlxpp_generate_normal(h, torch.empty(64 * 12, dtype=torch.float64, device="cuda"), 12, 9)
    with pytest.raises(rlx.RlxppError):
        rlx.rlxpp_set_state_ranlux(h, None)
    with pytest.raises(rlx.RlxppError):
        rlx.rlxpp_measure_hbm_write_pieces(33, 4096, 256, 1)  # rows must be a multiple of 32
    with pytest.raises(rlx.RlxppError):
        rlx.rlxpp_measure_hbm_write_pieces(64, 4096, 100, 1)  # pieces are multiples of 16 bytes
    rlx.rlxpp_generate_normal(h, torch.empty(1, dtype=torch.float64, device="cuda"), 0, rlx.RLXPP_STREAM_MAJOR)  # no-op
    assert rlx.rlxpp_measure_hbm_write_pieces(1 << 14, 4096, 256, 1) > 1e9  # the probe runs and reports bytes/s
    rlx.rlxpp_destroy(h)


@pytest.mark.parametrize("blocks", [1, 2, 3, 4, 7, 40])
@pytest.mark.parametrize("n", [3 * 128 + 44, 3 * 128 + 45])
def test_interleaved_floats_through_row_boxes(rlx, torch, oracle, nthreads, blocks, n):
    """rlxpp_generate_floats, interleaved, aligned cursors (UMMA engine: the CTA's block leaves as one TMA box of
    24 float rows x 128 streams, three boxes in flight; csrc/stages.cuh F32RowStage).  1, 2, 3 blocks (fewer than the ring),
    more; a ragged last tile the tensor map must clip; n not a multiple of 4 takes the direct stores; forced chunks;
    the guard band stays untouched; two calls in a row."""
    per = 12 * blocks
    h = rlx.rlxpp_create(n, 21, 2048)
    ref = oracle.streams(inputs.seeds(n, 21), 2048, 3 * per, want=("ints", "state"), nthreads=nthreads)
    want = _floats_of(ref["ints"])  # [n][2 * 3 per]
    for call in range(3):
        if call == 2:
            rlx.rlxpp_set_chunks(2)
        try:
            buf = torch.full((2 * per * n + 256,), -1.0, dtype=torch.float32, device="cuda")
            rlx.rlxpp_generate_floats(h, buf, 2 * per, rlx.RLXPP_INTERLEAVED)
            torch.cuda.synchronize()
        finally:
            rlx.rlxpp_set_chunks(0)
        raw = buf.cpu().numpy()
        got = raw[:2 * per * n].reshape(2 * per, n).T
        assert np.array_equal(got.view(np.uint32), want[:, call * 2 * per:(call + 1) * 2 * per].view(np.uint32)), \
            f"interleaved floats, {blocks} blocks, n = {n}, call {call}"
        assert np.all(raw[2 * per * n:] == -1.0), "wrote behind the output buffer"
    check_state(rlx, torch, h, ref, "interleaved floats")
    rlx.rlxpp_destroy(h)


# ------------------------------------------------------------------------------------- sharding
def test_eight_shard_handles_reproduce_one_generator(rlx, torch, oracle, nthreads):
    """The multi-GPU partition on one device, through librlxpp.so: a 2^13 + 37-stream job split into 8 contiguous ranges
    (paper_2106_02504_b200/shard.py), one handle per range seeded with rank_seed(seed, first); the concatenation of the
    shards' outputs (stream-major slabs, interleaved column blocks, fused sums, final states) is what ONE handle over
    all streams gives, and what the oracle gives.  No collective: the ranks never exchange anything."""
    from paper_2106_02504_b200 import shard
    world, n_total, per, p, seed = 8, (1 << 13) + 37, 96, 2048, 2**64 - 4000  # seeds wrap mod 2^64 inside the job
    one = rlx.rlxpp_create(n_total, seed, p)
    whole_sm = torch.empty((n_total, per), dtype=torch.float64, device="cuda")
    rlx.rlxpp_generate_doubles(one, whole_sm, per, rlx.RLXPP_STREAM_MAJOR)
    whole_s = torch.empty(n_total, dtype=torch.float64, device="cuda")
    whole_q = torch.empty(n_total, dtype=torch.float64, device="cuda")
    rlx.rlxpp_generate_reduce(one, whole_s, whole_q, 30)
    sm = torch.full((n_total, per), -1.0, dtype=torch.float64, device="cuda")
    il = torch.full((per, n_total), -1.0, dtype=torch.float64, device="cuda")
    S = torch.full((n_total,), -1.0, dtype=torch.float64, device="cuda")
    Q = torch.full((n_total,), -1.0, dtype=torch.float64, device="cuda")
    handles = []
    for r in range(world):
        first, count = shard.stream_range(r, world, n_total)
        h = rlx.rlxpp_create(count, shard.rank_seed(seed, first), p)
        handles.append((h, first, count))
        rlx.rlxpp_generate_doubles(h, sm[first:first + count], per, rlx.RLXPP_STREAM_MAJOR)  # its slab
        rlx.rlxpp_generate_reduce(h, S[first:first + count], Q[first:first + count], 30)
    torch.cuda.synchronize()
    assert_bits_equal(sm.cpu().numpy(), whole_sm.cpu().numpy(), "8 shards vs one handle, stream-major")
    assert_bits_equal(S.cpu().numpy(), whole_s.cpu().numpy(), "8 shards vs one handle, sums")
    assert_bits_equal(Q.cpu().numpy(), whole_q.cpu().numpy(), "8 shards vs one handle, sums of squares")
    # the interleaved column block of a rank is not contiguous in the job's array: each rank writes its own [per][count]
    for h, first, count in handles:
        blk = torch.empty((per, count), dtype=torch.float64, device="cuda")
        rlx.rlxpp_generate_doubles(h, blk, per, rlx.RLXPP_INTERLEAVED)
        il[:, first:first + count] = blk
    ref = oracle.streams(inputs.seeds(n_total, seed), p, per + 30 + per, want=("doubles", "state"), nthreads=nthreads)
    assert_bits_equal(sm.cpu().numpy(), ref["doubles"][:, :per], "8 shards vs oracle")
    assert_bits_equal(il.cpu().numpy().T, ref["doubles"][:, per + 30:], "8 shards vs oracle, interleaved blocks")
    for h, first, count in handles:
        sub = {k: v[first:first + count] for k, v in ref.items()}
        check_state(rlx, torch, h, sub, f"shard starting at stream {first}")
        rlx.rlxpp_destroy(h)
    rlx.rlxpp_destroy(one)


# ------------------------------------------------------------------------------------- short calls, time-parallel
@pytest.mark.parametrize("n, blocks", [(1024, 32), (128 * 20 + 77, 32), (128 * 60, 40), (5, 4), (128 * 140 + 3, 7), (700, 100)])
def test_short_calls_run_time_parallel(rlx, torch, oracle, nthreads, n, blocks):
    """UMMA engine, calls that leave most of the grid empty (cfg1's shape): K lanes per tile, lane j reaching block j with
    the byte matrix of A^(j+1) and striding with the one of A^K (csrc/kernels_umma.cuh tc_generate_lanes_kernel; reading D7: block b is
    to_ranlux(A^(b+1) X)).  One pass per lane (32 blocks, K = 32), several passes (K = 9 / 29 / 4: 60 or 21 tiles; 100 blocks),
    a 5-stream handle, a grid that is too full for lanes (141 tiles: the persistent path), ragged tiles; every output form
    and layout; the state each call leaves is the one the next call starts from; guard bands stay untouched."""
    per = 12 * blocks
    calls = [("doubles", "sm"), ("doubles", "il"), ("u48", "sm"), ("floats", "il"), ("normal", "il"), ("doubles", "sm")]
    ref = oracle.streams(inputs.seeds(n, 3), 2048, per * len(calls), want=("ints", "doubles", "state"), nthreads=nthreads)
    h = rlx.rlxpp_create(n, 3, 2048)
    for k, (form, lay) in enumerate(calls):
        sm = lay == "sm"
        layout = rlx.RLXPP_STREAM_MAJOR if sm else rlx.RLXPP_INTERLEAVED
        ints = ref["ints"][:, k * per:(k + 1) * per]
        words = 2 * per if form == "floats" else per
        dt = {"doubles": torch.float64, "u48": torch.int64, "floats": torch.float32, "normal": torch.float64}[form]
        buf = torch.full((n * words + 64,), -1, dtype=dt, device="cuda")
        if form == "doubles":
            rlx.rlxpp_generate_doubles(h, buf, per, layout)
        elif form == "u48":
            rlx.rlxpp_generate_u48(h, buf, per, layout)
        elif form == "floats":
            rlx.rlxpp_generate_floats(h, buf, 2 * per, layout)
        else:
            rlx.rlxpp_generate_normal(h, buf, per, layout)
        torch.cuda.synchronize()
        raw = buf.cpu().numpy()
        assert np.all(raw[n * words:] == -1), "wrote behind the output buffer"
        got = raw[:n * words].reshape(n, words) if sm else raw[:n * words].reshape(words, n).T
        what = f"time-parallel call {k} ({form}, {lay}), n = {n}, {blocks} blocks"
        if form == "doubles":
            assert_bits_equal(got, ref["doubles"][:, k * per:(k + 1) * per], what)
        elif form == "u48":
            assert np.array_equal(got.view(np.uint64), ints), what
        elif form == "floats":
            assert np.array_equal(np.ascontiguousarray(got).view(np.uint32), _floats_of(ints).view(np.uint32)), what
        else:
            assert_within_ulps(got, oracle.normals(ints), NORMAL_ULPS, what)
    check_state(rlx, torch, h, ref, "after time-parallel calls")
    rlx.rlxpp_destroy(h)


@pytest.mark.parametrize("per, n_chunks", [(2, 0), (30, 0), (96, 0), (250, 0), (1536, 0), (12 * 50 + 6, 3), (251, 0)])
def test_stream_major_per_stream_cursors_through_rings(rlx, torch, oracle, nthreads, per, n_chunks):
    """Stream-major output when the cursors are not at a block boundary (per-stream skips; one odd common cursor).  UMMA
    engine, even row length: every lane writes its 12 doubles at its own columns of a shared-memory ring and the warp sends
    128-byte granules of 32 rows as TMA boxes once its slowest lane has completed them (csrc/stages.cuh RingStage); row ends and
    rows past the launch are clipped by the tensor map.  Rows of 2 doubles up to cfg3's 1,536, a length that is not a
    multiple of 16, forced chunks (granule-aligned item starts), a ragged last tile, all 8-byte output forms, the guard
    band behind the buffer, two calls in a row; per = 251 (odd pitch) takes the element-wise row stage instead."""
    n = 3 * 128 + 45
    dist = inputs.splitmix64(777, n) % np.uint64(40)  # every cursor value occurs
    ref = oracle.streams(inputs.seeds(n, 17), 2048, 3 * per + 2, skips=dist, want=("ints", "doubles", "state"), nthreads=nthreads)
    h = rlx.rlxpp_create(n, 17, 2048)
    rlx.rlxpp_skip_each(h, torch.from_numpy(dist.view(np.int64)).cuda())
    rlx.rlxpp_set_chunks(n_chunks)
    try:
        at = 0
        for form in ("doubles", "u48", "doubles"):
            buf = torch.full((n * per + 512,), -1.0, dtype=torch.float64, device="cuda")
            if form == "doubles":
                rlx.rlxpp_generate_doubles(h, buf, per, rlx.RLXPP_STREAM_MAJOR)
            else:
                rlx.rlxpp_generate_u48(h, buf.view(torch.int64), per, rlx.RLXPP_STREAM_MAJOR)
            torch.cuda.synchronize()
            raw = buf.cpu().numpy()
            assert np.all(raw[n * per:] == -1.0), "wrote behind the output buffer"
            got = raw[:n * per].reshape(n, per)
            what = f"per-stream cursors, rows of {per}, {form}, draws {at}..{at + per}"
            if form == "doubles":
                assert_bits_equal(got, ref["doubles"][:, at:at + per], what)
            else:
                assert np.array_equal(got.view(np.uint64), ref["ints"][:, at:at + per]), what
            at += per
    finally:
        rlx.rlxpp_set_chunks(0)
    # normal deviates from the same cursors (pairs counted from each stream's first draw)
    z = torch.full((n, per + (per & 1)), np.nan, dtype=torch.float64, device="cuda")
    per_n = per + (per & 1)
    rlx.rlxpp_generate_normal(h, z, per_n, rlx.RLXPP_STREAM_MAJOR)
    g = dist + np.uint64(at)
    odd = (g & np.uint64(1)).astype(np.int64)
    k = oracle.streams(inputs.seeds(n, 17), 2048, per_n + 2, skips=g - odd.astype(np.uint64), want=("ints",), nthreads=nthreads)["ints"]
    zz = oracle.normals(k)
    want = np.stack([zz[i, odd[i]:odd[i] + per_n] for i in range(n)])
    assert_within_ulps(z.cpu().numpy(), want, NORMAL_ULPS, f"normals through rings, rows of {per_n}")
    ref2 = oracle.streams(inputs.seeds(n, 17), 2048, 0, skips=g + np.uint64(per_n), want=("state",), nthreads=nthreads)
    check_state(rlx, torch, h, ref2, "after ring calls")
    rlx.rlxpp_destroy(h)


@pytest.mark.parametrize("form", ["stream_major", "interleaved", "reduce", "lanes"])
def test_one_hot_state_bytes_reach_their_operand_column(rlx, torch, oracle, form):
    """The A operand of the tensor-core advance is written per thread into tensor memory (18 columns of 32 bits, four K
    bytes each; csrc/umma_path.cuh) or, for the raw advance, into a K-major shared-memory tile.  States with ONE non-zero
    byte -- 2^(8k) and 255 * 2^(8k) for every k < 72 -- pin byte order and column order of that operand: the block each
    produces is to_ranlux(A * x mod m) (D5, D6), row k of the byte matrix scaled.  Every kernel form that writes the
    operand: one tile per CTA (stream-major), two tiles per CTA (interleaved, fused reduce), time-parallel lanes."""
    xs = [v << (8 * k) for k in range(72) for v in (1, 255)] + [M - 1]
    xs = [x for x in xs if x < M]
    n = len(xs)
    states = np.stack([inputs.int_to_limbs(x) for x in xs])
    h = rlx.rlxpp_create(n, 1, 2048)
    rlx.rlxpp_set_state(h, torch.from_numpy(states.view(np.int64)).cuda(), None)
    blocks = 8 if form == "lanes" else 2
    per = 12 * blocks
    A = oracle.multiplier(2048)
    want = np.empty((n, per), dtype=np.uint64)
    for i, x in enumerate(xs):
        for b in range(blocks):
            x = oracle.mulmod(A, x)
            V, _ = oracle.to_ranlux(x)
            want[i, 12 * b:12 * b + 12] = [(V >> (48 * j)) & (2**48 - 1) for j in range(12)]
    if form == "reduce":
        s = torch.empty(n, dtype=torch.float64, device="cuda")
        q = torch.empty(n, dtype=torch.float64, device="cuda")
        rlx.rlxpp_generate_reduce(h, s, q, per)
        d = want.astype(np.float64) * 2.0**-48
        S = np.zeros(n)
        Q = np.zeros(n)
        for k in range(per):  # draw order, one rounding per step (c-14); d*d + Q in exact arithmetic, rounded once
            S = S + d[:, k]
            Q = np.array([float(Fraction(float(a)) * Fraction(float(a)) + Fraction(float(b))) for a, b in zip(d[:, k], Q)])
        assert_bits_equal(s.cpu().numpy(), S, "sum")
        assert_bits_equal(q.cpu().numpy(), Q, "sum of squares")
    else:
        if form == "interleaved":
            out = torch.empty((per, n), dtype=torch.float64, device="cuda")
            rlx.rlxpp_generate_doubles(h, out, per, rlx.RLXPP_INTERLEAVED)
            got = out.cpu().numpy().T
        else:
            if form == "stream_major":
                rlx.rlxpp_set_chunks(1)  # keep the call on the persistent kernel
            try:
                out = torch.empty((n, per), dtype=torch.float64, device="cuda")
                rlx.rlxpp_generate_doubles(h, out, per, rlx.RLXPP_STREAM_MAJOR)
            finally:
                rlx.rlxpp_set_chunks(0)
            got = out.cpu().numpy()
        assert np.array_equal((got * 2.0**48).astype(np.uint64), want)
    rlx.rlxpp_destroy(h)
