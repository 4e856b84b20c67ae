"""GPU parity on the RARE branches of the hot kernels, reached deterministically.

mod_m must give a result "smaller than m in all cases" and the conversion back to RANLUX
numbers (line 39) has cases that random data reaches with probability 2^-16 ... 2^-65 per advance.  The hot
kernels run both as fast forms with an exact fallback (csrc/arith.cuh fold_fast / to_ranlux_fast),
so the fallback plumbing of EVERY kernel variant has to be driven on purpose:

  * craft the state X_t that an advance must PRODUCE (one family per trigger: borrow out of limb 1, carry out of
    limb 9, top limb all ones, folded value in [m, 2^576) or above 2^576, carry out of the 8-limb addition,
    u - w in {-2 .. 2}, u = 2^32 - 1, v[0] = 0 with c = 1, reading D4's third combination),
  * take its pre-image X_0 = A^-d X_t mod m (Python pow), import it with rlxpp_set_state, and generate through
    every store mode, aligned and unaligned cursors, both engines, so that advance number d of that stream lands
    on X_t inside the hot loop,
  * compare doubles, sums, states, carries and cursors with the oracle, bit for bit, and
  * compare the library's rare-path counters (rlxpp_rare_counts) with a Python model of WHICH condition each
    advance of each stream raises, computed from the unreduced product z the engine forms (UMMA: sum of bytes x
    (A 2^(8k) mod m); IMAD: sum of 32-bit limbs x (A 2^(32 i) mod m)) -- so every branch is asserted to have fired,
    exactly as often as the arithmetic says.
"""
from fractions import Fraction

import numpy as np
import pytest

from paper_2106_02504_b200 import inputs

gpu = pytest.mark.gpu

M = (1 << 576) - (1 << 240) + 1
A1 = M - (M - 1) // (1 << 24)            # reading D2: a = b^-1 mod m
P = 2048
A = pow(A1, P, M)
MASK32 = (1 << 32) - 1
FULL = (1 << 576) - 1
NAMES = ("fold_borrow", "fold_carry", "fold_top", "ranlux_carry", "ranlux_near", "ranlux_umax", "ranlux_v0", "ranlux_third")
BORROW, CARRY, TOP, RCARRY, NEAR, UMAX, V0, THIRD = range(8)


@pytest.fixture(scope="module")
def torch():
    import torch as _torch
    if not _torch.cuda.is_available():
        pytest.fail("the gpu-marked tests need a CUDA device (there is no CPU fallback)")
    return _torch


@pytest.fixture(scope="module", params=["umma", "imad"])
def engine(request):
    return request.param


@pytest.fixture(scope="module")
def rlx(torch, engine):
    import paper_2106_02504_b200 as _rlx
    _rlx.load()
    _rlx.rlxpp_set_engine(_rlx.RLXPP_ENGINE_UMMA if engine == "umma" else _rlx.RLXPP_ENGINE_IMAD)
    yield _rlx
    _rlx.rlxpp_set_engine(_rlx.RLXPP_ENGINE_UMMA)


# ------------------------------------------------------------------------------------- the model of the decisions
R_BYTE = [(A << (8 * k)) % M for k in range(74)]    # UMMA engine: rows of the byte matrix; rows 72, 73
                                                    # serve operands that are unreduced products (< 2^591: raw advance)
R_LIMB = [(A << (32 * i)) % M for i in range(18)]   # IMAD engine: pre-reduced rows


def product(engine, x):
    """The unreduced value z == A x (mod m) the engine's multiply leaves for fold_fast."""
    if engine == "umma":
        assert x < 1 << 592
        return sum(((x >> (8 * k)) & 0xFF) * R_BYTE[k] for k in range(74))
    return sum(((x >> (32 * i)) & MASK32) * R_LIMB[i] for i in range(18))


def fold_mask(z):
    hi, lo = z >> 576, z & FULL
    m = 0
    if (lo & ((1 << 64) - 1)) < hi:
        m |= 1 << BORROW
    if ((lo >> 224) & ((1 << 96) - 1)) + (hi << 16) >= 1 << 96:
        m |= 1 << CARRY
    if lo >> 544 == MASK32:
        m |= 1 << TOP
    return m


def ranlux_mask(x, oracle):
    u, w = (x >> 304) & MASK32, x >> 544
    xh = x >> 336
    m = 0
    if (x & ((1 << 256) - 1)) + xh >= 1 << 256:
        m |= 1 << RCARRY
    if abs(u - w) <= 1:
        m |= 1 << NEAR
    if u == MASK32:
        m |= 1 << UMAX
    if ((x + xh) & MASK32) < (1 if u < w else 0):
        m |= 1 << V0
    V, c = oracle.to_ranlux(x)
    if c == 1 and V == x + xh:
        m |= 1 << THIRD
    return m


FAST_BITS = (1 << RCARRY) | (1 << NEAR) | (1 << UMAX) | (1 << V0)


def model_counts(engine, oracle, x0s, n_fold, n_hot, pad_to=128):
    """Expected rlxpp_rare_counts after a call in which stream i goes through n_fold[i] folds (advances whose product
    is reduced) of which the first n_hot[i] are also converted by to_ranlux_hot / advance_block.
    UMMA engine: the rows that pad the last tile (pad_to = 128 streams; 256 for the kernels that run two tiles per CTA)
    are advanced as x = 0, whose two leading words are equal (u = w = 0): every conversion of such a row takes the exact
    path and counts as `ranlux_near`; the IMAD engine has no such rows."""
    cnt = np.zeros(8, np.uint64)
    if engine == "umma" and max(n_hot, default=0) > 0:
        cnt[NEAR] += ((-len(x0s)) % pad_to) * max(n_hot)
    for x, nf, nh in zip(x0s, n_fold, n_hot):
        for a in range(1, nf + 1):
            fm = fold_mask(product(engine, x))
            x = A * x % M
            rm = ranlux_mask(x, oracle) if a <= nh else 0
            if engine == "umma":   # reduce_z and to_ranlux_hot count separately; the latter always sees the exact x
                mask = fm | (rm if rm & FAST_BITS else 0)
            elif a > nh:           # IMAD, raw advance (Fixed::advance)
                mask = fm
            elif fm:               # IMAD advance_block: one rare path; to_ranlux_fast saw a wrong x
                mask = fm | (rm & (1 << THIRD))
            else:
                mask = rm if rm & FAST_BITS else 0
            for k in range(8):
                cnt[k] += (mask >> k) & 1
    return cnt


def model_counts_lanes(oracle, x0s, nblk):
    """UMMA engine, time-parallel path with one lane per block (tc_generate_lanes_kernel, K = nblk): block j of a stream is
    ONE pass from the stored state against the byte matrix of A^(j+1), so the product that is folded is
    sum_k xb_k (A^(j+1) 2^(8k) mod m), not a chain of products by A."""
    cnt = np.zeros(8, np.uint64)
    cnt[NEAR] += ((-len(x0s)) % 128) * nblk
    for j in range(1, nblk + 1):
        Aj = pow(A, j, M)
        rows = [(Aj << (8 * k)) % M for k in range(72)]
        for x0 in x0s:
            fm = fold_mask(sum(((x0 >> (8 * k)) & 0xFF) * rows[k] for k in range(72)))
            rm = ranlux_mask(Aj * x0 % M, oracle)
            mask = fm | (rm if rm & FAST_BITS else 0)
            for k in range(8):
                cnt[k] += (mask >> k) & 1
    return cnt


# ------------------------------------------------------------------------------------- crafted target states
def crafted_targets():
    """(family, X_t) pairs; X_t canonical (< m)."""
    rng = np.random.default_rng(20210602)

    def rnd(bits):
        return int.from_bytes(rng.bytes(72), "little") >> (576 - bits)

    def put(x, lo, width, val):
        return (x & ~(((1 << width) - 1) << lo)) | ((val & ((1 << width) - 1)) << lo)

    out = []
    for s in (0, 1, 2, 5):                       # borrow of "- hi" out of limb 1: low 64 bits just below 2^64
        out.append(("fold_borrow", put(rnd(575), 0, 64, (1 << 64) - 1 - s)))
    for s in (0, 1, 0x1234, 1 << 20):            # carry of "+ hi 2^240" out of limb 9: bits 224..319 small
        out.append(("fold_carry", put(rnd(575), 224, 96, s)))
    for _ in range(4):                           # top limb all ones, still < m
        out.append(("fold_top", put(rnd(576), 544, 32, MASK32) & ~(1 << 400)))
    # A x lands below hi (2^240 - 1) (hi = z >> 576: ~2^12 UMMA, ~2^34 IMAD): the fold gives X_t + m, in [m, 2^576)
    # or above 2^576; 2^255 is past that for the UMMA engine only
    for x in (1, 2, (1 << 240) - 2, (1 << 240) - 1, 1 << 240, (1 << 241) + 5, 1 << 255, rnd(239), rnd(250), rnd(252)):
        out.append(("fold_small", x))
    for _ in range(4):                           # carry out of the 8-limb addition: limb 7 all ones, X >> 560 != 0
        out.append(("ranlux_carry", put(put(rnd(574), 224, 32, MASK32), 560, 14, 1 + rnd(13))))
    for delta in (-2, -1, 0, 1, 2):              # u - w = delta, with every fill below the two words
        for fill in ("ones", "zeros", "random"):
            w = 5 + rnd(31)
            x = rnd(575)
            if fill == "ones":
                x = put(put(x, 0, 304, (1 << 304) - 1), 336, 208, (1 << 208) - 1)
            elif fill == "zeros":
                x = put(put(x, 0, 304, 0), 336, 208, 0)
            out.append((f"near{delta:+d}", put(put(x, 544, 32, w), 304, 32, w + delta)))
    for w in (rnd(31), MASK32 - 1, 7):           # u = 2^32 - 1
        out.append(("ranlux_umax", put(put(rnd(575), 304, 32, MASK32), 544, 32, w)))
    for _ in range(4):                           # c = 1 and limb 0 of X + (X >> 336) is zero
        x = put(put(rnd(575), 544, 32, (1 << 31) + rnd(30)), 304, 32, rnd(30))
        out.append(("ranlux_v0", put(x, 0, 32, -((x >> 336) & MASK32))))
    for e in (0, 1, 3, 1 << 100):                # third combination: Xl + Xh crosses 2^336
        xh = rnd(239)
        out.append(("ranlux_third", (xh << 336) | ((1 << 336) - xh + e)))
    out.append(("max_hi", M - 2))                # bytes 0xFF except one 0xFE: the largest z[18] a canonical state gives
    for fam, x in out:
        assert 0 <= x < M, fam
    return out


def build_streams(n, depths, pad_seed=77):
    """n canonical start states: every crafted target at every depth d (X_0 = A^-d X_t), the rest random."""
    targets = crafted_targets()
    x0s, info = [], []
    for d in depths:
        inv = pow(A, -d, M)
        for fam, xt in targets:
            x0s.append(inv * xt % M)
            info.append((fam, d, xt))
    assert len(x0s) <= n, (len(x0s), n)
    rnd = inputs.cfg2_random_states(n - len(x0s), seed=pad_seed)
    x0s += [inputs.limbs_to_int(r) for r in rnd]
    info += [("random", 0, None)] * (n - len(info))
    order = np.random.default_rng(5).permutation(n)  # crafted rows spread over all tiles and warps
    return [x0s[i] for i in order], [info[i] for i in order]


def to_dev(torch, xs):
    return torch.from_numpy(np.stack([inputs.int_to_limbs(x) for x in xs]).view(np.int64)).cuda()


def oracle_run(oracle, x0s, pos, n_draws):
    """Per stream: (48-bit draws, final X, final pos) from the oracle's engine (D8)."""
    ints = np.zeros((len(x0s), n_draws), np.uint64)
    xe, pe = [], []
    for i, x in enumerate(x0s):
        X, p_, d = oracle.engine_run(x, int(pos[i]), P, [("draw", n_draws)])
        ints[i] = d
        xe.append(X)
        pe.append(p_)
    return ints, xe, pe


def check_final_state(rlx, torch, oracle, h, xe, pe, what):
    n = h.n_streams
    V = torch.empty((n, 9), dtype=torch.int64, device="cuda")
    X = torch.empty((n, 9), dtype=torch.int64, device="cuda")
    c = torch.empty(n, dtype=torch.int32, device="cuda")
    pos = torch.empty(n, dtype=torch.int32, device="cuda")
    rlx.rlxpp_get_state(h, V, c, pos, X)
    torch.cuda.synchronize()
    V, X, c, pos = V.cpu().numpy().view(np.uint64), X.cpu().numpy().view(np.uint64), c.cpu().numpy(), pos.cpu().numpy()
    for i in range(n):
        assert inputs.limbs_to_int(X[i]) == xe[i], f"{what}: LCG state of stream {i}"
        Vo, co = oracle.to_ranlux(xe[i])
        assert inputs.limbs_to_int(V[i]) == Vo and int(c[i]) == co, f"{what}: RANLUX numbers / carry of stream {i}"
        assert int(pos[i]) == pe[i], f"{what}: cursor of stream {i}"


def assert_counts(rlx, want, what, families_needed=()):
    got = rlx.rlxpp_rare_counts()
    assert got.tolist() == want.tolist(), f"{what}: rare-path counters {dict(zip(NAMES, got.tolist()))} != model " \
                                          f"{dict(zip(NAMES, want.tolist()))}"
    for k in families_needed:
        assert got[k] > 0, f"{what}: branch {NAMES[k]} never fired"


ALL_HOT = (BORROW, CARRY, TOP, RCARRY, NEAR, UMAX, V0, THIRD)


# ------------------------------------------------------------------------------------- the tests
def test_crafted_states_hit_what_they_are_crafted_for(oracle):
    """CPU: the Python model on the crafted targets alone.  Each family raises its own condition -- the to_ranlux ones
    on the canonical X_t, the fold ones on the product of its pre-image with either engine's rows -- and where no
    to_ranlux condition is raised (u - w = +-2 included) the fast decision V = X + Xh - [u < w] is the oracle's."""
    inv = pow(A, -1, M)
    for fam, xt in crafted_targets():
        for eng in ("umma", "imad"):
            fm = fold_mask(product(eng, inv * xt % M))
            if fam == "fold_borrow":
                assert fm & (1 << BORROW), (fam, eng)
            elif fam == "fold_carry":
                assert fm & (1 << CARRY), (fam, eng)
            elif fam == "fold_top":
                assert fm & (1 << TOP), (fam, eng)
            elif fam == "fold_small" and xt < 1 << 251:  # X_t < hi (2^240 - 1): the fold gives X_t + m, i.e. top limb
                assert fm & ((1 << TOP) | (1 << CARRY)), (fam, eng)  # all ones, or a carry that runs to the very top
        rm = ranlux_mask(xt, oracle)
        if fam == "ranlux_carry":
            assert rm & (1 << RCARRY)
        elif fam in ("near-1", "near+0", "near+1"):
            assert rm & (1 << NEAR)
        elif fam in ("near-2", "near+2"):
            assert not rm & (1 << NEAR)
        elif fam == "ranlux_umax":
            assert rm & (1 << UMAX)
        elif fam == "ranlux_v0":
            assert rm & (1 << V0)
        elif fam == "ranlux_third":
            assert rm & (1 << THIRD) and rm & (1 << UMAX)
        # the fast decision itself on the states it is allowed to decide: V = X + Xh - c with c = [u < w]
        if not rm & FAST_BITS:
            u, w = (xt >> 304) & MASK32, xt >> 544
            c = 1 if u < w else 0
            assert oracle.to_ranlux(xt) == (xt + (xt >> 336) - c, c), fam


@gpu
@pytest.mark.parametrize("mode", ["stream_major_short", "stream_major_tma", "interleaved", "interleaved_odd", "reduce",
                                  "floats_boxes", "u48", "chunked", "lanes"])
def test_rare_branches_aligned(rlx, torch, oracle, engine, mode):
    """Aligned cursors (pos = 12, whole blocks): the pipelined loops of tc_generate_kernel<.., aligned> (stream-major,
    floats), tc_pair_kernel<aligned, ..> (interleaved, even and odd stream counts; fused reduce) and generate_kernel<.., aligned> (IMAD), kept on the serial path with rlxpp_set_chunks; the crafted state is
    produced by advance d in {1, 2, 3, nblk}.  `lanes`: the time-parallel path such short calls take by default, where
    block d is one pass against the matrix of A^d."""
    nblk = {"stream_major_short": 4, "stream_major_tma": 17, "interleaved": 4, "interleaved_odd": 4, "reduce": 5,
            "floats_boxes": 4, "u48": 4, "chunked": 32, "lanes": 32}[mode]
    n = {"chunked": 3 * 128 + 44, "lanes": 3 * 128 + 44, "interleaved_odd": 4 * 128 + 45}.get(mode, 4 * 128 + 44)
    depths = {"chunked": (1, 16, 17, 32), "lanes": (1, 2, 17, 32)}.get(mode, (1, 2, 3, nblk))
    x0s, info = build_streams(n, depths)
    per = 12 * nblk
    h = rlx.rlxpp_create(n, 1, P)
    rlx.rlxpp_set_state(h, to_dev(torch, x0s), None)
    ints, xe, pe = oracle_run(oracle, x0s, [12] * n, per)
    want = ints.astype(np.float64) * 2.0**-48
    rlx.rlxpp_rare_counts(reset=True)
    if mode != "lanes":  # a forced chunk count keeps the call on the persistent kernels
        rlx.rlxpp_set_chunks(2 if mode == "chunked" else 1)
    try:
        if mode in ("stream_major_short", "stream_major_tma", "chunked", "lanes"):
            out = torch.empty((n, per), dtype=torch.float64, device="cuda")
            rlx.rlxpp_generate_doubles(h, out, per, rlx.RLXPP_STREAM_MAJOR)
            assert np.array_equal(out.cpu().numpy().view(np.uint64), want.view(np.uint64)), mode
        elif mode in ("interleaved", "interleaved_odd"):
            out = torch.empty((per, n), dtype=torch.float64, device="cuda")
            rlx.rlxpp_generate_doubles(h, out, per, rlx.RLXPP_INTERLEAVED)
            assert np.array_equal(out.cpu().numpy().T.copy().view(np.uint64), want.view(np.uint64)), mode
        elif mode == "u48":
            out = torch.empty((n, per), dtype=torch.int64, device="cuda")
            rlx.rlxpp_generate_u48(h, out, per, rlx.RLXPP_STREAM_MAJOR)
            assert np.array_equal(out.cpu().numpy().view(np.uint64), ints), mode
        elif mode == "floats_boxes":
            out = torch.empty((2 * per, n), dtype=torch.float32, device="cuda")
            rlx.rlxpp_generate_floats(h, out, 2 * per, rlx.RLXPP_INTERLEAVED)
            lo = (ints & np.uint64(0xFFFFFF)).astype(np.float32) * np.float32(2.0**-24)
            hi = (ints >> np.uint64(24)).astype(np.float32) * np.float32(2.0**-24)
            wantf = np.stack([lo, hi], axis=-1).reshape(n, 2 * per)
            assert np.array_equal(out.cpu().numpy().T.copy().view(np.uint32), wantf.view(np.uint32)), mode
        else:
            S = torch.empty(n, dtype=torch.float64, device="cuda")
            Q = torch.empty(n, dtype=torch.float64, device="cuda")
            rlx.rlxpp_generate_reduce(h, S, Q, per)
            Sw, Qw = sums_in_draw_order(want)
            assert np.array_equal(S.cpu().numpy().view(np.uint64), Sw.view(np.uint64)), "fused sum"
            assert np.array_equal(Q.cpu().numpy().view(np.uint64), Qw.view(np.uint64)), "fused sum of squares"
    finally:
        rlx.rlxpp_set_chunks(0)
    # u48 and floats always run the UMMA engine's kernels (include/rlxpp.h)
    eng = "umma" if mode in ("u48", "floats_boxes") else engine
    pad_to = 256 if mode in ("reduce", "interleaved", "interleaved_odd") else 128  # two tiles per CTA (tc_pair_kernel)
    if mode == "lanes" and eng == "umma":
        want_counts = model_counts_lanes(oracle, x0s, nblk)
    else:
        want_counts = model_counts(eng, oracle, x0s, [nblk] * n, [nblk] * n, pad_to)
    assert_counts(rlx, want_counts, f"aligned {mode}", ALL_HOT)
    check_final_state(rlx, torch, oracle, h, xe, pe, f"aligned {mode}")
    rlx.rlxpp_destroy(h)


def sums_in_draw_order(d):
    """S = S + d, Q = fma(d, d, Q) per row, in order (reading c-14), with exact rationals for the fma."""
    n = d.shape[0]
    S, Q = np.zeros(n), np.zeros(n)
    for i in range(n):
        a = b = 0.0
        for v in d[i]:
            v = float(v)
            a = a + v
            b = float(Fraction(v) * Fraction(v) + Fraction(b))
        S[i], Q[i] = a, b
    return S, Q


@gpu
@pytest.mark.parametrize("mode", ["stream_major", "interleaved", "reduce"])
@pytest.mark.parametrize("cursors", ["five", "random"])
def test_rare_branches_unaligned(rlx, torch, oracle, engine, mode, cursors):
    """Cursors inside a block (set_state with per-stream pos): block 0 is the current block (exact conversion), blocks
    1 .. smax - 2 run the unmasked middle loop, the last two the masked one; 48 draws from cursor 5 make the crafted
    state appear as block 1, 2 (middle), 3 or 4 (masked).  Stream-major goes through UnalignedRowStage."""
    n, per = 3 * 128 + 77, 48
    x0s, info = build_streams(n, (1, 2, 3, 4))
    if cursors == "five":
        pos = np.full(n, 5, np.int32)
    else:
        pos = (inputs.splitmix64(4711, n) % np.uint64(13)).astype(np.int32)
    h = rlx.rlxpp_create(n, 1, P)
    rlx.rlxpp_set_state(h, to_dev(torch, x0s), torch.from_numpy(pos).cuda())
    ints, xe, pe = oracle_run(oracle, x0s, pos, per)
    want = ints.astype(np.float64) * 2.0**-48
    rlx.rlxpp_rare_counts(reset=True)
    if mode == "stream_major":
        buf = torch.full((n * per + 64,), -1.0, dtype=torch.float64, device="cuda")
        rlx.rlxpp_generate_doubles(h, buf, per, rlx.RLXPP_STREAM_MAJOR)
        raw = buf.cpu().numpy()
        assert np.array_equal(raw[:n * per].reshape(n, per).view(np.uint64), want.view(np.uint64)), mode
        assert np.all(raw[n * per:] == -1.0)
    elif mode == "interleaved":
        out = torch.empty((per, n), dtype=torch.float64, device="cuda")
        rlx.rlxpp_generate_doubles(h, out, per, rlx.RLXPP_INTERLEAVED)
        assert np.array_equal(out.cpu().numpy().T.copy().view(np.uint64), want.view(np.uint64)), mode
    else:
        S = torch.empty(n, dtype=torch.float64, device="cuda")
        Q = torch.empty(n, dtype=torch.float64, device="cuda")
        rlx.rlxpp_generate_reduce(h, S, Q, per)
        Sw, Qw = sums_in_draw_order(want)
        assert np.array_equal(S.cpu().numpy().view(np.uint64), Sw.view(np.uint64)), "fused sum"
        assert np.array_equal(Q.cpu().numpy().view(np.uint64), Qw.view(np.uint64)), "fused sum of squares"
    last = [(int(p_) + per - 1) // 12 for p_ in pos]   # advances a stream takes (D8)
    smax = (12 + per - 1) // 12                        # trip count of every thread
    # UMMA: every thread reduces the product of all smax passes (a stream that ends one block early discards the last);
    # IMAD: a thread advances only up to its own last block
    n_fold = [smax] * n if engine == "umma" else last
    needed = ALL_HOT if cursors == "five" else ()
    pad_to = 256 if mode in ("reduce", "interleaved") else 128
    assert_counts(rlx, model_counts(engine, oracle, x0s, n_fold, last, pad_to), f"unaligned {mode} {cursors}", needed)
    check_final_state(rlx, torch, oracle, h, xe, pe, f"unaligned {mode}")
    rlx.rlxpp_destroy(h)


@gpu
@pytest.mark.parametrize("layout", ["aos", "soa"])
def test_rare_branches_raw_advance(rlx, torch, oracle, engine, layout):
    """rlxpp_advance_states (cfg2's kernel): only the fold.  Besides the pre-images, raw non-canonical inputs with the
    largest products: 2^576 - 1 (all bytes 0xFF: the largest z[18] the byte products can give), m, m + 1.  The UMMA
    kernel folds only the last of the `reps` products (the state stays an unreduced product in between), so the crafted
    state must be the FINAL one to reach its fold: depth d = reps."""
    reps = 4
    x0s, info = build_streams(3 * 128 + 61, (1, 2, 3, 4))
    x0s = x0s + [FULL, M, M + 1, FULL - 1, M - 2]
    n = len(x0s)
    states = np.stack([inputs.int_to_limbs(x) for x in x0s])
    want = oracle.advance_states(states, P, reps)
    rlx.rlxpp_rare_counts(reset=True)
    if layout == "aos":
        dev = torch.from_numpy(states.view(np.int64)).cuda()
        rlx.rlxpp_advance_states(dev, n, P, reps, rlx.RLXPP_AOS)
        got = dev.cpu().numpy().view(np.uint64)
    else:
        dev = torch.from_numpy(np.ascontiguousarray(states.T).view(np.int64)).cuda()
        rlx.rlxpp_advance_states(dev, n, P, reps, rlx.RLXPP_SOA)
        got = np.ascontiguousarray(dev.cpu().numpy().view(np.uint64).T)
    assert np.array_equal(got, want), f"raw advance {layout}"
    for i, x in enumerate(x0s):  # and against Python itself
        assert inputs.limbs_to_int(got[i]) == pow(A, reps, M) * x % M
    if engine == "umma":
        # the tensor-core raw advance keeps the state UNREDUCED between repetitions (the byte matrix has columns for
        # the two bytes above 2^576) and folds the last product only: one fold per state, of the reps-fold product chain
        want_counts = np.zeros(8, np.uint64)
        for x in x0s:
            z = x
            for _ in range(reps):
                z = product("umma", z)
            assert z % M == pow(A, reps, M) * x % M and z < 1 << 591
            for k in range(8):
                want_counts[k] += (fold_mask(z) >> k) & 1
    else:
        want_counts = model_counts(engine, oracle, x0s, [reps] * n, [0] * n)
    assert_counts(rlx, want_counts, f"raw advance {layout}", (BORROW, CARRY, TOP))
    # the largest overflow limb: z >> 576 for the all-ones input, as the model computes it
    assert 8000 < product("umma", FULL) >> 576 < 1 << 15 and product("imad", FULL) >> 576 < 1 << 37


@gpu
def test_counters_stay_zero_on_ordinary_streams_and_reset(rlx, torch):
    """A few thousand ordinary advances raise nothing but (possibly) the 2^-16 carry of the 8-limb addition; reset works."""
    rlx.rlxpp_rare_counts(reset=True)
    assert rlx.rlxpp_rare_counts().tolist() == [0] * 8
    h = rlx.rlxpp_create(256, 1, P)
    out = torch.empty((256, 120), dtype=torch.float64, device="cuda")
    rlx.rlxpp_generate_doubles(h, out, 120, rlx.RLXPP_STREAM_MAJOR)
    c = rlx.rlxpp_rare_counts(reset=True)
    assert sum(c.tolist()) == int(c[RCARRY]) <= 3
    assert rlx.rlxpp_rare_counts().tolist() == [0] * 8
    rlx.rlxpp_destroy(h)


@gpu
@pytest.mark.parametrize("coop", [1, 3])
def test_rare_branches_device_api(rlx, torch, oracle, engine, coop):
    """The public device headers on the crafted states: rlxpp_dev::TileStream (include/rlxpp_tile.cuh, coop = 3) runs the
    same fast forms with the same exact fallbacks inside its tensor-core pass (no counters there: parity only);
    rlxpp_dev::Stream (coop = 1) is exact arithmetic throughout.  Every stream draws its own count from its own cursor."""
    if engine != "umma":
        pytest.skip("the device API does not depend on the library's engine switch")
    n = 3 * 128 + 77
    x0s, info = build_streams(n, (1, 2, 3, 4))
    pos = (inputs.splitmix64(1234, n) % np.uint64(13)).astype(np.int32)
    pos[::3] = 12
    cnt = (40 + inputs.splitmix64(99, n) % np.uint64(20)).astype(np.uint32)  # 40 .. 59 draws: 4 or 5 passes
    ld = 64
    h = rlx.rlxpp_create(n, 1, P)
    rlx.rlxpp_set_state(h, to_dev(torch, x0s), torch.from_numpy(pos).cuda())
    out = torch.full((n, ld), -1.0, dtype=torch.float64, device="cuda")
    rlx.rlxpp_generate_ragged(h, torch.from_numpy(cnt.view(np.int32)).cuda(), out, ld, coop)
    torch.cuda.synchronize()
    got = out.cpu().numpy()
    xe, pe = [], []
    for i in range(n):
        X, p_, d = oracle.engine_run(x0s[i], int(pos[i]), P, [("draw", int(cnt[i]))])
        want = np.array(d, np.uint64).astype(np.float64) * 2.0**-48
        assert np.array_equal(got[i, :cnt[i]].view(np.uint64), want.view(np.uint64)), f"stream {i} ({info[i][0]})"
        assert np.all(got[i, cnt[i]:] == -1.0)
        xe.append(X)
        pe.append(p_)
    check_final_state(rlx, torch, oracle, h, xe, pe, f"device API coop = {coop}")
    rlx.rlxpp_destroy(h)
