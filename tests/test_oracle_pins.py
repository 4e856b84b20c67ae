"""Pins for the CPU oracle (oracle/rlxpp_oracle.cpp) -- everything here runs without a GPU.

The paper prints no algorithm bodies and no output values, so the
oracle is pinned against what the paper and the mathematics fix, using Python's
arbitrary-precision integers as the independent side:
  * m = 2^576 - 2^240 + 1; uint64[9]/uint64[18] layouts
  * mod_m result is the remainder and < m in all cases  -> Python %
  * RANLUX++ is the LCG equivalent of subtract-with-borrow RANLUX
      -> advance by a^p == p direct SWB steps (SWB stepper re-stated here in Python)
  * 48 bits per double, 12 per LCG advance -> lattice tests
  * skip "without generating them" -> skip(n) == n draws
The readings D1-D8 / c-1..c-18 referenced below are SURVEY.md section 8(c), restated in DESIGN.md.
"""
import json
import os
import random
from fractions import Fraction

import numpy as np
import pytest

from paper_2106_02504_b200 import inputs

B = 1 << 24
M = (1 << 576) - (1 << 240) + 1
A1 = M - (M - 1) // B  # b^-1 mod m  (D2)
GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "survey_vectors.json")))


# ----------------------------------------------------------------- Python side of the pins
def py_swb_step(x, c):
    """D1, literally: x = list of 24 numbers, oldest first."""
    t = x[24 - 10] - x[0] - c
    cn = 1 if t < 0 else 0
    return x[1:] + [t + (cn << 24)], cn


def pack(x):
    return sum(v << (24 * j) for j, v in enumerate(x))


def unpack(V):
    return [(V >> (24 * j)) & (B - 1) for j in range(24)]


def py_digits(X):
    """Row c-4: number j of V is (-(b^(24-j) X mod m)) mod b."""
    return [(-(pow(B, 24 - j, M) * X % M)) % B for j in range(24)]


def rand_recurrent_state(rng):
    x = [rng.randrange(B) for _ in range(24)]
    c = rng.randrange(2)
    for _ in range(48):
        x, c = py_swb_step(x, c)
    return x, c


EDGE = [0, 1, 2, M - 2, M - 1, M - (1 << 240), 1 << 240, (1 << 336) - 1, (1 << 336) + 1, (1 << 575), M >> 1]


# ----------------------------------------------------------------- constants
def test_modulus_and_multiplier_constants(oracle):
    assert oracle.modulus() == M
    assert A1 * B % M == 1
    assert A1 == (1 << 576) - (1 << 552) - (1 << 240) + (1 << 216) + 1
    assert oracle.multiplier(1) == A1
    for p in (1, 2, 24, 25, 389, 1024, 2048, 65537):
        assert oracle.multiplier(p) == pow(A1, p, M)
    gold = sum(int(v, 16) << (64 * i) for i, v in enumerate(GOLD["a_pow_2048_le_u64"]))
    assert oracle.multiplier(2048) == gold


def test_m_is_probably_prime():
    # Miller-Rabin, fixed bases: m prime => every seeded state is a unit, X = 0 unreachable (c-10)
    d, s = M - 1, 0
    while d % 2 == 0:
        d //= 2
        s += 1
    for a in (2, 3, 5, 7, 11, 13, 17, 19, 23, 29, 31, 37):
        x = pow(a, d, M)
        if x in (1, M - 1):
            continue
        for _ in range(s - 1):
            x = x * x % M
            if x == M - 1:
                break
        else:
            pytest.fail("m composite?")


# ----------------------------------------------------------------- multiply9x9 / mod_m
def test_multiply9x9_matches_bigint(oracle):
    rng = random.Random(11)
    top = (1 << 576) - 1
    cases = [(0, 0), (top, top), (1, top), (top, 1), (M - 1, M - 1), ((1 << 64) - 1, top)]
    cases += [(rng.getrandbits(576), rng.getrandbits(576)) for _ in range(300)]
    cases += [(rng.getrandbits(64 * rng.randrange(1, 10)), rng.getrandbits(576)) for _ in range(50)]
    for a, b in cases:
        assert oracle.multiply9x9(a, b) == a * b
    # not symmetric-only: a transposed operand order must still agree
    a, b = rng.getrandbits(576), rng.getrandbits(100)
    assert oracle.multiply9x9(a, b) == oracle.multiply9x9(b, a) == a * b


def test_mod_m_matches_bigint_remainder(oracle):
    rng = random.Random(12)
    zs = [0, 1, M - 1, M, M + 1, 2 * M - 1, 2 * M, (1 << 576) - 1, 1 << 576, (1 << 1152) - 1,
          (M - 1) * (M - 1), ((1 << 576) - 1) ** 2, M * M, M * M - 1, (1 << 816), (1 << 912) - 1]
    zs += [x * y for x in EDGE + [M, M + 1, (1 << 576) - 1] for y in EDGE + [M - 1]]
    zs += [rng.getrandbits(1152) for _ in range(400)]
    zs += [rng.getrandbits(576) for _ in range(100)]
    zs += [M + rng.getrandbits(239) for _ in range(50)]          # [m, 2^576)
    zs += [(rng.getrandbits(240) << 912) | rng.getrandbits(100) for _ in range(50)]  # large t1
    zs += [((1 << 576) - 1 - rng.getrandbits(200)) << 576 | rng.getrandbits(576) for _ in range(50)]
    for z in zs:
        r = oracle.mod_m(z)
        assert r == z % M, hex(z)
        assert r < M


def test_mod_m_fold_equals_long_division(oracle):
    rng = random.Random(13)
    for z in [0, M, (1 << 1152) - 1] + [rng.getrandbits(1152) for _ in range(40)]:
        assert oracle.mod_m_longdiv(z) == oracle.mod_m(z) == z % M


def test_mulmod_powmod(oracle):
    rng = random.Random(14)
    for _ in range(100):
        x, y = rng.randrange(M), rng.randrange(M)
        assert oracle.mulmod(x, y) == x * y % M
    # cfg2 allows non-canonical x in [m, 2^576)
    for _ in range(20):
        x, y = M + rng.getrandbits(239), rng.randrange(M)
        assert oracle.mulmod(y, x) == x * y % M
    for _ in range(10):
        x, e = rng.randrange(M), rng.getrandbits(rng.randrange(1, 200))
        assert oracle.powmod(x, e) == pow(x, e, M)
    assert oracle.powmod(rng.randrange(M), 0) == 1


# ----------------------------------------------------------------- state map (D3/D4), tiny-parameter exhaustive
@pytest.mark.parametrize("b,r,s", [(2, 5, 2), (3, 4, 1), (4, 4, 2), (5, 3, 1), (2, 9, 4)])
def test_state_map_exhaustive_small_parameters(b, r, s):
    """Row c-1/c-3/c-4 on generators small enough to enumerate: for EVERY state (x, c) of the
    SWB generator x_n = x_{n-s} - x_{n-r} - c (mod b), the map X = V - floor(V / b^(r-s)) + c
    commutes with the LCG X -> b^-1 X mod (b^r - b^s + 1), and the closed-form inverse returns
    exactly the recurrent states."""
    m = b**r - b**s + 1
    a = pow(b, -1, m)
    import itertools
    seen_recurrent = {}
    for digits in itertools.product(range(b), repeat=r):
        for c in (0, 1):
            x = list(digits)
            V = sum(v * b**j for j, v in enumerate(x))
            X = (V - V // b ** (r - s) + c) % m
            t = x[r - s] - x[0] - c
            cn = 1 if t < 0 else 0
            x2 = x[1:] + [t + cn * b]
            V2 = sum(v * b**j for j, v in enumerate(x2))
            X2 = (V2 - V2 // b ** (r - s) + cn) % m
            assert X2 == a * X % m
            # closed-form inverse
            if X != 0:
                Vc = (b**r * X) // m
                cc = X - Vc + Vc // b ** (r - s)
                assert cc in (0, 1)
                seen_recurrent[X] = (Vc, cc)
    # the closed form picks a state that the SWB map sends to the closed form of a X (i.e. it is closed
    # under the recurrence: a recurrent orbit), for every X in (0, m)
    assert len(seen_recurrent) == m - 1
    for X, (Vc, cc) in seen_recurrent.items():
        x = [(Vc // b**j) % b for j in range(r)]
        t = x[r - s] - x[0] - cc
        cn = 1 if t < 0 else 0
        x2 = x[1:] + [t + cn * b]
        V2 = sum(v * b**j for j, v in enumerate(x2))
        assert seen_recurrent[a * X % m] == (V2, cn)


# ----------------------------------------------------------------- SWB == LCG at full size
def test_swb_stepper_matches_definition(oracle):
    rng = random.Random(15)
    for _ in range(50):
        x = [rng.randrange(B) for _ in range(24)]
        c = rng.randrange(2)
        n = rng.randrange(0, 100)
        V, cc = oracle.swb_steps(pack(x), c, n)
        for _ in range(n):
            x, c = py_swb_step(x, c)
        assert (V, cc) == (pack(x), c)
    # borrow edge: all zero with carry -> wraps to b - 1
    V, cc = oracle.swb_steps(0, 1, 1)
    assert unpack(V)[23] == B - 1 and cc == 1


def test_to_lcg_commutes_with_one_swb_step(oracle):
    """D3: to_lcg(state_{n+1}) == a to_lcg(state_n) mod m for ANY state (not only recurrent),
    and b X_{n+1} = X_n + x_n m as integers."""
    rng = random.Random(16)
    for _ in range(300):
        x = [rng.randrange(B) for _ in range(24)]
        c = rng.randrange(2)
        X = oracle.to_lcg(pack(x), c)
        assert X == (pack(x) - (pack(x) >> 336) + c) % M
        x2, c2 = py_swb_step(x, c)
        X2 = oracle.to_lcg(pack(x2), c2)
        assert X2 == A1 * X % M
        if X:
            assert B * X2 == X + x2[23] * M
    assert oracle.to_lcg((1 << 576) - 1, 1) == 0  # V - Vh + c == m -> 0


@pytest.mark.parametrize("p", [1, 24, 25, 48, 389, 2048])
def test_advance_by_a_pow_p_equals_p_swb_steps(oracle, p):
    """the pin north_star asks for: LCG advance by a^p == p direct SWB steps."""
    rng = random.Random(17 + p)
    A = oracle.multiplier(p)
    for _ in range(12):
        x, c = rand_recurrent_state(rng)
        X = oracle.to_lcg(pack(x), c)
        Xn = oracle.mulmod(A, X)
        V_lcg, c_lcg = oracle.to_ranlux(Xn)
        V_swb, c_swb = oracle.swb_steps(pack(x), c, p)
        xs, cs = x, c
        for _ in range(p):
            xs, cs = py_swb_step(xs, cs)
        assert (V_swb, c_swb) == (pack(xs), cs)
        assert (V_lcg, c_lcg) == (V_swb, c_swb)


def crafted_lcg_states(rng):
    xs = list(range(1, 200)) + [M - k for k in range(1, 200)]
    xs += [(1 << k) + d for k in range(1, 576) for d in (-1, 0, 1) if 0 < (1 << k) + d < M]
    # near Xl + Xh = 2^336 (third combination T = Xh, c = 1; probability ~2^-96 at random)
    for _ in range(200):
        xh = rng.getrandbits(240)
        for d in (-2, -1, 0, 1, 2):
            xl = (1 << 336) - xh + d
            if 0 <= xl < (1 << 336):
                x = (xh << 336) | xl
                if 0 < x < M:
                    xs.append(x)
    # near D = 0:  S (2^240 - 1) ~ Xh 2^336, i.e. middle 240 bits ~ top 240 bits
    for _ in range(300):
        xh = rng.getrandbits(rng.choice([240, 240, 200, 100, 17]))
        for d in (-2, -1, 0, 1, 2):
            mid = xh + d
            if 0 <= mid < (1 << 240):
                for low in (0, 1, rng.getrandbits(96), (1 << 96) - 1):
                    x = (xh << 336) | (mid << 96) | low
                    if 0 < x < M:
                        xs.append(x)
    # top-limb collisions that defeat a "compare the leading 32 bits" shortcut
    for _ in range(200):
        w = rng.getrandbits(32)
        for dw in (-1, 0, 1):
            u = (w + dw) & 0xFFFFFFFF
            x = (w << 544) | (rng.getrandbits(208) << 336) | (u << 304) | rng.getrandbits(304)
            if 0 < x < M:
                xs.append(x)
    return xs


def test_to_ranlux_closed_form_long_division_and_digit_formula(oracle):
    rng = random.Random(18)
    xs = crafted_lcg_states(rng)[::7] + [rng.randrange(1, M) for _ in range(150)]
    for X in xs:
        V, c = oracle.to_ranlux(X)
        assert (V, c) == oracle.to_ranlux_def(X)
        assert V == (X << 576) // M and c == X - V + (V >> 336) and c in (0, 1)
        assert unpack(V) == py_digits(X)


def test_to_ranlux_shift_add_form_on_all_crafted_states(oracle):
    rng = random.Random(19)
    n_third = 0
    for X in crafted_lcg_states(rng) + [rng.randrange(1, M) for _ in range(3000)]:
        V, c = oracle.to_ranlux(X)
        Vd = (X << 576) // M
        cd = X - Vd + (Vd >> 336)
        assert (V, c) == (Vd, cd), hex(X)
        assert oracle.to_lcg(V, c) == X
        if c == 1 and V == X + (X >> 336):
            n_third += 1
    assert n_third > 0  # the (T = Xh, c = 1) combination was exercised
    assert oracle.to_ranlux(0) == (0, 0)
    assert oracle.to_ranlux(1) == (1, 0)
    assert oracle.to_ranlux(M - 1) == ((1 << 576) - 2, 1)


# ----------------------------------------------------------------- seeding / streams / cursor
def test_seeding_is_power_of_the_multiplier(oracle):
    """c-7: X_seed = (A^(2^96))^seed (parity with ROOT unpinned); with a small exponent the
    seeded state equals that many single advances from X = 1."""
    for p in (24, 2048):
        A = pow(A1, p, M)
        for seed in (0, 1, 2, 1024, (1 << 64) - 1, 0xDEADBEEFCAFE):
            assert oracle.seed_state(seed, p) == pow(A, seed << 96, M)
    A = oracle.multiplier(2048)
    for log2e in (0, 1, 3):
        X = 1
        for _ in range(5 * (1 << log2e)):
            X = oracle.mulmod(A, X)
        assert oracle.seed_state_exp(5, 2048, log2e) == X


def py_stream(seed, p, n, skip=0):
    """Big-int model of D5-D8 written independently of the oracle's engine: global draw index."""
    A = pow(A1, p, M)
    X0 = pow(A, seed << 96, M)
    out = []
    for t in range(skip, skip + n):
        blk, j = t // 12 + 1, t % 12
        X = pow(A, blk, M) * X0 % M
        V = (X << 576) // M
        out.append((V >> (48 * j)) & ((1 << 48) - 1))
    return out


def test_stream_draws_match_bigint_model_and_survey_vectors(oracle):
    for key, (p, seed) in {"p2048_seed1": (2048, 1), "p2048_seed2": (2048, 2), "p2048_seed1024": (2048, 1024),
                           "p24_seed1": (24, 1)}.items():
        got = oracle.streams([seed], p, 3, want=("ints",))["ints"][0]
        assert [int(v) for v in got] == [int(v, 16) for v in GOLD["first_draws_48bit"][key]]
    assert oracle.streams([1], 2048, 1)["doubles"][0, 0] == GOLD["first_double_p2048_seed1"]
    X = oracle.seed_state(1, 2048)
    assert X & (2**64 - 1) == int(GOLD["x_seed1_p2048_limb0"], 16) and X >> 512 == int(GOLD["x_seed1_p2048_limb8"], 16)
    for seed, p in ((3, 2048), (77, 389), ((1 << 64) - 1, 1024)):
        got = oracle.streams([seed], p, 40, want=("ints",))["ints"][0]
        assert [int(v) for v in got] == py_stream(seed, p, 40)


def test_stream_end_states_match_bigint_model(oracle):
    """The X / V / c / pos arrays oracle.streams returns with want=("state",) -- what every GPU check_state compares
    with -- against Python integers: after `skip` skipped and n taken draws from pos = 12 the stream has made
    k = ceil((skip + n) / 12) advances (D8), X = A^k X0, V = floor(2^576 X / m) (D4 by its definition, not the shift / add
    form) and c = X - V + (V >> 336) (D3 solved for the carry), cursor = skip + n - 12 (k - 1)."""
    for p, seed_list, n, skip_list in ((2048, (1, 2, 77), 29, (0, 5, 1000)), (2048, (3, 4), 36, (0, 12)),
                                       (24, (9, 2**64 - 1), 1, (0, 11)), (389, (5,), 0, (7,))):
        r = oracle.streams(np.array(seed_list, np.uint64), p, n, skips=np.array(skip_list, np.uint64), want=("state",))
        A = pow(A1, p, M)
        for i, (seed, skip) in enumerate(zip(seed_list, skip_list)):
            total = skip + n
            k = (total + 11) // 12
            X = pow(A, k, M) * pow(A, seed << 96, M) % M
            V = (X << 576) // M
            c = X - V + (V >> 336)
            assert c in (0, 1)
            assert inputs.limbs_to_int(r["X"][i]) == X, (p, seed, skip)
            assert inputs.limbs_to_int(r["V"][i]) == V, (p, seed, skip)
            assert int(r["c"][i]) == c and int(r["pos"][i]) == (total - 12 * (k - 1) if total else 12)


def test_cfg1_checksums(oracle):
    """BASELINE.json configs[0]: 1,024 streams x 384 draws, seeds 1..1024, p = 2048."""
    r = oracle.streams(inputs.seeds(1024), 2048, 384, want=("ints", "doubles", "state"), nthreads=4)
    ints = r["ints"]
    assert int(np.bitwise_xor.reduce(ints.reshape(-1))) == int(GOLD["cfg1_xor_of_48bit"], 16)
    assert int(ints.reshape(-1).sum(dtype=np.uint64)) == int(GOLD["cfg1_sum_mod_2_64"], 16)
    # lattice (c-11): exact k 2^-48, in [0, 1)
    d = r["doubles"]
    assert d.min() >= 0.0 and d.max() < 1.0
    assert np.array_equal(d * 2.0**48, ints.astype(np.float64)) and ints.max() < (1 << 48)
    assert np.all(r["pos"] == 12)  # 384 = 32 blocks exactly; cursor back at "block exhausted"


def test_p24_stream_is_the_raw_swb_sequence(oracle):
    """c-13: with p = 24 no numbers are skipped: the draws are the direct SWB numbers of the
    generator started from to_ranlux(X_seed), paired as x_{2j} + 2^24 x_{2j+1}."""
    for seed in (1, 5):
        X = oracle.seed_state(seed, 24)
        V, c = oracle.to_ranlux(X)
        x = unpack(V)
        nums = []
        for _ in range(24 * 6):
            x, c = py_swb_step(x, c)
            nums.append(x[23])
        want = [nums[2 * j] + (nums[2 * j + 1] << 24) for j in range(len(nums) // 2)]
        got = oracle.streams([seed], 24, len(want), want=("ints",))["ints"][0]
        assert [int(v) for v in got] == want


def test_skip_equals_single_draws(oracle):
    """P:47 / c-8: skip(n) == n draws, from every cursor position."""
    rng = random.Random(20)
    X0 = oracle.seed_state(9, 2048)
    for prior in list(range(0, 30)):
        for n in [0, 1, 2, 11, 12, 13, 23, 24, 25, rng.randrange(200)]:
            Xa, pa, da = oracle.engine_run(X0, 12, 2048, [("draw", prior), ("skip", n), ("draw", 3)])
            Xb, pb, db = oracle.engine_run(X0, 12, 2048, [("draw", prior), ("draw", n), ("draw", 3)])
            assert (Xa, pa) == (Xb, pb) and da[-3:] == db[-3:]
            assert 0 <= pa <= 12


def test_skip_64bit_distances_against_bigint_model(oracle):
    rng = random.Random(21)
    A = pow(A1, 2048, M)
    X0 = oracle.seed_state(4, 2048)
    for _ in range(20):
        n1, n2 = rng.getrandbits(64), rng.getrandbits(64)
        pos0 = rng.randrange(0, 13)
        X, pos, draws = oracle.engine_run(X0, pos0, 2048, [("skip", n1), ("skip", n2), ("draw", 2)])
        # model: global draw counter
        total = pos0 + n1 + n2  # draws consumed relative to the start of X0's block
        k = (total - 1) // 12 if total >= 1 else 0
        posm = total - 12 * k
        Xm = pow(A, k, M) * X0 % M
        # then two draws
        outs = []
        for _ in range(2):
            if posm == 12:
                Xm = A * Xm % M
                posm = 0
            V = (Xm << 576) // M
            outs.append((V >> (48 * posm)) & ((1 << 48) - 1))
            posm += 1
        assert (X, pos, draws) == (Xm, posm, outs)
    # all-ones distance from pos = 12 must not overflow (needs 65 bits)
    X, pos, _ = oracle.engine_run(X0, 12, 2048, [("skip", (1 << 64) - 1)])
    total = 12 + (1 << 64) - 1
    k = (total - 1) // 12
    assert (X, pos) == (pow(A, k, M) * X0 % M, total - 12 * k)


def _float_fma(d, q):
    return float(Fraction(d) * Fraction(d) + Fraction(q))  # exact, then ONE correct rounding


def test_fused_sums_rounding_and_survey_mini_vector(oracle):
    """c-14: S = S + d, Q = fma(d, d, Q) in draw order, round-to-nearest-even."""
    dist = inputs.cfg5_skip_distances(4)
    assert int(dist[0]) == int(GOLD["cfg5_mini"]["stream0"]["distance"], 16)
    assert int(dist[3]) == int(GOLD["cfg5_mini"]["stream3"]["distance"], 16)
    r = oracle.streams(inputs.seeds(4), 2048, 36, skips=dist, want=("doubles", "sums"))
    for i, key in ((0, "stream0"), (3, "stream3")):
        assert r["sum"][i] == float.fromhex(GOLD["cfg5_mini"][key]["S"])
        assert r["sumsq"][i] == float.fromhex(GOLD["cfg5_mini"][key]["Q"])
    pos_after_skip = oracle.streams(inputs.seeds(4), 2048, 0, skips=dist, want=("state",))["pos"]
    assert int(pos_after_skip[0]) == 2 and int(pos_after_skip[3]) == 5
    # exact-rational cross-check of the rounding order on a longer run (partial sums DO round)
    r = oracle.streams([7, 8], 2048, 500, skips=np.array([3, 100], np.uint64), want=("doubles", "sums"))
    rounded = False
    for i in range(2):
        S, Q = 0.0, 0.0
        for d in r["doubles"][i]:
            d = float(d)
            if Fraction(S) + Fraction(d) != Fraction(S + d):
                rounded = True
            S = S + d
            Q = _float_fma(d, Q)
        assert (S, Q) == (float(r["sum"][i]), float(r["sumsq"][i]))
    assert rounded


def test_degenerate_zero_state(oracle):
    """c-10: X = 0 is a fixed point; all draws 0.0."""
    X, pos, draws = oracle.engine_run(0, 12, 2048, [("draw", 13)])
    assert X == 0 and pos == 1 and draws == [0] * 13


# ----------------------------------------------------------------- workloads
def test_splitmix64_and_cfg2_inputs(oracle):
    assert int(inputs.splitmix64(0, 1)[0]) == int(GOLD["splitmix64_seed0_first"], 16)
    # scalar re-statement (c-15)
    s, outs = 12345, []
    for _ in range(5):
        s = (s + 0x9E3779B97F4A7C15) % 2**64
        z = s
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) % 2**64
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) % 2**64
        outs.append(z ^ (z >> 31))
    assert [int(v) for v in inputs.splitmix64(12345, 5)] == outs
    edge = inputs.cfg2_edge_states()
    vals = [inputs.limbs_to_int(e) for e in edge]
    assert vals[:4] == [0, 1, M - 1, M - (1 << 240)]
    assert all(M <= v < (1 << 576) for v in vals[4:24]) and vals[4] == M and vals[6] == M + (1 << 240) - 2
    assert vals[6] == (1 << 576) - 1
    assert all(v >> 512 == 2**64 - 1 and v < M for v in vals[24:])
    st = inputs.cfg2_states(256)
    assert st.shape == (256 + 64, 9) and all(inputs.limbs_to_int(s) < M for s in st[:256])
    out = oracle.advance_states(st, 2048, 16, nthreads=2)
    A16 = pow(A1, 2048 * 16, M)
    for i in list(range(0, 256, 17)) + list(range(256, 320)):
        assert inputs.limbs_to_int(out[i]) == A16 * inputs.limbs_to_int(st[i]) % M
    # reps == 0 only canonicalises (its own branch in orc_advance_states): Python's % on every edge state, incl. [m, 2^576)
    out0 = oracle.advance_states(st, 2048, 0)
    for i in range(320):
        assert inputs.limbs_to_int(out0[i]) == inputs.limbs_to_int(st[i]) % M
    assert any(inputs.limbs_to_int(s) >= M for s in st[256:])


# ----------------------------------------------------------------- normals (DESIGN reading N-1)
def _dec_pi_sin_cos(prec=60):
    """pi, sin, cos in `decimal` at `prec` digits (Machin's formula and Taylor series): the independent side."""
    import decimal
    D = decimal.Decimal
    ctx = decimal.Context(prec=prec)

    def atan_inv(n):  # atan(1 / n)
        x, total, k, n2 = D(1) / D(n), D(0), 0, D(n) * D(n)
        with decimal.localcontext(ctx):
            term = D(1) / D(n)
            while abs(term) > D(10) ** (-prec - 5):
                total += term / (2 * k + 1) if k % 2 == 0 else -term / (2 * k + 1)
                term /= n2
                k += 1
        return total

    with decimal.localcontext(ctx):
        pi = 16 * atan_inv(5) - 4 * atan_inv(239)

    def sincos(x):
        with decimal.localcontext(ctx):
            s, c, term, k = D(0), D(0), D(1), 0
            while abs(term) > D(10) ** (-prec - 5):
                if k % 2 == 0:
                    c += term if (k // 2) % 2 == 0 else -term
                else:
                    s += term if (k // 2) % 2 == 0 else -term
                k += 1
                term = term * x / k
            return s, c

    return ctx, pi, sincos


def test_normals_are_box_muller_to_the_last_bit_or_so(oracle):
    """orc_normals against 60-digit decimal arithmetic (ln and sqrt from `decimal`, pi / sin / cos above): the fp64
    result is within 1 ulp of the exact Box-Muller value, including arguments next to the zeros of sin and cos."""
    import decimal
    D = decimal.Decimal
    ctx, pi, sincos = _dec_pi_sin_cos()
    rng = random.Random(48)
    quarter = 1 << 46
    ks = [(rng.randrange(1 << 48), rng.randrange(1 << 48)) for _ in range(40)]
    ks += [(rng.randrange(1 << 48), q * quarter + d) for q in range(4) for d in (1, 2, 12345)]
    ks += [(rng.randrange(1 << 48), (q * quarter - d) % (1 << 48)) for q in range(4) for d in (1, 777)]
    ks += [(1, 5), ((1 << 48) - 1, 99), (1 << 47, 1 << 45)]
    z = oracle.normals(np.array(ks, dtype=np.uint64).reshape(-1))
    for i, (k0, k1) in enumerate(ks):
        with decimal.localcontext(ctx):
            u0, u1 = D(k0) / D(1 << 48), D(k1) / D(1 << 48)
            r = (-2 * (1 - u0).ln()).sqrt()
            s, c = sincos(2 * pi * u1)
            want = (r * c, r * s)
        for got, w in zip(z[2 * i:2 * i + 2], want):
            assert abs(D(float(got)) - w) <= D(float(np.spacing(abs(got)))), (k0, k1, got, w)


def test_normals_pairing_special_arguments_and_python_math(oracle):
    import math
    rng = random.Random(7)
    ks = [(rng.randrange(1 << 48), rng.randrange(1 << 48)) for _ in range(2000)]
    z = oracle.normals(np.array(ks, dtype=np.uint64).reshape(-1)).reshape(-1, 2)
    for (k0, k1), (z0, z1) in zip(ks, z):
        u0, u1 = k0 / 2**48, k1 / 2**48
        r2 = -2.0 * math.log(1.0 - u0)
        r = math.sqrt(r2)
        # the first draw of a pair sets the radius, the second the angle; cos first, sin second
        assert math.isclose(z0 * z0 + z1 * z1, r2, rel_tol=1e-14)
        dphi = (math.atan2(z1, z0) - 2 * math.pi * u1) % (2 * math.pi)
        assert min(dphi, 2 * math.pi - dphi) < 1e-14
        assert abs(z0 - r * math.cos(2 * math.pi * u1)) <= 4e-15 * max(r, 1.0)
        assert abs(z1 - r * math.sin(2 * math.pi * u1)) <= 4e-15 * max(r, 1.0)
    # exact zeros of the definition; u0 = 0 gives r = 0; the largest radius is sqrt(2 * 48 ln 2)
    k0 = 123456789 << 10
    r = math.sqrt(-2.0 * math.log(1.0 - k0 / 2**48))
    sp = oracle.normals(np.array([k0, 0, k0, 1 << 46, k0, 1 << 47, k0, 3 << 46, 0, 12345, (1 << 48) - 1, 0], dtype=np.uint64))
    assert list(sp[:8]) == [r, 0.0, 0.0, r, -r, 0.0, 0.0, -r]
    assert sp[8] == 0.0 and sp[9] == 0.0
    assert math.isclose(sp[10], math.sqrt(96 * math.log(2)), rel_tol=1e-15) and sp[11] == 0.0


def test_normals_are_standard_normal_in_distribution(oracle):
    """Sample moments of 4 x 10^5 deviates made from a RANLUX++ stream (5 sigma bands of the sampling error)."""
    n = 400_000
    k = oracle.streams(inputs.seeds(1, 2024), 2048, n, want=("ints",))["ints"].reshape(-1)
    z = oracle.normals(k)
    se = 1.0 / np.sqrt(n)
    assert abs(z.mean()) < 5 * se
    assert abs(z.var() - 1.0) < 5 * np.sqrt(2.0) * se
    assert abs((z**3).mean()) < 5 * np.sqrt(15.0) * se
    assert abs((z**4).mean() - 3.0) < 5 * np.sqrt(96.0) * se
    p1 = 0.6826894921370859  # P(|Z| < 1)
    assert abs((np.abs(z) < 1.0).mean() - p1) < 5 * np.sqrt(p1 * (1 - p1)) * se
    assert abs(np.mean(z[0::2] * z[1::2])) < 5 * np.sqrt(2.0) * se  # the two halves of a pair are uncorrelated
