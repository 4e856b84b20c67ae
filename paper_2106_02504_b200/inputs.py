"""Seeded synthetic inputs for the BASELINE.json workloads.

This module holds NO RANLUX++ arithmetic: it only draws the raw inputs (seeds,
raw 576-bit states, skip distances) that both the CUDA path and the CPU oracle
are fed.  The recipe is stated in DESIGN.md ("Input recipe") and follows
SURVEY.md 8(d).  The paper itself uses no dataset (every
thread generates 10^6 doubles from its own seeded state), so these generators
ARE the workloads; nothing here stands in for a public suite.
"""
import numpy as np

MASK64 = (1 << 64) - 1
#: the RANLUX modulus, needed only to classify / build edge inputs
M = (1 << 576) - (1 << 240) + 1
CFG2_SEED = 0x210602504
CFG5_SEED = 5


def splitmix64(seed: int, n: int) -> np.ndarray:
    """First n outputs of the public-domain splitmix64 generator started at `seed`
    (first output for seed 0 is 0xe220a8397b1dcdaf)."""
    with np.errstate(over="ignore"):
        k = np.arange(1, n + 1, dtype=np.uint64)
        z = np.uint64(seed & MASK64) + k * np.uint64(0x9E3779B97F4A7C15)
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        return z ^ (z >> np.uint64(31))


def int_to_limbs(x: int, n: int = 9) -> np.ndarray:
    return np.array([(x >> (64 * i)) & MASK64 for i in range(n)], dtype=np.uint64)


def limbs_to_int(a) -> int:
    return sum(int(v) << (64 * i) for i, v in enumerate(np.asarray(a).reshape(-1)))


def _ge_m(states: np.ndarray) -> np.ndarray:
    """Row-wise `state >= m` for [n][9] little-endian uint64 states.
    m = {1, 0, 0, 0xFFFF000000000000, ~0 x5}: x >= m  <=>  limbs 4..8 all ones,
    limb 3 >= 0xFFFF000000000000 and (limb 3 > that, or low 192 bits >= 1)."""
    ones = np.uint64(MASK64)
    top = np.all(states[:, 4:9] == ones, axis=1)
    l3 = states[:, 3]
    k = np.uint64(0xFFFF000000000000)
    low_nonzero = np.any(states[:, 0:3] != 0, axis=1)
    return top & ((l3 > k) | ((l3 == k) & low_nonzero))


def cfg2_random_states(n: int, seed: int = CFG2_SEED) -> np.ndarray:
    """n states uniform in [0, m): consecutive splitmix64 outputs, 9 per state, limb 0
    first; a state >= m is redrawn from the continuing stream (probability 2^-336)."""
    raw = splitmix64(seed, 9 * n).reshape(n, 9).copy()
    bad = _ge_m(raw)
    extra = 0
    while bad.any():  # practically never
        idx = np.nonzero(bad)[0]
        more = splitmix64(seed, 9 * (n + extra + len(idx)))[9 * (n + extra):].reshape(-1, 9)
        raw[idx] = more
        extra += len(idx)
        bad = _ge_m(raw)
    return raw


def cfg2_edge_states(seed: int = CFG2_SEED) -> np.ndarray:
    """The 64 edge states of BASELINE.json configs[1]: 0, 1, m-1, m-2^240; 20 values
    m + t covering [m, 2^576) (t in {0, 1, 2^240-2} and 17 splitmix-derived t); 40
    states with limb 8 all ones and limbs 0..7 from splitmix64."""
    rnd = splitmix64(seed ^ 0xEDBE5, 17 * 4 + 40 * 8)
    out = [0, 1, M - 1, M - (1 << 240)]
    ts = [0, 1, (1 << 240) - 2]
    for i in range(17):
        t = 0
        for j in range(4):
            t |= int(rnd[4 * i + j]) << (64 * j)
        ts.append(t % ((1 << 240) - 1))
    out += [M + t for t in ts]
    states = [int_to_limbs(x) for x in out]
    for i in range(40):
        limbs = np.empty(9, np.uint64)
        limbs[:8] = rnd[68 + 8 * i: 68 + 8 * i + 8]
        limbs[8] = np.uint64(MASK64)
        states.append(limbs)
    res = np.stack(states)
    assert res.shape == (64, 9)
    return res


def cfg2_states(n_random: int = 1 << 20, seed: int = CFG2_SEED) -> np.ndarray:
    """[n_random + 64][9] uint64: the random states followed by the 64 edge states."""
    return np.concatenate([cfg2_random_states(n_random, seed), cfg2_edge_states(seed)], axis=0)


def cfg5_skip_distances(n_streams: int, seed: int = CFG5_SEED) -> np.ndarray:
    """Per-stream skip distances of BASELINE.json configs[4]: uniform 64-bit, the i-th
    output of splitmix64(seed)."""
    return splitmix64(seed, n_streams)


def seeds(n_streams: int, first: int = 1) -> np.ndarray:
    """Stream i is seeded with first + i (BASELINE.json: seeds 1..N)."""
    with np.errstate(over="ignore"):
        return np.uint64(first) + np.arange(n_streams, dtype=np.uint64)
