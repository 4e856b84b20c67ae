"""rlxpp_generate_doubles_static: the entry point for callers that must not allocate device memory.

Who they are (include/rlxpp.h has the full contract): code that runs after a framework's memory pool has claimed the
whole GPU, code inside a latency budget that cannot take cudaMalloc's device-wide synchronisation, and code under a fixed
memory plan.  For them the library keeps its scratch -- a working copy of the states, the scheduler words of the
persistent kernel, the byte matrix of the luxury level -- in one fixed ~5 MB array of its device image instead of
allocating it, which caps a call at RLXPP_STATIC_MAX_STREAMS = 65,536 streams.

The check here is against the library's own handle path (rlxpp_create / rlxpp_set_state / rlxpp_generate_doubles /
rlxpp_get_state), which the parity tests pin to the oracle: same states in, the same doubles and the same advanced states
out, bit for bit (tolerance 0, as everywhere for the doubles) -- on two calls in a row, because the array is shared by all
calls and keeps what the last one left: the second call must not see the first one's scheduler counters, states or
matrix.  The file sorts last on purpose: `pytest -x` stops at the first failure, and a failure in this add-on must not
hide the parity tests.  It passes on its own in a fresh process (first use of the array on the device) and after the
other tests (the library already warm).
"""
import numpy as np
import pytest

import paper_2106_02504_b200 as rlx
from paper_2106_02504_b200 import inputs


def bits(t):
    return np.ascontiguousarray(t.cpu().numpy()).view(np.uint64)


def handle_path(torch, lcg0, p, calls):
    """The existing path: a handle loaded with the states lcg0, one rlxpp_generate_doubles per (count, layout)."""
    n = lcg0.shape[0]
    h = rlx.rlxpp_create(n, 1, p)
    rlx.rlxpp_set_state(h, lcg0)
    outs, states = [], []
    for per, layout in calls:
        out = torch.empty(n * per, dtype=torch.float64, device="cuda")
        rlx.rlxpp_generate_doubles(h, out, per, layout)
        X = torch.empty((n, 9), dtype=torch.int64, device="cuda")
        rlx.rlxpp_get_state(h, None, None, None, X)
        torch.cuda.synchronize()
        outs.append(bits(out))
        states.append(bits(X))
    rlx.rlxpp_destroy(h)
    return outs, states


@pytest.mark.gpu
def test_static_scratch_generation_matches_the_handle_path_on_two_calls_in_a_row():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("the gpu-marked tests need a CUDA device (there is no CPU fallback)")
    rlx.load()
    rlx.rlxpp_set_engine(rlx.RLXPP_ENGINE_UMMA)
    # 1,000 streams = 7 full tiles of 128 and a ragged one; random states plus the edge states of BASELINE configs[1]
    # (0, 1, m - 1, values >= m that the import must reduce)
    n = 1000
    lcg0 = torch.from_numpy(inputs.cfg2_states(n - 64).view(np.int64).reshape(n, 9).copy()).cuda()
    for p, calls in ((2048, ((36, rlx.RLXPP_INTERLEAVED), (1536, rlx.RLXPP_INTERLEAVED))),
                     (24, ((384, rlx.RLXPP_STREAM_MAJOR), (36, rlx.RLXPP_STREAM_MAJOR))),  # another p: the matrix is replaced
                     (2048, ((384, rlx.RLXPP_STREAM_MAJOR), (12, rlx.RLXPP_INTERLEAVED)))):
        want_out, want_state = handle_path(torch, lcg0, p, calls)
        lcg = lcg0.clone()
        for k, (per, layout) in enumerate(calls):  # two calls in a row on the same states
            out = torch.full((n * per,), -1.0, dtype=torch.float64, device="cuda")
            rlx.rlxpp_generate_doubles_static(lcg, n, p, out, per, layout)
            torch.cuda.synchronize()
            assert np.array_equal(bits(out), want_out[k]), f"p = {p}, call {k}: doubles differ from rlxpp_generate_doubles"
            assert np.array_equal(bits(lcg), want_state[k]), f"p = {p}, call {k}: advanced states differ from rlxpp_get_state"

    # the largest call the array holds, with forced chunks so that the per-tile counters in the array are used, twice:
    # the second call finds the first one's counters and states in the array and must clear / overwrite them
    n = rlx.RLXPP_STATIC_MAX_STREAMS
    per = 16 * 12 * 4
    lcg0 = torch.from_numpy(inputs.cfg2_states(n - 64).view(np.int64).reshape(n, 9).copy()).cuda()
    calls = ((per, rlx.RLXPP_INTERLEAVED), (per, rlx.RLXPP_STREAM_MAJOR))
    rlx.rlxpp_set_chunks(4)
    try:
        want_out, want_state = handle_path(torch, lcg0, 2048, calls)
        lcg = lcg0.clone()
        for k, (per, layout) in enumerate(calls):
            out = torch.full((n * per,), -1.0, dtype=torch.float64, device="cuda")
            rlx.rlxpp_generate_doubles_static(lcg, n, 2048, out, per, layout)
            torch.cuda.synchronize()
            assert np.array_equal(bits(out), want_out[k]), f"full size, call {k}: doubles differ"
            assert np.array_equal(bits(lcg), want_state[k]), f"full size, call {k}: states differ"
    finally:
        rlx.rlxpp_set_chunks(0)


def test_static_scratch_generation_rejects_what_does_not_fit():
    """Argument errors come before any CUDA call, so they are checked here without a device: one stream more than the
    array holds is refused with a message that names the limit, and a partial block (no cursor to keep it in) likewise."""
    rlx.load()
    with pytest.raises(rlx.RlxppError, match="exceeds the static scratch.*65536"):
        rlx.rlxpp_generate_doubles_static(256, rlx.RLXPP_STATIC_MAX_STREAMS + 1, 2048, 256, 12, rlx.RLXPP_INTERLEAVED, cuda_stream=0)
    with pytest.raises(rlx.RlxppError, match="multiple of 12"):
        rlx.rlxpp_generate_doubles_static(256, 128, 2048, 256, 13, rlx.RLXPP_INTERLEAVED, cuda_stream=0)
    with pytest.raises(rlx.RlxppError, match="p == 0"):
        rlx.rlxpp_generate_doubles_static(256, 128, 0, 256, 12, rlx.RLXPP_INTERLEAVED, cuda_stream=0)
    with pytest.raises(rlx.RlxppError, match="unknown layout"):
        rlx.rlxpp_generate_doubles_static(256, 128, 2048, 256, 12, 7, cuda_stream=0)
    # nothing to do is not an error, with or without a device
    rlx.rlxpp_generate_doubles_static(None, 0, 2048, None, 12, rlx.RLXPP_INTERLEAVED, cuda_stream=0)
    assert rlx.RLXPP_STATIC_SCRATCH_BYTES == 12288 + 80 * rlx.RLXPP_STATIC_MAX_STREAMS
