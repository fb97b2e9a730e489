"""mcdc_draws_noalloc: the random-number draws for callers that cannot hand the library any device memory.

Everything else in the library runs inside a workspace the caller allocated.  A caller may have none to give -- the GPU
is already filled by a running simulation so cudaMalloc fails, or it is a plug-in of a host program that keeps all
device memory in its own pool and forbids allocating -- and for those the library carries a fixed 1.5 MiB staging array
of its own (MCDC_NOALLOC_DRAWS_MAX = 65536 draws per call).  This file checks that entry point against the path that
already exists, Problem.draws (mcdc_test_draws, staged in the workspace; itself bit-equal to the CPU oracle in
test_gpu_parity.py::test_rng_bit_exact).  Draws are integer arithmetic turned into a float64 once, so the bar is the one
the existing draw test uses: every value equal bit for bit.

The calls come in pairs, the second smaller than and different from the first: the array keeps the first call's bytes,
and a result that depended on them would show here.  The file is named so that pytest collects it last (-x stops at the
first failure, and a failure here must not hide the other tests); it passes alone in a fresh process as well as after
the rest of the suite, because it depends on no state but the library's own.
"""
import numpy as np
import pytest

from paper_2501_05440_b200 import inputs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gpu():
    from paper_2501_05440_b200 import binding
    binding.load_library()
    return binding


def _request(rng, n):
    ids = rng.integers(0, 2 ** 63, n, dtype=np.uint64)
    ids[: min(n, 10)] = np.arange(min(n, 10))
    return ids, rng.integers(0, 1000, n).astype(np.uint32)


def test_noalloc_draws_equal_workspace_draws_on_two_calls_in_a_row(gpu):
    g = gpu.Problem(inputs.config1(n_particles=3000, n_inactive=1, n_active=1), max_particles=70000)
    rng = np.random.default_rng(11)
    # first call: the largest request the built-in array takes; second call right after it: smaller, other ids,
    # other stream key -- it must not see anything of the first
    calls = [(gpu.NOALLOC_DRAWS_MAX, 0, 7, 0xDEADBEEFCAFEF00D), (5000, 1, 3, 42)]
    for n, dom, cyc, seed in calls:
        ids, idx = _request(rng, n)
        got = gpu.draws_noalloc(seed, dom, cyc, ids, idx)
        want = g.draws(seed, dom, cyc, ids, idx)
        assert got.dtype == np.float64 and got.shape == want.shape
        assert (got == want).all()
        assert ((got > 0.0) & (got < 1.0)).all()
    # and once more with the very first request: same answer as before, whatever the array held in between
    rng = np.random.default_rng(11)
    ids, idx = _request(rng, gpu.NOALLOC_DRAWS_MAX)
    assert (gpu.draws_noalloc(0xDEADBEEFCAFEF00D, 0, 7, ids, idx) == g.draws(0xDEADBEEFCAFEF00D, 0, 7, ids, idx)).all()
    g.close()


def test_noalloc_draws_on_a_side_stream_and_without_any_problem(gpu):
    """No Problem (so no workspace) exists while these calls run; a non-default stream is accepted."""
    import torch
    rng = np.random.default_rng(12)
    st = torch.cuda.Stream()
    a_ids, a_idx = _request(rng, 4097)
    b_ids, b_idx = _request(rng, 33)
    a = gpu.draws_noalloc(1, 0, 0, a_ids, a_idx, stream=st.cuda_stream)
    b = gpu.draws_noalloc(1, 0, 0, b_ids, b_idx, stream=st.cuda_stream)
    g = gpu.Problem(inputs.config1(n_particles=3000, n_inactive=1, n_active=1), max_particles=20000)
    assert (a == g.draws(1, 0, 0, a_ids, a_idx)).all()
    assert (b == g.draws(1, 0, 0, b_ids, b_idx)).all()
    g.close()


def test_noalloc_draws_refuse_more_than_the_array_holds(gpu):
    n = gpu.NOALLOC_DRAWS_MAX + 1
    with pytest.raises(gpu.McdcError) as e:
        gpu.draws_noalloc(1, 0, 0, np.zeros(n, np.uint64), np.zeros(n, np.uint32))
    assert e.value.code == -1 and "at most 65536" in str(e.value)
    with pytest.raises(gpu.McdcError):
        gpu.draws_noalloc(1, 0, 0, np.zeros(4, np.uint64), np.zeros(4, np.uint32), device=64)
    assert len(gpu.draws_noalloc(1, 0, 0, np.zeros(0, np.uint64), np.zeros(0, np.uint32))) == 0
