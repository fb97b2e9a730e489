"""GPU parity for the continuous-energy time-dependent path (C5 and its closed-form reductions)."""
import numpy as np
import pytest

from paper_2501_05440_b200 import inputs
from tests.test_gpu_parity import ALWAYS, compare_traces

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gpu():
    from paper_2501_05440_b200 import binding
    binding.load_library()
    return binding


def compare_ce(r, ro, rtol=1e-9):
    assert np.allclose(r["k_cycle"], ro["k_cycle"], rtol=rtol)
    scale = np.abs(ro["flux_mean"]).max()
    assert np.allclose(r["flux_mean"], ro["flux_mean"], rtol=rtol, atol=1e-13 * scale)
    # events by type, tracks started and children banked are integers: exact
    assert (r["counters"][:12] == ro["counters"][:12]).all(), (r["counters"], ro["counters"])


CE_CASES = {
    "C5": lambda: inputs.config5(n_particles=1500, n_grid=50_000),
    "C5jitter": lambda: inputs.config5(n_particles=1201, n_grid=7000, jitter=True),
    "ce_1v": lambda: inputs.ce_one_over_v(n_particles=20000),
    "ce_scatter": lambda: inputs.ce_single_scatterer(A=16.0, n_particles=5000),
    "ce_scatterH": lambda: inputs.ce_single_scatterer(A=1.0, n_particles=5000),
    "ce_fission": lambda: _fis(),
    "ce_mix": lambda: inputs.ce_two_nuclide_mix(n_particles=3000, n_grid=3000),
    "ce_clock": lambda: inputs.ce_scatter_clock(n_particles=3000, n_grid=3000),
    # continuous energy in lattices (one level, two levels incl. non-square, an assembly with a gap around its pins)
    "ce_flat_lattice": lambda: inputs.ce_lattice("flat", n_particles=1500),
    "ce_two_level": lambda: inputs.ce_lattice("two_level", n_particles=1500),
    "ce_gap": lambda: inputs.ce_lattice("gap", n_particles=1500),
    "ce_clamp": lambda: inputs.ce_single_scatterer(A=1.0, n_particles=4000, E0=2.0e-5, sig_el=0.9, sig_c=0.1),
}


def _fis():
    P = inputs.ce_pure_fission(2000)
    P["t_edges"] = np.array([0.0, 1.0e-9])
    return P


@pytest.mark.parametrize("name", list(CE_CASES))
@pytest.mark.parametrize("schedule,persist,search", [(0, 0, 0), (0, -1, 1), (0, ALWAYS, 1), (1, 0, 0), (2, -1, 1), (0, 100, 0), (2, 1000, 1)])
def test_ce_parity(gpu, orc, name, schedule, persist, search):
    P = CE_CASES[name]()
    # the supercritical pure-fission pin grows by generation: give its waves room (capacity = 2 max + 1024)
    mp = 100_000 if name == "ce_fission" else None
    g = gpu.Problem(P, max_particles=mp, schedule=schedule, persist_threshold=persist, search=search)
    r = g.run()
    o = orc.Oracle(P)
    rc, ro = o.run()
    assert rc == 0
    compare_ce(r, ro)
    g.close()


@pytest.mark.parametrize("schedule,persist,search", [(0, -1, 0), (0, 0, 1), (1, 0, 1), (2, -1, 0), (0, 50, 1)])
def test_ce_traces_identical(gpu, orc, schedule, persist, search):
    """Source particles 0..99 of C5: identical event sequences incl. grid index, time, energy."""
    P = inputs.config5(n_particles=400, n_grid=20_000)
    g = gpu.Problem(P, schedule=schedule, persist_threshold=persist, search=search)
    g.set_trace(0, 100, 4096)
    r = g.run()
    o = orc.Oracle(P)
    o.set_trace(0, 100, 2_000_000)
    rc, ro = o.run()
    compare_traces(g.trace(), o.trace())
    compare_ce(r, ro)
    g.close()


@pytest.mark.parametrize("jitter", [False, True])
def test_grid_search_binary_equals_hash_equals_numpy(gpu, jitter):
    P = inputs.config5(n_particles=10, n_grid=50_000, jitter=jitter)
    g = gpu.Problem(P, max_particles=400_000)
    grid = P["grid"]
    rng = np.random.default_rng(3)
    E = np.concatenate([np.exp(rng.uniform(np.log(1e-6), np.log(1e8), 200_000)), grid, np.nextafter(grid, 0),
                        np.nextafter(grid, np.inf), [1e-7, 5e7, grid[0], grid[-1]]])
    ref = np.clip(np.searchsorted(grid, E, side="right") - 1, 0, len(grid) - 2)
    ob, oh = g.grid_index(E)
    assert (ob == ref).all()
    assert (oh == ref).all()
    g.close()


@pytest.mark.parametrize("persist", [-1, 0])
def test_ce_secondary_overflow_is_an_error_not_a_fault(gpu, persist):
    """A supercritical prompt chain outgrows the bank: MCDC_EBANK from the sweep kernels (regions meet) as well as
    from the persistent kernel (queue tail past the capacity), never an out-of-bounds access; the problem stays
    usable afterwards."""
    P = inputs.ce_pure_fission(3000)
    P["t_edges"] = np.array([0.0, 1.0e-6])  # dozens of generations of nu = 2.5
    g = gpu.Problem(P, max_particles=3000, persist_threshold=persist)
    with pytest.raises(gpu.McdcError) as e:
        g.run()
    assert e.value.code == -3
    P2 = _fis()
    g.close()
    g = gpu.Problem(P2, max_particles=100_000, persist_threshold=persist)
    r = g.run()
    assert r["counters"][0] > 2000
    g.close()


def test_ce_source_traces_with_secondaries_in_flight(gpu, orc):
    """Source histories 300..399 of a C5 run (ids beyond the first warp's worth), persistent kernel with queue pushes."""
    P = inputs.config5(n_particles=500, n_grid=10_000)
    g = gpu.Problem(P, search=1)
    g.set_trace(300, 100, 4096)
    r = g.run()
    o = orc.Oracle(P)
    o.set_trace(300, 100, 2_000_000)
    rc, ro = o.run()
    compare_traces(g.trace(), o.trace())
    compare_ce(r, ro)
    g.close()


@pytest.mark.parametrize("kind", ["flat", "two_level", "gap"])
@pytest.mark.parametrize("schedule,persist", [(0, 0), (0, -1), (1, 0)])
def test_ce_lattice_traces(gpu, orc, kind, schedule, persist):
    """Continuous energy inside one- and two-level lattices: event sequences of source particles 0..199 (lattice walls
    of both levels, packed element locations, time and energy) equal the oracle's."""
    P = inputs.ce_lattice(kind, n_particles=600)
    g = gpu.Problem(P, schedule=schedule, persist_threshold=persist, search=1)
    g.set_trace(0, 200, 1024)
    r = g.run()
    o = orc.Oracle(P)
    o.set_trace(0, 200, 1_000_000)
    rc, ro = o.run()
    tg = g.trace()
    assert (tg["ev"] == 7).sum() > 50
    compare_traces(tg, o.trace())
    compare_ce(r, ro)
    g.close()
