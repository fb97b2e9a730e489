"""GPU parity for SURVEY.md 8f row f2 -- time-dependent multi-group with delayed-neutron precursors and census
population control ("fully dynamic simulations"; R38-R40) -- and for mcdc_run_cycle on
fixed-source problems (one census interval per call)."""
import numpy as np
import pytest

from paper_2501_05440_b200 import inputs
from tests.test_gpu_parity import compare_traces
from tests.test_gpu_ce import compare_ce
from tests.test_gpu_f4 import compare_balance

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gpu():
    from paper_2501_05440_b200 import binding
    binding.load_library()
    return binding


def _with(P, **kw):
    P.update(kw)
    return P


TD_CASES = {
    "cube_G1": lambda: inputs.td_infinite(n_particles=3000, G=1),
    "cube_G2": lambda: inputs.td_infinite(n_particles=3000, G=2),
    "cube_G1_comb_half": lambda: inputs.td_infinite(n_particles=3000, G=1, census_target=1500),
    "cube_G2_comb_double": lambda: inputs.td_infinite(n_particles=2000, G=2, census_target=4000),
    "pin_G2": lambda: inputs.td_infinite(n_particles=3000, G=2, geom="pin"),
    "pin_G2_comb": lambda: inputs.td_infinite(n_particles=3000, G=2, geom="pin", census_target=2500),
    "pin_G1_implicit_comb": lambda: _with(inputs.td_infinite(n_particles=2500, G=1, geom="pin", census_target=2500),
                                          implicit_capture=1),
    "lattice2_G2_comb": lambda: inputs.td_infinite(n_particles=3000, G=2, geom="lattice2", census_target=2000, t_end=4.0e-4),
    "cube_G2_two_bins": lambda: inputs.td_infinite(n_particles=3000, G=2, n_t=2),
    "cube_G2_fine": lambda: inputs.td_infinite(n_particles=2000, G=2, t_end=8.0e-5, n_t=16),  # time bins << a lifetime
    "cube_G1_late_source": lambda: _with(inputs.td_infinite(n_particles=2000, G=1, census_target=1000), src_t=1.2e-3),
}


def compare_census(cg, co):
    assert len(cg) == len(co)
    for a, b in zip(cg, co):
        assert a[0] == b[0] and a[1] == b[1], (cg, co)
        assert a[2] == pytest.approx(b[2], rel=1e-11, abs=1e-300) and a[3] == pytest.approx(b[3], rel=1e-11, abs=1e-300)


@pytest.mark.parametrize("name", list(TD_CASES))
def test_td_parity(gpu, orc, name):
    """Flux by (bin, time bin, group), event counters, tracks, weight balance and the population / weight entering
    every census interval (before and after the comb) equal the oracle's."""
    P = TD_CASES[name]()
    g = gpu.Problem(P)
    r = g.run()
    o = orc.Oracle(P)
    rc, ro = o.run()
    assert rc == 0
    compare_ce(r, ro)
    compare_census(g.census(), o.census())
    compare_balance(g.balance(), o.balance())
    g.close()


@pytest.mark.parametrize("name", ["cube_G2", "pin_G2", "pin_G1_implicit_comb", "cube_G2_fine", "lattice2_G2_comb"])
def test_td_traces(gpu, orc, name):
    """Event sequences of source particles 0..99 (up to the first comb, which re-keys the tracks): time, time-edge
    events, group transfers, the census interruptions."""
    P = TD_CASES[name]()
    g = gpu.Problem(P)
    g.set_trace(0, 100, 4096)
    g.run()
    o = orc.Oracle(P)
    o.set_trace(0, 100, 2_000_000)
    o.run()
    tg, to = g.trace(), o.trace()
    if name == "cube_G2_fine":
        assert (tg["ev"] == 8).sum() > 50  # traced histories cross time edges (census interruptions)
    compare_traces(tg, to)
    g.close()


def test_td_run_cycle_interval_by_interval(gpu, orc):
    """mcdc_run_cycle on a time-dependent problem = one census interval per call; the calls in order reproduce
    mcdc_run_fixed_source; out-of-order calls are refused."""
    P = TD_CASES["pin_G2_comb"]()
    g = gpu.Problem(P)
    ref = g.run()
    cen = g.census()
    N, nt = P["run"]["n_particles"], len(P["t_edges"]) - 1
    with pytest.raises(gpu.McdcError) as e:
        g.run_cycle(N, 3, 1, P["run"]["seed"])  # the run was finished: interval 3 is not the next one
    assert e.value.code == -1
    for k in range(nt):
        g.run_cycle(N, k, 1, P["run"]["seed"])
        if k == 1:
            with pytest.raises(gpu.McdcError):
                g.run_cycle(N, 1, 1, P["run"]["seed"])  # the same interval twice
    r = g.results()
    assert np.allclose(r["flux_mean"], ref["flux_mean"], rtol=1e-12, atol=0) and (r["counters"][:12] == ref["counters"][:12]).all()
    compare_census(g.census(), cen)
    g.close()


@pytest.mark.parametrize("schedule", [0, 2])
def test_ce_run_cycle_equals_one_call(gpu, orc, schedule):
    """Continuous energy (C5): the run made one census interval per call (bank carried between calls, sorted by id)
    gives the one-call run's tallies -- and the oracle's -- to 1e-9; every counter is the same."""
    P = inputs.config5(n_particles=1200, n_grid=8000)
    g = gpu.Problem(P, schedule=schedule, search=1)
    one = g.run()
    N, nt = P["run"]["n_particles"], len(P["t_edges"]) - 1
    for k in range(nt):
        g.run_cycle(N, k, 1, P["run"]["seed"])
        assert g.dims().n_cycles == 1
    r = g.results()
    compare_ce(r, one)
    o = orc.Oracle(P)
    rc, ro = o.run()
    compare_ce(r, ro)
    compare_balance(g.balance(), o.balance())
    cen = g.census()
    assert len(cen) == nt and cen[0][0] == N and all(c[0] == c[1] for c in cen)  # no population control
    assert sum(c[0] for c in cen[1:]) == ro["counters"][8]  # every time-edge event is one census crossing
    g.close()


def test_td_validation(gpu):
    P = inputs.td_infinite(n_particles=500, G=1)
    with pytest.raises(gpu.McdcError) as e:
        gpu.Problem(P, schedule=1)
    assert e.value.code == -1
    bad = dict(P)
    bad["td"] = dict(P["td"], speed=np.array([0.0]))
    with pytest.raises(gpu.McdcError):
        gpu.Problem(bad)
    bad = dict(P)
    bad["td"] = dict(P["td"], decay=np.array([[-1.0]]))
    with pytest.raises(gpu.McdcError):
        gpu.Problem(bad)
    g = gpu.Problem(P)
    with pytest.raises(gpu.McdcError):
        g.L.mcdc_run_eigenvalue(g.h, 500, 1, 1, 1) and g._check(-1)
    g.close()


def _supercritical_td(n=500):
    """The G = 1 kinetics medium with its prompt yield raised to k_prompt = 1.47: the population grows about tenfold per
    census interval, so a run of a few intervals ends in the runaway guard (R25a) -- in a LATER interval than the first."""
    P = inputs.td_infinite(n_particles=n, G=1, t_end=8.0e-4, n_t=8)
    P["mg_nu"] = P["mg_nu"] * 1.6
    return P


def test_td_failed_interval_leaves_the_last_successful_results(gpu):
    """mcdc.h: a failed run call leaves the results of the last successful call readable.  Interval by interval, the
    flux of the failed interval must not reach the published accumulators; mcdc_run_fixed_source publishes once, at the
    end, so a failure part-way leaves the previous call's results; after a failure the run has to start again."""
    P = _supercritical_td()
    N, seed, nt = P["run"]["n_particles"], P["run"]["seed"], len(P["t_edges"]) - 1
    g = gpu.Problem(P, max_particles=200000)
    good, failed_at = None, None
    for k in range(nt):
        try:
            g.run_cycle(N, k, 1, seed)
        except gpu.McdcError as e:
            assert e.code == -3  # MCDC_EBANK: the secondaries limit, raised on the device
            failed_at = k
            break
        good = g.results()
        cen = g.census()
    assert failed_at is not None and failed_at >= 1, failed_at
    after = g.results()
    assert (after["flux_mean"] == good["flux_mean"]).all() and (after["counters"] == good["counters"]).all()
    assert after["k_mean"] == good["k_mean"] and g.census() == cen
    with pytest.raises(gpu.McdcError) as e:
        g.run_cycle(N, failed_at, 1, seed)  # the run is over: the failed interval cannot be tried again
    assert e.value.code == -1 and "start again" in str(e.value)
    # a new run from the first interval works, and reproduces the first run's intervals
    for k in range(failed_at):
        g.run_cycle(N, k, 1, seed)
    again = g.results()
    assert np.allclose(again["flux_mean"], good["flux_mean"], rtol=1e-12, atol=0) and (again["counters"] == good["counters"]).all()
    # the same run as ONE call fails as a whole and publishes nothing of it
    with pytest.raises(gpu.McdcError) as e:
        g.run()
    assert e.value.code == -3
    kept = g.results()
    assert (kept["flux_mean"] == again["flux_mean"]).all() and (kept["counters"] == again["counters"]).all()
    g.close()
