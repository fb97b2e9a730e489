"""GPU parity for SURVEY.md 8f row f4: free-gas thermal scattering with a constant cross section (R35)
and implicit capture with weight roulette (R36), against the oracle on the same seeded inputs.  Same tolerances as
the analog path: discrete trace fields and event counters exact, floats / k / flux / weight balance 1e-9 relative."""
import numpy as np
import pytest

from paper_2501_05440_b200 import inputs
from tests.test_gpu_parity import ALWAYS, compare_results, compare_traces
from tests.test_gpu_ce import compare_ce

pytestmark = pytest.mark.gpu

KT = 0.0253
BAL = ("source", "absorbed", "leaked", "cutoff", "roulette_loss", "roulette_gain")


@pytest.fixture(scope="module")
def gpu():
    from paper_2501_05440_b200 import binding
    binding.load_library()
    return binding


def compare_balance(bg, bo, rtol=1e-9):
    for k in BAL:
        assert bg[k] == pytest.approx(bo[k], rel=rtol, abs=1e-9 * bo["source"]), (k, bg, bo)
    rhs = bg["absorbed"] + bg["leaked"] + bg["cutoff"] + bg["roulette_loss"] - bg["roulette_gain"]
    assert rhs == pytest.approx(bg["source"], rel=1e-10)


def _with(P, **kw):
    P.update(kw)
    return P


MG_CASES = {
    "C1": lambda: inputs.config1(n_particles=3000, n_inactive=2, n_active=3),
    "C1_no_roulette": lambda: _with(inputs.config1(n_particles=2000, n_inactive=1, n_active=2), w_roulette=0.0),
    "C2": lambda: inputs.config2(n_particles=4000, n_inactive=1, n_active=3),
    "C3": lambda: inputs.config3(n_particles=4000, n_inactive=1, n_active=3),
    "C4small": lambda: inputs.config4(n_particles=3001, n_inactive=1, n_active=2, n_asm=1, n_pin=3, n_refl=1),
    "C4": lambda: inputs.config4(n_particles=5000, n_inactive=1, n_active=2),
    "mixed": lambda: inputs.mixed_surfaces(n_particles=3000),
    "slab": lambda: _with(inputs.slab_beam(L=2.0, sig_t=1.3, n_particles=5000), mg_S=np.array([[[0.8]]])),
    "C3_thresholds": lambda: _with(inputs.config3(n_particles=3000, n_inactive=1, n_active=2), w_roulette=0.6, w_survive=1.5),
}
SCHEDULES = [(0, 0), (0, -1), (1, 0), (2, -1), (0, 300)]


@pytest.mark.parametrize("name", list(MG_CASES))
@pytest.mark.parametrize("schedule,persist", SCHEDULES)
def test_mg_implicit_capture_parity(gpu, orc, name, schedule, persist):
    """Survival biasing in every schedule: k per cycle, flux, leakage, event counters, fission bank and the weight
    balance (source, absorbed, leaked, roulette loss / gain) equal the oracle's."""
    P = MG_CASES[name]()
    P["implicit_capture"] = 1
    g = gpu.Problem(P, schedule=schedule, persist_threshold=persist)
    r = g.run()
    o = orc.Oracle(P)
    rc, ro = o.run()
    assert rc == 0
    compare_results(r, ro)
    compare_balance(g.balance(), o.balance())
    bg, bo = g.bank(), o.bank()
    assert len(bg) == len(bo) and (bg["g"] == bo["g"]).all()
    for f in ("x", "y", "z", "ux", "uy", "uz"):
        assert np.allclose(bg[f], bo[f], rtol=1e-9, atol=1e-11), f
    g.close()


@pytest.mark.parametrize("name", ["C1", "C3", "C4small", "mixed"])
@pytest.mark.parametrize("schedule,persist", [(0, 0), (0, -1), (1, 0), (0, 100)])
def test_mg_implicit_capture_traces(gpu, orc, name, schedule, persist):
    """100 particles x 2 cycles: identical event sequences (the roulette draw sits between the reaction draw and the
    scatter draws; a roulette kill is traced as a capture)."""
    P = MG_CASES[name]()
    P["implicit_capture"] = 1
    N = 1000
    g = gpu.Problem(P, max_particles=N, schedule=schedule, persist_threshold=persist)
    g.set_trace(0, 100, 2048)
    r = g.run(n_particles=N, n_inactive=0, n_active=2)
    o = orc.Oracle(P)
    o.set_trace(0, 100, 800000)
    rc, ro = o.run(n_particles=N, n_inactive=0, n_active=2)
    compare_traces(g.trace(), o.trace())
    compare_results(r, ro)
    g.close()


def test_analog_balance_matches_oracle(gpu, orc):
    """The analog path reports the same balance terms (from its event counters and the launch weight)."""
    P = MG_CASES["C4small"]()
    g = gpu.Problem(P)
    g.run()
    o = orc.Oracle(P)
    o.run()
    compare_balance(g.balance(), o.balance())
    g.close()
    Pc = inputs.config5(n_particles=300, n_grid=3000)
    g = gpu.Problem(Pc)
    g.run()
    o = orc.Oracle(Pc)
    o.run()
    compare_balance(g.balance(), o.balance())
    g.close()


def free_gas_medium(A=1.0, n_particles=1500, n_grid=2000, T_end=4.0e-4, sig_c=0.0):
    """Infinite free-gas scatterer with a constant elastic cross section, source at 10 kT (the oracle pin's medium)."""
    P = inputs.ce_single_scatterer(A=A, n_particles=n_particles, E0=10 * KT, sig_el=1.0, sig_c=sig_c, n_grid=n_grid)
    P["kT"] = KT
    P["t_edges"] = np.array([0.0, 0.25 * T_end, T_end])
    P["e_edges"] = np.concatenate([[1e-5], KT * np.linspace(0.1, 8.0, 40), [2e7]])
    P["name"] = "free_gas"
    return P


CE_CASES = {
    "free_gas_H": lambda: free_gas_medium(A=1.0),
    "free_gas_C": lambda: free_gas_medium(A=12.0),
    "free_gas_abs": lambda: free_gas_medium(A=1.0, sig_c=0.05),
    "C5_thermal": lambda: _with(inputs.config5(n_particles=800, n_grid=8000), kT=KT),
    "C5_implicit": lambda: _with(inputs.config5(n_particles=800, n_grid=8000), implicit_capture=1),
    "C5_both": lambda: _with(inputs.config5(n_particles=800, n_grid=8000), kT=KT, implicit_capture=1),
    "mix_implicit": lambda: _with(inputs.ce_two_nuclide_mix(n_particles=2000, n_grid=3000), implicit_capture=1),
    "free_gas_implicit": lambda: _with(free_gas_medium(A=1.0, sig_c=0.05), implicit_capture=1, w_roulette=0.3),
}


@pytest.mark.parametrize("name", list(CE_CASES))
@pytest.mark.parametrize("schedule,persist,search", [(0, 0, 1), (0, -1, 0), (1, 0, 1), (0, 200, 0)])
def test_ce_f4_parity(gpu, orc, name, schedule, persist, search):
    P = CE_CASES[name]()
    g = gpu.Problem(P, schedule=schedule, persist_threshold=persist, search=search)
    r = g.run()
    o = orc.Oracle(P)
    rc, ro = o.run()
    assert rc == 0
    compare_ce(r, ro)
    compare_balance(g.balance(), o.balance())
    g.close()


@pytest.mark.parametrize("name", ["free_gas_H", "free_gas_C", "C5_both", "free_gas_implicit"])
@pytest.mark.parametrize("schedule,persist", [(0, 0), (0, -1), (1, 0)])
def test_ce_f4_traces(gpu, orc, name, schedule, persist):
    """Event sequences of source particles 0..99: the energy after every free-gas collision (a variable number of
    draws: rejection loop), grid index, time and position agree record by record."""
    P = CE_CASES[name]()
    g = gpu.Problem(P, schedule=schedule, persist_threshold=persist)
    g.set_trace(0, 100, 4096)
    r = g.run()
    o = orc.Oracle(P)
    o.set_trace(0, 100, 3_000_000)
    rc, ro = o.run()
    compare_traces(g.trace(), o.trace())
    compare_ce(r, ro)
    g.close()


def test_set_physics_validation(gpu):
    P = MG_CASES["C1"]()
    g = gpu.Problem(P)
    with pytest.raises(gpu.McdcError) as e:
        g.set_physics(kT=-1.0)
    assert e.value.code == -1
    with pytest.raises(gpu.McdcError) as e:
        g.set_physics(implicit_capture=1, w_roulette=0.5, w_survive=0.25)
    assert e.value.code == -1
    # switching the option on and off again gives back the analog result
    r0 = g.run()
    g.set_physics(implicit_capture=1)
    r1 = g.run()
    g.set_physics()
    r2 = g.run()
    assert np.allclose(r0["k_cycle"], r2["k_cycle"], rtol=1e-12) and (r0["counters"][:12] == r2["counters"][:12]).all()
    assert not np.allclose(r0["k_cycle"], r1["k_cycle"], rtol=1e-6)
    g.close()
