"""Pins of the oracle's free-gas thermal scattering (R35; "free-gas scattering model with constant
cross-sections") and implicit capture with weight roulette (R36) -- no GPU."""
import math

import numpy as np
import pytest
from scipy import integrate, special

from paper_2501_05440_b200 import inputs

EV = dict(scatter=1, fission=2, capture=3, transmit=4, reflect=5, leak=6, lattice=7, time_edge=8, cutoff=9, lost=10)
KT = 0.0253


def collision_density(E, A, kT):
    """Equilibrium density of pre-collision energies in an infinite free-gas scatterer whose cross section is constant
    in the TARGET frame while flights use the constant table value: Maxwellian flux E exp(-E/kT) times the free-gas
    rate factor g(y) = (1 + 1/(2 y^2)) erf(y) + exp(-y^2) / (sqrt(pi) y), y = sqrt(A E / kT) (detailed balance of the
    kernel holds for the Maxwellian density with the effective cross section Sigma_0 g(y))."""
    y = np.sqrt(A * E / kT)
    g = (1.0 + 0.5 / (y * y)) * special.erf(y) + np.exp(-y * y) / (math.sqrt(math.pi) * y)
    return E * np.exp(-E / kT) * g


@pytest.mark.parametrize("A", [1.0, 12.0])
def test_free_gas_chain_equilibrium(orc, A):
    """A long chain of free-gas collisions of ONE neutron: its pre-collision energies are distributed as the exact
    equilibrium collision density above (chi-square over 12 bins, thinned to decorrelate)."""
    u = np.array([0.0, 0.0, 1.0])
    E, ctr, es = 5.0 * KT, 0, []
    n = 60000
    for k in range(n):
        E, u, used = orc.free_gas(E, u, A, KT, 11, 3, 0, ctr)
        ctr += used
        assert 6 <= used and E > 0 and abs(np.dot(u, u) - 1) < 1e-12
        es.append(E)
    thin = 4 if A == 1.0 else 40  # heavy targets change the energy slowly
    es = np.array(es[2000::thin])
    edges = KT * np.array([0, 0.3, 0.6, 0.9, 1.2, 1.6, 2.0, 2.5, 3.0, 3.8, 4.8, 6.5, 60.0])
    edges[0] = 1e-9 * KT
    norm = integrate.quad(collision_density, edges[0], edges[-1], args=(A, KT), limit=200)[0]
    pr = np.array([integrate.quad(collision_density, a, b, args=(A, KT), limit=200)[0] for a, b in zip(edges[:-1], edges[1:])]) / norm
    obs = np.histogram(es, edges)[0]
    chi2 = ((obs - len(es) * pr) ** 2 / (len(es) * pr)).sum()
    assert chi2 < 40.0, (chi2, obs, len(es) * pr)  # 11 degrees of freedom; residual correlation allowed for
    mean_want = integrate.quad(lambda e: e * collision_density(e, A, KT), edges[0], edges[-1], limit=200)[0] / norm
    assert abs(es.mean() / mean_want - 1) < 0.05


def test_free_gas_cold_limit_is_target_at_rest(orc):
    """kT -> 0: the free-gas collision reduces to the target-at-rest kinematics: E'/E uniform on [alpha, 1]."""
    A, E0 = 12.0, 1.0
    alpha = ((A - 1) / (A + 1)) ** 2
    r = np.array([orc.free_gas(E0, [0.6, 0.0, 0.8], A, 1e-12, 5, i)[0] for i in range(20000)])
    assert r.min() >= alpha - 1e-5 and r.max() <= 1 + 1e-5
    assert abs(r.mean() - (1 + alpha) / 2) < 4 * (1 - alpha) / math.sqrt(12 * len(r))
    assert abs(np.mean(r < (alpha + 1) / 2) - 0.5) < 4 * 0.5 / math.sqrt(len(r))


def test_free_gas_upscatter_below_kT(orc):
    """A neutron much slower than the gas gains energy on average (mean E' -> about 3/2 kT x 2A/(A+1)^2 ... > E)."""
    out = np.array([orc.free_gas(0.01 * KT, [0, 0, 1.0], 1.0, KT, 9, i)[0] for i in range(5000)])
    assert out.mean() > 0.3 * KT and (out > 0.01 * KT).mean() > 0.95


def free_gas_medium(A=1.0, n_particles=3000, n_grid=2000, T_end=2.0e-3):
    """Infinite pure free-gas scatterer (constant elastic cross section, nothing else), source at 10 kT, run long
    enough to thermalise; the flux spectrum of the last time bin is tallied in 40 energy bins."""
    P = inputs.ce_single_scatterer(A=A, n_particles=n_particles, E0=10 * KT, sig_el=1.0, sig_c=0.0, n_grid=n_grid)
    P["kT"] = KT
    P["t_edges"] = np.array([0.0, 0.25 * T_end, T_end])
    P["e_edges"] = np.concatenate([[1e-5], KT * np.linspace(0.1, 8.0, 40), [2e7]])
    P["name"] = "free_gas"
    return P


def test_free_gas_flux_spectrum_in_transport(orc):
    """The same equilibrium through the transport loop: after ~100 collisions the track-length flux spectrum (last
    time bin) is proportional to the equilibrium collision density (the flight cross section is constant)."""
    P = free_gas_medium()
    o = orc.Oracle(P)
    rc, r = o.run()
    assert rc == 0
    c = r["counters"]
    assert c[EV["scatter"]] / c[0] > 80 and c[EV["capture"]] == 0 and c[EV["cutoff"]] == c[0]
    f = r["flux_mean"].reshape(2, -1)[1]
    edges = P["e_edges"]
    pr = np.array([integrate.quad(collision_density, a, b, args=(1.0, KT), limit=200)[0] for a, b in zip(edges[:-1], edges[1:])])
    pr[-1] = integrate.quad(collision_density, edges[-2], 60 * KT, args=(1.0, KT), limit=200)[0]
    pr /= pr.sum()
    got = f / f.sum()
    # per-bin noise: ~3000 histories x ~75 collisions in the bin window, strongly correlated within a history
    assert np.abs(got - pr).max() < 0.012, np.abs(got - pr).max()
    assert abs((got * 0.5 * (edges[:-1] + np.minimum(edges[1:], 20 * KT))).sum() / (pr * 0.5 * (edges[:-1] + np.minimum(edges[1:], 20 * KT))).sum() - 1) < 0.03


# --------------------------------------------------------------------------- implicit capture (R36)
def _balance_ok(b, rel=1e-11):
    rhs = b["absorbed"] + b["leaked"] + b["cutoff"] + b["roulette_loss"] - b["roulette_gain"]
    assert rhs == pytest.approx(b["source"], rel=rel)


@pytest.mark.parametrize("implicit", [0, 1])
def test_weight_balance_identity(orc, implicit):
    """source weight = absorbed + leaked + cut off + roulette losses - roulette gains, exactly (to rounding), history
    by history: analog and implicit capture, multi-group (lattice, vacuum faces) and continuous energy."""
    P = inputs.config4(n_particles=4000, n_inactive=1, n_active=2, n_asm=1, n_pin=3, n_refl=1)
    P["implicit_capture"] = implicit
    o = orc.Oracle(P)
    rc, r = o.run()
    assert rc == 0
    b = o.balance()
    _balance_ok(b)
    assert b["source"] == pytest.approx(3 * 4000.0, rel=1e-12) and b["leaked"] > 0
    if implicit:
        assert b["roulette_loss"] > 0 and b["roulette_gain"] > 0
        assert abs(b["roulette_loss"] - b["roulette_gain"]) < 0.1 * b["roulette_loss"] + 30  # roulette is fair
    else:
        assert b["roulette_loss"] == 0 and b["roulette_gain"] == 0
    Pc = inputs.config5(n_particles=300, n_grid=3000)
    Pc["implicit_capture"] = implicit
    oc = orc.Oracle(Pc)
    rc, rcx = oc.run()
    assert rc == 0
    _balance_ok(oc.balance())


def test_implicit_capture_preserves_k_and_flux(orc):
    """Survival biasing changes no expectation: C1 k = 1.3 within 3 sigma, flux 1/Sigma_a, and (roulette off) no
    history ends in a capture."""
    P = inputs.config1(n_particles=10000, n_inactive=3, n_active=12)
    P["implicit_capture"] = 1
    o = orc.Oracle(P)
    rc, r = o.run()
    assert rc == 0
    assert abs(r["k_mean"] - 1.3) < 3.5 * r["k_sdev"]
    assert abs(r["flux_mean"][0] - 1 / 0.3) < 4 * r["flux_sdev"][0]
    P["w_roulette"] = 0.0
    o2 = orc.Oracle(P)
    rc, r2 = o2.run(n_particles=2000, n_inactive=0, n_active=2)
    c = r2["counters"]
    assert c[EV["capture"]] == 0 and c[EV["fission"]] == c[0]
    b = o2.balance()
    assert b["roulette_loss"] == 0 and b["roulette_gain"] == 0
    _balance_ok(b)


def test_implicit_capture_slab_leakage_agrees_with_analog(orc):
    """Scattering slab, normal beam: transmitted + reflected weight per source particle is the same with and without
    survival biasing (within 4 combined sigma over 10 batches)."""
    vals = {}
    for implicit in (0, 1):
        P = inputs.slab_beam(L=2.0, sig_t=1.3, n_particles=4000)
        P["mg_S"] = np.array([[[0.8]]])  # Sigma_s = 0.8 of 1.3
        P["implicit_capture"] = implicit
        leaks = []
        for seed in range(10):
            o = orc.Oracle(P)
            rc, r = o.run(n_inactive=0, n_active=1, seed=100 + seed)
            leaks.append(r["leak_mean"])
        vals[implicit] = (np.mean(leaks), np.std(leaks, ddof=1) / math.sqrt(10))
    assert abs(vals[0][0] - vals[1][0]) < 4 * math.hypot(vals[0][1], vals[1][1])
    assert vals[1][1] < vals[0][1] * 1.1  # and it does not raise the variance
