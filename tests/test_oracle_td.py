"""Pins of the oracle's time-dependent multi-group path with delayed-neutron precursors and census population
control ("fully dynamic simulations"; R38-R40) -- no GPU.

The pin is the exact kinetics of an infinite homogeneous medium: with n_g(t) the neutrons of group g and C_j(t) the
precursors of group j per source neutron,
    dn_g/dt = -v_g Sigma_t,g n_g + sum_g' v_g' n_g' (S_g'g + chi_g nu_p,g' Sigma_f,g') + sum_j chi_d,jg lambda_j C_j
    dC_j/dt = sum_g' nu_d,jg' Sigma_f,g' v_g' n_g' - lambda_j C_j
a linear system y' = A y whose integral over a time bin gives the expected track-length flux v_g int n_g dt (for one
group and one precursor group these are the point-kinetics equations, exact here because the medium is infinite)."""
import numpy as np
import pytest
from scipy.linalg import expm

from paper_2501_05440_b200 import inputs

EV = dict(scatter=1, fission=2, capture=3, reflect=5, time_edge=8, cutoff=9)


def kinetics_flux(P):
    """expected flux[time bin][g] per source neutron of the infinite-medium problem P (material 0)"""
    G, td = P["G"], P["td"]
    J = td["J"]
    st, S, sf, nup = P["mg_sig_t"][0], P["mg_S"][0], P["mg_sig_f"][0], P["mg_nu"][0]
    chi, v = P["mg_chi"][0] / P["mg_chi"][0].sum(), td["speed"]
    nud, lam, chid = td["nu_d"][0], td["decay"][0], td["chi_d"][0]
    chid = chid / chid.sum(axis=1, keepdims=True)
    A = np.zeros((G + J, G + J))
    for g in range(G):
        A[g, g] -= v[g] * st[g]
        for gp in range(G):
            A[g, gp] += v[gp] * (S[gp, g] + chi[g] * nup[gp] * sf[gp])
        for j in range(J):
            A[g, G + j] += chid[j, g] * lam[j]
    for j in range(J):
        A[G + j, G + j] -= lam[j]
        for gp in range(G):
            A[G + j, gp] += nud[j, gp] * sf[gp] * v[gp]
    y0 = np.zeros(G + J)
    y0[:G] = P["src_group_pdf"] / P["src_group_pdf"].sum()
    t = P["t_edges"]
    Ai = np.linalg.inv(A)
    out = np.zeros((len(t) - 1, G))
    for k in range(len(t) - 1):
        integ = Ai @ (expm(A * t[k + 1]) - expm(A * t[k])) @ y0
        out[k] = v * integ[:G]
    return out


def _run(orc, P, seeds):
    fl = []
    for s in seeds:
        o = orc.Oracle(P)
        rc, r = o.run(seed=s)
        assert rc == 0
        fl.append(r["flux_mean"].reshape(len(P["t_edges"]) - 1, P["G"]))
    fl = np.array(fl)
    return fl.mean(0), fl.std(0, ddof=1) / np.sqrt(len(seeds)), o, r


def test_comb_against_brute_force(orc):
    """The comb on plain arrays: copies per particle = teeth of the grid (xi + j) W / N inside the particle's interval
    of the running weight sum (numpy searchsorted), exactly N copies, weight N * delta = W; and the expected number of
    copies over the offset is w_i N / W."""
    rng = np.random.default_rng(5)
    w = rng.uniform(0.05, 3.0, 500)
    W, N = w.sum(), 137
    exp = np.zeros(len(w))
    for xi in rng.uniform(0, 1, 400):
        copies, delta = orc.comb(w, N, xi)
        teeth = (xi + np.arange(N)) * (W / N)
        ref = np.bincount(np.searchsorted(np.cumsum(w), teeth, side="right"), minlength=len(w))[: len(w)]
        assert (copies == ref).all() and copies.sum() == N
        assert delta * N == pytest.approx(W, rel=1e-14)
        exp += copies
    assert np.abs(exp / 400 - w * N / W).max() < 0.12
    # equal weights, N = M: everybody survives exactly once; N = 2 M: exactly twice
    assert (orc.comb(np.ones(50), 50, 0.37)[0] == 1).all() and (orc.comb(np.ones(50), 100, 0.9)[0] == 2).all()


@pytest.mark.parametrize("G", [1, 2])
def test_td_flux_equals_kinetics(orc, G):
    """Pulse at t = 0 in an infinite medium with delayed neutrons, no population control: the flux in every time bin
    (and group) equals the kinetics integral within 4 sigma over 6 seeds; the slow tail is carried by the delayed
    neutrons alone (prompt-only kinetics would be lower by orders of magnitude)."""
    P = inputs.td_infinite(n_particles=6000, G=G)
    ref = kinetics_flux(P)
    mean, sd, o, r = _run(orc, P, range(100, 106))
    assert (np.abs(mean - ref) < 4 * sd + 1e-4 * ref).all(), (mean, ref, sd)
    assert np.abs(mean.sum() / ref.sum() - 1) < 0.02
    prompt_only = dict(P)
    prompt_only["td"] = dict(P["td"], nu_d=P["td"]["nu_d"] * 0.0)
    assert kinetics_flux(prompt_only)[-1].sum() < 0.05 * ref[-1].sum() and mean[-1].sum() > 0.5 * ref[-1].sum()
    c = r["counters"]
    assert c[EV["time_edge"]] > 0 and c[EV["cutoff"]] > 0 and c[10] == 0


def test_td_population_control_is_unbiased_and_conserves_weight(orc):
    """Combing to half / twice the source size at every census: the flux still equals the kinetics integral, the
    population entering each later interval is exactly the target, and the comb conserves the total weight to
    rounding."""
    for target in (3000, 12000):
        P = inputs.td_infinite(n_particles=6000, G=1, census_target=target)
        ref = kinetics_flux(P)
        mean, sd, o, r = _run(orc, P, range(200, 206))
        assert (np.abs(mean - ref) < 4 * sd + 1e-4 * ref).all(), (target, mean, ref, sd)
        cen = o.census()
        assert len(cen) == 8 and cen[0][0] == cen[0][1] == 6000
        for before, after, w_before, w_after in cen[1:]:
            assert after == target and before > 0
            assert w_after == pytest.approx(w_before, rel=1e-12)
        b = o.balance()  # tracks replaced by the comb are neither lost nor counted twice
        assert b["absorbed"] + b["leaked"] + b["cutoff"] + b["roulette_loss"] - b["roulette_gain"] == pytest.approx(b["source"], rel=1e-10)


def test_td_time_edges_are_census_points(orc):
    """Without population control the census only interrupts a history: total events and the flux do not depend on
    how many time edges cut the same time span (2 bins against 8: the 8-bin flux summed in fours), except for the
    time-edge events themselves."""
    P8 = inputs.td_infinite(n_particles=3000, G=2, n_t=8)
    P2 = inputs.td_infinite(n_particles=3000, G=2, n_t=2)
    o8, o2 = orc.Oracle(P8), orc.Oracle(P2)
    rc8, r8 = o8.run()
    rc2, r2 = o2.run()
    assert rc8 == 0 and rc2 == 0
    # a time edge restarts the segment (one more d_coll draw), so the histories differ: statistical agreement only
    f8 = r8["flux_mean"].reshape(8, 2).reshape(2, 4, 2).sum(1)
    f2 = r2["flux_mean"].reshape(2, 2)
    assert np.abs(f8[0] / f2[0] - 1).max() < 0.02 and np.abs(f8[1] / f2[1] - 1).max() < 0.35  # the tail is a few histories
    assert r8["counters"][EV["time_edge"]] > r2["counters"][EV["time_edge"]]


def test_td_delayed_neutron_after_cutoff_is_not_born(orc):
    """Decay much slower than the run: almost every delayed neutron would be emitted after the last edge and must not
    appear; the children banked equal the prompt fraction within counting noise."""
    P = inputs.td_infinite(n_particles=4000, G=1, t_end=2.0e-4, n_t=2)
    P["td"] = dict(P["td"], decay=np.array([[1.0e-2]]))
    o = orc.Oracle(P)
    rc, r = o.run()
    assert rc == 0
    c = r["counters"]
    nu_p, nu_d = 2.3, 0.15
    born_per_fission = c[11] / c[EV["fission"]]
    assert abs(born_per_fission - nu_p) < 0.05 and born_per_fission < nu_p + 0.5 * nu_d
