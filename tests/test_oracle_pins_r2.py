"""Round-2 pins of the oracle (no GPU): the parts VERDICT r01 listed as unpinned.

  - reflect(), non-axis branch: closed forms behind a reflecting sphere / cylinders (k_inf, zero leakage, uniform
    flux); event-by-event pins are in tests/test_oracle_traces.py (brute-force tracer);
  - the continuous-energy elastic branch INSIDE transport(): which nuclide a sampled column names, the energy clamp,
    the clock t += d / v with a changing v;
  - edge_bin() over 100 bins against numpy.searchsorted, as used by the tally inside the loop.
Citations: SURVEY.md 8(c) readings 13 (reflection), 19 (clamp), 21 (elastic), 23 (speed), 24 (bins by bisection)."""
import math

import numpy as np
import pytest

from paper_2501_05440_b200 import inputs

EV = dict(scatter=1, fission=2, capture=3, transmit=4, reflect=5, leak=6, lattice=7, time_edge=8, cutoff=9, lost=10)


@pytest.mark.parametrize("kind", ["sphere", "cyl_z", "cyl_x", "cyl_y"])
def test_curved_mirror_closed_forms(orc, kind):
    """C1's material behind a specular curved wall is an infinite medium: nothing leaks, k -> nuSigma_f / Sigma_a = 1.3,
    and the converged flux is uniform, so inner / outer track length = volume ratio (r_in^3 / (1 - r_in^3) for the
    sphere, r_in^2 / (1 - r_in^2) for a cylinder).  A wrong sign or a missing normalisation in the reflection formula
    sends particles out of the cell (lost) or piles flux up at the wall."""
    P = inputs.curved_mirror(kind, n_particles=20000, n_inactive=3, n_active=12)
    o = orc.Oracle(P)
    rc, r = o.run()
    assert rc == 0
    c = r["counters"].astype(np.int64)
    assert c[EV["lost"]] == 0 and c[EV["leak"]] == 0 and r["leak_mean"] == 0.0
    assert c[EV["reflect"]] > 100000
    assert c[EV["capture"]] + c[EV["fission"]] == c[0]
    assert abs(r["k_mean"] - 1.3) < 3.5 * r["k_sdev"]
    f, s = r["flux_mean"], r["flux_sdev"]
    want = 0.6 ** 3 / (1 - 0.6 ** 3) if kind == "sphere" else 0.36 / 0.64
    ratio = f[0] / f[1]
    sig = ratio * math.hypot(s[0] / f[0], s[1] / f[1])
    assert abs(ratio - want) < 4 * sig + 2e-3
    assert abs(f.sum() - 1 / 0.3) < 4 * math.hypot(s[0], s[1])  # track length per source particle = 1 / Sigma_a


def _ratios_of_scatters(tr):
    """E'/E of every scatter event of every traced history: E' is the flight energy of the history's next event."""
    out = []
    for pid in np.unique(tr["id"]):
        h = tr[tr["id"] == pid]
        h = h[np.argsort(h["seq"])]
        for a, b in zip(h[:-1], h[1:]):
            if a["ev"] == EV["scatter"]:
                out.append(b["E"] / a["E"])
    return np.array(out)


def test_ce_elastic_branch_names_the_right_nuclide(orc):
    """Mixture of A = 1 (30 % of Sigma_el, first in the material's list, LAST in the nuclide table) and A = 238: a
    collision with the heavy nuclide keeps E'/E >= alpha_238 = (237/239)^2, one with the light nuclide spreads E'/E
    uniformly over [0, 1].  So the fraction of scatters with E'/E < alpha_238 is p_light * alpha_238, the ones above
    it are uniform on [alpha_238, 1] for the heavy nuclide (mean (1 + alpha)/2).  A wrong column -> nuclide map (e.g.
    the column used as the nuclide id) gives 0.70 * alpha or a third mass instead."""
    P = inputs.ce_two_nuclide_mix(n_particles=3000)
    o = orc.Oracle(P)
    o.set_trace(0, 3000, 400000)
    rc, r = o.run()
    assert rc == 0
    ratio = _ratios_of_scatters(o.trace())
    n = len(ratio)
    assert n > 50000
    alpha = (237.0 / 239.0) ** 2
    p = 0.3 * alpha
    frac = (ratio < alpha).mean()
    assert abs(frac - p) < 4 * math.sqrt(p * (1 - p) / n)
    assert ratio.max() <= 1.0 and ratio.min() >= 0.0
    # light-nuclide collisions below alpha: uniform on [0, alpha)
    low = ratio[ratio < alpha]
    assert abs(low.mean() - alpha / 2) < 4 * alpha / math.sqrt(12 * len(low))
    # above alpha: heavy-nuclide collisions (uniform on [alpha, 1]) plus the light ones' share (1 - alpha) p_light
    hi = ratio[ratio >= alpha]
    assert abs(hi.mean() - (1 + alpha) / 2) < 4 * (1 - alpha) / math.sqrt(12 * len(hi))
    # every history is captured at its first collision below E_cut (capture is 10^7 times the elastic there)
    c = r["counters"].astype(np.int64)
    assert c[EV["capture"]] == c[0] == 3000 and c[EV["cutoff"]] == 0


def test_ce_slowing_down_collision_count(orc):
    """Pure hydrogen-like scatterer (E'/E uniform): the lethargy gain per collision is Exp(1), so the number of
    collisions needed to fall from E0 below E_cut is Poisson(ln(E0/E_cut)) + 1: mean ln(E0/E_cut) + 1 scatters per
    history (all collisions above E_cut are scatters; the next one is the capture)."""
    N = 20000
    P = inputs.ce_two_nuclide_mix(n_particles=N, p_light=1.0, E0=1.0e6, E_cut=1.0)
    rc, r = orc.Oracle(P).run()
    assert rc == 0
    c = r["counters"].astype(np.float64)
    lam = math.log(1.0e6 / 1.0)
    assert c[EV["capture"]] == N
    assert abs(c[EV["scatter"]] / N - (lam + 1.0)) < 4 * math.sqrt(lam / N) + 2e-3  # + grid-interval smear of the step


@pytest.mark.parametrize("A", [1.0, 12.0])
def test_ce_clock_advances_with_the_flight_speed(orc, A):
    """Sigma_el = lam / v(E): collisions happen at rate lam per unit time whatever the energy, so the number of
    scatters up to the time cutoff T is Poisson(lam T) -- mean AND variance -- only if each flight adds d / v(E of
    that flight) to the clock (with A = 1 the speed changes by large factors from flight to flight)."""
    N, lam, T = 20000, 3.0e6, 4.0e-6
    P = inputs.ce_scatter_clock(lam=lam, T=T, A=A, n_particles=N)
    o = orc.Oracle(P)
    o.set_trace(0, 2000, 200000)
    rc, r = o.run()
    assert rc == 0
    c = r["counters"].astype(np.float64)
    assert c[EV["cutoff"]] == N and c[EV["capture"]] == 0
    mean = c[EV["scatter"]] / N
    assert abs(mean - lam * T) < 4 * math.sqrt(lam * T / N)
    tr = o.trace()
    per = np.array([((tr["id"] == i) & (tr["ev"] == EV["scatter"])).sum() for i in range(300)])
    assert abs(per.var(ddof=1) / (lam * T) - 1.0) < 0.35  # Poisson: variance = mean (300 histories: +- 8 % one sigma)
    # the clock itself: t after each event = sum of d / v(E_flight) along the history
    h = tr[tr["id"] == 7]
    h = h[np.argsort(h["seq"])]
    v = 2.99792458e10 * np.sqrt(2.0 * h["E"] / 939.56542052e6)
    t = np.cumsum(h["d"] / v)
    assert np.allclose(h["t"][:-1], t[:-1], rtol=1e-12) and h["t"][-1] == T


def test_ce_energy_clamp_at_grid_floor(orc):
    """A = 1 at E0 = 2 E_min: E'/E is uniform on [0, 1], so half of the first collisions fall below the grid and are
    clamped to E_min exactly (reading 19); no energy below the floor ever appears."""
    P = inputs.ce_single_scatterer(A=1.0, n_particles=4000, E0=2.0e-5, sig_el=0.9, sig_c=0.1)
    o = orc.Oracle(P)
    o.set_trace(0, 4000, 400000)
    rc, r = o.run()
    assert rc == 0
    tr = o.trace()
    assert tr["E"].min() == 1.0e-5
    first = tr[tr["seq"] == 0]
    second = tr[tr["seq"] == 1]
    ids = first["id"][first["ev"] == EV["scatter"]]
    e2 = second["E"][np.isin(second["id"], ids)]
    n = len(e2)
    assert n > 3000
    frac = (e2 == 1.0e-5).mean()
    assert abs(frac - 0.5) < 4 * math.sqrt(0.25 / n)
    rest = e2[e2 > 1.0e-5]
    assert abs(rest.mean() - 1.5e-5) < 4 * (1.0e-5 / math.sqrt(12 * len(rest)))


def test_edge_bin_100_bins_vs_searchsorted(orc):
    """The (time bin, energy bin) every segment is tallied into equals numpy.searchsorted on the edge arrays: rebuild
    the whole 10 x 100 flux tally of a C5 run from its event trace (flight energy, flight length, time) and compare
    bin by bin.  An off-by-one anywhere in the oracle's bisection moves track length to a neighbouring bin."""
    n = 40
    P = inputs.config5(n_particles=n, n_grid=4000, absorber=1.0e-4)
    P["nuc_f"] = P["nuc_f"] * 0.0  # no fission: every track is a traced source history
    o = orc.Oracle(P)
    o.set_trace(0, n, 2_000_000)
    rc, r = o.run()
    assert rc == 0 and r["counters"][11] == 0
    tr = o.trace()
    te, ee = P["t_edges"], P["e_edges"]
    v = 2.99792458e10 * np.sqrt(2.0 * tr["E"] / 939.56542052e6)
    t_mid = tr["t"] - 0.5 * tr["d"] / v
    tb = np.clip(np.searchsorted(te, t_mid, side="right") - 1, 0, len(te) - 2)
    eb = np.clip(np.searchsorted(ee, tr["E"], side="right") - 1, 0, len(ee) - 2)
    want = np.zeros((len(te) - 1, len(ee) - 1))
    np.add.at(want, (tb, eb), tr["d"])
    got = r["flux_mean"].reshape(want.shape) * n
    assert (want > 0).sum() > 100  # the run visits many bins
    assert np.allclose(got, want, rtol=1e-9, atol=1e-12 * want.max())
    # energies sitting exactly on an edge belong to the bin that starts there
    Pe = inputs.ce_single_scatterer(A=200.0, n_particles=50, E0=float(ee[37]), sig_el=0.0, sig_c=1.0)
    Pe["e_edges"] = ee
    rc, re = orc.Oracle(Pe).run()
    f = re["flux_mean"]
    assert f[37] > 0 and f[36] == 0 and f[38] == 0
