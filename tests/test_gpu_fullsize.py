"""Full-size parity (BASELINE.json sizes, in the launch configuration bench.py times): sampled per-particle event
sequences the oracle can compute one by one, invariants that hold at any size, k within 3 combined sigma of the
closed form (C1, C2) or of the oracle at reduced N (C3, C4), C5 flux per time bin within 4 sigma."""
import math

import numpy as np
import pytest

from paper_2501_05440_b200 import inputs
from tests.test_gpu_parity import compare_results, compare_traces
from tests.test_oracle_transport import EV, kinf_dense

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gpu():
    from paper_2501_05440_b200 import binding
    binding.load_library()
    return binding


def invariants(r, n_hist_expected=None):
    c = r["counters"].astype(np.int64)
    assert c[EV["lost"]] == 0
    assert c[EV["capture"]] + c[EV["fission"]] + c[EV["leak"]] + c[EV["cutoff"]] == c[0]
    assert np.isfinite(r["flux_mean"]).all() and (r["flux_mean"] >= 0).all()
    if n_hist_expected is not None:
        assert c[0] == n_hist_expected


def test_c1_full(gpu, orc):
    P = inputs.config1()
    g = gpu.Problem(P)
    r = g.run()
    rc, ro = orc.Oracle(P).run()
    compare_results(r, ro)
    invariants(r)
    assert abs(r["k_mean"] - 1.3) < 3 * r["k_sdev"]
    g.close()


def test_c2_full(gpu, orc):
    P = inputs.config2()
    g = gpu.Problem(P)
    r = g.run()
    rc, ro = orc.Oracle(P).run()
    compare_results(r, ro)
    invariants(r)
    assert abs(r["k_mean"] - kinf_dense(P)) < 3 * r["k_sdev"]
    g.close()


def test_c3_full(gpu, orc):
    """10^6 particles x (20 + 80) cycles on the GPU; oracle at 5*10^4 x (10 + 30)."""
    P = inputs.config3()
    g = gpu.Problem(P)
    r = g.run()
    invariants(r)
    assert len(r["k_cycle"]) == 100
    Po = inputs.config3(n_particles=50_000, n_inactive=10, n_active=30)
    rc, ro = orc.Oracle(Po).run()
    assert abs(r["k_mean"] - ro["k_mean"]) < 3 * math.hypot(r["k_sdev"], ro["k_sdev"])
    comb = np.hypot(r["flux_sdev"], ro["flux_sdev"])
    assert (np.abs(r["flux_mean"] - ro["flux_mean"]) < 4.5 * comb + 1e-12).all()
    # sum over cycles of source weight = N per cycle: flux per source particle is O(1/Sigma_a)
    assert 1.0 < r["flux_mean"].sum() < 100.0
    g.close()


@pytest.mark.parametrize("first", [0, 250_000])
def test_c4_full_sampled_traces(gpu, orc, first):
    """C4 at 10^7 particles per cycle (bench configuration): the event sequences of 150 sampled histories of
    cycle 0 equal the oracle's, which can follow them one by one (cycle-0 histories depend on (seed, id) only)."""
    P = inputs.config4()
    g = gpu.Problem(P)
    g.set_trace(first, 150, 2048)
    k0 = g.run_cycle(10_000_000, 0, 1, 1)
    tg = g.trace()
    r = g.results()
    invariants(r, 10_000_000)
    o = orc.Oracle(P)
    o.set_trace(first, 150, 1_000_000)
    o.run(n_particles=first + 150, n_inactive=0, n_active=1)
    compare_traces(tg, o.trace())
    # k of cycle 0 (a mean over source histories, which depend on (seed, id) only) against the oracle's cycle-0 k at 10^5
    # histories: within 4 sigma of a 10^5 run, sigma measured from eight GPU seeds at that size
    rc, ro = orc.Oracle(P).run(n_particles=100_000, n_inactive=0, n_active=1)
    gs = gpu.Problem(inputs.config4(n_particles=100_000))
    sig = np.std([gs.run_cycle(100_000, 0, 1, seed) for seed in range(2, 10)], ddof=1)
    gs.close()
    assert 0.0 < sig < 0.02 and abs(k0 - ro["k_cycle"][0]) < 4 * sig * math.sqrt(1.01)
    g.close()


REFILL_LANES = 444 * 256  # resident lanes of k_persist (3 blocks of 256 on each of 148 SMs): more particles than this
                          # and lanes are refilled from the ticket queue while their neighbours are mid-history


@pytest.mark.parametrize("name", ["C4", "C3", "C4_2l", "C4_implicit", "C3_implicit", "C4_3d_axial"])
def test_mg_parity_refill_regime(gpu, orc, name):
    """Element-by-element tally parity in the regime the benchmark runs in (finding 1): 3 x 10^5 particles
    per cycle is 2.6 x the resident lanes of the persistent kernel, so every lane ends a history, takes a new ticket and
    re-initialises its state and random-number stream next to running neighbours, and (global tally flavour) all 64
    replicated tally copies are written.  Default schedule, 1 inactive + 2 active cycles; k per cycle, every flux bin and
    the leakage within 1e-9 of the serial oracle, counters equal, the fission bank site by site."""
    N = 300_000
    kw = dict(n_particles=N, n_inactive=1, n_active=2)
    P = {"C4": lambda: inputs.config4(**kw), "C3": lambda: inputs.config3(**kw),
         "C4_2l": lambda: inputs.config4(two_level=True, **kw),
         "C4_implicit": lambda: inputs.config4(**kw), "C3_implicit": lambda: inputs.config3(**kw),
         "C4_3d_axial": lambda: inputs.config4(height=64.26, axial_reflector=21.42, **kw)}[name]()
    if name.endswith("implicit"):
        P["implicit_capture"] = 1
    g = gpu.Problem(P)
    r = g.run()
    o = orc.Oracle(P)
    rc, ro = o.run()
    assert rc == 0
    compare_results(r, ro)
    invariants(r) if not name.endswith("implicit") else None
    # lanes were refilled: the persistent kernel took every history of every cycle from its queue, far more than it has lanes
    assert r["counters"][13] == 3                      # one persistent launch per cycle
    assert r["counters"][14] == r["counters"][0] > 3 * 2 * REFILL_LANES
    # The fission bank, site by site (same order by construction: sorted by parent, child).  Group exact; directions are
    # fresh isotropic samples: 1e-12.  Positions carry the history's rounding differences (FMA contraction, libm),
    # amplified where a distance is ill-conditioned -- a flight almost parallel to z in these 2-D geometries
    # (d = (p - x) / u_x: a last-bit difference in the numerator is divided by sin(polar angle); z, which no surface
    # bounds, takes all of it) or a near-tangent cylinder crossing (divided by the chord's half-length).  Over ~5e7
    # events per run such events do occur (measured on B200: 99.9 % of the sites within 1e-11, worst
    # x / y 2.5e-10, worst z 3.0e-9), so: at most 0.5 % of the sites beyond 1e-11, none beyond 1e-9 (x, y) / 1e-8 (z).
    bg, bo = g.bank(), o.bank()
    assert len(bg) == len(bo) and len(bo) > REFILL_LANES
    assert (bg["g"] == bo["g"]).all()
    for f in ("ux", "uy", "uz"):
        assert np.abs(bg[f] - bo[f]).max() < 1e-12, f
    for f, worst in (("x", 1e-9), ("y", 1e-9), ("z", 1e-8)):
        d = np.abs(bg[f] - bo[f]) - 1e-9 * np.abs(bo[f])
        assert d.max() < worst, (f, d.max())
        assert (d > 1e-11).mean() < 5e-3, (f, int((d > 1e-11).sum()))
    g.close()


def test_c4_full_k_and_flux(gpu, orc):
    """10^7 x (3 + 6) cycles on the GPU against the oracle at 10^5 x (3 + 6): k within 3 combined sigma, total
    flux per source particle within 4 sigma, leakage tiny and consistent."""
    P = inputs.config4(n_inactive=3, n_active=6)
    g = gpu.Problem(P)
    r = g.run()
    invariants(r)
    Po = inputs.config4(n_particles=100_000, n_inactive=3, n_active=6)  # same cycles: the source is still converging
    rc, ro = orc.Oracle(Po).run()
    # Two runs of different size: the GPU's 10^7 and the oracle's 10^5 particles per cycle.  The difference of their k
    # means has the statistical spread (3 combined sigma of the mean over 6 active cycles) plus the well-known 1/N
    # bias of power iteration with a finite population (source renormalisation, R6), which at N = 10^5 is of order
    # 1/N x (a few hundred) ~ 1e-3 for a loosely coupled core like C4.  The exact-parity check of the same kernels is
    # test_mg_parity_refill_regime; this one only guards the statistics at full size.
    assert abs(r["k_mean"] - ro["k_mean"]) < 3 * math.hypot(r["k_sdev"], ro["k_sdev"]) + 1e-3
    fg, fo = r["flux_mean"].reshape(-1, 7), ro["flux_mean"].reshape(-1, 7)
    tg, to = fg.sum(), fo.sum()
    assert abs(tg - to) / to < 0.01
    # per-group spectrum summed over space
    assert np.allclose(fg.sum(0) / tg, fo.sum(0) / to, atol=3e-3)
    assert r["leak_mean"] < 1e-2
    g.close()


def test_c5_full(gpu, orc):
    """10^6 source particles: sampled source histories identical to the oracle's; flux per time bin within 4 sigma of
    the oracle at 2*10^4 (sigma from 8 independent GPU seeds at that size)."""
    P = inputs.config5()
    g = gpu.Problem(P, search=1)
    g.set_trace(0, 60, 8192)
    r = g.run()
    invariants(r)
    tg = g.trace()
    o = orc.Oracle(P)
    o.set_trace(0, 60, 2_000_000)
    o.run(n_particles=60)
    compare_traces(tg, o.trace())
    g.close()
    n = 20_000
    Ps = inputs.config5(n_particles=n)
    gs = gpu.Problem(Ps, search=1)
    per_t = []
    for seed in range(2, 10):
        rs = gs.run(seed=seed)
        per_t.append(rs["flux_mean"].reshape(10, 100).sum(1))
    gs.close()
    sig = np.std(per_t, axis=0, ddof=1)
    rc, ro = orc.Oracle(Ps).run()
    ft_o = ro["flux_mean"].reshape(10, 100).sum(1)
    ft_g = r["flux_mean"].reshape(10, 100).sum(1)
    assert (np.abs(ft_g - ft_o) < 4 * sig * math.sqrt(1 + n / 1e6) + 1e-12).all()
    # tracks per source history (prompt chain k) agree statistically
    kg = r["counters"][11] / r["counters"][0]
    ko = ro["counters"][11] / ro["counters"][0]
    assert abs(kg - ko) < 0.02


def test_c4_two_level_full_equals_flat(gpu, orc):
    """C4 at 10^7 particles per cycle described as a lattice of assemblies of 17 x 17 pin lattices (R37): the same
    random numbers meet the same geometry, so counters and the fission bank size equal the flat run's, k and the per-pin
    flux agree to rounding; 150 sampled histories equal the oracle's event by event."""
    N = 10_000_000
    gf = gpu.Problem(inputs.config4())
    kf = [gf.run_cycle(N, c, 1, 1) for c in range(2)]
    rf = gf.results()
    nf = gf.dims().bank_count
    gf.close()
    P2 = inputs.config4(two_level=True)
    g2 = gpu.Problem(P2)
    g2.set_trace(77_000, 150, 2048)
    k2 = [g2.run_cycle(N, c, 1, 1) for c in range(2)]
    r2 = g2.results()
    assert g2.dims().bank_count == nf
    assert np.allclose(kf, k2, rtol=1e-10)
    assert (rf["counters"][:12] == r2["counters"][:12]).all()
    assert np.allclose(rf["flux_mean"], r2["flux_mean"], rtol=1e-8, atol=1e-12 * rf["flux_mean"].max())
    invariants(r2)
    tg = g2.trace()
    tg = tg[tg["cycle"] == 0]
    o = orc.Oracle(P2)
    o.set_trace(77_000, 150, 1_000_000)
    o.run(n_particles=77_150, n_inactive=0, n_active=1)
    compare_traces(tg, o.trace())
    g2.close()


def test_td_full_equals_kinetics(gpu):
    """Time-dependent multi-group at 10^6 source particles with the comb on (census_target 5 x 10^5): the flux in every
    time bin and group equals the closed-form kinetics integral of the infinite medium (tests/test_oracle_td.py) within
    5 sigma, sigma from 8 seeds at 10^5; population and weight at every census as the comb prescribes."""
    from tests.test_oracle_td import kinetics_flux
    P = inputs.td_infinite(n_particles=1_000_000, G=2, census_target=500_000)
    ref = kinetics_flux(P)
    g = gpu.Problem(P)
    r = g.run()
    f = r["flux_mean"].reshape(8, 2)
    cen = g.census()
    assert len(cen) == 8 and cen[0][1] == 1_000_000 and all(c[1] == 500_000 for c in cen[1:])
    assert all(abs(c[3] - c[2]) <= 1e-9 * c[2] for c in cen)
    g.close()
    Ps = inputs.td_infinite(n_particles=100_000, G=2, census_target=50_000)
    gs = gpu.Problem(Ps)
    runs = np.array([gs.run(seed=s)["flux_mean"].reshape(8, 2) for s in range(10, 18)])
    gs.close()
    sig = runs.std(0, ddof=1)
    assert (np.abs(runs.mean(0) - ref) < 5 * sig / math.sqrt(8) + 1e-4 * ref).all()
    assert (np.abs(f - ref) < 5 * sig / math.sqrt(10) + 1e-4 * ref).all(), (f, ref, sig)
