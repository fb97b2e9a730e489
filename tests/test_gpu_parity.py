"""GPU parity: the CUDA library (through the C-ABI) against the CPU oracle on the same seeded inputs.

Tolerances (BASELINE.json north_star): per-particle event sequences identical for tiny runs (discrete fields
exact, floats 1e-9), k per cycle and flux within 1e-9 relative in float64 (accumulation order only), k_eff within
3 combined standard deviations on large runs."""
import math

import numpy as np
import pytest

from paper_2501_05440_b200 import inputs

pytestmark = pytest.mark.gpu

DISCRETE = ["id", "cycle", "seq", "ev", "c0", "elem", "c1", "surf", "gi"]
FLOATS = ["x", "y", "z", "d", "E", "t"]


@pytest.fixture(scope="module")
def gpu():
    from paper_2501_05440_b200 import binding
    binding.load_library()
    return binding


def compare_results(r, ro, rtol=1e-9):
    assert np.allclose(r["k_cycle"], ro["k_cycle"], rtol=rtol, atol=0), (r["k_cycle"], ro["k_cycle"])
    scale = np.abs(ro["flux_mean"]).max()
    assert np.allclose(r["flux_mean"], ro["flux_mean"], rtol=rtol, atol=1e-13 * scale)
    assert np.allclose(r["flux_sdev"], ro["flux_sdev"], rtol=1e-5, atol=1e-9 * scale)
    assert r["k_mean"] == pytest.approx(ro["k_mean"], rel=rtol)
    assert r["leak_mean"] == pytest.approx(ro["leak_mean"], rel=rtol, abs=1e-300)
    assert (r["counters"][:12] == ro["counters"][:12]).all(), (r["counters"], ro["counters"])


def compare_traces(tg, to):
    assert len(tg) == len(to) and len(to) > 0
    kg = np.lexsort((tg["seq"], tg["id"], tg["cycle"]))
    ko = np.lexsort((to["seq"], to["id"], to["cycle"]))
    tg, to = tg[kg], to[ko]
    for f in DISCRETE:
        assert (tg[f] == to[f]).all(), f
    for f in FLOATS:
        assert np.allclose(tg[f], to[f], rtol=1e-9, atol=1e-11), f


CASES = {
    "C1": lambda: inputs.config1(n_particles=3000, n_inactive=2, n_active=4),
    "C2": lambda: inputs.config2(n_particles=5000, n_inactive=2, n_active=3),
    "C3": lambda: inputs.config3(n_particles=4000, n_inactive=1, n_active=3),
    "C4": lambda: inputs.config4(n_particles=6000, n_inactive=1, n_active=2),
    "C4small": lambda: inputs.config4(n_particles=3001, n_inactive=1, n_active=2, n_asm=1, n_pin=3, n_refl=1),
    "mixed": lambda: inputs.mixed_surfaces(n_particles=4000),
    "C4_3d": lambda: inputs.config4(n_particles=4000, n_inactive=1, n_active=2, n_asm=1, n_pin=4, n_refl=1, height=6.0),
    "slab": lambda: inputs.slab_beam(n_particles=5000),
    "sphere": lambda: inputs.sphere_absorber(n_particles=5000),
}


@pytest.mark.parametrize("name", list(CASES))
@pytest.mark.parametrize("schedule,tail,fuse", [(0, 0, 0), (0, -1, -1), (0, 1 << 30, 0), (1, 0, 0), (0, -1, 1 << 30), (0, 300, 2000)])
def test_mg_parity(gpu, orc, name, schedule, tail, fuse):
    """Default schedule, pure per-event kernels (no tail, no fused sweeps), tail-only (histories in registers),
    the monolithic schedule, fused sweeps only, and a mix of all three stages all reproduce the oracle."""
    P = CASES[name]()
    g = gpu.Problem(P, schedule=schedule, tail_threshold=tail, fuse_threshold=fuse, fuse_segments=3)
    r = g.run()
    o = orc.Oracle(P)
    rc, ro = o.run()
    assert rc == 0
    compare_results(r, ro)
    bg, bo = g.bank(), o.bank()
    assert len(bg) == len(bo)
    assert (bg["g"] == bo["g"]).all()
    for f in ("x", "y", "z", "ux", "uy", "uz"):
        assert np.allclose(bg[f], bo[f], rtol=1e-9, atol=1e-11), f
    g.close()


@pytest.mark.parametrize("name", ["C1", "C2", "C3", "C4", "C4small", "mixed", "C4_3d"])
@pytest.mark.parametrize("schedule,tail,fuse", [(0, -1, -1), (0, 0, 0), (1, 0, 0), (0, 100, 500)])
def test_mg_traces_identical(gpu, orc, name, schedule, tail, fuse):
    """100 particles x 2 cycles: identical per-particle event sequences (SURVEY.md 8d parity protocol 1)."""
    P = CASES[name]()
    N = 1000
    g = gpu.Problem(P, max_particles=N, schedule=schedule, tail_threshold=tail, fuse_threshold=fuse)
    g.set_trace(0, 100, 1024)
    r = g.run(n_particles=N, n_inactive=0, n_active=2)
    o = orc.Oracle(P)
    o.set_trace(0, 100, 400000)
    rc, ro = o.run(n_particles=N, n_inactive=0, n_active=2)
    compare_traces(g.trace(), o.trace())
    compare_results(r, ro)
    g.close()


def test_run_cycle_matches_run_eigenvalue(gpu, orc):
    P = CASES["C3"]()
    g = gpu.Problem(P)
    ks = [g.run_cycle(4000, c, c >= 1, 1) for c in range(4)]
    r = g.results()
    o = orc.Oracle(P)
    rc, ro = o.run()
    assert np.allclose(ks, ro["k_cycle"], rtol=1e-9)
    compare_results(r, ro)
    g.close()


def test_run_cycle_host_roundtrip(gpu, orc):
    """Host-buffer cycle: bank out of cycle c fed back as the source of cycle c+1 reproduces the in-device run."""
    P = CASES["C3"]()
    N = 4000
    g = gpu.Problem(P)
    sites = np.zeros(2 * N + 1024, gpu.SITE_DTYPE)
    flux = np.zeros(g.n_tally)
    k, leak, n = g.run_cycle_host(N, 0, 1, 1.0, None, sites, flux)
    ks = [k]
    for c in range(1, 4):
        src = sites[:n].copy()
        k, leak, n = g.run_cycle_host(N, c, 1, ks[-1], src, sites, flux)
        ks.append(k)
    o = orc.Oracle(P)
    rc, ro = o.run(n_inactive=0, n_active=4)
    assert np.allclose(ks, ro["k_cycle"], rtol=1e-9)
    bo = o.bank()
    assert n == len(bo) and np.allclose(sites["x"][:n], bo["x"], rtol=1e-9, atol=1e-11)
    g.close()


def test_rng_bit_exact(gpu, orc):
    P = CASES["C1"]()
    g = gpu.Problem(P, max_particles=20000)
    rng = np.random.default_rng(0)
    ids = rng.integers(0, 2 ** 63, 5000, dtype=np.uint64)
    ids[:10] = np.arange(10)
    idx = rng.integers(0, 1000, 5000).astype(np.uint32)
    for dom, cyc, seed in ((0, 0, 1), (0, 7, 0xDEADBEEFCAFEF00D), (1, 3, 42)):
        got = g.draws(seed, dom, cyc, ids, idx)
        ref = np.array([orc.draw(seed, int(i), dom, cyc, int(j)) for i, j in zip(ids, idx)])
        assert (got == ref).all()
    g.close()


def test_geometry_unit_parity(gpu, orc):
    P = inputs.config4(n_particles=1000)
    g = gpu.Problem(P, max_particles=20000)
    o = orc.Oracle(P)
    rng = np.random.default_rng(5)
    n = 4000
    side = 51 * 1.26
    x = np.column_stack([rng.uniform(0, side, n), rng.uniform(0, side, n), rng.uniform(-1, 1, n)])
    mu, phi = rng.uniform(-1, 1, n), rng.uniform(0, 2 * np.pi, n)
    s = np.sqrt(1 - mu * mu)
    u = np.column_stack([s * np.cos(phi), s * np.sin(phi), mu])
    loc, dist, surf = g.geometry(x, u)
    for i in range(n):
        rc, lo = o.locate(x[i], u[i])
        assert rc == 0 and tuple(lo) == tuple(loc[i])
        d, sh = o.distance(x[i], u[i], lo)
        assert sh == surf[i] and dist[i] == pytest.approx(d, rel=1e-13)
    g.close()


def test_empty_and_error_paths(gpu):
    P = CASES["C1"]()
    g = gpu.Problem(P, max_particles=100)
    with pytest.raises(gpu.McdcError) as e:
        g.run(n_particles=1000)
    assert e.value.code == -1
    r = g.run(n_particles=1, n_inactive=0, n_active=1)  # one particle: ragged single thread
    assert r["counters"][0] == 1
    g.close()
    bad = dict(P)
    bad["mg_sig_t"] = P["mg_sig_t"] * 0.5  # Sigma_s + Sigma_f > Sigma_t
    with pytest.raises(gpu.McdcError):
        gpu.Problem(bad)
    # vacuum everywhere, pure absorber, bank empties -> EBANK on the next cycle
    P2 = inputs.slab_beam(n_particles=100)
    g2 = gpu.Problem(P2)
    with pytest.raises(gpu.McdcError) as e:
        g2.run(n_inactive=0, n_active=2)
    assert e.value.code == -3
    g2.close()


def test_bank_overflow_and_lost_particle_errors(gpu):
    """R6: more than 2N fission sites is MCDC_EBANK; a source point in no cell is MCDC_EGEOM; both leave the
    problem usable for a later valid run."""
    P = inputs.config1(n_particles=2000, n_inactive=0, n_active=2)
    P["mg_nu"] = P["mg_nu"] * 4.0  # k_inf = 5.2: the first cycle banks about 5 N sites
    g = gpu.Problem(P)
    with pytest.raises(gpu.McdcError) as e:
        g.run()
    assert e.value.code == -3
    g.close()
    P = inputs.config1(n_particles=500, n_inactive=0, n_active=1)
    P["src_hi"] = np.array([1.5, 1.0, 1.0])  # a third of the source box lies outside the cube
    g = gpu.Problem(P)
    with pytest.raises(gpu.McdcError) as e:
        g.run()
    assert e.value.code == -2
    g.close()
