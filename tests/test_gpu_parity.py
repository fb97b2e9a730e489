"""GPU parity: the CUDA library (through the C-ABI) against the CPU oracle on the same seeded inputs.

Tolerances (BASELINE.json north_star): per-particle event sequences identical for tiny runs (discrete fields
exact, floats 1e-9), k per cycle and flux within 1e-9 relative in float64 (accumulation order only), k_eff within
3 combined standard deviations on large runs."""
import math

import numpy as np
import pytest

from paper_2501_05440_b200 import inputs

pytestmark = pytest.mark.gpu

ALWAYS = 0x7FFFFFFF  # persist_threshold: the persistent kernel from the first segment on
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


def compare_traces(tg, to, atol=1e-11):
    assert len(tg) == len(to) and len(to) > 0
    kg = np.lexsort((tg["seq"], tg["id"], tg["cycle"]))
    ko = np.lexsort((to["seq"], to["id"], to["cycle"]))
    tg, to = tg[kg], to[ko]
    for f in DISCRETE:
        assert (tg[f] == to[f]).all(), f
    for f in FLOATS:
        assert np.allclose(tg[f], to[f], rtol=1e-9, atol=atol), f


def float_atol(name):
    """Absolute tolerance on positions.  Specular reflection off a CURVED wall amplifies the last-bit differences
    between the two implementations (FMA contraction, libm) along near-tangent multi-bounce paths (a
    direction error e becomes up to ~(1 + 2 L / (r cos theta)) e at a bounce with chord L, radius r and incidence theta;
    dozens of bounces of an ulp-level 1e-16 reach 1e-9): measured worst case 1.2e-9 cm.  The bound is ten times the
    measured worst case (VERDICT r2 finding 2: it was 1e-7 before); tallies and k still agree to 1e-9 relative."""
    return 1e-8 if name.startswith("mirror") else 1e-11


CASES = {
    "C1": lambda: inputs.config1(n_particles=3000, n_inactive=2, n_active=4),
    "C2": lambda: inputs.config2(n_particles=5000, n_inactive=2, n_active=3),
    "C3": lambda: inputs.config3(n_particles=4000, n_inactive=1, n_active=3),
    "C4": lambda: inputs.config4(n_particles=6000, n_inactive=1, n_active=2),
    "C4small": lambda: inputs.config4(n_particles=3001, n_inactive=1, n_active=2, n_asm=1, n_pin=3, n_refl=1),
    "mixed": lambda: inputs.mixed_surfaces(n_particles=4000),
    "C4_3d": lambda: inputs.config4(n_particles=4000, n_inactive=1, n_active=2, n_asm=1, n_pin=4, n_refl=1, height=6.0),
    # fully 3-D cores with an axial reflector (row f1): a z plane inside every pin universe (fuel below, moderator above)
    "C4_3d_axial": lambda: inputs.config4(n_particles=4000, n_inactive=1, n_active=2, n_asm=1, n_pin=4, n_refl=1, height=6.0,
                                         axial_reflector=2.0),
    "C4_2l_3d_axial": lambda: inputs.config4(n_particles=3000, n_inactive=1, n_active=2, n_asm=1, n_pin=4, n_refl=4, two_level=True,
                                            height=6.0, axial_reflector=2.0),
    "lat1x6": lambda: inputs.rect_lattice(1, 6),
    "lat5x1": lambda: inputs.rect_lattice(5, 1),
    "lat3x5": lambda: inputs.rect_lattice(3, 5),
    "mirror_sphere": lambda: inputs.curved_mirror("sphere", n_particles=3000, n_inactive=1, n_active=2),
    "mirror_cyl_z": lambda: inputs.curved_mirror("cyl_z", n_particles=3000, n_inactive=1, n_active=2),
    "mirror_cyl_x": lambda: inputs.curved_mirror("cyl_x", n_particles=3000, n_inactive=1, n_active=2),
    # two-level lattices (R37): assemblies of pin lattices, 2-D and finite height, a homogeneous reflector assembly, an
    # assembly universe with a moderator gap around its pin lattice (surfaces of the cell the inner lattice fills)
    "C4_2l": lambda: inputs.config4(n_particles=4000, n_inactive=1, n_active=2, n_asm=2, n_pin=3, n_refl=3, two_level=True),
    "C4_2l_3d": lambda: inputs.config4(n_particles=3000, n_inactive=1, n_active=2, n_asm=1, n_pin=4, n_refl=4, two_level=True,
                                      height=6.0),
    "C4_2l_homog": lambda: inputs.config4(n_particles=3000, n_inactive=1, n_active=2, n_asm=2, n_pin=3, n_refl=3, two_level=True,
                                         reflector_lattice=False),
    "C4_2l_17": lambda: inputs.config4(n_particles=5000, n_inactive=1, n_active=2, two_level=True),
    "rect_2l": lambda: inputs.two_level_rect(2, 3, 3, 2),
    "rect_2l_1col": lambda: inputs.two_level_rect(1, 2, 1, 4),
    "asm_gap": lambda: inputs.assembly_gap(2, 3),
    "asm_gap_wide": lambda: inputs.assembly_gap(3, 2, gap=0.6),
    "slab": lambda: inputs.slab_beam(n_particles=5000),
    "sphere": lambda: inputs.sphere_absorber(n_particles=5000),
}


SCHEDULES = [(0, 0), (0, -1), (0, ALWAYS), (1, 0), (2, -1), (0, 300), (2, 700)]


@pytest.mark.parametrize("name", list(CASES))
@pytest.mark.parametrize("schedule,persist", SCHEDULES)
def test_mg_parity(gpu, orc, name, schedule, persist):
    """Default schedule, event sweeps only (no persistent kernel), the persistent kernel alone (whole histories in
    registers, lanes refilled from the queue), the monolithic schedule, split per-event kernels, and sweeps handing
    over to the persistent kernel part-way all reproduce the oracle."""
    P = CASES[name]()
    g = gpu.Problem(P, schedule=schedule, persist_threshold=persist)
    r = g.run()
    o = orc.Oracle(P)
    rc, ro = o.run()
    assert rc == 0
    compare_results(r, ro)
    bg, bo = g.bank(), o.bank()
    assert len(bg) == len(bo)
    assert (bg["g"] == bo["g"]).all()
    for f in ("x", "y", "z", "ux", "uy", "uz"):
        assert np.allclose(bg[f], bo[f], rtol=1e-9, atol=float_atol(name)), f
    g.close()


@pytest.mark.parametrize("name", ["C1", "C2", "C3", "C4", "C4small", "mixed", "C4_3d", "C4_3d_axial", "C4_2l_3d_axial", "lat1x6", "lat3x5", "mirror_sphere",
                                  "mirror_cyl_x", "C4_2l", "C4_2l_3d", "C4_2l_homog", "asm_gap", "asm_gap_wide", "rect_2l", "rect_2l_1col"])
@pytest.mark.parametrize("schedule,persist", [(0, -1), (0, 0), (1, 0), (2, -1), (0, 100)])
def test_mg_traces_identical(gpu, orc, name, schedule, persist):
    """100 particles x 2 cycles: identical per-particle event sequences (SURVEY.md 8d parity protocol 1)."""
    P = CASES[name]()
    N = 1000
    g = gpu.Problem(P, max_particles=N, schedule=schedule, persist_threshold=persist)
    g.set_trace(0, 100, 1024)
    r = g.run(n_particles=N, n_inactive=0, n_active=2)
    o = orc.Oracle(P)
    o.set_trace(0, 100, 400000)
    rc, ro = o.run(n_particles=N, n_inactive=0, n_active=2)
    compare_traces(g.trace(), o.trace(), atol=float_atol(name))
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


@pytest.mark.parametrize("height,axial", [(None, None), (3.0, None), (3.0, 1.0)])
def test_geometry_unit_parity(gpu, orc, height, axial):
    P = inputs.config4(n_particles=1000, height=height, axial_reflector=axial)
    g = gpu.Problem(P, max_particles=20000)
    o = orc.Oracle(P)
    rng = np.random.default_rng(5)
    n = 4000
    side = 51 * 1.26
    x = np.column_stack([rng.uniform(0, side, n), rng.uniform(0, side, n), rng.uniform(0, 1, n) * (height or 1.0)])
    x[: n // 4, 0] = rng.uniform(0, 1.26, n // 4)           # edge elements: the enclosing cell's planes matter there
    x[n // 4: n // 2, 1] = rng.uniform(50 * 1.26, side, n // 4)
    mu, phi = rng.uniform(-1, 1, n), rng.uniform(0, 2 * np.pi, n)
    s = np.sqrt(1 - mu * mu)
    u = np.column_stack([s * np.cos(phi), s * np.sin(phi), mu])
    # all three device paths: straight-line / pruned list as the kernels choose, generic loops with the pruned list of
    # the enclosing cell's surfaces, generic loops over every surface
    res = [g.geometry(x, u, path=k) for k in (0, 1, 2)]
    for i in range(n):
        rc, lo = o.locate(x[i], u[i])
        d, sh = o.distance(x[i], u[i], lo)
        for loc, dist, surf in res:
            assert rc == 0 and tuple(lo) == tuple(loc[i])
            assert sh == surf[i] and dist[i] == pytest.approx(d, rel=1e-13)
    g.close()


@pytest.mark.parametrize("name", ["C1", "C3", "mixed", "mirror_cyl_z", "lat3x5", "C4_2l", "C4_2l_3d", "C4_3d_axial", "C4_2l_3d_axial",
                                  "asm_gap", "C4_2l_17", "rect_2l"])
def test_geometry_unit_parity_plain_cells(gpu, orc, name):
    """Cells outside a lattice (box, pin cell: straight-line path; mixed surfaces: generic loops) and a small lattice:
    locate + nearest boundary of random points, every device path against the oracle."""
    P = CASES[name]()
    g = gpu.Problem(P, max_particles=20000)
    o = orc.Oracle(P)
    rng = np.random.default_rng(11)
    n = 3000
    lo, hi = np.array(P["src_lo"], float), np.array(P["src_hi"], float)
    hi = np.where(hi > lo, hi, lo + 1.0)
    x = lo + rng.uniform(0, 1, (n, 3)) * (hi - lo)
    mu, phi = rng.uniform(-1, 1, n), rng.uniform(0, 2 * np.pi, n)
    sq = np.sqrt(1 - mu * mu)
    u = np.column_stack([sq * np.cos(phi), sq * np.sin(phi), mu])
    res = [g.geometry(x, u, path=k) for k in (0, 1, 2)]
    for i in range(n):
        rc, lo_ = o.locate(x[i], u[i])
        d, sh = o.distance(x[i], u[i], lo_)
        for loc, dist, surf in res:
            assert rc == 0 and tuple(lo_) == tuple(loc[i])
            assert sh == surf[i] and (dist[i] == pytest.approx(d, rel=1e-12) or (np.isinf(d) and np.isinf(dist[i])))
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


def test_bank_overflow_and_lost_particle_errors(gpu, orc):
    """R6: more than 2N fission sites is MCDC_EBANK and leaves the problem usable; a source box that is not inside
    the geometry is MCDC_EGEOM at create; a failed run leaves the last successful run's results readable."""
    P = inputs.config1(n_particles=2000, n_inactive=1, n_active=2)
    g = gpu.Problem(P)
    good = g.run()
    # cycle 0 of a new run samples 2000 source particles as before; then feed a cycle more particles than it can bank
    with pytest.raises(gpu.McdcError) as e:
        g.run(n_particles=5000)  # exceeds the capacity the problem was created for: refused before any device work
    assert e.value.code == -1
    after = g.results()
    assert (after["k_cycle"] == good["k_cycle"]).all() and (after["flux_mean"] == good["flux_mean"]).all()
    g.close()
    P2 = inputs.config1(n_particles=2000, n_inactive=0, n_active=2)
    P2["mg_nu"] = P2["mg_nu"] * 4.0  # k_inf = 5.2: the first cycle banks about 5 N sites
    g = gpu.Problem(P2)
    with pytest.raises(gpu.McdcError) as e:
        g.run()
    assert e.value.code == -3
    assert g.dims().n_cycles == 0  # nothing was published
    r = g.run(n_particles=300, n_inactive=0, n_active=1)  # 300 x 5.2 sites fit: the problem is still usable
    assert r["counters"][0] == 300 and len(r["k_cycle"]) == 1
    with pytest.raises(gpu.McdcError):
        g.run()
    again = g.results()  # the failed run did not touch what the last good one published
    assert (again["k_cycle"] == r["k_cycle"]).all() and (again["flux_mean"] == r["flux_mean"]).all()
    assert (again["counters"] == r["counters"]).all()
    g.close()
    P = inputs.config1(n_particles=500, n_inactive=0, n_active=1)
    P["src_hi"] = np.array([1.5, 1.0, 1.0])  # a third of the source box lies outside the cube
    with pytest.raises(gpu.McdcError) as e:
        gpu.Problem(P)
    assert e.value.code == -2


def test_segment_guard(gpu, orc):
    """R11: a history that never ends (pure scatterer in a reflecting box) is cut at 10^6 segments with MCDC_ELOST;
    the oracle reports the same error and the same number of events."""
    P = inputs.config1(n_particles=3, n_inactive=0, n_active=1)
    P["mg_S"] = P["mg_sig_t"].reshape(1, 1, 1).copy()  # Sigma_s = Sigma_t: nothing absorbs
    P["mg_sig_f"] = P["mg_sig_f"] * 0.0
    o = orc.Oracle(P)
    rc, ro = o.run()
    assert rc == -4 and ro["counters"][10] == 3
    g = gpu.Problem(P, persist_threshold=ALWAYS)
    with pytest.raises(gpu.McdcError) as e:
        g.run()
    assert e.value.code == -4
    g.close()


def test_two_level_equals_flat_on_gpu(gpu):
    """The same quarter core as one flat lattice (straight-line geometry path) and as a lattice of lattices (generic
    path): identical event counters and fission bank, k per cycle and per-pin flux to rounding."""
    kw = dict(n_particles=20000, n_inactive=1, n_active=2)
    gf = gpu.Problem(inputs.config4(**kw))
    g2 = gpu.Problem(inputs.config4(two_level=True, **kw))
    rf, r2 = gf.run(), g2.run()
    assert np.allclose(rf["k_cycle"], r2["k_cycle"], rtol=1e-11)
    assert (rf["counters"][:12] == r2["counters"][:12]).all()
    assert np.allclose(rf["flux_mean"], r2["flux_mean"], rtol=1e-9, atol=1e-13 * rf["flux_mean"].max())
    bf, b2 = gf.bank(), g2.bank()
    assert len(bf) == len(b2) and (bf["g"] == b2["g"]).all() and np.allclose(bf["x"], b2["x"], rtol=0, atol=1e-10)
    gf.close()
    g2.close()


def test_two_level_validation(gpu):
    P = inputs.assembly_gap(2, 3)
    for key, val in (("lat2_off", np.array([0, 8], np.int32)), ("lat2_univ", np.full(9, 3, np.int32)),
                     ("lat2_bin", np.full(9, 10_000, np.int32)), ("lat2_nx", np.array([0], np.int32))):
        bad = dict(P)
        bad[key] = val
        with pytest.raises(gpu.McdcError) as e:
            gpu.Problem(bad)
        assert e.value.code in (-1, -2), key
    bad = dict(P)
    bad["cell_fill"] = P["cell_fill"].copy()
    bad["cell_fill"][P["cell_fill_type"] == 2] = 1  # names a second-level lattice that does not exist
    with pytest.raises(gpu.McdcError) as e:
        gpu.Problem(bad)
    assert e.value.code == -2


def test_validation_errors(gpu):
    P = inputs.rect_lattice(3, 2)
    bad = dict(P)
    bad["cell_bin"] = P["cell_bin"].copy()
    bad["cell_bin"][1:] = 1  # cell_bin + max lat_bin reaches n_bins
    with pytest.raises(gpu.McdcError) as e:
        gpu.Problem(bad)
    assert e.value.code == -1
    bad = dict(P)
    bad["univ_cell_off"] = P["univ_cell_off"].copy()
    bad["univ_cell_off"][-1] += 1
    with pytest.raises(gpu.McdcError) as e:
        gpu.Problem(bad)
    assert e.value.code == -1
