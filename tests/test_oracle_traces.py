"""Event-sequence and geometry pins of the oracle by brute force on tiny inputs (no GPU).
SURVEY.md 8(c): "independent tiny Python tracer ... for the first <= 100 histories of C1 and C3" and
"brute-force geometry: distance/next-cell from the fast path vs min over all surfaces / point-in-cell"."""
import math

import numpy as np
import pytest

from paper_2501_05440_b200 import inputs
from tests import brute_tracer


def _compare(orc, P, n_hist, N):
    o = orc.Oracle(P)
    o.set_trace(0, n_hist, 200000)
    rc, _ = o.run(n_particles=N, n_inactive=0, n_active=1)
    assert rc == 0
    tr = o.trace()
    tr = tr[tr["cycle"] == 0]
    ref = brute_tracer.trace_cycle0(P, P["run"]["seed"], n_hist)
    assert len(tr) == len(ref) and len(ref) >= n_hist
    for a, b in zip(tr, ref):
        assert (int(a["id"]), int(a["seq"]), int(a["ev"]), int(a["surf"]), int(a["gi"])) == b[:5]
        assert (int(a["elem"]), int(a["c1"])) == b[9:11]
        assert a["x"] == pytest.approx(b[5], abs=1e-11) and a["y"] == pytest.approx(b[6], abs=1e-11)
        assert a["z"] == pytest.approx(b[7], abs=1e-9) and a["d"] == pytest.approx(b[8], rel=1e-9, abs=1e-12)
    return tr


def test_trace_c1_vs_brute_force(orc):
    _compare(orc, inputs.config1(), 100, 100)


def test_trace_c3_vs_brute_force(orc):
    _compare(orc, inputs.config3(), 100, 100)


def test_trace_sphere_and_slab_vs_brute_force(orc):
    _compare(orc, inputs.sphere_absorber(n_particles=60), 60, 60)
    P = inputs.slab_beam(n_particles=60)
    _compare(orc, P, 60, 60)


def test_trace_all_surface_types_vs_brute_force(orc):
    """PLANE, PLANE_Z, SPHERE, CYL_X, CYL_Y, reflect + vacuum + transmit in one geometry, incl. reflections off the
    general plane x + y + z = 5 (surface 10: non-axis branch of the oracle's reflect())."""
    tr = _compare(orc, inputs.mixed_surfaces(), 400, 400)
    assert ((tr["ev"] == 5) & (tr["surf"] == 10)).sum() >= 5


@pytest.mark.parametrize("kind", ["sphere", "cyl_z", "cyl_x", "cyl_y"])
def test_trace_curved_mirrors_vs_brute_force(orc, kind):
    """Specular reflection off a sphere and off cylinders along each axis (non-axis branch of reflect(): normal
    from the gradient, Omega' = Omega - 2 (Omega.n) n), event by event against the brute-force tracer."""
    tr = _compare(orc, inputs.curved_mirror(kind), 120, 120)
    curved = 0  # the reflecting quadric is surface 0 in geom_mirror
    assert ((tr["ev"] == 5) & (tr["surf"] == curved)).sum() >= 100


@pytest.mark.parametrize("case", ["C4small", "C4_3d", "C4_3d_axial", "lat1x6", "lat5x1", "lat3x5", "C4edge"])
def test_trace_lattice_vs_brute_force(orc, case):
    """One-level lattices, event by event (incl. element and local cell of every event): the oracle's neighbour /
    wall-ahead logic (R14) against brute force over every grid line and every pin of the lattice."""
    P = dict(C4small=lambda: inputs.config4(n_particles=60, n_asm=1, n_pin=3, n_refl=1),
             C4_3d=lambda: inputs.config4(n_particles=60, n_asm=1, n_pin=4, n_refl=1, height=6.0),
             C4_3d_axial=lambda: inputs.config4(n_particles=60, n_asm=1, n_pin=4, n_refl=1, height=6.0, axial_reflector=2.0),
             lat1x6=lambda: inputs.rect_lattice(1, 6), lat5x1=lambda: inputs.rect_lattice(5, 1),
             lat3x5=lambda: inputs.rect_lattice(3, 5),
             C4edge=lambda: inputs.config4(n_particles=40, n_asm=2, n_pin=5, n_refl=2))[case]()
    tr = _compare(orc, P, 60, 60)
    assert (tr["ev"] == 7).sum() >= 50  # lattice-wall events
    if case == "C4_3d_axial":  # the plane between fuel and axial reflector (the last surface) was crossed from all three
        zf = len(P["surf_type"]) - 1          # cells of a pin universe: fuel, the moderator beside it, the reflector above
        hit = tr[(tr["ev"] == 4) & (tr["surf"] == zf)]
        assert len(hit) >= 20 and len(set(int(c) for c in hit["c1"])) >= 3


def _compare_ce(orc, P, n_src):
    """CE time-dependent fixed source: source histories event by event, integer event counters of ALL tracks (source
    particles and every prompt secondary below them) and the (time bin x energy bin) flux tally."""
    o = orc.Oracle(P)
    o.set_trace(0, n_src, 2_000_000)
    rc, r = o.run(n_particles=n_src)
    assert rc == 0
    tr = o.trace()
    ev, cnt, flux = brute_tracer.trace_ce(P, P["run"]["seed"], n_src)
    assert len(tr) == len(ev) and len(ev) >= n_src
    for a, b in zip(tr, ev):
        assert (int(a["id"]), int(a["seq"]), int(a["ev"]), int(a["surf"]), int(a["gi"])) == b[:5]
        for k, f in enumerate(("x", "y", "z", "d", "E", "t")):
            assert a[f] == pytest.approx(b[5 + k], rel=1e-9, abs=1e-11), f
    assert [int(v) for v in r["counters"][:12]] == cnt[:12]
    got = r["flux_mean"].reshape(len(flux), -1) * n_src
    want = np.array(flux)
    assert np.allclose(got, want, rtol=1e-9, atol=1e-13 * want.max())
    return tr, r


def test_trace_ce_c5_vs_brute_force(orc):
    """C5 (pin cell, 5 nuclides, resonances, Watt fission, 10 time x 100 energy bins): 25 source histories and their
    whole prompt-fission families against the pure-Python tracer.  Pins, inside the transport loop: the column ->
    nuclide map of the elastic branch, the energy clamp, t += d / v, the time-edge logic, edge_bin() over 100 bins
    (every track length lands in the bin numpy-style bisection names), secondaries' ids and streams."""
    P = inputs.config5(n_particles=25, n_grid=3000)
    tr, r = _compare_ce(orc, P, 25)
    assert r["counters"][11] > 10 and (tr["ev"] == 8).sum() > 5


def test_trace_ce_jittered_grid_and_light_nuclide(orc):
    P = inputs.config5(n_particles=12, n_grid=1500, jitter=True)
    _compare_ce(orc, P, 12)
    P = inputs.ce_two_nuclide_mix(n_particles=15, n_grid=800)
    _compare_ce(orc, P, 15)


def test_geometry_brute_force_quarter_core(orc):
    """Lattice fast path (element walls + local cell + enclosing cell) vs brute force: the distance returned
    must be the smallest positive distance to ANY pin cylinder / lattice line / outer plane along the ray that
    actually bounds the current region, and the midpoint of the segment must lie in the same element/cell."""
    P = inputs.config4(n_particles=10, n_asm=1, n_pin=3, n_refl=2)
    o = orc.Oracle(P)
    lat = P["lat"]
    n, p, r = lat["nx"], lat["px"], 0.54
    rng = np.random.default_rng(8)
    for _ in range(3000):
        x = np.array([rng.uniform(0, n * p), rng.uniform(0, n * p), rng.uniform(-1, 1)])
        mu, phi = rng.uniform(-1, 1), rng.uniform(0, 2 * np.pi)
        u = np.array([math.sqrt(1 - mu * mu) * math.cos(phi), math.sqrt(1 - mu * mu) * math.sin(phi), mu])
        rc, loc = o.locate(x, u)
        assert rc == 0
        ix, iy = int(x[0] // p), int(x[1] // p)
        assert loc[1] == iy * n + ix
        univ = lat["univ"][iy, ix]
        cx, cy = (ix + 0.5) * p, (iy + 0.5) * p
        inside = (x[0] - cx) ** 2 + (x[1] - cy) ** 2 < r * r
        c_lo = P["univ_cell_off"][univ]
        assert loc[2] == (c_lo if (inside or univ == 7) else c_lo + 1)
        d, s = o.distance(x, u, loc)
        # brute force: all grid lines (incl. the outer planes) and this element's cylinder
        cands = []
        for ax in (0, 1):
            if u[ax] != 0:
                for kk in range(n + 1):
                    t = (kk * p - x[ax]) / u[ax]
                    if t > 0:
                        cands.append(t)
        if univ != 7:
            a = u[0] ** 2 + u[1] ** 2
            k = (x[0] - cx) * u[0] + (x[1] - cy) * u[1]
            c = (x[0] - cx) ** 2 + (x[1] - cy) ** 2 - r * r
            disc = k * k - a * c
            if a > 0 and disc >= 0:
                cands += [t for t in ((-k - math.sqrt(disc)) / a, (-k + math.sqrt(disc)) / a) if t > 0]
        assert d == pytest.approx(min(cands), rel=1e-12)
        # midpoint stays in the same element and cell
        rc2, loc2 = o.locate(x + 0.5 * d * u, u)
        assert rc2 == 0 and tuple(loc2) == tuple(loc)
        # surface id class: outer plane / cylinder -> real surface (< n_surf); inner wall -> n_surf + k
        ns = len(P["surf_type"])
        xe = x + d * u
        on_outer = min(abs(xe[0]), abs(xe[1]), abs(xe[0] - n * p), abs(xe[1] - n * p)) < 1e-9
        on_cyl = univ != 7 and abs(math.hypot(xe[0] - cx, xe[1] - cy) - r) < 1e-9
        if on_outer:
            assert s < 4
        elif on_cyl:
            assert s == 4
        else:
            assert s >= ns


def test_last_surface_logic(orc):
    """R11/R13: a particle sitting on a surface never re-hits it at d = 0: planes are skipped, quadrics give
    only the far root and only when heading inward."""
    P = inputs.config3()
    o = orc.Oracle(P)
    cyl = 4
    x = np.array([0.54, 0.0, 0.0])
    inward = np.array([-1.0, 0.0, 0.0])
    rc, loc = o.locate(x, inward, last_surf=cyl)
    assert rc == 0 and loc[0] == 0  # entering the fuel
    d, s = o.distance(x, inward, loc, last_surf=cyl)
    assert s == cyl and d == pytest.approx(1.08, rel=1e-14)
    outward = -inward
    rc, loc = o.locate(x, outward, last_surf=cyl)
    assert rc == 0 and loc[0] == 1  # entering the moderator
    d, s = o.distance(x, outward, loc, last_surf=cyl)
    assert s == 1 and d == pytest.approx(0.09, rel=1e-12)  # the +x plane, not the cylinder
    # on the +x plane after a reflection: that plane is skipped
    x = np.array([0.63, 0.1, 0.0])
    u = np.array([-0.6, 0.8, 0.0])
    rc, loc = o.locate(x, u, last_surf=1)
    d, s = o.distance(x, u, loc, last_surf=1)
    assert s != 1 and d > 0.05
    # tangent / miss: ray in the moderator passing outside the cylinder
    x = np.array([-0.6, 0.58, 0.0])
    u = np.array([1.0, 0.0, 0.0])
    rc, loc = o.locate(x, u)
    d, s = o.distance(x, u, loc)
    assert s == 1 and d == pytest.approx(1.23, rel=1e-12)
