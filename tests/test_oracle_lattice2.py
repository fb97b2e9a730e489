"""Pins of the oracle's two-level lattices (the multi-group benchmark is a core of
assemblies of pin lattices; R37) -- no GPU.  Two independent checks: (1) the same physical core described
as ONE flat lattice and as a lattice of lattices must give the same histories, event for event; (2) the brute-force
tracer (every grid line of both levels, every pin of every assembly, no neighbour logic)."""
import numpy as np
import pytest

from paper_2501_05440_b200 import inputs
from tests import brute_tracer
from tests.test_oracle_traces import _compare


def _flat_elem(packed, n_outer, n_pin):
    """flat-lattice element index of a two-level (outer | (inner + 1) << 20) location"""
    outer, inner = packed & 0xFFFFF, (packed >> 20) - 1
    ax, ay = outer % n_outer, outer // n_outer
    px, py = inner % n_pin, inner // n_pin
    return (ay * n_pin + py) * (n_outer * n_pin) + ax * n_pin + px


@pytest.mark.parametrize("n_asm,n_pin,n_refl,height,axial", [(2, 3, 3, None, None), (1, 4, 4, 6.0, None), (2, 5, 5, None, None),
                                                              (1, 3, 3, 6.0, 2.0)])
def test_two_level_equals_flat_lattice(orc, n_asm, n_pin, n_refl, height, axial):
    """A core of (n_asm + 1)^2 assemblies of n_pin^2 pins, flat (one lattice) and two-level: identical k per cycle,
    event counters and fission bank; per-pin flux to rounding; and the traced histories agree event by event once the
    two-level locations and wall codes are mapped to the flat ones (second-level wall n_surf+4+w and first-level wall
    n_surf+w are both flat wall n_surf+w)."""
    kw = dict(n_particles=1500, n_inactive=1, n_active=2, n_asm=n_asm, n_pin=n_pin, n_refl=n_refl, height=height,
              axial_reflector=axial)
    Pf, P2 = inputs.config4(**kw), inputs.config4(two_level=True, **kw)
    assert "lat2_nx" in P2 and "lat2_nx" not in Pf
    of, o2 = orc.Oracle(Pf), orc.Oracle(P2)
    of.set_trace(0, 150, 400000)
    o2.set_trace(0, 150, 400000)
    rcf, rf = of.run()
    rc2, r2 = o2.run()
    assert rcf == 0 and rc2 == 0
    assert np.allclose(rf["k_cycle"], r2["k_cycle"], rtol=1e-12)
    assert (rf["counters"][:13] == r2["counters"][:13]).all()
    assert np.allclose(rf["flux_mean"], r2["flux_mean"], rtol=1e-10, atol=1e-14)
    bf, b2 = of.bank(), o2.bank()
    assert len(bf) == len(b2) and (bf["g"] == b2["g"]).all()
    assert np.allclose(bf["x"], b2["x"], rtol=0, atol=1e-11) and np.allclose(bf["ux"], b2["ux"], rtol=0, atol=1e-11)
    tf, t2 = of.trace(), o2.trace()
    assert len(tf) == len(t2) > 1000
    ns = len(Pf["surf_type"])
    n_outer = n_asm + n_refl // n_pin
    for a, b in zip(tf, t2):
        assert (a["id"], a["cycle"], a["seq"], a["ev"], a["gi"], a["c1"]) == (b["id"], b["cycle"], b["seq"], b["ev"], b["gi"], b["c1"])
        sb = int(b["surf"])
        assert int(a["surf"]) == (ns + (sb - ns) % 4 if sb >= ns else sb)
        assert int(a["elem"]) == _flat_elem(int(b["elem"]), n_outer, n_pin)
        assert abs(a["x"] - b["x"]) < 1e-11 and abs(a["y"] - b["y"]) < 1e-11 and abs(a["d"] - b["d"]) < 1e-11
    lat = t2[t2["ev"] == 7]
    assert (lat["surf"] >= ns + 4).sum() > 200 and (lat["surf"] < ns + 4).sum() > 20  # walls of both levels were crossed


@pytest.mark.parametrize("case", ["core2l", "core2l_3d", "core2l_3d_axial", "gap", "gap_wide", "core2l_homog_reflector", "rect", "rect_1col"])
def test_trace_two_level_vs_brute_force(orc, case):
    """Two-level lattices event by event (packed element, local cell, wall codes of both levels, surfaces of the cell
    the inner lattice fills) against brute force over all grid lines and all pins."""
    P = dict(core2l=lambda: inputs.config4(n_particles=50, n_asm=1, n_pin=3, n_refl=3, two_level=True),
             core2l_3d=lambda: inputs.config4(n_particles=40, n_asm=2, n_pin=2, n_refl=2, two_level=True, height=5.0),
             core2l_3d_axial=lambda: inputs.config4(n_particles=40, n_asm=2, n_pin=2, n_refl=2, two_level=True, height=5.0,
                                                    axial_reflector=1.5),
             gap=lambda: inputs.assembly_gap(2, 3), gap_wide=lambda: inputs.assembly_gap(3, 2, gap=0.6),
             rect=lambda: inputs.two_level_rect(2, 3, 3, 2), rect_1col=lambda: inputs.two_level_rect(1, 2, 1, 4),
             core2l_homog_reflector=lambda: inputs.config4(n_particles=50, n_asm=1, n_pin=3, n_refl=3, two_level=True,
                                                           reflector_lattice=False))[case]()
    tr = _compare(orc, P, 50, 50)
    ns = len(P["surf_type"])
    assert ((tr["ev"] == 7) & (tr["surf"] >= ns + 4)).sum() >= 30 and ((tr["ev"] == 7) & (tr["surf"] < ns + 4)).sum() >= 5
    assert (tr["elem"] >> 20).max() >= 1
    if case.startswith("gap"):
        mid = {5, 6, 7, 8}  # the four planes that bound the pin lattice inside the assembly
        assert np.isin(tr["surf"][tr["ev"] == 4], list(mid)).sum() >= 20


def test_two_level_uniform_core_flat_flux(orc):
    """All materials identical, all faces reflecting: the two-level core is an infinite homogeneous medium: k = the
    dense 7-group eigenvalue (1.2 by construction) and a flat per-pin flux."""
    P = inputs.config4(n_particles=30000, n_inactive=3, n_active=8, n_asm=1, n_pin=2, n_refl=2, uniform=True, two_level=True)
    o = orc.Oracle(P)
    rc, r = o.run()
    assert rc == 0
    assert abs(r["k_mean"] - 1.2) < 3 * r["k_sdev"] + 1e-3
    f = r["flux_mean"].reshape(-1, 7).sum(axis=1)
    per_elem = np.concatenate([f[:4], [f[4] / 12]])  # 4 fuelled pins + 16 - 4 reflector pins sharing one bin
    assert np.allclose(per_elem / per_elem.mean(), 1.0, atol=0.05)
    c = r["counters"]
    assert c[7] > 0 and c[10] == 0 and c[6] == 0
