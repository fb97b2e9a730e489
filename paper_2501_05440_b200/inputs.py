"""Seeded synthetic problem generators (BASELINE.json configs C1..C5 and the pin problems).

This module serves BOTH the CPU oracle (``oracle/``) and the CUDA library: it only builds
plain NumPy arrays that describe a problem (surfaces, cells, lattice, cross sections,
source, tally edges).  It holds none of the transport method's arithmetic: no RNG stream,
no distance/collision sampling, no cumulative tables, no tallies.  It imports neither side.

A *problem* is a dict of NumPy arrays / scalars ("problem dict"):

geometry (SURVEY.md 8b/8c rules 11-16; "constructive solid geometry ... surface tracking")
  surf_type  i32[ns]    0 PLANE_X, 1 PLANE_Y, 2 PLANE_Z, 3 PLANE(a,b,c,d), 4 CYL_X, 5 CYL_Y,
                        6 CYL_Z, 7 SPHERE
  surf_param f64[ns,4]  PLANE_X/Y/Z: (p,-,-,-); PLANE: (a,b,c,d) with a x+b y+c z = d;
                        CYL_Z: (x0,y0,r,-) (CYL_X: (y0,z0,r), CYL_Y: (x0,z0,r)); SPHERE: (x0,y0,z0,r)
  surf_bc    i32[ns]    0 TRANSMIT, 1 REFLECT, 2 VACUUM
  cell_surf_off i32[nc+1], cell_surf_id i32[], cell_surf_sense i32[] (+1: f>0, -1: f<0)
  cell_fill_type i32[nc] 0 material, 1 lattice, 2 second-level lattice;  cell_fill i32[nc] material id (0 for the
                        lattice; the second-level lattice's index)
  cell_bin   i32[nc]    spatial tally bin of the cell (added to the lattice element's bin)
  univ_cell_off i32[nu+1]  cells are sorted by universe; universe 0 is the root
  lat        None | dict(x0,y0,px,py,nx,ny, univ i32[ny,nx], bin i32[ny,nx])
  lat2_nx, lat2_ny i32[n2], lat2_px, lat2_py f64[n2], lat2_off i32[n2+1], lat2_univ, lat2_bin i32[]  (optional)
                        second-level lattices: lattice k fills a cell (fill type 2) of a first-level element's
                        universe, centred on that universe's origin; element (ix,iy) is entry lat2_off[k]+iy*nx+ix
  n_bins     number of spatial tally bins
physics
  mode 'mg': G, n_mat, mg_sig_t/mg_sig_c/mg_sig_f/mg_nu/mg_chi f64[nm,G], mg_S f64[nm,G,G] (row = from)
  mode 'ce': grid f64[n], nuc_A f64[nn], nuc_el/nuc_c/nuc_f f64[nn,n] (barns),
             mat_nuc_off i32[nm+1], mat_nuc_id i32[], mat_nuc_dens f64[] (1/(b cm)),
             nu0, nu1 (nu = nu0 + nu1*E[MeV]), watt_a [MeV], watt_b [1/MeV],
             t_edges f64[nt+1] (s), e_edges f64[ne+1] (eV)
  td (optional, mode 'mg'): time-dependent multi-group with delayed neutrons (run kind 'td'; tally flux[bin][time bin][g]):
             dict(speed f64[G] cm/s, J precursor groups, nu_d f64[nm,J,G] delayed yields (mg_nu = prompt yield),
             decay f64[nm,J] 1/s, chi_d f64[nm,J,G], census_target (0 = no population control)); t_edges f64[nt+1]
source
  src_lo, src_hi f64[3]; src_iso (1/0); src_dir f64[3]; src_group_pdf f64[G] | src_E (eV); src_t (s)
run
  run: dict(kind 'eigen'|'fixed'|'td', n_particles, n_inactive, n_active, seed)
"""
from __future__ import annotations

import numpy as np

PLANE_X, PLANE_Y, PLANE_Z, PLANE, CYL_X, CYL_Y, CYL_Z, SPHERE = range(8)
TRANSMIT, REFLECT, VACUUM = range(3)


# --------------------------------------------------------------------------- geometry builders
class _Geom:
    """Accumulates surfaces and cells; universe 0 (root) must be added first."""

    def __init__(self):
        self.st, self.sp, self.sb = [], [], []
        self.cells = []  # (universe, [(surf, sense)], fill_type, fill, bin)

    def surf(self, typ, params, bc=TRANSMIT):
        p = list(params) + [0.0] * (4 - len(params))
        self.st.append(typ)
        self.sp.append(p)
        self.sb.append(bc)
        return len(self.st) - 1

    def cell(self, univ, region, fill, bin_=0, lattice=False, lattice2=False):
        self.cells.append((univ, list(region), 2 if lattice2 else (1 if lattice else 0), fill, bin_))

    def finish(self, lat=None, n_bins=1, lat2=None):
        """lat2: list of dict(nx, ny, px, py, univ i32[ny,nx], bin i32[ny,nx]) -- the second-level lattices."""
        out = self._finish(lat, n_bins)
        if lat2:
            out["lat2_nx"] = np.array([L["nx"] for L in lat2], np.int32)
            out["lat2_ny"] = np.array([L["ny"] for L in lat2], np.int32)
            out["lat2_px"] = np.array([L["px"] for L in lat2], np.float64)
            out["lat2_py"] = np.array([L["py"] for L in lat2], np.float64)
            out["lat2_off"] = np.concatenate([[0], np.cumsum([L["nx"] * L["ny"] for L in lat2])]).astype(np.int32)
            out["lat2_univ"] = np.concatenate([np.asarray(L["univ"], np.int32).ravel() for L in lat2])
            out["lat2_bin"] = np.concatenate([np.asarray(L["bin"], np.int32).ravel() for L in lat2])
        return out

    def _finish(self, lat=None, n_bins=1):
        cells = sorted(enumerate(self.cells), key=lambda t: (t[1][0], t[0]))
        nu = max(c[1][0] for c in cells) + 1
        off, sid, sse, ft, fl, cb = [0], [], [], [], [], []
        uoff = [0] * (nu + 1)
        for _, (u, region, ftype, fill, b) in cells:
            uoff[u + 1] += 1
            for s, sense in region:
                sid.append(s)
                sse.append(sense)
            off.append(len(sid))
            ft.append(ftype)
            fl.append(fill)
            cb.append(b)
        uoff = np.cumsum(uoff)
        return dict(
            surf_type=np.array(self.st, np.int32),
            surf_param=np.array(self.sp, np.float64).reshape(-1, 4),
            surf_bc=np.array(self.sb, np.int32),
            cell_surf_off=np.array(off, np.int32),
            cell_surf_id=np.array(sid, np.int32),
            cell_surf_sense=np.array(sse, np.int32),
            cell_fill_type=np.array(ft, np.int32),
            cell_fill=np.array(fl, np.int32),
            cell_bin=np.array(cb, np.int32),
            univ_cell_off=uoff.astype(np.int32),
            lat=lat,
            n_bins=int(n_bins),
        )


def geom_box(lo, hi, bc=REFLECT, material=0):
    """Rectangular box [lo,hi] bounded by six axis planes, one cell."""
    g = _Geom()
    bcs = bc if isinstance(bc, (list, tuple)) else [bc] * 6
    reg = []
    for ax, typ in enumerate((PLANE_X, PLANE_Y, PLANE_Z)):
        s0 = g.surf(typ, [lo[ax]], bcs[2 * ax])
        s1 = g.surf(typ, [hi[ax]], bcs[2 * ax + 1])
        reg += [(s0, +1), (s1, -1)]
    g.cell(0, reg, material)
    return g.finish()


def geom_infinite(material=0):
    """All space, one cell without surfaces."""
    g = _Geom()
    g.cell(0, [], material)
    return g.finish()


def geom_slab(L, material=0):
    """Slab 0<x<L, vacuum on both faces, infinite in y,z."""
    g = _Geom()
    s0 = g.surf(PLANE_X, [0.0], VACUUM)
    s1 = g.surf(PLANE_X, [L], VACUUM)
    g.cell(0, [(s0, +1), (s1, -1)], material)
    return g.finish()


def geom_sphere(r, bc=VACUUM, material=0):
    g = _Geom()
    s = g.surf(SPHERE, [0.0, 0.0, 0.0, r], bc)
    g.cell(0, [(s, -1)], material)
    return g.finish()


def geom_pincell(pitch=1.26, r=0.54, fuel=0, mod=1):
    """C3: fuel cylinder (CYL_Z) centred in a reflecting square; infinite in z (rule 15)."""
    g = _Geom()
    h = 0.5 * pitch
    xm = g.surf(PLANE_X, [-h], REFLECT)
    xp = g.surf(PLANE_X, [h], REFLECT)
    ym = g.surf(PLANE_Y, [-h], REFLECT)
    yp = g.surf(PLANE_Y, [h], REFLECT)
    cy = g.surf(CYL_Z, [0.0, 0.0, r], TRANSMIT)
    g.cell(0, [(cy, -1)], fuel, bin_=0)
    g.cell(0, [(xm, +1), (xp, -1), (ym, +1), (yp, -1), (cy, +1)], mod, bin_=1)
    return g.finish(n_bins=2)


def geom_mixed(material_a=0, material_b=1):
    """Every surface type in one problem (parity / pin geometry, not a BASELINE config): a reflecting box
    [-2,2]^3 (PLANE_X/Y/Z) holding a sphere (r = 0.9 at (0.3,-0.2,0.1)), an x-axis cylinder (CYL_X, r = 0.5 through
    (y,z) = (-1.3, 1.3)), a y-axis cylinder (CYL_Y, r = 0.4 through (x,z) = (1.2,-1.1)), and a general plane
    x + 2y - z = 0.8 that splits the remaining volume in two cells; vacuum on the +z face; a REFLECTING general plane
    x + y + z = 5 cuts off the (+,+,+) corner (non-axis reflection)."""
    g = _Geom()
    xm = g.surf(PLANE_X, [-2.0], REFLECT); xp = g.surf(PLANE_X, [2.0], REFLECT)
    ym = g.surf(PLANE_Y, [-2.0], REFLECT); yp = g.surf(PLANE_Y, [2.0], REFLECT)
    zm = g.surf(PLANE_Z, [-2.0], REFLECT); zp = g.surf(PLANE_Z, [2.0], VACUUM)
    sp = g.surf(SPHERE, [0.3, -0.2, 0.1, 0.9])
    cx = g.surf(CYL_X, [-1.3, 1.3, 0.5])
    cy = g.surf(CYL_Y, [1.2, -1.1, 0.4])
    pl = g.surf(PLANE, [1.0, 2.0, -1.0, 0.8])
    mir = g.surf(PLANE, [1.0, 1.0, 1.0, 5.0], REFLECT)  # a mirror that cuts the (+,+,+) corner off the box
    box = [(xm, +1), (xp, -1), (ym, +1), (yp, -1), (zm, +1), (zp, -1), (mir, -1)]
    g.cell(0, [(sp, -1)], material_a, bin_=0)
    g.cell(0, [(cx, -1), (xm, +1), (xp, -1)], material_a, bin_=1)
    g.cell(0, [(cy, -1), (ym, +1), (yp, -1)], material_b, bin_=2)
    g.cell(0, box + [(sp, +1), (cx, +1), (cy, +1), (pl, -1)], material_b, bin_=3)
    g.cell(0, box + [(sp, +1), (cx, +1), (cy, +1), (pl, +1)], material_a, bin_=4)
    return g.finish(n_bins=5)


def mixed_surfaces(n_particles=20_000, n_inactive=1, n_active=3, seed=23, G=3):
    """Two synthetic 3-group materials in geom_mixed(); eigenvalue run."""
    rng = np.random.default_rng(6)
    mats = [mg_fuel(rng, G, 1.4), mg_moderator(rng, G)]
    P = geom_mixed()
    P.update(_mg_pack(mats))
    P.update(_src([-1.9, -1.9, -1.9], [1.6, 1.6, 1.6], G=G, pdf=mats[0]["chi"]))
    P["run"] = dict(kind="eigen", n_particles=n_particles, n_inactive=n_inactive, n_active=n_active, seed=seed)
    P["name"] = "mixed"
    return P


def geom_mirror(kind, r=1.0, r_in=0.6):
    """Homogeneous medium inside ONE reflecting curved surface (non-axis specular reflection, R13): 'sphere' (radius
    r), 'cyl_z' / 'cyl_x' / 'cyl_y' (radius r, closed by two reflecting axis planes at +-1).  A concentric transmitting
    surface of radius r_in splits it in two tally bins (same material): with specular walls the flux stays uniform, so
    the bins' track lengths are in the ratio of their volumes."""
    g = _Geom()
    if kind == "sphere":
        so = g.surf(SPHERE, [0.0, 0.0, 0.0, r], REFLECT)
        si = g.surf(SPHERE, [0.0, 0.0, 0.0, r_in])
        caps = []
    else:
        typ = dict(cyl_x=CYL_X, cyl_y=CYL_Y, cyl_z=CYL_Z)[kind]
        ptyp = dict(cyl_x=PLANE_X, cyl_y=PLANE_Y, cyl_z=PLANE_Z)[kind]
        so = g.surf(typ, [0.0, 0.0, r], REFLECT)
        si = g.surf(typ, [0.0, 0.0, r_in])
        c0 = g.surf(ptyp, [-1.0], REFLECT)
        c1 = g.surf(ptyp, [1.0], REFLECT)
        caps = [(c0, +1), (c1, -1)]
    g.cell(0, [(si, -1)] + caps, 0, bin_=0)
    g.cell(0, [(si, +1), (so, -1)] + caps, 0, bin_=1)
    return g.finish(n_bins=2)


def curved_mirror(kind="sphere", n_particles=20_000, n_inactive=2, n_active=10, seed=31):
    """C1's one-group material inside geom_mirror(kind): leakage 0, k -> 1.3, flux ratio = volume ratio.  The source
    is a small box at the centre (the inner cell); the fission source spreads out over the cycles."""
    P = geom_mirror(kind)
    P.update(_mg_pack([one_group_material()]))
    P.update(_src([-0.3, -0.3, -0.3], [0.3, 0.3, 0.3], G=1))
    P["run"] = dict(kind="eigen", n_particles=n_particles, n_inactive=n_inactive, n_active=n_active, seed=seed)
    P["name"] = "mirror_" + kind
    return P


def tube_positions():
    """25 moderator-filled tube positions of a 17x17 assembly: our own 8-fold-symmetric
    choice (a regular 5x5 sub-grid, spacing 3) -- NOT any published benchmark's pin map."""
    return [(8 + i, 8 + j) for i in (-6, -3, 0, 3, 6) for j in (-6, -3, 0, 3, 6)]


def _pin_universes(g, cy, zf):
    """Universes 1..6 (pins: material u - 1 inside the cylinder, moderator 6 outside) and 7 (moderator only).  zf = the
    z plane that ends the fuel (axial reflector above it: "fully 3D"), or None: with it every pin universe
    has three cells -- fuel (inside the cylinder AND below zf), moderator beside it (outside the cylinder, below zf) and
    the moderator of the axial reflector (above zf, the whole element)."""
    for u in range(1, 7):
        if zf is None:
            g.cell(u, [(cy, -1)], u - 1)
            g.cell(u, [(cy, +1)], 6)
        else:
            g.cell(u, [(cy, -1), (zf, -1)], u - 1)
            g.cell(u, [(cy, +1), (zf, -1)], 6)
            g.cell(u, [(zf, +1)], 6)
    g.cell(7, [], 6)


def geom_quarter_core(pitch=1.26, r=0.54, n_asm=2, n_pin=17, n_refl=17, all_reflect=False, height=None, axial_reflector=None):
    """C4: one (n_asm*n_pin+n_refl)^2 lattice; elements [0,n_asm*n_pin)^2
    are fuelled assemblies, the rest moderator 'reflector' elements.  x=0,y=0 REFLECT,
    outer faces VACUUM.  Materials: 0,1,2 fuel variants; 3,4 alternate fuel; 5 tube fill; 6 moderator.
    Universes: 1..5 fuel pins (material u-1), 6 tube pin, 7 moderator-only."""
    g = _Geom()
    nfuel = n_asm * n_pin
    n = nfuel + n_refl
    side = n * pitch
    outer = REFLECT if all_reflect else VACUUM
    x0 = g.surf(PLANE_X, [0.0], REFLECT)
    x1 = g.surf(PLANE_X, [side], outer)
    y0 = g.surf(PLANE_Y, [0.0], REFLECT)
    y1 = g.surf(PLANE_Y, [side], outer)
    cy = g.surf(CYL_Z, [0.0, 0.0, r], TRANSMIT)
    root = [(x0, +1), (x1, -1), (y0, +1), (y1, -1)]
    zf = None
    if height is not None:  # finite height: reflecting mid-plane at z = 0, vacuum top at z = height
        z0 = g.surf(PLANE_Z, [0.0], REFLECT)
        z1 = g.surf(PLANE_Z, [float(height)], outer)
        root += [(z0, +1), (z1, -1)]
        if axial_reflector:  # the top `axial_reflector` cm of every pin are moderator
            assert 0.0 < axial_reflector < height
            zf = g.surf(PLANE_Z, [float(height - axial_reflector)], TRANSMIT)
    g.cell(0, root, 0, lattice=True)
    _pin_universes(g, cy, zf)
    univ = np.full((n, n), 7, np.int32)
    bins = np.full((n, n), nfuel * nfuel, np.int32)
    tubes = set(tube_positions()) if n_pin == 17 else set()
    for iy in range(nfuel):
        for ix in range(nfuel):
            ax, ay = ix // n_pin, iy // n_pin
            px, py = ix % n_pin, iy % n_pin
            edge = min(px, py, n_pin - 1 - px, n_pin - 1 - py)  # Chebyshev distance from assembly edge
            if (px, py) in tubes:
                u = 6
            elif (ax + ay) % 2 == 0:
                u = 1 if edge < 2 else (2 if edge < 5 else 3)
            else:
                u = 4 if edge < 3 else 5
            univ[iy, ix] = u
            bins[iy, ix] = iy * nfuel + ix
    lat = dict(x0=0.0, y0=0.0, px=float(pitch), py=float(pitch), nx=n, ny=n, univ=univ, bin=bins)
    return g.finish(lat=lat, n_bins=nfuel * nfuel + 1)


def geom_quarter_core_2l(pitch=1.26, r=0.54, n_asm=2, n_pin=17, n_refl_asm=1, all_reflect=False, height=None,
                         reflector_lattice=True, axial_reflector=None):
    """The quarter core of geom_quarter_core as a TWO-LEVEL lattice (the paper's multi-group benchmark
    is a core of assemblies of pins): a first-level (n_asm + n_refl_asm)^2 lattice of assemblies of pitch n_pin * pitch;
    every assembly universe is one cell without surfaces filled by a second-level n_pin x n_pin pin lattice.  Same pin
    map, materials and per-pin tally bins as the flat geometry with n_refl = n_refl_asm * n_pin, so both describe the
    same physical problem.  Universes 1..7 as there; 8, 9 = the two fuel assembly types, 10 = reflector assembly
    (reflector_lattice=False: reflector assemblies are one moderator cell with no inner walls)."""
    g = _Geom()
    na = n_asm + n_refl_asm
    nfuel = n_asm * n_pin
    ap = n_pin * pitch
    side = na * ap
    outer = REFLECT if all_reflect else VACUUM
    x0 = g.surf(PLANE_X, [0.0], REFLECT)
    x1 = g.surf(PLANE_X, [side], outer)
    y0 = g.surf(PLANE_Y, [0.0], REFLECT)
    y1 = g.surf(PLANE_Y, [side], outer)
    cy = g.surf(CYL_Z, [0.0, 0.0, r], TRANSMIT)
    root = [(x0, +1), (x1, -1), (y0, +1), (y1, -1)]
    zf = None
    if height is not None:
        z0 = g.surf(PLANE_Z, [0.0], REFLECT)
        z1 = g.surf(PLANE_Z, [float(height)], outer)
        root += [(z0, +1), (z1, -1)]
        if axial_reflector:
            assert 0.0 < axial_reflector < height
            zf = g.surf(PLANE_Z, [float(height - axial_reflector)], TRANSMIT)
    g.cell(0, root, 0, lattice=True)
    _pin_universes(g, cy, zf)
    g.cell(8, [], 0, lattice2=True)
    g.cell(9, [], 1, lattice2=True)
    if reflector_lattice:
        g.cell(10, [], 2, lattice2=True)
    else:
        g.cell(10, [], 6)
    tubes = set(tube_positions()) if n_pin == 17 else set()
    inner = []
    for kind in (0, 1):
        un = np.zeros((n_pin, n_pin), np.int32)
        for py in range(n_pin):
            for px in range(n_pin):
                edge = min(px, py, n_pin - 1 - px, n_pin - 1 - py)
                if (px, py) in tubes:
                    u = 6
                elif kind == 0:
                    u = 1 if edge < 2 else (2 if edge < 5 else 3)
                else:
                    u = 4 if edge < 3 else 5
                un[py, px] = u
        bins = (np.arange(n_pin)[:, None] * nfuel + np.arange(n_pin)[None, :]).astype(np.int32)
        inner.append(dict(nx=n_pin, ny=n_pin, px=float(pitch), py=float(pitch), univ=un, bin=bins))
    if reflector_lattice:
        inner.append(dict(nx=n_pin, ny=n_pin, px=float(pitch), py=float(pitch), univ=np.full((n_pin, n_pin), 7, np.int32),
                          bin=np.zeros((n_pin, n_pin), np.int32)))
    univ = np.full((na, na), 10, np.int32)
    bins = np.full((na, na), nfuel * nfuel, np.int32)
    for ay in range(n_asm):
        for ax in range(n_asm):
            univ[ay, ax] = 8 if (ax + ay) % 2 == 0 else 9
            bins[ay, ax] = ay * n_pin * nfuel + ax * n_pin
    lat = dict(x0=0.0, y0=0.0, px=float(ap), py=float(ap), nx=na, ny=na, univ=univ, bin=bins)
    return g.finish(lat=lat, n_bins=nfuel * nfuel + 1, lat2=inner)


def geom_assembly_gap(n_asm=2, n_pin=3, pitch=1.26, r=0.54, gap=0.2):
    """Two-level lattice whose assembly universe has structure of its own: the pin lattice fills a square cell
    |x|, |y| < n_pin * pitch / 2 (four planes in assembly coordinates) and a moderator gap of width `gap` surrounds it
    (four conjunctive cells).  n_asm x n_asm assemblies; x = 0, y = 0 reflect, the far faces are vacuum.  Materials:
    0 fuel, 1 moderator.  One tally bin per pin plus one gap bin per assembly."""
    g = _Geom()
    h = 0.5 * n_pin * pitch
    ap = 2.0 * (h + gap)
    side = n_asm * ap
    x0 = g.surf(PLANE_X, [0.0], REFLECT)
    x1 = g.surf(PLANE_X, [side], VACUUM)
    y0 = g.surf(PLANE_Y, [0.0], REFLECT)
    y1 = g.surf(PLANE_Y, [side], VACUUM)
    cy = g.surf(CYL_Z, [0.0, 0.0, r], TRANSMIT)
    xl = g.surf(PLANE_X, [-h], TRANSMIT)
    xh = g.surf(PLANE_X, [h], TRANSMIT)
    yl = g.surf(PLANE_Y, [-h], TRANSMIT)
    yh = g.surf(PLANE_Y, [h], TRANSMIT)
    g.cell(0, [(x0, +1), (x1, -1), (y0, +1), (y1, -1)], 0, lattice=True)
    g.cell(1, [(cy, -1)], 0)
    g.cell(1, [(cy, +1)], 1)
    g.cell(2, [], 1)
    npp = n_pin * n_pin
    # assembly universe 3: the lattice cell first, then the four gap cells (bin offset npp = the assembly's gap bin)
    g.cell(3, [(xl, +1), (xh, -1), (yl, +1), (yh, -1)], 0, lattice2=True)
    g.cell(3, [(xl, -1)], 1, bin_=npp)
    g.cell(3, [(xh, +1)], 1, bin_=npp)
    g.cell(3, [(xl, +1), (xh, -1), (yl, -1)], 1, bin_=npp)
    g.cell(3, [(xl, +1), (xh, -1), (yh, +1)], 1, bin_=npp)
    un = np.array([[1 if (ix + iy) % 3 else 2 for ix in range(n_pin)] for iy in range(n_pin)], np.int32)
    inner = [dict(nx=n_pin, ny=n_pin, px=float(pitch), py=float(pitch), univ=un,
                  bin=np.arange(npp, dtype=np.int32).reshape(n_pin, n_pin))]
    univ = np.full((n_asm, n_asm), 3, np.int32)
    bins = (np.arange(n_asm * n_asm, dtype=np.int32) * (npp + 1)).reshape(n_asm, n_asm)
    lat = dict(x0=0.0, y0=0.0, px=float(ap), py=float(ap), nx=n_asm, ny=n_asm, univ=univ, bin=bins)
    return g.finish(lat=lat, n_bins=n_asm * n_asm * (npp + 1), lat2=inner)


def assembly_gap(n_asm=2, n_pin=3, n_particles=4000, n_inactive=1, n_active=2, seed=43, G=3, gap=0.2):
    """Two synthetic 3-group materials in geom_assembly_gap; eigenvalue run."""
    rng = np.random.default_rng(7)
    mats = [mg_fuel(rng, G, 1.5), mg_moderator(rng, G)]
    P = geom_assembly_gap(n_asm, n_pin, gap=gap)
    P.update(_mg_pack(mats))
    side = n_asm * (n_pin * 1.26 + 2 * gap)
    P.update(_src([0, 0, 0], [side, side, 0], G=G, pdf=mats[0]["chi"]))
    P["run"] = dict(kind="eigen", n_particles=n_particles, n_inactive=n_inactive, n_active=n_active, seed=seed)
    P["name"] = "asm_gap"
    return P


def two_level_rect(nxo=2, nyo=3, nxi=3, nyi=2, n_particles=4000, n_inactive=1, n_active=2, seed=53, G=3, pitch=1.26, r=0.54):
    """Non-square lattices at both levels (index-transposition check): nxo x nyo assemblies, each one cell filled by one
    of two nxi x nyi pin lattices (different pin maps); rectangular pins of pitch (pitch, 0.9 pitch).  x = 0, y = 0
    reflect, the far faces are vacuum.  One tally bin per pin."""
    g = _Geom()
    px, py = float(pitch), float(0.9 * pitch)
    ax, ay = nxi * px, nyi * py
    x0 = g.surf(PLANE_X, [0.0], REFLECT)
    x1 = g.surf(PLANE_X, [nxo * ax], VACUUM)
    y0 = g.surf(PLANE_Y, [0.0], REFLECT)
    y1 = g.surf(PLANE_Y, [nyo * ay], VACUUM)
    cy = g.surf(CYL_Z, [0.0, 0.0, r], TRANSMIT)
    g.cell(0, [(x0, +1), (x1, -1), (y0, +1), (y1, -1)], 0, lattice=True)
    g.cell(1, [(cy, -1)], 0)
    g.cell(1, [(cy, +1)], 1)
    g.cell(2, [], 1)
    g.cell(3, [], 0, lattice2=True)
    g.cell(4, [], 1, lattice2=True)
    npi = nxi * nyi
    inner = []
    for kind in (0, 1):
        un = np.array([[1 if (ix + 2 * iy + kind) % 3 else 2 for ix in range(nxi)] for iy in range(nyi)], np.int32)
        inner.append(dict(nx=nxi, ny=nyi, px=px, py=py, univ=un, bin=np.arange(npi, dtype=np.int32).reshape(nyi, nxi)))
    univ = np.array([[3 + (ix + iy) % 2 for ix in range(nxo)] for iy in range(nyo)], np.int32)
    bins = (np.arange(nxo * nyo, dtype=np.int32) * npi).reshape(nyo, nxo)
    lat = dict(x0=0.0, y0=0.0, px=float(ax), py=float(ay), nx=nxo, ny=nyo, univ=univ, bin=bins)
    P = g.finish(lat=lat, n_bins=nxo * nyo * npi, lat2=inner)
    rng = np.random.default_rng(7)
    mats = [mg_fuel(rng, G, 1.5), mg_moderator(rng, G)]
    P.update(_mg_pack(mats))
    P.update(_src([0, 0, 0], [nxo * ax, nyo * ay, 0], G=G, pdf=mats[0]["chi"]))
    P["run"] = dict(kind="eigen", n_particles=n_particles, n_inactive=n_inactive, n_active=n_active, seed=seed)
    P["name"] = "two_level_rect"
    return P


def geom_rect_lattice(nx, ny, pitch=1.26, r=0.54, x_hi=VACUUM, y_hi=REFLECT):
    """nx x ny pin lattice filling the box [0, nx p] x [0, ny p] (parity geometry for non-square and one-column /
    one-row lattices): universes 1 = fuel pin (material 0 in a cylinder, 1 outside), 2 = moderator only, in a
    checker pattern; x = 0 and y = 0 reflect; one tally bin per element."""
    g = _Geom()
    x0 = g.surf(PLANE_X, [0.0], REFLECT)
    x1 = g.surf(PLANE_X, [nx * pitch], x_hi)
    y0 = g.surf(PLANE_Y, [0.0], REFLECT)
    y1 = g.surf(PLANE_Y, [ny * pitch], y_hi)
    cy = g.surf(CYL_Z, [0.0, 0.0, r], TRANSMIT)
    g.cell(0, [(x0, +1), (x1, -1), (y0, +1), (y1, -1)], 0, lattice=True)
    g.cell(1, [(cy, -1)], 0)
    g.cell(1, [(cy, +1)], 1)
    g.cell(2, [], 1)
    univ = np.array([[1 if (ix + 2 * iy) % 3 else 2 for ix in range(nx)] for iy in range(ny)], np.int32)
    bins = np.arange(nx * ny, dtype=np.int32).reshape(ny, nx)
    lat = dict(x0=0.0, y0=0.0, px=float(pitch), py=float(pitch), nx=nx, ny=ny, univ=univ, bin=bins)
    return g.finish(lat=lat, n_bins=nx * ny)


def rect_lattice(nx, ny, n_particles=4000, n_inactive=1, n_active=2, seed=29, G=3):
    """Two synthetic 3-group materials in geom_rect_lattice(nx, ny); eigenvalue run."""
    rng = np.random.default_rng(7)
    mats = [mg_fuel(rng, G, 1.5), mg_moderator(rng, G)]
    P = geom_rect_lattice(nx, ny)
    P.update(_mg_pack(mats))
    P.update(_src([0, 0, 0], [nx * 1.26, ny * 1.26, 0], G=G, pdf=mats[0]["chi"]))
    P["run"] = dict(kind="eigen", n_particles=n_particles, n_inactive=n_inactive, n_active=n_active, seed=seed)
    P["name"] = f"lat{nx}x{ny}"
    return P


# --------------------------------------------------------------------------- MG materials
def mg_kinf(sig_t, S, nusf, chi):
    """Input-design helper (used to scale Sigma_f to a target k); tests re-derive k independently."""
    A = np.diag(sig_t) - S.T
    return float(nusf @ np.linalg.solve(A, chi))


def mg_fuel(rng, G=7, k_target=1.2, thermal_boost=1.0):
    """SURVEY.md 8d C2 recipe: Sigma_t~U(0.2,1.5), c~U(0.6,0.95), downscatter + 2 upscatter terms,
    nu~U(2.4,2.9), Sigma_f scaled so the infinite-medium k equals k_target, chi in groups 0-2."""
    while True:
        sig_t = rng.uniform(0.2, 1.5, G)
        c = rng.uniform(0.6, 0.95, G)
        sig_s = c * sig_t
        S = np.zeros((G, G))
        for g in range(G):
            for gp in range(g, G):
                S[g, gp] = np.exp(-0.9 * (gp - g)) * rng.uniform(0.5, 1.5)
        if G >= 3:
            S[G - 1, G - 2] = 0.05 * rng.uniform(0.5, 1.5)
            S[G - 2, G - 3] = 0.02 * rng.uniform(0.5, 1.5)
        S *= (sig_s / S.sum(axis=1))[:, None]
        nu = rng.uniform(2.4, 2.9, G)
        ramp = np.linspace(0.3, 1.0, G) if G > 1 else np.ones(1)
        f = rng.uniform(0.2, 0.5, G) * ramp
        if thermal_boost != 1.0 and G >= 2:
            f[-2:] *= thermal_boost
        chi = np.zeros(G)
        w = np.array([3.0, 2.0, 0.2])[: min(3, G)]
        chi[: len(w)] = rng.uniform(0.5, 1.0, len(w)) * w
        chi /= chi.sum()
        rem = sig_t - S.sum(axis=1)
        k1 = mg_kinf(sig_t, S, nu * f * rem, chi)
        s = k_target / k1
        if s * f.max() <= 0.95:
            break
    sig_f = s * f * rem
    sig_c = sig_t - S.sum(axis=1) - sig_f
    return dict(sig_t=sig_t, sig_c=sig_c, sig_f=sig_f, nu=nu, chi=chi, S=S)


def mg_moderator(rng, G=7):
    """SURVEY.md 8d C3 recipe: Sigma_t~U(0.5,3), c~U(0.97,0.998), strong downscatter, no fission."""
    sig_t = rng.uniform(0.5, 3.0, G)
    c = rng.uniform(0.97, 0.998, G)
    S = np.zeros((G, G))
    for g in range(G):
        for gp in range(g, G):
            S[g, gp] = np.exp(-0.4 * (gp - g)) * rng.uniform(0.5, 1.5) * (1.0 if gp > g else 0.6)
    if G >= 3:
        S[G - 1, G - 2] = 0.05 * rng.uniform(0.5, 1.5)
        S[G - 2, G - 3] = 0.02 * rng.uniform(0.5, 1.5)
    S *= (c * sig_t / S.sum(axis=1))[:, None]
    z = np.zeros(G)
    return dict(sig_t=sig_t, sig_c=sig_t - S.sum(axis=1), sig_f=z.copy(), nu=z.copy(), chi=z.copy(), S=S)


def _mg_pack(mats):
    G = len(mats[0]["sig_t"])
    out = dict(mode="mg", G=G, n_mat=len(mats))
    for k in ("sig_t", "sig_c", "sig_f", "nu", "chi"):
        out["mg_" + k] = np.ascontiguousarray(np.stack([m[k] for m in mats]), np.float64)
    out["mg_S"] = np.ascontiguousarray(np.stack([m["S"] for m in mats]), np.float64)
    return out


def _src(lo, hi, G=None, pdf=None, iso=True, direction=(0.0, 0.0, 1.0), E=None, t=0.0):
    d = dict(src_lo=np.array(lo, np.float64), src_hi=np.array(hi, np.float64), src_iso=int(iso),
             src_dir=np.array(direction, np.float64), src_t=float(t))
    if G is not None:
        d["src_group_pdf"] = np.array(pdf if pdf is not None else [1.0] + [0.0] * (G - 1), np.float64)
    if E is not None:
        d["src_E"] = float(E)
    return d


def one_group_material(sig_t=1.0, sig_s=0.7, sig_f=0.15, nu=2.6):
    return dict(sig_t=np.array([sig_t]), sig_c=np.array([sig_t - sig_s - sig_f]), sig_f=np.array([sig_f]),
                nu=np.array([nu]), chi=np.array([1.0]), S=np.array([[sig_s]]))


# --------------------------------------------------------------------------- the five configs
def config1(n_particles=10_000, n_inactive=5, n_active=15, seed=1):
    """C1: 1-group infinite medium, unit reflecting cube; Sigma_t 1.0, Sigma_s 0.7, nuSigma_f 0.39
    (split nu=2.6, Sigma_f=0.15, Sigma_c=0.15) -> k_inf = 1.3."""
    P = geom_box([0, 0, 0], [1, 1, 1], REFLECT)
    P.update(_mg_pack([one_group_material()]))
    P.update(_src([0, 0, 0], [1, 1, 1], G=1))
    P["run"] = dict(kind="eigen", n_particles=n_particles, n_inactive=n_inactive, n_active=n_active, seed=seed)
    P["name"] = "C1"
    return P


def config2(n_particles=100_000, n_inactive=10, n_active=40, seed=1, mat_seed=2, G=7):
    """C2: 7-group infinite medium (reflecting unit cube), synthetic fuel from seed 2, k_inf = 1.2."""
    rng = np.random.default_rng(mat_seed)
    m = mg_fuel(rng, G, 1.2)
    P = geom_box([0, 0, 0], [1, 1, 1], REFLECT)
    P.update(_mg_pack([m]))
    P.update(_src([0, 0, 0], [1, 1, 1], G=G, pdf=m["chi"]))
    P["run"] = dict(kind="eigen", n_particles=n_particles, n_inactive=n_inactive, n_active=n_active, seed=seed)
    P["name"] = "C2"
    return P


def config3(n_particles=1_000_000, n_inactive=20, n_active=80, seed=1, same_material=False, G=7):
    """C3: 2-D pin cell, fuel = C2 material, moderator from seed 3.  same_material=True fills the
    moderator with the fuel (pin: flux fraction -> area fraction, k -> C2 closed form)."""
    fuel = mg_fuel(np.random.default_rng(2), G, 1.2)
    mod = fuel if same_material else mg_moderator(np.random.default_rng(3), G)
    P = geom_pincell()
    P.update(_mg_pack([fuel, mod]))
    P.update(_src([-0.63, -0.63, 0], [0.63, 0.63, 0], G=G, pdf=fuel["chi"]))
    P["run"] = dict(kind="eigen", n_particles=n_particles, n_inactive=n_inactive, n_active=n_active, seed=seed)
    P["name"] = "C3"
    return P


def config4(n_particles=10_000_000, n_inactive=20, n_active=100, seed=1, uniform=False,
            n_asm=2, n_pin=17, n_refl=17, G=7, height=None, two_level=False, reflector_lattice=True, axial_reflector=None):
    """C4: 2-D quarter core stand-in for the paper's C5G7 workload: 7 synthetic
    materials from seed 4.  uniform=True: all materials identical + all faces reflecting (pin).
    two_level=True: the same core described as a lattice of assemblies of pin lattices (n_refl must be a
    multiple of n_pin).  height: the fully 3-D core (reflecting mid-plane z = 0, vacuum top); axial_reflector: the top
    so many cm of every pin are moderator (the source then lies in the fuelled part)."""
    rng = np.random.default_rng(4)
    mats = [mg_fuel(rng, G, kt) for kt in (1.05, 1.15, 1.25)]
    mats += [mg_fuel(rng, G, kt, thermal_boost=1.5) for kt in (1.10, 1.20)]
    mats += [mg_moderator(rng, G), mg_moderator(rng, G)]
    if uniform:
        mats = [mg_fuel(np.random.default_rng(2), G, 1.2)] * 7
    if two_level:
        assert n_refl % n_pin == 0
        P = geom_quarter_core_2l(n_asm=n_asm, n_pin=n_pin, n_refl_asm=n_refl // n_pin, all_reflect=uniform, height=height,
                                 reflector_lattice=reflector_lattice, axial_reflector=axial_reflector)
    else:
        P = geom_quarter_core(n_asm=n_asm, n_pin=n_pin, n_refl=n_refl, all_reflect=uniform, height=height,
                              axial_reflector=axial_reflector)
    P.update(_mg_pack(mats))
    side = n_asm * n_pin * 1.26
    z_src = 0.9 * ((height - axial_reflector) if axial_reflector else height) if height else 0
    P.update(_src([0, 0, 0], [side, side, z_src], G=G, pdf=mats[0]["chi"]))
    P["run"] = dict(kind="eigen", n_particles=n_particles, n_inactive=n_inactive, n_active=n_active, seed=seed)
    P["name"] = "C4"
    return P


# --------------------------------------------------------------------------- time-dependent multi-group
def td_infinite(n_particles=20_000, seed=47, G=1, J=1, t_end=4.0e-3, n_t=8, census_target=0, geom="cube"):
    """Infinite homogeneous medium (reflecting unit cube) with delayed neutrons, a pulse of neutrons at t = 0:
    the kinetics problem whose expected flux per time bin is a linear ODE solution (tests integrate it).
    G = 1, J = 1: Sigma_t 1.0, Sigma_s 0.5, Sigma_f 0.2, prompt yield 2.3, delayed yield 0.15 (k = 0.98, prompt
    k = 0.92), decay 500 /s, speed 1e5 cm/s.  G = 2, J = 2: a fast and a slow group with down- and up-scatter, two
    precursor groups with different spectra.  geom 'pin': the same materials in the C3 pin cell (fuel = the medium,
    moderator = its non-fissile twin) for the geometry-coupled parity cases."""
    if G == 1:
        sig_t, S, sig_f = np.array([1.0]), np.array([[0.5]]), np.array([0.2])
        nu_p, speed = np.array([2.3]), np.array([1.0e5])
        nu_d, decay, chi_d = np.array([[0.15]]), np.array([500.0]), np.array([[1.0]])
        chi = np.array([1.0])
    else:
        assert G == 2
        sig_t, S = np.array([0.8, 1.6]), np.array([[0.30, 0.25], [0.05, 0.95]])
        sig_f, nu_p = np.array([0.05, 0.30]), np.array([2.5, 2.2])
        speed = np.array([4.0e5, 1.0e5])
        nu_d, decay = np.array([[0.10, 0.08], [0.06, 0.05]]), np.array([300.0, 2500.0])
        chi, chi_d = np.array([0.9, 0.1]), np.array([[0.3, 0.7], [0.6, 0.4]])
    J = nu_d.shape[0]
    mat = dict(sig_t=sig_t, S=S, sig_f=sig_f, nu=nu_p, chi=chi, sig_c=sig_t - S.sum(1) - sig_f)
    mats = [mat]
    td = dict(speed=speed, J=J, nu_d=nu_d[None], decay=decay[None], chi_d=chi_d[None], census_target=int(census_target))
    if geom == "cube":
        P = geom_box([0, 0, 0], [1, 1, 1], REFLECT)
        lo, hi = [0, 0, 0], [1, 1, 1]
    else:
        if geom == "lattice2":  # a two-level lattice with vacuum faces (fuel 0 / moderator 1 as in the pin cell)
            P = _geometry_of(two_level_rect(2, 2, 3, 2))
            lo, hi = [0, 0, 0], [2 * 3 * 1.26, 2 * 2 * 0.9 * 1.26, 0]
        else:
            P = geom_pincell()
            lo, hi = [-0.63, -0.63, 0], [0.63, 0.63, 0]
        mod = dict(sig_t=sig_t * 1.3, S=S * 1.5, sig_f=sig_f * 0.0, nu=nu_p, chi=chi, sig_c=sig_t * 1.3 - (S * 1.5).sum(1))
        mats = [mat, mod]
        td = dict(speed=speed, J=J, nu_d=np.stack([nu_d, nu_d * 0.0]), decay=np.stack([decay, decay]),
                  chi_d=np.stack([chi_d, chi_d]), census_target=int(census_target))
    P.update(_mg_pack(mats))
    P.update(_src(lo, hi, G=G, pdf=chi))
    P["td"] = td
    P["t_edges"] = np.linspace(0.0, t_end, n_t + 1)
    P["run"] = dict(kind="td", n_particles=n_particles, n_inactive=0, n_active=1, seed=seed)
    P["name"] = f"td_{geom}_G{G}"
    return P


# --------------------------------------------------------------------------- CE data
def ce_nuclides(seed=5, n_grid=50_000, jitter=False, n_res=200):
    """SURVEY.md 8d C5 recipe: five synthetic nuclides on a log-spaced union grid (eV), flat
    potential + 1/v + (heavy only) single-level Breit-Wigner resonances, Lorentzian, no interference."""
    rng = np.random.default_rng(seed)
    lg = np.linspace(np.log(1e-5), np.log(2e7), n_grid)
    if jitter:
        step = lg[1] - lg[0]
        lg[1:-1] += rng.uniform(-0.4, 0.4, n_grid - 2) * step
    E = np.exp(lg)
    E[0], E[-1] = 1e-5, 2e7
    inv_v = np.sqrt(0.0253 / E)

    def resonances(lo_pk, hi_pk):
        E0 = np.exp(rng.uniform(np.log(1.0), np.log(1e4), n_res))
        gam = E0 * np.exp(rng.uniform(np.log(3e-3), np.log(1e-2), n_res))
        pk = np.exp(rng.uniform(np.log(lo_pk), np.log(hi_pk), n_res)) / np.sqrt(E0)
        out = np.zeros_like(E)
        for e0, gm, p in zip(E0, gam, pk):
            out += p / (1.0 + ((E - e0) / (0.5 * gm)) ** 2)
        return out

    nn = 5
    A = np.array([235.0, 238.0, 16.0, 1.0, 10.0])
    el = np.zeros((nn, n_grid))
    ca = np.zeros((nn, n_grid))
    fi = np.zeros((nn, n_grid))
    r_fis = resonances(20.0, 500.0)
    r_fer = resonances(10.0, 400.0)
    # fissile
    el[0] = 11.5 + 0.05 * r_fis
    ca[0] = 100.0 * inv_v + 0.40 * r_fis
    fi[0] = 580.0 * inv_v + 1.2 + 0.55 * r_fis
    # fertile
    ramp = np.clip((E - 0.8e6) / (1.5e6 - 0.8e6), 0.0, 1.0)
    el[1] = 9.0 + 0.10 * r_fer
    ca[1] = 2.7 * inv_v + 0.90 * r_fer
    fi[1] = 0.5 * ramp
    # oxygen-like
    el[2] = 3.8
    # hydrogen-like
    el[3] = 20.0 / np.sqrt(1.0 + E / 1e5)
    ca[3] = 0.33 * inv_v
    # absorber-like
    el[4] = 2.0
    ca[4] = 3840.0 * inv_v
    return dict(grid=E, nuc_A=A, nuc_el=el, nuc_c=ca, nuc_f=fi)


def config5(n_particles=1_000_000, seed=1, n_grid=50_000, jitter=False, absorber=1.0e-4, data_seed=5):
    """C5: CE time-dependent infinite pin cell; stand-in for the paper's UO2 pin cell with the
    OpenMC data library, which is not in this container."""
    P = geom_pincell(fuel=0, mod=1)
    P["cell_bin"][:] = 0
    P["n_bins"] = 1
    P.update(ce_nuclides(data_seed, n_grid, jitter))
    P["mode"] = "ce"
    P["n_mat"] = 2
    P["mat_nuc_off"] = np.array([0, 3, 5], np.int32)
    P["mat_nuc_id"] = np.array([0, 1, 2, 3, 4], np.int32)
    P["mat_nuc_dens"] = np.array([5.5e-4, 2.24e-2, 4.6e-2, 6.68e-2, absorber], np.float64)
    P.update(nu0=2.4, nu1=0.1, watt_a=0.988, watt_b=2.249)
    P["t_edges"] = np.concatenate([[0.0], 10.0 ** (-8.0 + 0.5 * np.arange(1, 11))])
    P["e_edges"] = np.exp(np.linspace(np.log(1e-5), np.log(2e7), 101))
    P["e_edges"][0], P["e_edges"][-1] = 1e-5, 2e7
    P.update(_src([-0.63, -0.63, 0], [0.63, 0.63, 0], E=2.0e6, t=0.0))
    P["run"] = dict(kind="fixed", n_particles=n_particles, n_inactive=0, n_active=1, seed=seed)
    P["name"] = "C5"
    return P


GEO_KEYS = ("surf_type", "surf_param", "surf_bc", "cell_surf_off", "cell_surf_id", "cell_surf_sense", "cell_fill_type",
            "cell_fill", "cell_bin", "univ_cell_off", "lat", "n_bins", "lat2_nx", "lat2_ny", "lat2_px", "lat2_py",
            "lat2_off", "lat2_univ", "lat2_bin")


def _geometry_of(G):
    """the geometry and spatial-tally part of a problem dict"""
    return {k: G[k] for k in GEO_KEYS if k in G}


def ce_lattice(kind="two_level", n_particles=2000, seed=1, n_grid=6000):
    """The C5 nuclide data and time / energy bins in a lattice geometry with vacuum faces (continuous-energy kernels with
    lattice and second-level lattice geometry): kind 'two_level' = two_level_rect(2, 2, 3, 2), 'gap' = geom_assembly_gap,
    'flat' = geom_rect_lattice(4, 3).  Material 0 fuel, 1 moderator as in C5; one spatial bin per pin."""
    if kind == "two_level":
        G = two_level_rect(2, 2, 3, 2)
        side = (2 * 3 * 1.26, 2 * 2 * 0.9 * 1.26)
    elif kind == "gap":
        G = assembly_gap(2, 3)
        side = (2 * (3 * 1.26 + 0.4),) * 2
    else:
        G = rect_lattice(4, 3)
        side = (4 * 1.26, 3 * 1.26)
    P = _geometry_of(G)
    C = config5(n_particles=n_particles, seed=seed, n_grid=n_grid)
    for k, v in C.items():
        if k not in GEO_KEYS:
            P[k] = v
    P.update(_src([0, 0, 0], [side[0], side[1], 0], E=2.0e6, t=0.0))
    P["name"] = "ce_" + kind
    return P


# --------------------------------------------------------------------------- pin problems (closed forms)
def slab_beam(L=2.0, sig_t=1.3, n_particles=100_000, seed=7):
    """Pure absorber slab, mono-directional normal beam born on x=0+: leakage = exp(-Sigma_t L)."""
    P = geom_slab(L)
    P.update(_mg_pack([one_group_material(sig_t=sig_t, sig_s=0.0, sig_f=0.0, nu=0.0)]))
    P.update(_src([1e-12, 0, 0], [1e-12, 0, 0], G=1, iso=False, direction=(1.0, 0.0, 0.0)))
    P["run"] = dict(kind="eigen", n_particles=n_particles, n_inactive=0, n_active=1, seed=seed)
    P["name"] = "slab"
    return P


def sphere_absorber(r=1.5, sig_t=0.8, n_particles=100_000, seed=11):
    """Pure absorber sphere, isotropic point source at the centre: leakage = exp(-Sigma_t r)."""
    P = geom_sphere(r)
    P.update(_mg_pack([one_group_material(sig_t=sig_t, sig_s=0.0, sig_f=0.0, nu=0.0)]))
    P.update(_src([0, 0, 0], [0, 0, 0], G=1))
    P["run"] = dict(kind="eigen", n_particles=n_particles, n_inactive=0, n_active=1, seed=seed)
    P["name"] = "sphere"
    return P


def ce_one_over_v(lam=2.0e5, n_particles=100_000, seed=13, E0=1.0e3, n_grid=2000):
    """Single nuclide, pure 1/v absorber (Sigma_a v = lam [1/s]), no scatter, infinite medium:
    track length in [t1,t2] per source neutron = (v/lam)(exp(-lam t1)-exp(-lam t2))."""
    P = geom_infinite()
    E = np.exp(np.linspace(np.log(1e-5), np.log(2e7), n_grid))
    E[0], E[-1] = 1e-5, 2e7
    c_cm = 2.99792458e10
    v = c_cm * np.sqrt(2.0 * E / 939.56542052e6)
    P.update(mode="ce", n_mat=1, grid=E, nuc_A=np.array([10.0]), nuc_el=np.zeros((1, n_grid)),
             nuc_c=(lam / v)[None, :].copy(), nuc_f=np.zeros((1, n_grid)),
             mat_nuc_off=np.array([0, 1], np.int32), mat_nuc_id=np.array([0], np.int32),
             mat_nuc_dens=np.array([1.0]), nu0=0.0, nu1=0.0, watt_a=0.988, watt_b=2.249)
    P["t_edges"] = np.concatenate([[0.0], 10.0 ** (-6.5 + 0.25 * np.arange(1, 9))])
    P["e_edges"] = np.array([1e-5, 1.0, 2e7])
    P.update(_src([0, 0, 0], [0, 0, 0], E=E0, t=0.0))
    P["run"] = dict(kind="fixed", n_particles=n_particles, n_inactive=0, n_active=1, seed=seed)
    P["name"] = "ce_1v"
    return P


def ce_single_scatterer(A=16.0, n_particles=50_000, seed=17, E0=1.0e6, sig_el=0.5, sig_c=0.5, n_grid=500):
    """One nuclide with flat elastic + flat capture in an infinite medium (elastic-kinematics pin:
    the first-collision energy/angle moments are read from the event trace)."""
    P = geom_infinite()
    E = np.exp(np.linspace(np.log(1e-5), np.log(2e7), n_grid))
    E[0], E[-1] = 1e-5, 2e7
    P.update(mode="ce", n_mat=1, grid=E, nuc_A=np.array([float(A)]), nuc_el=np.full((1, n_grid), sig_el),
             nuc_c=np.full((1, n_grid), sig_c), nuc_f=np.zeros((1, n_grid)),
             mat_nuc_off=np.array([0, 1], np.int32), mat_nuc_id=np.array([0], np.int32),
             mat_nuc_dens=np.array([1.0]), nu0=0.0, nu1=0.0, watt_a=0.988, watt_b=2.249)
    P["t_edges"] = np.array([0.0, 1.0])
    P["e_edges"] = np.array([1e-5, 2e7])
    P.update(_src([0, 0, 0], [0, 0, 0], E=E0, t=0.0))
    P["run"] = dict(kind="fixed", n_particles=n_particles, n_inactive=0, n_active=1, seed=seed)
    P["name"] = "ce_scatter"
    return P


def ce_two_nuclide_mix(n_particles=20_000, seed=37, E0=1.0e6, E_cut=1.0e3, p_light=0.3, n_grid=4000):
    """Elastic-branch pin of the transport loop: a mixture of a light (A = 1) and a heavy (A = 238) nuclide with flat
    elastic cross sections (light share p_light of Sigma_el), listed in the material in the order [light, heavy] while
    the nuclide table holds [heavy, dummy A = 16, light] -- so the column -> nuclide map matters.  Capture (on the
    heavy nuclide) is zero above E_cut and overwhelming below: a history slows down by elastic collisions only and is
    captured at its first collision below E_cut."""
    P = geom_infinite()
    E = np.exp(np.linspace(np.log(1e-5), np.log(2e7), n_grid))
    E[0], E[-1] = 1e-5, 2e7
    el = np.zeros((3, n_grid))
    ca = np.zeros((3, n_grid))
    el[0] = 1.0 - p_light      # heavy
    el[1] = 123.0              # never used by the material
    el[2] = p_light            # light
    ca[0] = np.where(E < E_cut, 1.0e7, 0.0)
    P.update(mode="ce", n_mat=1, grid=E, nuc_A=np.array([238.0, 16.0, 1.0]), nuc_el=el, nuc_c=ca,
             nuc_f=np.zeros((3, n_grid)), mat_nuc_off=np.array([0, 2], np.int32), mat_nuc_id=np.array([2, 0], np.int32),
             mat_nuc_dens=np.array([1.0, 1.0]), nu0=0.0, nu1=0.0, watt_a=0.988, watt_b=2.249)
    P["t_edges"] = np.array([0.0, 1.0e3])
    P["e_edges"] = np.exp(np.linspace(np.log(1e-5), np.log(2e7), 101))
    P["e_edges"][0], P["e_edges"][-1] = 1e-5, 2e7
    P.update(_src([0, 0, 0], [0, 0, 0], E=E0, t=0.0))
    P["run"] = dict(kind="fixed", n_particles=n_particles, n_inactive=0, n_active=1, seed=seed)
    P["name"] = "ce_mix"
    return P


def ce_scatter_clock(lam=3.0e6, T=4.0e-6, A=1.0, n_particles=20_000, seed=41, E0=1.0e5, n_grid=6000):
    """Time pin of the elastic branch: one nuclide (mass ratio A) whose only reaction is elastic scattering with
    Sigma_el(E) = lam / v(E), in an infinite medium, run to the single time edge T.  The collision rate per unit TIME
    is then lam whatever the energy history, so collisions per history ~ Poisson(lam T) -- only if every flight
    advances the clock by d / v(E of that flight).  (Lin-lin interpolation of a 1/v curve on the fine log grid is
    accurate to < 1e-6 relative; the energy floor E_min is never reached: the mean lethargy gain lam T is far less than
    ln(E0 / E_min).)"""
    P = geom_infinite()
    E = np.exp(np.linspace(np.log(1e-5), np.log(2e7), n_grid))
    E[0], E[-1] = 1e-5, 2e7
    v = 2.99792458e10 * np.sqrt(2.0 * E / 939.56542052e6)
    P.update(mode="ce", n_mat=1, grid=E, nuc_A=np.array([float(A)]), nuc_el=(lam / v)[None, :].copy(),
             nuc_c=np.zeros((1, n_grid)), nuc_f=np.zeros((1, n_grid)), mat_nuc_off=np.array([0, 1], np.int32),
             mat_nuc_id=np.array([0], np.int32), mat_nuc_dens=np.array([1.0]), nu0=0.0, nu1=0.0, watt_a=0.988,
             watt_b=2.249)
    P["t_edges"] = np.array([0.0, float(T)])
    P["e_edges"] = np.array([1e-5, 2e7])
    P.update(_src([0, 0, 0], [0, 0, 0], E=E0, t=0.0))
    P["run"] = dict(kind="fixed", n_particles=n_particles, n_inactive=0, n_active=1, seed=seed)
    P["name"] = "ce_clock"
    return P


def ce_pure_fission(n_particles=50_000, seed=19, E0=1.0e6, n_grid=500):
    """One nuclide whose only reaction is fission, children killed by the first time edge
    (Watt/nu pin: child energies and multiplicities are read from the trace/counters)."""
    P = ce_single_scatterer(A=235.0, n_particles=n_particles, seed=seed, E0=E0, n_grid=n_grid)
    P["nuc_el"][:] = 0.0
    P["nuc_c"][:] = 0.0
    P["nuc_f"][:] = 1.0
    P.update(nu0=2.4, nu1=0.1)
    P["t_edges"] = np.array([0.0, 1.0e-12])
    P["name"] = "ce_fission"
    return P


CONFIGS = dict(C1=config1, C2=config2, C3=config3, C4=config4, C5=config5)
