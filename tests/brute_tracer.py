"""Independent tiny pure-Python tracer used ONLY to pin the oracle's event sequences (SURVEY.md 8c "Event
sequences").  Different structure from oracle/mcdc_oracle.c on purpose: Philox on Python integers, geometry by
brute force over ALL surfaces of the problem -- with a lattice: every root surface, every grid line and the
surfaces of EVERY element's universe moved to that element's centre -- no per-cell surface lists, no neighbour or
last-surface logic (a root closer than 1e-9 is the surface the particle sits on), location by point-in-cell test a
little way along the flight, and an event is the first crossing after which the location differs.
Multi-group eigenvalue cycle 0 (`trace_cycle0`) and the continuous-energy time-dependent fixed-source run with its
prompt secondaries (`trace_ce`, physics per SURVEY.md 8c: union-grid lin-lin interpolation nuclide by nuclide, target-
at-rest elastic kinematics, Watt spectrum, time edges)."""
import bisect
import math

M32 = 0xFFFFFFFF


def philox(c, k):
    c0, c1, c2, c3 = c
    k0, k1 = k
    for _ in range(10):
        p0 = 0xD2511F53 * c0
        p1 = 0xCD9E8D57 * c2
        c0, c1, c2, c3 = ((p1 >> 32) ^ c1 ^ k0) & M32, p1 & M32, ((p0 >> 32) ^ c3 ^ k1) & M32, p0 & M32
        k0 = (k0 + 0x9E3779B9) & M32
        k1 = (k1 + 0xBB67AE85) & M32
    return c0, c1, c2, c3


class Stream:
    def __init__(self, seed, pid, cycle):
        self.key = (seed & M32, seed >> 32)
        self.base = (pid & M32, pid >> 32, cycle)
        self.n = 0

    def __call__(self):
        o = philox(self.base + (self.n >> 1,), self.key)
        u = (o[3] << 32 | o[2]) if self.n & 1 else (o[1] << 32 | o[0])
        self.n += 1
        return ((u >> 11) + 0.5) / 9007199254740992.0


def child_id(seed, parent, parent_ctr, j):
    o = philox((parent & M32, parent >> 32, (1 << 24) | j, parent_ctr), (seed & M32, seed >> 32))
    return o[1] << 32 | o[0]


# --------------------------------------------------------------------------- brute-force geometry
def _f(t, q, x):
    if t <= 2:
        return x[t] - q[0]
    if t == 3:
        return q[0] * x[0] + q[1] * x[1] + q[2] * x[2] - q[3]
    if t == 7:
        return sum((x[i] - q[i]) ** 2 for i in range(3)) - q[3] ** 2
    ax = [i for i in range(3) if i != t - 4]
    return (x[ax[0]] - q[0]) ** 2 + (x[ax[1]] - q[1]) ** 2 - q[2] ** 2


def _roots(t, q, x, u):
    if t <= 2:
        return [] if u[t] == 0 else [(q[0] - x[t]) / u[t]]
    if t == 3:
        den = q[0] * u[0] + q[1] * u[1] + q[2] * u[2]
        return [] if den == 0 else [(q[3] - (q[0] * x[0] + q[1] * x[1] + q[2] * x[2])) / den]
    if t == 7:
        ax, ctr, r = [0, 1, 2], q[:3], q[3]
    else:
        ax, ctr, r = [i for i in range(3) if i != t - 4], q[:2], q[2]
    a = sum(u[i] ** 2 for i in ax)
    k = sum((x[i] - c) * u[i] for i, c in zip(ax, ctr))
    cc = sum((x[i] - c) ** 2 for i, c in zip(ax, ctr)) - r * r
    disc = k * k - a * cc
    if a == 0 or disc < 0:
        return []
    sq = math.sqrt(disc)
    return [(-k - sq) / a, (-k + sq) / a]


def _normal(t, q, x):
    n = [0.0, 0.0, 0.0]
    if t <= 2:
        n[t] = 1.0
    elif t == 3:
        n = list(q[:3])
    elif t == 7:
        n = [x[i] - q[i] for i in range(3)]
    else:
        ax = [i for i in range(3) if i != t - 4]
        n[ax[0]], n[ax[1]] = x[ax[0]] - q[0], x[ax[1]] - q[1]
    nn = math.sqrt(sum(v * v for v in n))
    return [v / nn for v in n]


class World:
    """The whole problem as one flat list of crossing candidates."""

    def __init__(self, P):
        self.P = P
        self.st = [int(t) for t in P["surf_type"]]
        self.sq = [[float(v) for v in q] for q in P["surf_param"]]
        self.bc = [int(b) for b in P["surf_bc"]]
        self.ns = len(self.st)
        self.uoff = [int(v) for v in P["univ_cell_off"]]
        self.lat = P.get("lat")
        if self.lat:
            L = self.lat
            self.nx, self.ny = int(L["nx"]), int(L["ny"])
            self.x0, self.y0, self.px, self.py = float(L["x0"]), float(L["y0"]), float(L["px"]), float(L["py"])
            self.univ = [[int(v) for v in row] for row in L["univ"]]
        # second-level lattices: (nx, ny, px, py, x0, y0, universes[iy][ix], bins[iy][ix]), centred on the origin of the
        # universe whose cell (fill type 2) they fill
        self.lat2 = []
        for k in range(len(P.get("lat2_nx", []))):
            nx, ny = int(P["lat2_nx"][k]), int(P["lat2_ny"][k])
            px, py, o = float(P["lat2_px"][k]), float(P["lat2_py"][k]), int(P["lat2_off"][k])
            un = [[int(P["lat2_univ"][o + iy * nx + ix]) for ix in range(nx)] for iy in range(ny)]
            bn = [[int(P["lat2_bin"][o + iy * nx + ix]) for ix in range(nx)] for iy in range(ny)]
            self.lat2.append((nx, ny, px, py, -0.5 * nx * px, -0.5 * ny * py, un, bn))

    def _lat2_of(self, univ):
        """(cell, lattice) of the second-level lattice that fills a cell of `univ`, or None."""
        for c in range(self.uoff[univ], self.uoff[univ + 1]):
            if int(self.P["cell_fill_type"][c]) == 2:
                return c, self.lat2[int(self.P["cell_fill"][c])]
        return None

    def _in_cell(self, c, x):
        P = self.P
        lo, hi = P["cell_surf_off"][c], P["cell_surf_off"][c + 1]
        return all((_f(self.st[P["cell_surf_id"][k]], self.sq[P["cell_surf_id"][k]], x) > 0) == (P["cell_surf_sense"][k] > 0)
                   for k in range(lo, hi))

    def _cell_in(self, univ, x):
        for c in range(self.uoff[univ], self.uoff[univ + 1]):
            if self._in_cell(c, x):
                return c
        return -1

    def where(self, x):
        """(c0, elem, c1) of a point, or None when it is in no cell."""
        c0 = self._cell_in(0, x)
        if c0 < 0:
            return None
        if int(self.P["cell_fill_type"][c0]) != 1:
            return (c0, -1, -1)
        ix, iy = math.floor((x[0] - self.x0) / self.px), math.floor((x[1] - self.y0) / self.py)
        if not (0 <= ix < self.nx and 0 <= iy < self.ny):
            return None
        xl = [x[0] - (self.x0 + (ix + 0.5) * self.px), x[1] - (self.y0 + (iy + 0.5) * self.py), x[2]]
        c1 = self._cell_in(self.univ[iy][ix], xl)
        if c1 < 0:
            return None
        elem = iy * self.nx + ix
        if int(self.P["cell_fill_type"][c1]) == 2:  # a lattice of its own fills this cell of the element's universe
            nx, ny, px, py, x0, y0, un, _ = self.lat2[int(self.P["cell_fill"][c1])]
            jx, jy = math.floor((xl[0] - x0) / px), math.floor((xl[1] - y0) / py)
            if not (0 <= jx < nx and 0 <= jy < ny):
                return None
            x2 = [xl[0] - (x0 + (jx + 0.5) * px), xl[1] - (y0 + (jy + 0.5) * py), xl[2]]
            c2 = self._cell_in(un[jy][jx], x2)
            return None if c2 < 0 else (c0, elem | ((jy * nx + jx + 1) << 20), c2)
        return (c0, elem, c1)

    def material(self, loc):
        return int(self.P["cell_fill"][loc[2] if loc[1] >= 0 else loc[0]])

    def spatial_bin(self, loc):
        b = int(self.P["cell_bin"][loc[2] if loc[1] >= 0 else loc[0]])
        if loc[1] >= 0:
            outer, inner = loc[1] & 0xFFFFF, (loc[1] >> 20) - 1
            b += int(self.lat["bin"].ravel()[outer])
            if inner >= 0:
                nx, _, _, _, _, _, _, bn = self._lat2_of(self.univ[outer // self.nx][outer % self.nx])[1]
                b += bn[inner // nx][inner % nx]
        return b

    def candidates(self, x, u):
        """Every positive crossing distance along the ray: (d, kind, id); kind 0 = a surface (root surfaces in
        global coordinates, universe surfaces moved to every element that holds the universe), 1 = a grid line
        (id = wall code n_surf + 0..3 by axis and direction of flight)."""
        P, out = self.P, []
        root_surfs = {int(P["cell_surf_id"][k]) for c in range(self.uoff[0], self.uoff[1])
                      for k in range(P["cell_surf_off"][c], P["cell_surf_off"][c + 1])}
        for s in root_surfs:
            out += [(d, 0, s) for d in _roots(self.st[s], self.sq[s], x, u) if d > 1e-9]
        if self.lat:
            for ax, (o, p, n) in enumerate(((self.x0, self.px, self.nx), (self.y0, self.py, self.ny))):
                if u[ax] != 0:
                    for k in range(n + 1):
                        d = (o + k * p - x[ax]) / u[ax]
                        if d > 1e-9:
                            out.append((d, 1, self.ns + 2 * ax + (1 if u[ax] > 0 else 0)))
            for iy in range(self.ny):
                for ix in range(self.nx):
                    un = self.univ[iy][ix]
                    surfs = {int(P["cell_surf_id"][k]) for c in range(self.uoff[un], self.uoff[un + 1])
                             for k in range(P["cell_surf_off"][c], P["cell_surf_off"][c + 1])}
                    xl = [x[0] - (self.x0 + (ix + 0.5) * self.px), x[1] - (self.y0 + (iy + 0.5) * self.py), x[2]]
                    for s in surfs:
                        out += [(d, 0, s) for d in _roots(self.st[s], self.sq[s], xl, u) if d > 1e-9]
                    l2 = self._lat2_of(un)
                    if l2 is None:
                        continue
                    # second level: every grid line of the inner lattice (wall codes n_surf + 4..7) and the surfaces of
                    # every inner element's universe, moved to that element's centre
                    nx2, ny2, px2, py2, x02, y02, un2, _ = l2[1]
                    for ax, (o, p, n) in enumerate(((x02, px2, nx2), (y02, py2, ny2))):
                        if u[ax] != 0:
                            for k in range(n + 1):
                                d = (o + k * p - xl[ax]) / u[ax]
                                if d > 1e-9:
                                    out.append((d, 1, self.ns + 4 + 2 * ax + (1 if u[ax] > 0 else 0)))
                    for jy in range(ny2):
                        for jx in range(nx2):
                            uu = un2[jy][jx]
                            surfs2 = {int(P["cell_surf_id"][k]) for c in range(self.uoff[uu], self.uoff[uu + 1])
                                      for k in range(P["cell_surf_off"][c], P["cell_surf_off"][c + 1])}
                            x2 = [xl[0] - (x02 + (jx + 0.5) * px2), xl[1] - (y02 + (jy + 0.5) * py2), xl[2]]
                            for s in surfs2:
                                out += [(d, 0, s) for d in _roots(self.st[s], self.sq[s], x2, u) if d > 1e-9]
        return sorted(out)

    def next_event(self, x, u):
        """(location now, distance, surface / wall code) of the first crossing that changes the location or meets a
        boundary condition; surface -1 and distance inf when there is none."""
        cands = self.candidates(x, u)
        probe = min(cands[0][0], 1.0) * 0.5e-3 if cands else 0.0
        here = self.where([x[i] + probe * u[i] for i in range(3)])
        i = 0
        while i < len(cands):
            d = cands[i][0]
            group = [c for c in cands[i:] if c[0] - d <= 1e-9 * (1.0 + d)]
            i += len(group)
            # a real surface with a boundary condition wins over a grid line at the same place (the lattice's outermost
            # lines are never events: the enclosing cell's surfaces bound it there, R14)
            real = [c for c in group if c[1] == 0]
            beyond = self.where([x[k] + (d + 1e-7) * u[k] for k in range(3)])
            for c in real:
                if self.bc[c[2]] != 0 and (beyond is None or beyond != here):
                    return here, c[0], c[2]
            if beyond is None or beyond == here:
                continue
            for c in real:
                return here, c[0], c[2]
            # grid lines only: where a first-level line and the rim of a second-level lattice coincide, the first-level
            # wall is the event (a lattice's outermost lines never are, R14 / R37)
            first = min(group, key=lambda c: c[2])
            return here, first[0], first[2]
        return here, math.inf, -1

    def reflect(self, s, x, u, loc):
        xl = list(x)
        if loc[1] >= 0 and not self._surface_of_root(s):
            ix, iy = (loc[1] & 0xFFFFF) % self.nx, (loc[1] & 0xFFFFF) // self.nx
            xl = [x[0] - (self.x0 + (ix + 0.5) * self.px), x[1] - (self.y0 + (iy + 0.5) * self.py), x[2]]
        n = _normal(self.st[s], self.sq[s], xl)
        dot = sum(u[i] * n[i] for i in range(3))
        return [u[i] - 2 * dot * n[i] for i in range(3)]

    def _surface_of_root(self, s):
        P = self.P
        return any(int(P["cell_surf_id"][k]) == s for c in range(self.uoff[0], self.uoff[1])
                   for k in range(P["cell_surf_off"][c], P["cell_surf_off"][c + 1]))


def _iso(a, b):
    mu, phi = 2 * a - 1, 2 * math.pi * b
    s = math.sqrt(1 - mu * mu)
    return [s * math.cos(phi), s * math.sin(phi), mu]


def _pick(row, v):
    acc = 0.0
    for i, r in enumerate(row):
        acc += r
        if acc > v:
            return i
    return len(row) - 1


def trace_cycle0(P, seed, n_hist, k_prev=1.0):
    """Multi-group: events of histories 0..n_hist-1 of cycle 0:
    list of (id, seq, ev, surf, g_before, x, y, z, d, elem, c1)."""
    W = World(P)
    out = []
    for pid in range(n_hist):
        xi = Stream(seed, pid, 0)
        r = [xi() for _ in range(6)]
        x = [P["src_lo"][i] + r[i] * (P["src_hi"][i] - P["src_lo"][i]) for i in range(3)]
        u = _iso(r[3], r[4]) if P["src_iso"] else list(P["src_dir"])
        pdf = list(P["src_group_pdf"])
        g = _pick(pdf, r[5] * sum(pdf))
        w, seq, alive = 1.0, 0, True
        while alive:
            loc, d_surf, s_hit = W.next_event(x, u)
            m = W.material(loc)
            st = float(P["mg_sig_t"][m][g])
            d_coll = -math.log(xi()) / st
            g0 = g
            if d_coll < d_surf:
                d = d_coll
                x = [x[i] + d * u[i] for i in range(3)]
                row = [float(v) for v in P["mg_S"][m][g]]
                ss, sf = sum(row), float(P["mg_sig_f"][m][g])
                t = xi() * st
                if t < ss:
                    ev = 1
                    g = _pick(row, xi() * ss)
                    a, b = xi(), xi()
                    u = _iso(a, b)
                elif t < ss + sf:
                    ev = 2
                    n = int(math.floor(w * float(P["mg_nu"][m][g]) / k_prev + xi()))
                    for _ in range(n):
                        xi(), xi(), xi()
                    alive = False
                else:
                    ev, alive = 3, False
                out.append((pid, seq, ev, -1, g0, x[0], x[1], x[2], d, loc[1], loc[2]))
            else:
                d = d_surf
                x = [x[i] + d * u[i] for i in range(3)]
                if s_hit >= W.ns:
                    ev = 7
                else:
                    bc = W.bc[s_hit]
                    if bc == 2:
                        ev, alive = 6, False
                    elif bc == 1:
                        ev = 5
                        u = W.reflect(s_hit, x, u, loc)
                    else:
                        ev = 4
                out.append((pid, seq, ev, s_hit, g0, x[0], x[1], x[2], d, loc[1], loc[2]))
            seq += 1
    return out


# --------------------------------------------------------------------------- continuous energy, time dependent
C_LIGHT, MN_C2 = 2.99792458e10, 939.56542052e6


def _interp(col, i, f):
    return float(col[i]) + f * (float(col[i + 1]) - float(col[i]))


def trace_ce(P, seed, n_src):
    """Fixed-source run of source particles 0..n_src-1 and all their prompt secondaries (depth first).
    Returns (events, counters, flux): events of the SOURCE particles as (id, seq, ev, surf, grid index, x, y, z, d,
    E of the flight, t after the move); counters[ev] over all tracks, counters[0] = tracks, counters[11] = secondaries;
    flux[tbin][ebin] = track length (unnormalised)."""
    W = World(P)
    grid = [float(v) for v in P["grid"]]
    ng = len(grid)
    te = [float(v) for v in P["t_edges"]]
    ee = [float(v) for v in P["e_edges"]]
    nt, ne = len(te) - 1, len(ee) - 1
    flux = [[0.0] * ne for _ in range(nt)]
    cnt = [0] * 16
    events = []
    A_of = [float(a) for a in P["nuc_A"]]
    a_w, b_w = float(P["watt_a"]), float(P["watt_b"])

    def clampE(E):
        return min(max(E, grid[0]), grid[-1])

    for src in range(n_src):
        xi = Stream(seed, src, 0)
        r = [xi() for _ in range(6)]
        x = [P["src_lo"][i] + r[i] * (P["src_hi"][i] - P["src_lo"][i]) for i in range(3)]
        u = _iso(r[3], r[4]) if P["src_iso"] else list(P["src_dir"])
        t0 = float(P.get("src_t", 0.0))
        tb0 = min(max(bisect.bisect_right(te, t0) - 1, 0), nt - 1)
        stack = [dict(id=src, x=x, u=u, E=float(P["src_E"]), t=t0, tb=tb0, xi=xi, traced=True)]
        while stack:
            q = stack.pop()
            cnt[0] += 1
            x, u, E, t, tb, xi, pid = q["x"], q["u"], q["E"], q["t"], q["tb"], q["xi"], q["id"]
            seq, alive = 0, True
            while alive:
                loc, d_surf, s_hit = W.next_event(x, u)
                m = W.material(loc)
                gi = min(max(bisect.bisect_right(grid, E) - 1, 0), ng - 2)
                f = (E - grid[gi]) / (grid[gi + 1] - grid[gi])
                n0, n1 = int(P["mat_nuc_off"][m]), int(P["mat_nuc_off"][m + 1])
                parts, sf, sc = [], 0.0, 0.0
                for j in range(n0, n1):  # nuclide by nuclide: interpolate the microscopic value, then the density
                    nuc, dens = int(P["mat_nuc_id"][j]), float(P["mat_nuc_dens"][j])
                    parts.append(dens * _interp(P["nuc_el"][nuc], gi, f))
                    sf += dens * _interp(P["nuc_f"][nuc], gi, f)
                    sc += dens * _interp(P["nuc_c"][nuc], gi, f)
                parts += [sf, sc]
                sig_t = sum(parts)
                v = C_LIGHT * math.sqrt(2.0 * E / MN_C2)
                d_coll = -math.log(xi()) / sig_t
                d_time = v * (te[tb + 1] - t)
                ebin = min(max(bisect.bisect_right(ee, E) - 1, 0), ne - 1)
                E_fl = E
                if d_coll < d_surf and d_coll < d_time:
                    d, kind = d_coll, 0
                elif d_surf <= d_time:
                    d, kind = d_surf, 1
                else:
                    d, kind = d_time, 2
                x = [x[i] + d * u[i] for i in range(3)]
                flux[tb][ebin] += d
                t = te[tb + 1] if kind == 2 else t + d / v
                surf = -1
                if kind == 0:
                    rsel = _pick(parts, xi() * sig_t)
                    if rsel < len(parts) - 2:
                        ev = 1
                        A = A_of[int(P["mat_nuc_id"][n0 + rsel])]
                        mu_cm = 2.0 * xi() - 1.0
                        den = A * A + 2.0 * A * mu_cm + 1.0
                        mu = (1.0 + A * mu_cm) / math.sqrt(den) if den > 0.0 else 0.0
                        E = clampE(E * den / ((A + 1.0) ** 2))
                        phi = 2.0 * math.pi * xi()
                        s = math.sqrt(max(1.0 - mu * mu, 0.0))
                        a2 = 1.0 - u[2] * u[2]
                        if a2 < 1e-10:
                            o = [s * math.cos(phi), s * math.sin(phi), mu if u[2] > 0 else -mu]
                        else:
                            rr = math.sqrt(a2)
                            o = [mu * u[0] + s * (u[0] * u[2] * math.cos(phi) - u[1] * math.sin(phi)) / rr,
                                 mu * u[1] + s * (u[1] * u[2] * math.cos(phi) + u[0] * math.sin(phi)) / rr,
                                 mu * u[2] - s * rr * math.cos(phi)]
                        nn = math.sqrt(sum(c * c for c in o))
                        u = [c / nn for c in o]
                    elif rsel == len(parts) - 2:
                        ev, alive = 2, False
                        nch = int(math.floor(float(P["nu0"]) + float(P["nu1"]) * (E * 1e-6) + xi()))
                        ctr_birth = xi.n
                        kids = []
                        for j in range(nch):
                            x1, x2, x3, x4 = xi(), xi(), xi(), xi()
                            cs = math.cos(0.5 * math.pi * x3)
                            Wm = -a_w * (math.log(x1) + math.log(x2) * cs * cs)
                            Ec = 1e6 * (Wm + 0.25 * a_w * a_w * b_w + (2.0 * x4 - 1.0) * math.sqrt(a_w * a_w * b_w * Wm))
                            da, db = xi(), xi()
                            cid = child_id(seed, pid, ctr_birth, j)
                            kids.append(dict(id=cid, x=list(x), u=_iso(da, db), E=clampE(Ec), t=t, tb=tb,
                                             xi=Stream(seed, cid, 0), traced=False))
                            cnt[11] += 1
                        stack += kids  # LIFO: the last child runs first
                    else:
                        ev, alive = 3, False
                elif kind == 1:
                    surf = s_hit
                    if s_hit >= W.ns:
                        ev = 7
                    elif W.bc[s_hit] == 2:
                        ev, alive = 6, False
                    elif W.bc[s_hit] == 1:
                        ev = 5
                        u = W.reflect(s_hit, x, u, loc)
                    else:
                        ev = 4
                else:
                    tb += 1
                    if tb == nt:
                        ev, alive = 9, False
                    else:
                        ev = 8
                cnt[ev] += 1
                if q["traced"]:
                    events.append((pid, seq, ev, surf, gi, x[0], x[1], x[2], d, E_fl, t))
                seq += 1
    return events, cnt, flux
