"""Independent tiny pure-Python tracer used ONLY to pin the oracle's event sequences (SURVEY.md 8c "Event
sequences").  Different structure from oracle/mcdc_oracle.c on purpose: Philox on Python integers, geometry
by brute force over ALL surfaces of the problem (no per-cell surface lists, no last-surface logic: a root closer
than 1e-9 is the surface the particle sits on), cell by point-in-cell test a little way along the flight.
Multi-group, single-level geometry only (C1, C3, slab, sphere)."""
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


def _f(P, s, x):
    t, q = int(P["surf_type"][s]), P["surf_param"][s]
    if t <= 2:
        return x[t] - q[0]
    if t == 3:
        return q[0] * x[0] + q[1] * x[1] + q[2] * x[2] - q[3]
    if t == 7:
        return sum((x[i] - q[i]) ** 2 for i in range(3)) - q[3] ** 2
    ax = [i for i in range(3) if i != t - 4]
    return (x[ax[0]] - q[0]) ** 2 + (x[ax[1]] - q[1]) ** 2 - q[2] ** 2


def _roots(P, s, x, u):
    t, q = int(P["surf_type"][s]), P["surf_param"][s]
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


def _cell_at(P, x):
    for c in range(len(P["cell_fill"])):
        lo, hi = P["cell_surf_off"][c], P["cell_surf_off"][c + 1]
        if all((_f(P, P["cell_surf_id"][k], x) > 0) == (P["cell_surf_sense"][k] > 0) for k in range(lo, hi)):
            return c
    return -1


def _normal(P, s, x):
    t, q = int(P["surf_type"][s]), P["surf_param"][s]
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
    """Events of histories 0..n_hist-1 of cycle 0: list of (id, seq, ev, surf, g_before, x, y, z, d)."""
    G = P["G"]
    out = []
    ns = len(P["surf_type"])
    for pid in range(n_hist):
        xi = Stream(seed, pid, 0)
        r = [xi() for _ in range(6)]
        x = [P["src_lo"][i] + r[i] * (P["src_hi"][i] - P["src_lo"][i]) for i in range(3)]
        u = _iso(r[3], r[4]) if P["src_iso"] else list(P["src_dir"])
        pdf = list(P["src_group_pdf"])
        g = _pick(pdf, r[5] * sum(pdf))
        w, seq, alive = 1.0, 0, True
        while alive:
            cands = sorted((d, s) for s in range(ns) for d in _roots(P, s, x, u) if d > 1e-9)
            probe = min(cands[0][0], 1.0) * 0.5 if cands else 0.0
            cell = _cell_at(P, [x[i] + probe * 1e-3 * u[i] for i in range(3)])
            # the event is the first crossing that changes the cell (or meets a boundary condition): a surface
            # that merely passes through a cell which does not list it is not a boundary there
            d_surf, s_hit = math.inf, -1
            for dc, sc in cands:
                if int(P["surf_bc"][sc]) != 0 or _cell_at(P, [x[i] + (dc + 1e-7) * u[i] for i in range(3)]) != cell:
                    d_surf, s_hit = dc, sc
                    break
            m = int(P["cell_fill"][cell])
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
                out.append((pid, seq, ev, -1, g0, x[0], x[1], x[2], d))
            else:
                d = d_surf
                x = [x[i] + d * u[i] for i in range(3)]
                bc = int(P["surf_bc"][s_hit])
                if bc == 2:
                    ev, alive = 6, False
                elif bc == 1:
                    ev = 5
                    n = _normal(P, s_hit, x)
                    dot = sum(u[i] * n[i] for i in range(3))
                    u = [u[i] - 2 * dot * n[i] for i in range(3)]
                else:
                    ev = 4
                out.append((pid, seq, ev, s_hit, g0, x[0], x[1], x[2], d))
            seq += 1
    return out
