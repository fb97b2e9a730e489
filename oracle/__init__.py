"""ctypes loader for the CPU ORACLE (test infrastructure, not the product).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It builds oracle/mcdc_oracle.c with gcc (-O2, no -ffast-math, no -march:
so no FMA contraction) and exposes the C entry points.  Nothing here is imported by, or imports,
paper_2501_05440_b200's CUDA binding.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libmcdc_oracle.so")
_SRC = [os.path.join(_HERE, "mcdc_oracle.c"), os.path.join(_HERE, "mcdc_oracle.h")]

N_COUNTERS = 16
EV_NAMES = {1: "scatter", 2: "fission", 3: "capture", 4: "transmit", 5: "reflect", 6: "leak", 7: "lattice",
            8: "time_edge", 9: "cutoff", 10: "lost"}

_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int32)


class OrcInput(C.Structure):
    _fields_ = [
        ("mode", C.c_int32),
        ("n_surf", C.c_int32), ("surf_type", _ip), ("surf_param", _dp), ("surf_bc", _ip),
        ("n_cell", C.c_int32), ("cell_surf_off", _ip), ("cell_surf_id", _ip), ("cell_surf_sense", _ip),
        ("cell_fill_type", _ip), ("cell_fill", _ip), ("cell_bin", _ip),
        ("n_univ", C.c_int32), ("univ_cell_off", _ip),
        ("has_lat", C.c_int32), ("lat_x0", C.c_double), ("lat_y0", C.c_double), ("lat_px", C.c_double),
        ("lat_py", C.c_double), ("lat_nx", C.c_int32), ("lat_ny", C.c_int32), ("lat_univ", _ip), ("lat_bin", _ip),
        ("n_lat2", C.c_int32), ("lat2_nx", _ip), ("lat2_ny", _ip), ("lat2_px", _dp), ("lat2_py", _dp), ("lat2_off", _ip),
        ("lat2_univ", _ip), ("lat2_bin", _ip),
        ("n_bins", C.c_int32), ("n_mat", C.c_int32),
        ("G", C.c_int32), ("sig_t", _dp), ("sig_f", _dp), ("nu", _dp), ("chi", _dp), ("S", _dp),
        ("n_grid", C.c_int32), ("grid", _dp), ("n_nuc", C.c_int32), ("nuc_A", _dp),
        ("nuc_el", _dp), ("nuc_c", _dp), ("nuc_f", _dp),
        ("mat_nuc_off", _ip), ("mat_nuc_id", _ip), ("mat_nuc_dens", _dp),
        ("nu0", C.c_double), ("nu1", C.c_double), ("watt_a", C.c_double), ("watt_b", C.c_double),
        ("n_t", C.c_int32), ("t_edges", _dp), ("n_e", C.c_int32), ("e_edges", _dp),
        ("src_lo", C.c_double * 3), ("src_hi", C.c_double * 3), ("src_iso", C.c_int32),
        ("src_dir", C.c_double * 3), ("src_group_pdf", _dp), ("src_E", C.c_double), ("src_t", C.c_double),
        ("kT", C.c_double), ("implicit_capture", C.c_int32), ("w_roulette", C.c_double), ("w_survive", C.c_double),
        ("td", C.c_int32), ("n_dgroup", C.c_int32), ("speed", _dp), ("nu_d", _dp), ("decay", _dp), ("chi_d", _dp),
        ("census_target", C.c_int64),
    ]


TRACE_DTYPE = np.dtype([("id", "<u8"), ("cycle", "<u4"), ("seq", "<u4"), ("ev", "<i4"), ("c0", "<i4"),
                        ("elem", "<i4"), ("c1", "<i4"), ("surf", "<i4"), ("gi", "<i4"), ("x", "<f8"), ("y", "<f8"),
                        ("z", "<f8"), ("d", "<f8"), ("E", "<f8"), ("t", "<f8")], align=True)
SITE_DTYPE = np.dtype([("x", "<f8"), ("y", "<f8"), ("z", "<f8"), ("ux", "<f8"), ("uy", "<f8"), ("uz", "<f8"),
                       ("g", "<i4"), ("pad", "<i4")], align=True)


_SO_SAN = os.path.join(_HERE, "libmcdc_oracle_san.so")


def build(force: bool = False) -> str:
    """Compile the oracle (gcc -O2).  Building the checker is not using it.

    MCDC_ORACLE_SANITIZE=1 in the environment builds and loads an AddressSanitizer + UndefinedBehaviorSanitizer
    instrumented copy instead (profiles/r03_oracle_sanitizers.md gives the command and its result)."""
    if os.environ.get("MCDC_ORACLE_SANITIZE") == "1":
        if force or not os.path.exists(_SO_SAN) or any(os.path.getmtime(s) > os.path.getmtime(_SO_SAN) for s in _SRC):
            subprocess.check_call(["gcc", "-O1", "-g", "-std=c99", "-fopenmp", "-fPIC", "-shared", "-fno-omit-frame-pointer",
                                   "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined",
                                   "-o", _SO_SAN, _SRC[0], "-lm"])
        return _SO_SAN
    if force or not os.path.exists(_SO) or any(os.path.getmtime(s) > os.path.getmtime(_SO) for s in _SRC):
        subprocess.check_call(["gcc", "-O2", "-std=c99", "-fopenmp", "-fPIC", "-shared", "-o", _SO, _SRC[0], "-lm"])
    return _SO


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.orc_create.restype = C.c_void_p
        L.orc_create.argtypes = [C.POINTER(OrcInput)]
        L.orc_destroy.argtypes = [C.c_void_p]
        L.orc_set_trace.argtypes = [C.c_void_p, C.c_uint64, C.c_uint64, C.c_uint64]
        L.orc_run_eigenvalue.argtypes = [C.c_void_p, C.c_uint64, C.c_int, C.c_int, C.c_uint64]
        L.orc_run_eigenvalue_mt.argtypes = [C.c_void_p, C.c_uint64, C.c_int, C.c_int, C.c_uint64, C.c_int]
        L.orc_run_fixed_source.argtypes = [C.c_void_p, C.c_uint64, C.c_uint64]
        L.orc_run_td.argtypes = [C.c_void_p, C.c_uint64, C.c_uint64]
        L.orc_get_census.argtypes = [C.c_void_p, C.POINTER(C.c_uint64), _dp, C.c_int]
        L.orc_comb.restype = C.c_double
        L.orc_comb.argtypes = [_dp, C.c_uint64, C.c_uint64, C.c_double, C.POINTER(C.c_uint32)]
        L.orc_n_tally.restype = C.c_int64
        L.orc_n_tally.argtypes = [C.c_void_p]
        L.orc_get_results.argtypes = [C.c_void_p, _dp, _dp, _dp, _dp, _dp, _dp, _dp, C.POINTER(C.c_uint64)]
        L.orc_get_trace.restype = C.c_uint64
        L.orc_get_trace.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64]
        L.orc_get_bank.restype = C.c_uint64
        L.orc_get_bank.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64]
        L.orc_get_balance.argtypes = [C.c_void_p, _dp]
        L.orc_free_gas.argtypes = [C.c_double, _dp, C.c_double, C.c_double, C.c_uint64, C.c_uint64, C.c_uint32,
                                   C.POINTER(C.c_uint32), _dp, _dp]
        L.orc_philox4x32_10.argtypes = [C.POINTER(C.c_uint32), C.POINTER(C.c_uint32), C.POINTER(C.c_uint32)]
        L.orc_draw.restype = C.c_double
        L.orc_draw.argtypes = [C.c_uint64, C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32]
        L.orc_child_id.restype = C.c_uint64
        L.orc_child_id.argtypes = [C.c_uint64, C.c_uint64, C.c_uint32, C.c_uint32]
        L.orc_grid_index.restype = C.c_int32
        L.orc_grid_index.argtypes = [C.c_void_p, C.c_double]
        L.orc_ce_xs.argtypes = [C.c_void_p, C.c_int32, C.c_double, _dp]
        L.orc_locate.argtypes = [C.c_void_p, _dp, _dp, C.c_int32, _ip]
        L.orc_distance.restype = C.c_double
        L.orc_distance.argtypes = [C.c_void_p, _dp, _dp, _ip, C.c_int32, _ip]
        L.orc_iso_dir.argtypes = [C.c_double, C.c_double, _dp]
        L.orc_elastic.argtypes = [C.c_double, _dp, C.c_double, C.c_double, C.c_double, _dp, _dp]
        L.orc_watt.restype = C.c_double
        L.orc_watt.argtypes = [C.c_double] * 6
        L.orc_speed.restype = C.c_double
        L.orc_speed.argtypes = [C.c_double]
        _lib = L
    return _lib


def _d(a):
    return np.ascontiguousarray(a, np.float64)


def _i(a):
    return np.ascontiguousarray(a, np.int32)


class Oracle:
    """One oracle problem built from a problem dict (paper_2501_05440_b200.inputs)."""

    def __init__(self, P: dict):
        self.P = P
        self._keep = []
        inp = OrcInput()

        def dp(a):
            a = _d(a)
            self._keep.append(a)
            return a.ctypes.data_as(_dp)

        def ip(a):
            a = _i(a)
            self._keep.append(a)
            return a.ctypes.data_as(_ip)

        ce = P["mode"] == "ce"
        inp.mode = 1 if ce else 0
        inp.n_surf = len(P["surf_type"])
        inp.surf_type, inp.surf_param, inp.surf_bc = ip(P["surf_type"]), dp(P["surf_param"]), ip(P["surf_bc"])
        inp.n_cell = len(P["cell_fill"])
        inp.cell_surf_off, inp.cell_surf_id = ip(P["cell_surf_off"]), ip(P["cell_surf_id"])
        inp.cell_surf_sense = ip(P["cell_surf_sense"])
        inp.cell_fill_type, inp.cell_fill, inp.cell_bin = ip(P["cell_fill_type"]), ip(P["cell_fill"]), ip(P["cell_bin"])
        inp.n_univ = len(P["univ_cell_off"]) - 1
        inp.univ_cell_off = ip(P["univ_cell_off"])
        lat = P.get("lat")
        inp.has_lat = 1 if lat else 0
        if lat:
            inp.lat_x0, inp.lat_y0, inp.lat_px, inp.lat_py = lat["x0"], lat["y0"], lat["px"], lat["py"]
            inp.lat_nx, inp.lat_ny = lat["nx"], lat["ny"]
            inp.lat_univ, inp.lat_bin = ip(lat["univ"]), ip(lat["bin"])
        inp.n_lat2 = len(P["lat2_nx"]) if "lat2_nx" in P else 0
        if inp.n_lat2:
            inp.lat2_nx, inp.lat2_ny, inp.lat2_off = ip(P["lat2_nx"]), ip(P["lat2_ny"]), ip(P["lat2_off"])
            inp.lat2_px, inp.lat2_py = dp(P["lat2_px"]), dp(P["lat2_py"])
            inp.lat2_univ, inp.lat2_bin = ip(P["lat2_univ"]), ip(P["lat2_bin"])
        inp.n_bins, inp.n_mat = P["n_bins"], P["n_mat"]
        if not ce:
            inp.G = P["G"]
            inp.sig_t, inp.sig_f, inp.nu, inp.chi = dp(P["mg_sig_t"]), dp(P["mg_sig_f"]), dp(P["mg_nu"]), dp(P["mg_chi"])
            inp.S = dp(P["mg_S"])
            inp.src_group_pdf = dp(P["src_group_pdf"])
        else:
            inp.n_grid, inp.grid = len(P["grid"]), dp(P["grid"])
            inp.n_nuc, inp.nuc_A = len(P["nuc_A"]), dp(P["nuc_A"])
            inp.nuc_el, inp.nuc_c, inp.nuc_f = dp(P["nuc_el"]), dp(P["nuc_c"]), dp(P["nuc_f"])
            inp.mat_nuc_off, inp.mat_nuc_id = ip(P["mat_nuc_off"]), ip(P["mat_nuc_id"])
            inp.mat_nuc_dens = dp(P["mat_nuc_dens"])
            inp.nu0, inp.nu1, inp.watt_a, inp.watt_b = P["nu0"], P["nu1"], P["watt_a"], P["watt_b"]
            inp.n_t, inp.t_edges = len(P["t_edges"]) - 1, dp(P["t_edges"])
            inp.n_e, inp.e_edges = len(P["e_edges"]) - 1, dp(P["e_edges"])
            inp.src_E = P["src_E"]
        inp.src_lo = (C.c_double * 3)(*P["src_lo"])
        inp.src_hi = (C.c_double * 3)(*P["src_hi"])
        inp.src_iso = int(P["src_iso"])
        inp.src_dir = (C.c_double * 3)(*P["src_dir"])
        inp.src_t = P.get("src_t", 0.0)
        inp.kT = float(P.get("kT", 0.0))
        inp.implicit_capture = int(P.get("implicit_capture", 0))
        inp.w_roulette = float(P.get("w_roulette", 0.25))
        inp.w_survive = float(P.get("w_survive", 1.0))
        td = P.get("td")
        inp.td = 1 if td else 0
        if td:  # time-dependent multi-group: speeds, delayed-neutron data, time edges, census population target
            inp.n_dgroup = int(td["J"])
            inp.speed, inp.nu_d, inp.decay, inp.chi_d = dp(td["speed"]), dp(td["nu_d"]), dp(td["decay"]), dp(td["chi_d"])
            inp.census_target = int(td.get("census_target", 0))
            inp.n_t, inp.t_edges = len(P["t_edges"]) - 1, dp(P["t_edges"])
        self.L = lib()
        self.h = self.L.orc_create(C.byref(inp))
        self.n_tally = self.L.orc_n_tally(self.h)
        self.n_cycles = 0

    def __del__(self):
        try:
            if self.h:
                self.L.orc_destroy(self.h)
                self.h = None
        except Exception:
            pass

    def set_trace(self, first_id=0, n_ids=100, max_records=1_000_000):
        self.L.orc_set_trace(self.h, first_id, n_ids, max_records)
        self._tr_max = max_records

    def run_mt(self, n_threads, n_particles=None, n_inactive=None, n_active=None, seed=None):
        """All-core timing variant of the eigenvalue run (see mcdc_oracle.c); not used by the parity tests."""
        r = self.P["run"]
        N = int(n_particles if n_particles is not None else r["n_particles"])
        ni = int(n_inactive if n_inactive is not None else r["n_inactive"])
        na = int(n_active if n_active is not None else r["n_active"])
        sd = int(seed if seed is not None else r["seed"])
        rc = self.L.orc_run_eigenvalue_mt(self.h, N, ni, na, sd, int(n_threads))
        self.n_cycles = ni + na
        return rc, self.results()

    def run(self, n_particles=None, n_inactive=None, n_active=None, seed=None):
        r = self.P["run"]
        N = int(n_particles if n_particles is not None else r["n_particles"])
        ni = int(n_inactive if n_inactive is not None else r["n_inactive"])
        na = int(n_active if n_active is not None else r["n_active"])
        sd = int(seed if seed is not None else r["seed"])
        if r["kind"] == "eigen":
            rc = self.L.orc_run_eigenvalue(self.h, N, ni, na, sd)
            self.n_cycles = ni + na
        elif r["kind"] == "td":
            rc = self.L.orc_run_td(self.h, N, sd)
            self.n_cycles = 1
        else:
            rc = self.L.orc_run_fixed_source(self.h, N, sd)
            self.n_cycles = 1
        return rc, self.results()

    def results(self):
        kc = np.zeros(max(self.n_cycles, 1))
        fm, fs = np.zeros(self.n_tally), np.zeros(self.n_tally)
        sc = [C.c_double() for _ in range(4)]
        cnt = np.zeros(N_COUNTERS, np.uint64)
        rc = self.L.orc_get_results(self.h, kc.ctypes.data_as(_dp), C.byref(sc[0]), C.byref(sc[1]),
                                    fm.ctypes.data_as(_dp), fs.ctypes.data_as(_dp), C.byref(sc[2]), C.byref(sc[3]),
                                    cnt.ctypes.data_as(C.POINTER(C.c_uint64)))
        return dict(rc=rc, k_cycle=kc[: self.n_cycles], k_mean=sc[0].value, k_sdev=sc[1].value, flux_mean=fm,
                    flux_sdev=fs, leak_mean=sc[2].value, leak_sdev=sc[3].value, counters=cnt)

    def balance(self):
        """Weight balance of the last run: dict(source, absorbed, leaked, cutoff, roulette_loss, roulette_gain)."""
        out = np.zeros(6)
        self.L.orc_get_balance(self.h, out.ctypes.data_as(_dp))
        return dict(zip(("source", "absorbed", "leaked", "cutoff", "roulette_loss", "roulette_gain"), out))

    def census(self):
        """Population entering each census interval of the last time-dependent multi-group run:
        (particles before the comb, after it, weight before, weight after) per interval."""
        cnt, w = np.zeros(128, np.uint64), np.zeros(128)
        n = self.L.orc_get_census(self.h, cnt.ctypes.data_as(C.POINTER(C.c_uint64)), w.ctypes.data_as(_dp), 64)
        return [(int(cnt[2 * k]), int(cnt[2 * k + 1]), float(w[2 * k]), float(w[2 * k + 1])) for k in range(n)]

    def trace(self):
        n = self.L.orc_get_trace(self.h, None, 0)
        n = min(n, self._tr_max)
        out = np.zeros(n, TRACE_DTYPE)
        if n:
            self.L.orc_get_trace(self.h, out.ctypes.data, n)
        return out

    def bank(self):
        n = self.L.orc_get_bank(self.h, None, 0)
        out = np.zeros(n, SITE_DTYPE)
        if n:
            self.L.orc_get_bank(self.h, out.ctypes.data, n)
        return out

    # unit-level helpers for the pins
    def grid_index(self, E):
        return int(self.L.orc_grid_index(self.h, float(E)))

    def ce_xs(self, m, E):
        out = np.zeros(64)
        nc = self.L.orc_ce_xs(self.h, int(m), float(E), out.ctypes.data_as(_dp))
        return out[: nc + 1].copy()

    def locate(self, x, u, last_surf=-1):
        x, u = _d(x), _d(u)
        loc = np.zeros(3, np.int32)
        rc = self.L.orc_locate(self.h, x.ctypes.data_as(_dp), u.ctypes.data_as(_dp), last_surf, loc.ctypes.data_as(_ip))
        return rc, loc

    def distance(self, x, u, loc, last_surf=-1):
        x, u, loc = _d(x), _d(u), _i(loc)
        s = C.c_int32()
        d = self.L.orc_distance(self.h, x.ctypes.data_as(_dp), u.ctypes.data_as(_dp), loc.ctypes.data_as(_ip),
                                last_surf, C.byref(s))
        return d, s.value


def philox(ctr, key):
    c = (C.c_uint32 * 4)(*ctr)
    k = (C.c_uint32 * 2)(*key)
    o = (C.c_uint32 * 4)()
    lib().orc_philox4x32_10(c, k, o)
    return [int(v) for v in o]


def draw(seed, pid, domain, cycle, index):
    return lib().orc_draw(seed, pid, domain, cycle, index)


def iso_dir(a, b):
    o = np.zeros(3)
    lib().orc_iso_dir(a, b, o.ctypes.data_as(_dp))
    return o


def elastic(E, u, A, a, b):
    u = _d(u)
    o = np.zeros(3)
    e = C.c_double()
    lib().orc_elastic(E, u.ctypes.data_as(_dp), A, a, b, C.byref(e), o.ctypes.data_as(_dp))
    return e.value, o


def free_gas(E, u, A, kT, seed, pid, cycle=0, ctr=0):
    """One free-gas collision drawn from stream (seed, pid, 0, cycle) starting at draw ctr: (E', u', draws used)."""
    u = _d(u)
    o = np.zeros(3)
    e = C.c_double()
    c = C.c_uint32(ctr)
    lib().orc_free_gas(E, u.ctypes.data_as(_dp), A, kT, seed, pid, cycle, C.byref(c), C.byref(e), o.ctypes.data_as(_dp))
    return e.value, o, c.value - ctr


def watt(a, b, x1, x2, x3, x4):
    return lib().orc_watt(a, b, x1, x2, x3, x4)


def speed(E):
    return lib().orc_speed(E)


def comb(w, n_teeth, xi):
    """The population-control comb on plain arrays (orc_comb): copies per particle and the tooth spacing."""
    w = _d(w)
    copies = np.zeros(len(w), np.uint32)
    delta = lib().orc_comb(w.ctypes.data_as(_dp), len(w), int(n_teeth), float(xi), copies.ctypes.data_as(C.POINTER(C.c_uint32)))
    return copies, delta
