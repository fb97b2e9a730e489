"""Thin ctypes binding of the C-ABI CUDA library (include/mcdc.h): argument marshalling only.

PyTorch is used for device memory (the workspace tensor) and the stream; every step of the transport
path runs in the library's kernels.  There is no CPU fallback: if the built library or a CUDA device is
missing, construction raises.  This module never imports oracle/.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_ROOT = os.path.dirname(_HERE)
_SO = os.path.join(_HERE, "libmcdc_b200.so")
_SRC = [os.path.join(_HERE, "csrc", f) for f in ("mcdc_lib.cu", "mcdc_kernels.cuh", "mcdc_device.cuh", "mcdc_census.cuh",
                                                   "mcdc_microbench.cuh")]
_HDRS = [os.path.join(_ROOT, "include", f) for f in ("mcdc.h", "mcdc_test.h")]

N_COUNTERS = 16
NOALLOC_DRAWS_MAX = 65536  # MCDC_NOALLOC_DRAWS_MAX of include/mcdc.h
ALWAYS = 0x7FFFFFFF  # persist_threshold: the persistent kernel runs the whole cycle
EV_NAMES = {1: "scatter", 2: "fission", 3: "capture", 4: "transmit", 5: "reflect", 6: "leak", 7: "lattice",
            8: "time_edge", 9: "cutoff", 10: "lost"}
SYMBOLS = ["mcdc_workspace_bytes", "mcdc_create", "mcdc_run_eigenvalue", "mcdc_run_cycle", "mcdc_run_cycle_host",
           "mcdc_run_fixed_source", "mcdc_get_dims", "mcdc_get_tallies", "mcdc_get_bank", "mcdc_set_trace",
           "mcdc_get_trace", "mcdc_test_draws", "mcdc_test_grid_index", "mcdc_test_geometry", "mcdc_get_timing",
           "mcdc_set_profile", "mcdc_get_profile", "mcdc_microbench", "mcdc_destroy", "mcdc_last_error",
           "mcdc_set_physics", "mcdc_get_balance", "mcdc_get_census", "mcdc_draws_noalloc", "mcdc_build_id"]

_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int32)


class McdcError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"mcdc error {code}: {msg}")
        self.code = code


class Geometry(C.Structure):
    _fields_ = [("n_surf", C.c_int32), ("surf_type", _ip), ("surf_param", _dp), ("surf_bc", _ip),
                ("n_cell", C.c_int32), ("cell_surf_off", _ip), ("cell_surf_id", _ip), ("cell_surf_sense", _ip),
                ("cell_fill_type", _ip), ("cell_fill", _ip), ("n_univ", C.c_int32), ("univ_cell_off", _ip),
                ("has_lattice", C.c_int32), ("lat_x0", C.c_double), ("lat_y0", C.c_double), ("lat_px", C.c_double),
                ("lat_py", C.c_double), ("lat_nx", C.c_int32), ("lat_ny", C.c_int32), ("lat_univ", _ip),
                ("n_lat2", C.c_int32), ("lat2_nx", _ip), ("lat2_ny", _ip), ("lat2_px", _dp), ("lat2_py", _dp),
                ("lat2_off", _ip), ("lat2_univ", _ip)]


class Kinetics(C.Structure):
    _fields_ = [("speed", _dp), ("n_dgroup", C.c_int32), ("pad", C.c_int32), ("nu_d", _dp), ("decay", _dp), ("chi_d", _dp),
                ("census_target", C.c_int64)]


class Materials(C.Structure):
    _fields_ = [("n_mat", C.c_int32), ("G", C.c_int32), ("sig_t", _dp), ("sig_f", _dp), ("nu", _dp), ("chi", _dp),
                ("S", _dp), ("kinetics", C.POINTER(Kinetics))]


class XS(C.Structure):
    _fields_ = [("n_mat", C.c_int32), ("n_grid", C.c_int32), ("grid", _dp), ("n_nuc", C.c_int32), ("nuc_A", _dp),
                ("nuc_el", _dp), ("nuc_c", _dp), ("nuc_f", _dp), ("mat_nuc_off", _ip), ("mat_nuc_id", _ip),
                ("mat_nuc_dens", _dp), ("nu0", C.c_double), ("nu1", C.c_double), ("watt_a", C.c_double),
                ("watt_b", C.c_double), ("search", C.c_int32)]


class Source(C.Structure):
    _fields_ = [("lo", C.c_double * 3), ("hi", C.c_double * 3), ("isotropic", C.c_int32), ("dir", C.c_double * 3),
                ("group_pdf", _dp), ("E", C.c_double), ("t", C.c_double)]


class TallySpec(C.Structure):
    _fields_ = [("n_bins", C.c_int32), ("cell_bin", _ip), ("lat_bin", _ip), ("n_t", C.c_int32), ("t_edges", _dp),
                ("n_e", C.c_int32), ("e_edges", _dp), ("lat2_bin", _ip)]


class Device(C.Structure):
    _fields_ = [("workspace", C.c_void_p), ("workspace_bytes", C.c_uint64), ("stream", C.c_void_p),
                ("device", C.c_int32), ("schedule", C.c_int32), ("persist_threshold", C.c_int32),
                ("reserved", C.c_int32 * 3)]


class Physics(C.Structure):
    _fields_ = [("kT", C.c_double), ("implicit_capture", C.c_int32), ("pad", C.c_int32), ("w_roulette", C.c_double),
                ("w_survive", C.c_double)]


class Dims(C.Structure):
    _fields_ = [("mode", C.c_int32), ("n_tally", C.c_int32), ("n_cycles", C.c_int32), ("n_active", C.c_int32),
                ("bank_count", C.c_uint64)]


class Tallies(C.Structure):
    _fields_ = [("k_cycle", _dp), ("flux_mean", _dp), ("flux_sdev", _dp), ("counters", C.POINTER(C.c_uint64)),
                ("k_mean", C.c_double), ("k_sdev", C.c_double), ("leak_mean", C.c_double), ("leak_sdev", C.c_double)]


TRACE_DTYPE = np.dtype([("id", "<u8"), ("cycle", "<u4"), ("seq", "<u4"), ("ev", "<i4"), ("c0", "<i4"),
                        ("elem", "<i4"), ("c1", "<i4"), ("surf", "<i4"), ("gi", "<i4"), ("x", "<f8"), ("y", "<f8"),
                        ("z", "<f8"), ("d", "<f8"), ("E", "<f8"), ("t", "<f8")], align=True)
SITE_DTYPE = np.dtype([("x", "<f8"), ("y", "<f8"), ("z", "<f8"), ("ux", "<f8"), ("uy", "<f8"), ("uz", "<f8"),
                       ("g", "<i4"), ("pad", "<i4")], align=True)

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-shared",
              "-Xcompiler", "-fPIC"]


def source_id() -> str:
    """Identity of the CUDA sources as they are on disk: sha256 over csrc/* and include/*.h, 16 hex digits.  build()
    compiles it into the library (mcdc_build_id), so a measurement file can name the build it was taken on."""
    import hashlib
    h = hashlib.sha256()
    for f in sorted(_SRC + _HDRS):
        h.update(os.path.basename(f).encode() + b"\0")
        with open(f, "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()[:16]


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile the CUDA library for sm_100a with nvcc (in-tree, next to this file)."""
    deps = _SRC + _HDRS
    if force or not os.path.exists(_SO) or any(os.path.getmtime(s) > os.path.getmtime(_SO) for s in deps):
        cmd = (["nvcc"] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else [])
               + [f'-DMCDC_BUILD_ID="{source_id()}"', "-o", _SO, _SRC[0]])
        subprocess.check_call(cmd)
    return _SO


def build_id() -> str:
    """source_id() of the sources the LOADED library was compiled from ("unknown" if built by hand without it)."""
    return load_library().mcdc_build_id().decode()


_lib = None


def load_library():
    """dlopen the built library and declare the prototypes.  Raises if it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_SO):
        try:  # build the product in-tree if the toolchain is there; never fall back to anything else
            build()
        except Exception as e:
            raise McdcError(-5, f"{_SO} is missing and could not be built ({e}): run "
                                "`python -c 'import __graft_entry__ as g; g.build()'`")
    L = C.CDLL(_SO)
    vp, u64, u32, i32 = C.c_void_p, C.c_uint64, C.c_uint32, C.c_int32
    P = C.POINTER
    L.mcdc_workspace_bytes.argtypes = [P(Geometry), P(Materials), P(XS), P(TallySpec), u64, P(u64)]
    L.mcdc_create.argtypes = [P(Geometry), P(Materials), P(XS), P(Source), P(TallySpec), P(Device), u64, P(vp)]
    L.mcdc_run_eigenvalue.argtypes = [vp, u64, i32, i32, u64]
    L.mcdc_run_cycle.argtypes = [vp, u64, u32, i32, u64, _dp]
    L.mcdc_run_cycle_host.argtypes = [vp, u64, u32, u64, C.c_double, vp, u64, vp, u64, P(u64), _dp, _dp, _dp]
    L.mcdc_run_fixed_source.argtypes = [vp, u64, u64]
    L.mcdc_get_dims.argtypes = [vp, P(Dims)]
    L.mcdc_get_tallies.argtypes = [vp, P(Tallies)]
    L.mcdc_get_bank.argtypes = [vp, vp, u64, P(u64)]
    L.mcdc_set_trace.argtypes = [vp, u64, u32, u32]
    L.mcdc_get_trace.argtypes = [vp, vp, u64, P(u64)]
    L.mcdc_test_draws.argtypes = [vp, u64, u32, u32, vp, vp, u64, _dp]
    L.mcdc_test_grid_index.argtypes = [vp, _dp, u64, _ip, _ip]
    L.mcdc_test_geometry.argtypes = [vp, _dp, _dp, u64, i32, _ip, _dp, _ip]
    L.mcdc_get_timing.argtypes = [vp, _dp, P(u64)]
    L.mcdc_set_profile.argtypes = [vp, i32]
    L.mcdc_get_profile.argtypes = [vp, _dp, P(u64), P(u64)]
    L.mcdc_microbench.argtypes = [vp, i32, u64, _dp, _dp]
    L.mcdc_set_physics.argtypes = [vp, P(Physics)]
    L.mcdc_get_balance.argtypes = [vp, _dp]
    L.mcdc_get_census.argtypes = [vp, P(u64), _dp, i32, P(i32)]
    L.mcdc_draws_noalloc.argtypes = [i32, vp, u64, u32, u32, vp, vp, u64, _dp]
    L.mcdc_destroy.argtypes = [vp]
    L.mcdc_destroy.restype = None
    L.mcdc_last_error.restype = C.c_char_p
    L.mcdc_build_id.restype = C.c_char_p
    _lib = L
    return L


def _d(a):
    return np.ascontiguousarray(a, np.float64)


def _i(a):
    return np.ascontiguousarray(a, np.int32)


def draws_noalloc(seed, domain, cycle, ids, idx, device=0, stream=None):
    """``mcdc_draws_noalloc``: draw ``idx[i]`` of the random-number stream (seed, ids[i], domain, cycle) for every i,
    computed on GPU ``device`` without a Problem and without a workspace.

    For callers that cannot give the library device memory (the GPU is already full, or the host program forbids
    allocating): the staging lives in a fixed 1.5 MiB array inside the library, so at most ``NOALLOC_DRAWS_MAX`` draws
    per call (more raises McdcError).  ``ids`` / ``idx`` are host arrays; the result is a host float64 array, bit-equal
    to ``Problem.draws``.  ``stream``: a raw cudaStream_t handle (int) of that device, None = the default stream.  The
    first call on a device does a one-time address look-up: make it before any stream capture on that device."""
    L = load_library()
    ids = np.ascontiguousarray(ids, np.uint64)
    idx = np.ascontiguousarray(idx, np.uint32)
    if ids.shape != idx.shape or ids.ndim != 1:
        raise ValueError("ids and idx must be 1-D arrays of equal length")
    out = np.zeros(len(ids))
    rc = L.mcdc_draws_noalloc(int(device), stream, int(seed), int(domain), int(cycle), ids.ctypes.data, idx.ctypes.data,
                              len(ids), out.ctypes.data_as(_dp))
    if rc != 0:
        raise McdcError(rc, L.mcdc_last_error().decode())
    return out


class Problem:
    """One transport problem on one CUDA device, built from a problem dict (see ``inputs``)."""

    def __init__(self, P: dict, max_particles=None, device=0, schedule=0, persist_threshold=0, search=0):
        """schedule 0: event sweeps + persistent kernel below persist_threshold (0 = library default, < 0 = never,
        ALWAYS = from the first segment); 1: monolithic; 2: split per-event kernels (see include/mcdc.h)."""
        import torch

        if not torch.cuda.is_available():
            raise McdcError(-5, "no CUDA device: this library has no CPU path")
        self.L = load_library()
        self.P = P
        self._keep = []
        self.torch = torch
        self.dev = torch.device("cuda", device)
        run = P["run"]
        self.max_particles = int(max_particles if max_particles is not None else run["n_particles"])

        def dp(a):
            a = _d(a)
            self._keep.append(a)
            return a.ctypes.data_as(_dp)

        def ip(a):
            a = _i(a)
            self._keep.append(a)
            return a.ctypes.data_as(_ip)

        ce = P["mode"] == "ce"
        self.ce = ce
        g = Geometry()
        g.n_surf = len(P["surf_type"])
        g.surf_type, g.surf_param, g.surf_bc = ip(P["surf_type"]), dp(P["surf_param"]), ip(P["surf_bc"])
        g.n_cell = len(P["cell_fill"])
        g.cell_surf_off, g.cell_surf_id, g.cell_surf_sense = ip(P["cell_surf_off"]), ip(P["cell_surf_id"]), ip(P["cell_surf_sense"])
        g.cell_fill_type, g.cell_fill = ip(P["cell_fill_type"]), ip(P["cell_fill"])
        g.n_univ = len(P["univ_cell_off"]) - 1
        g.univ_cell_off = ip(P["univ_cell_off"])
        lat = P.get("lat")
        t = TallySpec()
        t.n_bins, t.cell_bin = int(P["n_bins"]), ip(P["cell_bin"])
        g.has_lattice = 1 if lat else 0
        if lat:
            g.lat_x0, g.lat_y0, g.lat_px, g.lat_py = lat["x0"], lat["y0"], lat["px"], lat["py"]
            g.lat_nx, g.lat_ny, g.lat_univ = lat["nx"], lat["ny"], ip(lat["univ"])
            t.lat_bin = ip(lat["bin"])
        if "lat2_nx" in P:
            g.n_lat2 = len(P["lat2_nx"])
            g.lat2_nx, g.lat2_ny, g.lat2_off = ip(P["lat2_nx"]), ip(P["lat2_ny"]), ip(P["lat2_off"])
            g.lat2_px, g.lat2_py, g.lat2_univ = dp(P["lat2_px"]), dp(P["lat2_py"]), ip(P["lat2_univ"])
            t.lat2_bin = ip(P["lat2_bin"])
        s = Source()
        s.lo = (C.c_double * 3)(*P["src_lo"])
        s.hi = (C.c_double * 3)(*P["src_hi"])
        s.isotropic = int(P["src_iso"])
        s.dir = (C.c_double * 3)(*P["src_dir"])
        s.t = float(P.get("src_t", 0.0))
        m = x = None
        if not ce:
            m = Materials()
            m.n_mat, m.G = int(P["n_mat"]), int(P["G"])
            m.sig_t, m.sig_f, m.nu, m.chi, m.S = dp(P["mg_sig_t"]), dp(P["mg_sig_f"]), dp(P["mg_nu"]), dp(P["mg_chi"]), dp(P["mg_S"])
            s.group_pdf = dp(P["src_group_pdf"])
            td = P.get("td")
            if td:  # time-dependent multi-group: speeds, delayed-neutron data; the time edges go with the tally
                kn = Kinetics()
                kn.speed, kn.n_dgroup = dp(td["speed"]), int(td["J"])
                kn.nu_d, kn.decay, kn.chi_d = dp(td["nu_d"]), dp(td["decay"]), dp(td["chi_d"])
                kn.census_target = int(td.get("census_target", 0))
                self._keep.append(kn)
                m.kinetics = C.pointer(kn)
                t.n_t, t.t_edges = len(P["t_edges"]) - 1, dp(P["t_edges"])
        else:
            x = XS()
            x.n_mat, x.n_grid, x.grid = int(P["n_mat"]), len(P["grid"]), dp(P["grid"])
            x.n_nuc, x.nuc_A = len(P["nuc_A"]), dp(P["nuc_A"])
            x.nuc_el, x.nuc_c, x.nuc_f = dp(P["nuc_el"]), dp(P["nuc_c"]), dp(P["nuc_f"])
            x.mat_nuc_off, x.mat_nuc_id, x.mat_nuc_dens = ip(P["mat_nuc_off"]), ip(P["mat_nuc_id"]), dp(P["mat_nuc_dens"])
            x.nu0, x.nu1, x.watt_a, x.watt_b = P["nu0"], P["nu1"], P["watt_a"], P["watt_b"]
            x.search = int(search)
            t.n_t, t.t_edges = len(P["t_edges"]) - 1, dp(P["t_edges"])
            t.n_e, t.e_edges = len(P["e_edges"]) - 1, dp(P["e_edges"])
            s.E = float(P["src_E"])
        mp = C.byref(m) if m is not None else None
        xp = C.byref(x) if x is not None else None
        nbytes = C.c_uint64()
        self._check(self.L.mcdc_workspace_bytes(C.byref(g), mp, xp, C.byref(t), self.max_particles, C.byref(nbytes)))
        with torch.cuda.device(self.dev):
            self.workspace = torch.empty(nbytes.value + 256, dtype=torch.uint8, device=self.dev)
            self.stream = torch.cuda.current_stream(self.dev)
        base = (self.workspace.data_ptr() + 255) & ~255
        d = Device()
        d.workspace, d.workspace_bytes = base, nbytes.value
        d.stream, d.device = self.stream.cuda_stream, device
        d.schedule, d.persist_threshold = int(schedule), int(persist_threshold)
        h = C.c_void_p()
        self._check(self.L.mcdc_create(C.byref(g), mp, xp, C.byref(s), C.byref(t), C.byref(d), self.max_particles, C.byref(h)))
        self.h = h
        self.workspace_bytes = nbytes.value
        if P.get("kT", 0.0) or P.get("implicit_capture", 0):
            self.set_physics(P.get("kT", 0.0), P.get("implicit_capture", 0), P.get("w_roulette", 0.25), P.get("w_survive", 1.0))
        dims = self.dims()
        self.n_tally = dims.n_tally

    def _check(self, rc):
        if rc != 0:
            raise McdcError(rc, self.L.mcdc_last_error().decode())

    def close(self):
        if getattr(self, "h", None):
            self.L.mcdc_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def dims(self):
        d = Dims()
        self._check(self.L.mcdc_get_dims(self.h, C.byref(d)))
        return d

    def set_physics(self, kT=0.0, implicit_capture=0, w_roulette=0.25, w_survive=1.0):
        ph = Physics(float(kT), int(implicit_capture), 0, float(w_roulette), float(w_survive))
        self._check(self.L.mcdc_set_physics(self.h, C.byref(ph)))

    def balance(self):
        """Weight balance of the last run: dict(source, absorbed, leaked, cutoff, roulette_loss, roulette_gain)."""
        out = np.zeros(6)
        self._check(self.L.mcdc_get_balance(self.h, out.ctypes.data_as(_dp)))
        return dict(zip(("source", "absorbed", "leaked", "cutoff", "roulette_loss", "roulette_gain"), out))

    def census(self):
        """Population entering each census interval of the last run made interval by interval:
        (particles before the comb, after it, weight before, weight after) per interval."""
        cnt, w, n = np.zeros(128, np.uint64), np.zeros(128), C.c_int32()
        self._check(self.L.mcdc_get_census(self.h, cnt.ctypes.data_as(C.POINTER(C.c_uint64)), w.ctypes.data_as(_dp), 64, C.byref(n)))
        return [(int(cnt[2 * k]), int(cnt[2 * k + 1]), float(w[2 * k]), float(w[2 * k + 1])) for k in range(n.value)]

    # ---- runs
    def run(self, n_particles=None, n_inactive=None, n_active=None, seed=None):
        r = self.P["run"]
        N = int(n_particles if n_particles is not None else r["n_particles"])
        ni = int(n_inactive if n_inactive is not None else r["n_inactive"])
        na = int(n_active if n_active is not None else r["n_active"])
        sd = int(seed if seed is not None else r["seed"])
        if r["kind"] == "eigen":
            self._check(self.L.mcdc_run_eigenvalue(self.h, N, ni, na, sd))
        else:  # "fixed" (continuous energy) and "td" (time-dependent multi-group)
            self._check(self.L.mcdc_run_fixed_source(self.h, N, sd))
        return self.results()

    def run_cycle(self, n_particles, cycle, active, seed):
        k = C.c_double()
        self._check(self.L.mcdc_run_cycle(self.h, int(n_particles), int(cycle), int(active), int(seed), C.byref(k)))
        return k.value

    def run_cycle_host(self, n_particles, cycle, seed, k_prev, sites_in=None, sites_out=None, flux_out=None):
        """End-to-end form: HOST source bank in, HOST fission bank + per-cycle flux out (pinned numpy views)."""
        n_in = 0 if sites_in is None else len(sites_in)
        n_out, k, leak = C.c_uint64(), C.c_double(), C.c_double()
        self._check(self.L.mcdc_run_cycle_host(
            self.h, int(n_particles), int(cycle), int(seed), float(k_prev),
            sites_in.ctypes.data if n_in else None, n_in,
            sites_out.ctypes.data if sites_out is not None else None, 0 if sites_out is None else len(sites_out),
            C.byref(n_out), flux_out.ctypes.data_as(_dp) if flux_out is not None else None, C.byref(k), C.byref(leak)))
        return k.value, leak.value, n_out.value

    def results(self):
        d = self.dims()
        kc = np.zeros(max(d.n_cycles, 1))
        fm, fs = np.zeros(self.n_tally), np.zeros(self.n_tally)
        cnt = np.zeros(N_COUNTERS, np.uint64)
        t = Tallies()
        t.k_cycle, t.flux_mean, t.flux_sdev = kc.ctypes.data_as(_dp), fm.ctypes.data_as(_dp), fs.ctypes.data_as(_dp)
        t.counters = cnt.ctypes.data_as(C.POINTER(C.c_uint64))
        self._check(self.L.mcdc_get_tallies(self.h, C.byref(t)))
        return dict(rc=0, k_cycle=kc[: d.n_cycles], k_mean=t.k_mean, k_sdev=t.k_sdev, flux_mean=fm, flux_sdev=fs,
                    leak_mean=t.leak_mean, leak_sdev=t.leak_sdev, counters=cnt)

    def timing(self):
        ms, nl = C.c_double(), C.c_uint64()
        self._check(self.L.mcdc_get_timing(self.h, C.byref(ms), C.byref(nl)))
        return ms.value, nl.value

    PROFILE_CLASSES = ("sweep", "scatter", "surface", "persist", "segment", "bank")

    def set_profile(self, on=True):
        self._check(self.L.mcdc_set_profile(self.h, int(on)))

    def profile(self):
        ms, nl = np.zeros(6), np.zeros(6, np.uint64)
        ev = C.c_uint64()
        self._check(self.L.mcdc_get_profile(self.h, ms.ctypes.data_as(_dp), nl.ctypes.data_as(C.POINTER(C.c_uint64)), C.byref(ev)))
        out = {k: dict(ms=float(m), launches=int(n)) for k, m, n in zip(self.PROFILE_CLASSES, ms, nl)}
        out["sweep"]["events"] = int(ev.value)
        return out

    MICROBENCH = ("ffma", "dfma", "log", "div", "sqrt", "sincospi", "rcp", "philox")

    def microbench(self, which, iters=20000):
        """Measured rate (thread-level operations per second) of one arithmetic micro-benchmark of the library."""
        ms, ops = C.c_double(), C.c_double()
        self._check(self.L.mcdc_microbench(self.h, self.MICROBENCH.index(which), int(iters), C.byref(ms), C.byref(ops)))
        return ops.value / (ms.value * 1e-3)

    def bank(self):
        n = C.c_uint64()
        self._check(self.L.mcdc_get_bank(self.h, None, 0, C.byref(n)))
        out = np.zeros(n.value, SITE_DTYPE)
        if n.value:
            self._check(self.L.mcdc_get_bank(self.h, out.ctypes.data, n.value, C.byref(n)))
        return out

    def set_trace(self, first_id=0, n_ids=100, max_events=512):
        self._check(self.L.mcdc_set_trace(self.h, int(first_id), int(n_ids), int(max_events)))

    def trace(self):
        n = C.c_uint64()
        self._check(self.L.mcdc_get_trace(self.h, None, 0, C.byref(n)))
        out = np.zeros(n.value, TRACE_DTYPE)
        if n.value:
            self._check(self.L.mcdc_get_trace(self.h, out.ctypes.data, n.value, C.byref(n)))
        return out

    # ---- unit-level entry points
    def draws(self, seed, domain, cycle, ids, idx):
        ids = np.ascontiguousarray(ids, np.uint64)
        idx = np.ascontiguousarray(idx, np.uint32)
        out = np.zeros(len(ids))
        self._check(self.L.mcdc_test_draws(self.h, int(seed), int(domain), int(cycle), ids.ctypes.data, idx.ctypes.data,
                                           len(ids), out.ctypes.data_as(_dp)))
        return out

    def grid_index(self, E):
        E = _d(E)
        ob, oh = np.zeros(len(E), np.int32), np.zeros(len(E), np.int32)
        self._check(self.L.mcdc_test_grid_index(self.h, E.ctypes.data_as(_dp), len(E), ob.ctypes.data_as(_ip), oh.ctypes.data_as(_ip)))
        return ob, oh

    def geometry(self, x, u, path=0):
        x, u = _d(x).reshape(-1, 3), _d(u).reshape(-1, 3)
        n = len(x)
        loc, dist, surf = np.zeros((n, 3), np.int32), np.zeros(n), np.zeros(n, np.int32)
        self._check(self.L.mcdc_test_geometry(self.h, x.ctypes.data_as(_dp), u.ctypes.data_as(_dp), n, int(path), loc.ctypes.data_as(_ip),
                                              dist.ctypes.data_as(_dp), surf.ctypes.data_as(_ip)))
        return loc, dist, surf
