"""Pins of the oracle's transport loop against closed forms and invariants (no GPU).

Citations: BASELINE.json north_star ("k_inf = nuSigma_f/Sigma_a ... dominant eigenvalue of
(diag(Sigma_t) - S^T)^-1 chi nuSigma_f^T ... exp(-Sigma_t L) ... particle-weight conservation");
SURVEY.md 8(c) "What pins each part"; DESIGN.md section 3.
"""
import math

import numpy as np
import pytest

from paper_2501_05440_b200 import inputs

EV = dict(scatter=1, fission=2, capture=3, transmit=4, reflect=5, leak=6, lattice=7, time_edge=8, cutoff=9, lost=10)


def kinf_dense(P, m=0):
    """Dominant eigenvalue of (diag Sigma_t - S^T)^-1 chi nuSigma_f^T, by a dense eigen-solve (numpy)."""
    st, S = P["mg_sig_t"][m], P["mg_S"][m]
    F = np.outer(P["mg_chi"][m], P["mg_nu"][m] * P["mg_sig_f"][m])
    M = np.linalg.solve(np.diag(st) - S.T, F)
    w = np.linalg.eigvals(M)
    return float(w.real[np.argmax(np.abs(w))])


@pytest.fixture(scope="module")
def c1(orc):
    P = inputs.config1()
    o = orc.Oracle(P)
    rc, r = o.run()
    assert rc == 0
    return P, o, r


def test_c1_k_closed_form(c1):
    """1-group infinite medium: k_inf = nuSigma_f / Sigma_a = 0.39/0.3 = 1.3 within 3 sigma."""
    P, o, r = c1
    assert r["k_sdev"] > 0 and r["k_sdev"] < 0.01
    assert abs(r["k_mean"] - 1.3) < 3 * r["k_sdev"]
    assert kinf_dense(P) == pytest.approx(1.3, rel=1e-12)


def test_c1_event_rates(c1):
    """collisions/history = Sigma_t/Sigma_a = 3.333, track length/history = 1/Sigma_a, reflections/history
    = (1/Sigma_a) S/(4V) = 5 for the unit cube (mean chord theorem); all within 4 sigma of counting noise."""
    P, o, r = c1
    c = r["counters"].astype(float)
    M = c[0]
    coll = c[EV["scatter"]] + c[EV["fission"]] + c[EV["capture"]]
    assert abs(coll / M - 1 / 0.3) < 4 * math.sqrt((0.7 / 0.09) / M) + 1e-3
    assert abs(c[EV["reflect"]] / M - 5.0) < 0.05
    # flux (track length per source particle, normalised per cycle by N): 1/Sigma_a
    assert abs(r["flux_mean"][0] - 1 / 0.3) < 4 * r["flux_sdev"][0] + 1e-9
    # reaction branching: fission : capture = 0.15 : 0.15, scatter fraction 0.7
    assert abs(c[EV["scatter"]] / coll - 0.7) < 4 * math.sqrt(0.21 / coll)
    assert abs(c[EV["fission"]] / (c[EV["fission"]] + c[EV["capture"]]) - 0.5) < 4 * math.sqrt(0.25 / (0.3 * coll))


def test_c1_integer_invariant(c1):
    """Every history ends in exactly one of capture / fission / leak / cutoff: counts sum to the tracks started."""
    P, o, r = c1
    c = r["counters"]
    assert c[EV["capture"]] + c[EV["fission"]] + c[EV["leak"]] + c[EV["cutoff"]] == c[0]
    assert c[EV["lost"]] == 0 and c[EV["leak"]] == 0 and c[EV["lattice"]] == 0
    assert c[12] <= 2 * P["run"]["n_particles"]


def test_c1_k_estimators_agree(orc):
    """Track-length k_c vs the analog estimator M_next k_prev / N: E[children] = w nu/k_prev per fission, so
    bank size * k_prev / N estimates k too; the two agree within combined noise."""
    P = inputs.config1(n_particles=20000, n_inactive=0, n_active=6)
    o = orc.Oracle(P)
    L = o.L
    # run cycle by cycle lengths 1..6 to read the bank size after each (the run is deterministic)
    ks, Ms = None, []
    for n in range(1, 7):
        rc = L.orc_run_eigenvalue(o.h, 20000, 0, n, 1)
        o.n_cycles = n
        Ms.append(len(o.bank()))
        ks = o.results()["k_cycle"]
    kprev = np.concatenate([[1.0], ks[:-1]])
    analog = np.array(Ms) * kprev / 20000.0
    # per cycle both are ~1.3 +- 0.015
    assert np.all(np.abs(analog - ks) < 0.06)
    assert abs(analog.mean() - ks.mean()) < 0.02
    assert abs(analog.mean() - 1.3) < 0.02


def test_weight_conservation_c1(orc):
    """Per cycle: source weight N = absorbed weight (+ leaked).  With equal weights w0 = N/M per cycle the
    absorbed weight is w0 * (captures + fissions): check exactly in integers, cycle by cycle."""
    P = inputs.config1(n_particles=5000, n_inactive=0, n_active=1)
    o = orc.Oracle(P)
    prev_c = None
    for n in range(1, 4):
        o.L.orc_run_eigenvalue(o.h, 5000, 0, n, 3)
        o.n_cycles = n
        c = o.results()["counters"].astype(np.int64)
        d = c if prev_c is None else c - prev_c
        M = d[0]
        assert d[EV["capture"]] + d[EV["fission"]] + d[EV["leak"]] == M
        w0 = 5000.0 / M
        assert w0 * (d[EV["capture"]] + d[EV["fission"]] + d[EV["leak"]]) == pytest.approx(5000.0, rel=1e-12)
        prev_c = c


@pytest.fixture(scope="module")
def c2(orc):
    P = inputs.config2(n_particles=40000, n_inactive=5, n_active=25)
    o = orc.Oracle(P)
    rc, r = o.run()
    assert rc == 0
    return P, o, r


def test_c2_k_dense_eigenvalue(c2):
    """7-group infinite medium: k within 3 sigma of the dominant eigenvalue of the dense 7x7 operator,
    and that eigenvalue equals nuSigma_f^T (diag Sigma_t - S^T)^-1 chi (rank one)."""
    P, o, r = c2
    k = kinf_dense(P)
    st, S = P["mg_sig_t"][0], P["mg_S"][0]
    phi = np.linalg.solve(np.diag(st) - S.T, P["mg_chi"][0])
    assert k == pytest.approx(float((P["mg_nu"][0] * P["mg_sig_f"][0]) @ phi), rel=1e-12)
    assert 1.1 <= k <= 1.3
    assert abs(r["k_mean"] - k) < 3 * r["k_sdev"]
    assert r["k_sdev"] < 0.004


def test_c2_spectrum(c2):
    """Group flux per source neutron -> k * ((diag Sigma_t - S^T)^-1 chi)_g: with the bank renormalised to
    total weight N each cycle, flux/N is the flux per unit source = phi_g for a chi-distributed source."""
    P, o, r = c2
    st, S = P["mg_sig_t"][0], P["mg_S"][0]
    phi = np.linalg.solve(np.diag(st) - S.T, P["mg_chi"][0])
    f, s = r["flux_mean"], r["flux_sdev"]
    assert np.all(np.abs(f - phi) < 4 * s + 1e-3 * phi)
    # shape (independent of normalisation)
    assert np.allclose(f / f.sum(), phi / phi.sum(), atol=4e-3)


def test_slab_transmission(orc):
    """Uncollided transmission of a normal beam through a pure absorber slab: leakage = exp(-Sigma_t L) within
    3 sigma, track length = (1 - exp(-Sigma_t L))/Sigma_t."""
    Lx, st, N = 2.0, 1.3, 100000
    P = inputs.slab_beam(Lx, st, N)
    o = orc.Oracle(P)
    rc, r = o.run()
    assert rc == 0
    p = math.exp(-st * Lx)
    assert abs(r["leak_mean"] - p) < 3 * math.sqrt(p * (1 - p) / N)
    tl = (1 - p) / st
    # per-history track length = min(Exp(st), L): variance <= 1/st^2
    assert abs(r["flux_mean"][0] - tl) < 4 / st / math.sqrt(N)
    c = r["counters"]
    assert c[EV["leak"]] + c[EV["capture"]] == N and c[EV["scatter"]] == 0 and c[EV["fission"]] == 0
    assert r["k_cycle"][0] == 0.0


def test_sphere_transmission(orc):
    """Isotropic point source at the centre of a pure-absorber sphere (quadric distance, vacuum BC):
    leakage = exp(-Sigma_t r)."""
    rr, st, N = 1.5, 0.8, 100000
    P = inputs.sphere_absorber(rr, st, N)
    o = orc.Oracle(P)
    rc, r = o.run()
    assert rc == 0
    p = math.exp(-st * rr)
    assert abs(r["leak_mean"] - p) < 3 * math.sqrt(p * (1 - p) / N)


def test_pincell_same_material_area_fraction(orc):
    """C3 with fuel == moderator material: track length is uniform in an infinite homogeneous medium, so
    flux_fuel/flux_total -> pi r^2/p^2 = 0.577027 and k -> the C2 closed form (pins cell lookup, cylinder
    distance, transmission and reflection)."""
    P = inputs.config3(n_particles=20000, n_inactive=3, n_active=12, same_material=True)
    o = orc.Oracle(P)
    rc, r = o.run()
    assert rc == 0
    f = r["flux_mean"].reshape(2, 7)
    frac = f[0].sum() / f.sum()
    area = math.pi * 0.54 ** 2 / 1.26 ** 2
    assert area == pytest.approx(0.577027, abs=1e-6)
    # relative sdev of the fraction from the per-bin sdevs (upper bound, bins positively correlated)
    sd = np.sqrt((r["flux_sdev"].reshape(2, 7) ** 2).sum()) / f.sum()
    assert abs(frac - area) < 4 * sd + 2e-3
    # per group too
    assert np.allclose(f[0] / (f[0] + f[1]), area, atol=0.02)
    k = kinf_dense(P)
    assert abs(r["k_mean"] - k) < 3 * r["k_sdev"] + 1e-3
    c = r["counters"]
    assert c[EV["lost"]] == 0 and c[EV["transmit"]] > 0 and c[EV["reflect"]] > 0


def test_quarter_core_uniform(orc):
    """C4 geometry with all 7 materials identical and all faces reflecting: k -> C2 closed form and the
    per-element flux is uniform (pins lattice indexing, lattice walls, local cells, per-pin bins)."""
    P = inputs.config4(n_particles=30000, n_inactive=2, n_active=10, uniform=True, n_asm=1, n_pin=3, n_refl=2)
    o = orc.Oracle(P)
    rc, r = o.run()
    assert rc == 0
    k = kinf_dense(P)
    assert abs(r["k_mean"] - k) < 3 * r["k_sdev"] + 1e-3
    f = r["flux_mean"].reshape(-1, 7).sum(1)
    # 9 fuelled-element bins of equal area + one reflector bin with 25-9=16 elements
    per_elem = np.concatenate([f[:9], [f[9] / 16]])
    assert np.allclose(per_elem / per_elem.mean(), 1.0, atol=0.05)
    c = r["counters"]
    assert c[EV["lattice"]] > 0 and c[EV["lost"]] == 0 and c[EV["leak"]] == 0
    # the source lives only in the fuelled 3x3 corner, the cycle-0 source too
    assert r["leak_mean"] == 0.0


def test_quarter_core_vacuum_leakage_pure_absorber(orc):
    """Lattice + vacuum BC special case that reduces to a slab: pure absorber everywhere, beam along +x born
    at x = 0+: leakage through the outer face = exp(-Sigma_t * side) exactly as for a slab."""
    P = inputs.config4(n_particles=40000, n_inactive=0, n_active=1, n_asm=1, n_pin=2, n_refl=1, G=1)
    st = 0.45
    for k in ("mg_sig_t", "mg_sig_c"):
        P[k][:] = st
    for k in ("mg_sig_f", "mg_nu", "mg_S"):
        P[k][:] = 0.0
    P["mg_chi"][:] = 1.0
    side = 3 * 1.26
    P["src_lo"][:] = [1e-9, 0.3, 0.0]
    P["src_hi"][:] = [1e-9, 3.2, 0.0]
    P["src_iso"] = 0
    P["src_dir"][:] = [1.0, 0.0, 0.0]
    o = orc.Oracle(P)
    rc, r = o.run()
    assert rc == 0
    p = math.exp(-st * side)
    assert abs(r["leak_mean"] - p) < 3 * math.sqrt(p * (1 - p) / 40000)
    assert r["counters"][EV["lattice"]] > 0


def test_ce_one_over_v_time_dependence(orc):
    """Single pure 1/v absorber (Sigma_a v = lambda), no scatter: track length in [t1,t2] per source neutron
    = (v/lambda)(exp(-lambda t1) - exp(-lambda t2)); survivors at cutoff = exp(-lambda t_max)."""
    lam, N, E0 = 2.0e5, 60000, 1.0e3
    P = inputs.ce_one_over_v(lam, N, E0=E0)
    o = orc.Oracle(P)
    rc, r = o.run()
    assert rc == 0
    v = orc.speed(E0)
    te = P["t_edges"]
    exp = v / lam * (np.exp(-lam * te[:-1]) - np.exp(-lam * te[1:]))
    f = r["flux_mean"].reshape(len(te) - 1, 2)
    assert np.all(f[:, 0] == 0)  # 1 keV falls in the second energy bin
    got = f[:, 1]
    # per-history contribution to a bin is <= v*dt; use a generous binomial-style bound
    for b in range(len(exp)):
        dt = te[b + 1] - te[b]
        sig = v * dt * math.sqrt(max(math.exp(-lam * te[b]), 1e-12) / N)
        assert abs(got[b] - exp[b]) < 5 * sig + 1e-6 * exp[b], b
    surv = r["counters"][EV["cutoff"]] / N
    p = math.exp(-lam * te[-1])
    assert abs(surv - p) < 4 * math.sqrt(p * (1 - p) / N) + 1e-4
    assert r["counters"][EV["cutoff"]] + r["counters"][EV["capture"]] == N
    # exactly one time-edge event per bin boundary crossed
    assert r["counters"][EV["time_edge"]] > 0


def test_ce_fission_multiplicity_and_watt(orc):
    """Pure fission nuclide: children per fission = floor(nu(E) + xi), nu = 2.4 + 0.1 E[MeV], so the total
    number of children equals sum nu(E_fission) within the rounding noise (variance <= 1/4 per fission);
    child energies follow the Watt spectrum (mean 2.03084 MeV) (R4, R5, R22)."""
    N = 3000
    P = inputs.ce_pure_fission(N, E0=1.0e6)
    P["t_edges"] = np.array([0.0, 1.0e-9])
    o = orc.Oracle(P)
    o.set_trace(0, 2 ** 64 - 1, 2_000_000)
    rc, r = o.run()
    assert rc == 0
    c = r["counters"]
    tr = o.trace()
    assert len(tr) == c[1:11].sum()
    fis = tr[tr["ev"] == EV["fission"]]
    nfis = len(fis)
    assert nfis == c[EV["fission"]] and nfis > 2000
    nu = 2.4 + 0.1 * fis["E"] * 1e-6
    assert abs(float(c[11]) - nu.sum()) < 4 * math.sqrt(0.25 * nfis)
    # a source particle at exactly 1 MeV has nu = 2.5: 2 or 3 children, half each
    kids_id, first = np.unique(tr["id"][tr["id"] >= N], return_index=True)
    assert len(kids_id) == c[11]
    Ek = tr["E"][tr["id"] >= N][first] * 1e-6
    assert abs(Ek.mean() - 2.03084) < 4 * Ek.std() / math.sqrt(len(Ek))
    # children are born at the parent's fission site: first record of a child starts from a fission site
    assert c[EV["capture"]] == 0 and c[EV["scatter"]] == 0
    assert c[EV["fission"]] + c[EV["cutoff"]] == c[0] == N + c[11]


def test_c5_subcritical_and_bounded(orc):
    """R25: the synthetic C5 mixture must be subcritical (prompt chain terminates): secondaries < 10 N, no
    lost particle, every track ends in capture / fission / cutoff."""
    N = 400
    P = inputs.config5(n_particles=N)
    o = orc.Oracle(P)
    rc, r = o.run()
    assert rc == 0
    c = r["counters"]
    assert c[11] < 10 * N and c[EV["lost"]] == 0 and c[EV["leak"]] == 0
    assert c[EV["capture"]] + c[EV["fission"]] + c[EV["cutoff"]] == c[0] == N + c[11]
    k_chain = c[11] / c[0]  # secondaries per track = k of the prompt chain
    assert 0.5 < k_chain < 0.95
    # flux tallies: total track length per source history = sum over bins; positive, finite
    f = r["flux_mean"]
    assert np.isfinite(f).all() and f.sum() > 0


def test_quarter_core_finite_height_leakage(orc):
    """Lattice inside z planes (reflecting z = 0, vacuum top): pure absorber, beam along +z from z = 0+: leakage
    through the top = exp(-Sigma_t * height); no lattice wall is ever crossed."""
    hgt, st = 3.0, 0.5
    P = inputs.config4(n_particles=40000, n_inactive=0, n_active=1, n_asm=1, n_pin=2, n_refl=1, G=1, height=hgt)
    for k in ("mg_sig_t", "mg_sig_c"):
        P[k][:] = st
    for k in ("mg_sig_f", "mg_nu", "mg_S"):
        P[k][:] = 0.0
    P["mg_chi"][:] = 1.0
    P["src_lo"][:] = [0.1, 0.1, 1e-9]
    P["src_hi"][:] = [3.6, 3.6, 1e-9]
    P["src_iso"] = 0
    P["src_dir"][:] = [0.0, 0.0, 1.0]
    rc, r = orc.Oracle(P).run()
    assert rc == 0
    p = math.exp(-st * hgt)
    assert abs(r["leak_mean"] - p) < 3 * math.sqrt(p * (1 - p) / 40000)
    assert r["counters"][EV["lattice"]] == 0


@pytest.mark.parametrize("two_level", [False, True])
@pytest.mark.parametrize("start", ["fuel", "moderator"])
def test_axial_reflector_beam_leakage(orc, two_level, start):
    """Fully 3-D core with an axial reflector: every pin universe has a z plane that
    ends the fuel (fuel below it inside the cylinder, moderator beside and above).  Pure absorbers with different cross
    sections in fuel and moderator, a beam along +z from the mid-plane: started inside a fuel cylinder it leaks through
    the top with probability exp(-Sigma_fuel h_fuel - Sigma_mod h_refl), started beside it with exp(-Sigma_mod height);
    a survivor of the fuelled part crosses the new plane exactly once (transmit events); no lattice wall, no cylinder."""
    hgt, h_r, s_fuel, s_mod, N = 3.0, 1.0, 0.5, 0.2, 40000
    P = inputs.config4(n_particles=N, n_inactive=0, n_active=1, n_asm=1, n_pin=2, n_refl=2, G=1, height=hgt,
                       axial_reflector=h_r, two_level=two_level)
    P["mg_sig_t"][:5] = s_fuel; P["mg_sig_t"][5:] = s_mod
    P["mg_sig_c"][:] = P["mg_sig_t"]
    for k in ("mg_sig_f", "mg_nu", "mg_S"):
        P[k][:] = 0.0
    P["mg_chi"][:] = 1.0
    if start == "fuel":   # a square well inside the cylinder of pin (0, 0) (centre 0.63, 0.63; r = 0.54)
        P["src_lo"][:] = [0.33, 0.33, 1e-9]; P["src_hi"][:] = [0.93, 0.93, 1e-9]
        p_plane = math.exp(-s_fuel * (hgt - h_r))
        p = p_plane * math.exp(-s_mod * h_r)
    else:                 # the corner of the same element, outside the cylinder
        P["src_lo"][:] = [0.02, 0.02, 1e-9]; P["src_hi"][:] = [0.12, 0.12, 1e-9]
        p_plane = math.exp(-s_mod * (hgt - h_r))
        p = math.exp(-s_mod * hgt)
    P["src_iso"] = 0
    P["src_dir"][:] = [0.0, 0.0, 1.0]
    rc, r = orc.Oracle(P).run()
    assert rc == 0
    assert abs(r["leak_mean"] - p) < 3.5 * math.sqrt(p * (1 - p) / N)
    c = r["counters"]
    assert abs(c[EV["transmit"]] / N - p_plane) < 3.5 * math.sqrt(p_plane * (1 - p_plane) / N)
    assert c[EV["lattice"]] == 0 and c[EV["reflect"]] == 0 and c[EV["lost"]] == 0
    assert c[EV["capture"]] + c[EV["leak"]] == N


def test_axial_reflector_returns_neutrons(orc):
    """A core of fuelled height 4 with 2 cm of axial reflector on top against the bare core of the same fuelled height,
    same seed: the reflector scatters neutrons back, so k is higher and fewer histories leak (the ordering any transport
    code must reproduce; a reflector cell filled with the wrong material or never entered would not)."""
    kw = dict(n_particles=20000, n_inactive=2, n_active=6, n_asm=1, n_pin=3, n_refl=1)
    rc, refl = orc.Oracle(inputs.config4(height=6.0, axial_reflector=2.0, **kw)).run()
    rc, bare = orc.Oracle(inputs.config4(height=4.0, **kw)).run()
    assert refl["k_mean"] > bare["k_mean"] + 3 * math.hypot(refl["k_sdev"], bare["k_sdev"])
    assert refl["leak_mean"] < bare["leak_mean"] - 3 * math.hypot(refl["leak_sdev"], bare["leak_sdev"])


def test_all_core_variant_equals_serial_run(orc):
    """orc_run_eigenvalue_mt (bench.py's all-core cpu_baseline) splits the source particles in contiguous id ranges:
    identical integer counters and bank, tallies equal to summation order; one thread = the serial run bit for bit."""
    P = inputs.config4(n_particles=6000, n_inactive=1, n_active=2, n_asm=1, n_pin=5, n_refl=2)
    o = orc.Oracle(P)
    rc, r1 = o.run()
    b1 = o.bank().copy()
    rc3, r3 = o.run_mt(3)
    b3 = o.bank().copy()
    assert rc == 0 and rc3 == 0
    assert (r1["counters"] == r3["counters"]).all()
    assert len(b1) == len(b3) and (b1["x"] == b3["x"]).all() and (b1["g"] == b3["g"]).all()
    assert np.allclose(r1["k_cycle"], r3["k_cycle"], rtol=1e-12)
    assert np.allclose(r1["flux_mean"], r3["flux_mean"], rtol=1e-11, atol=1e-15)
    rc1, r1b = o.run_mt(1)
    assert (r1["k_cycle"] == r1b["k_cycle"]).all() and (r1["flux_mean"] == r1b["flux_mean"]).all()
