"""Pins of the oracle's unit-level pieces against what the mathematics fixes (no GPU).

Citations: SURVEY.md 8(c) "What pins each part" table; DESIGN.md section 3 (readings R8-R10, R19-R23).
"""
import math
import os

import numpy as np
import pytest

from paper_2501_05440_b200 import inputs

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def test_philox_known_answers(orc):
    """R10: Philox4x32-10 reproduces the published known-answer vectors (tests/golden)."""
    n = 0
    for line in open(os.path.join(GOLD, "philox4x32_10_kat.txt")):
        if line.startswith("#") or not line.strip():
            continue
        w = [int(x, 16) for x in line.split()]
        assert orc.philox(w[:4], w[4:6]) == w[6:]
        n += 1
    assert n == 3


def test_draw_layout_and_range(orc):
    """R9/R10: draw 2b and 2b+1 are the two u64 halves of block b of counter (id_lo,id_hi,domain<<24|cycle,b);
    xi = ((u>>11)+0.5) 2^-53 lies strictly inside (0,1)."""
    seed, pid, cyc = 0x123456789ABCDEF0, 0xFEDCBA9876543210, 7
    for idx in range(6):
        o = orc.philox([pid & 0xFFFFFFFF, pid >> 32, cyc, idx >> 1], [seed & 0xFFFFFFFF, seed >> 32])
        u = (o[3] << 32 | o[2]) if idx & 1 else (o[1] << 32 | o[0])
        assert orc.draw(seed, pid, 0, cyc, idx) == ((u >> 11) + 0.5) * 2.0 ** -53
    # domain enters the third counter word
    o = orc.philox([5, 0, (1 << 24) | 3, 0], [9, 0])
    assert orc.draw(9, 5, 1, 3, 0) == (((o[1] << 32 | o[0]) >> 11) + 0.5) * 2.0 ** -53


def test_draw_uniformity(orc):
    xs = np.array([orc.draw(1, i, 0, 0, j) for i in range(4000) for j in range(5)])
    assert xs.min() > 0.0 and xs.max() < 1.0
    n = len(xs)
    assert abs(xs.mean() - 0.5) < 4 / math.sqrt(12 * n)
    assert abs(xs.var() - 1 / 12) < 4 * math.sqrt(1 / 180 / n)
    h, _ = np.histogram(xs, 20, (0, 1))
    chi2 = ((h - n / 20) ** 2 / (n / 20)).sum()
    assert chi2 < 50  # 19 dof, p ~ 1e-4
    # streams of neighbouring ids / cycles are uncorrelated
    a = np.array([orc.draw(1, i, 0, 0, 0) for i in range(4000)])
    b = np.array([orc.draw(1, i + 1, 0, 0, 0) for i in range(4000)])
    c = np.array([orc.draw(1, i, 0, 1, 0) for i in range(4000)])
    assert abs(np.corrcoef(a, b)[0, 1]) < 0.07 and abs(np.corrcoef(a, c)[0, 1]) < 0.07


def test_child_id_is_domain1_block(orc):
    """R10: secondary id = first u64 of the domain-1 block (parent id, 1<<24|j, parent ctr)."""
    L = orc.lib()
    seed, pid, ctr, j = 77, 0x1_0000_0005, 19, 2
    o = orc.philox([pid & 0xFFFFFFFF, pid >> 32, (1 << 24) | j, ctr], [seed, 0])
    assert L.orc_child_id(seed, pid, ctr, j) == (o[1] << 32 | o[0])


def test_isotropic_direction(orc):
    """R8: mu = 2 xi1 - 1, phi = 2 pi xi2; unit vectors with <mu>=0, <mu^2>=1/3, <Omega_x Omega_y>=0."""
    rng = np.random.default_rng(0)
    xi = rng.random((20000, 2))
    d = np.array([orc.iso_dir(a, b) for a, b in xi])
    assert np.allclose((d ** 2).sum(1), 1.0, atol=1e-14)
    assert np.allclose(d[:, 2], 2 * xi[:, 0] - 1)
    assert np.allclose(np.arctan2(d[:, 1], d[:, 0]) % (2 * np.pi), 2 * np.pi * xi[:, 1], atol=1e-9)
    n = len(d)
    for ax in range(3):
        assert abs(d[:, ax].mean()) < 4 / math.sqrt(3 * n)
        assert abs((d[:, ax] ** 2).mean() - 1 / 3) < 4 * math.sqrt(4 / 45 / n)
    assert abs((d[:, 0] * d[:, 1]).mean()) < 4 / (3 * math.sqrt(n))
    # fixed points
    assert np.allclose(orc.iso_dir(0.5, 0.0), [1, 0, 0], atol=1e-15)
    assert np.allclose(orc.iso_dir(0.5, 0.25), [0, 1, 0], atol=1e-15)


def test_speed(orc):
    """R23: non-relativistic v = c sqrt(2E / m_n c^2); 2 MeV -> 1.956e9 cm/s."""
    v = orc.speed(2.0e6)
    assert abs(v - 1.956e9) / 1.956e9 < 1e-3
    assert v == pytest.approx(2.99792458e10 * math.sqrt(4.0e6 / 939.56542052e6), rel=1e-15)
    assert orc.speed(8.0e6) == pytest.approx(2 * v, rel=1e-15)


@pytest.mark.parametrize("A", [1.0, 16.0, 238.0])
def test_elastic_kinematics_moments(orc, A):
    """Target-at-rest elastic: E'/E uniform on [alpha,1] (mean (1+alpha)/2), mean lab cosine 2/(3A),
    mean lethargy gain 1 + alpha ln alpha/(1-alpha); the polar angle between Omega and Omega' is mu_lab;
    the azimuth is uniform (SURVEY.md 8c pins, R21)."""
    rng = np.random.default_rng(int(A))
    n = 20000
    alpha = ((A - 1) / (A + 1)) ** 2
    u0 = orc.iso_dir(0.3, 0.7)
    E0 = 1.0e6
    xi = rng.random((n, 2))
    out = [orc.elastic(E0, u0, A, a, b) for a, b in xi]
    r = np.array([o[0] for o in out]) / E0
    un = np.array([o[1] for o in out])
    assert np.allclose((un ** 2).sum(1), 1.0, atol=1e-13)
    assert r.min() >= alpha - 1e-15 and r.max() <= 1.0
    assert abs(r.mean() - (1 + alpha) / 2) < 4 * (1 - alpha) / math.sqrt(12 * n)
    mu = un @ u0
    assert abs(mu.mean() - 2 / (3 * A)) < 4 * mu.std() / math.sqrt(n)
    # closed form for each sample: E'/E = (A^2+2A mu_cm+1)/(A+1)^2, mu_lab = (1+A mu_cm)/sqrt(A^2+2A mu_cm+1)
    mucm = 2 * xi[:, 0] - 1
    den = A * A + 2 * A * mucm + 1
    assert np.allclose(r, den / (A + 1) ** 2, rtol=1e-14)
    assert np.allclose(mu, (1 + A * mucm) / np.sqrt(den), atol=1e-12)
    xi_leth = -np.log(r[r > 0])
    leth = 1.0 if A == 1.0 else 1 + alpha * math.log(alpha) / (1 - alpha)
    assert abs(xi_leth.mean() - leth) < 5 * xi_leth.std() / math.sqrt(n)
    # azimuth about the incoming direction is uniform: component along a fixed perpendicular averages to 0
    e1 = np.cross(u0, [0, 0, 1.0])
    e1 /= np.linalg.norm(e1)
    s = np.sqrt(np.maximum(1 - mu ** 2, 1e-300))
    assert abs(((un @ e1) / s).mean()) < 4 * math.sqrt(0.5 / n)


def test_elastic_polar_special_cases(orc):
    """R21: polar branch when 1-u_z^2 < 1e-10, and A=1 back-scatter (den <= 0 -> mu_lab := 0, E' = 0)."""
    for uz in (1.0, -1.0):
        E1, o = orc.elastic(1.0, [0, 0, uz], 12.0, 0.8, 0.1)
        mucm = 0.6
        den = 144 + 24 * mucm + 1
        mu = (1 + 12 * mucm) / math.sqrt(den)
        assert o[2] == pytest.approx(mu * uz, abs=1e-14)
        assert np.hypot(o[0], o[1]) == pytest.approx(math.sqrt(1 - mu * mu), abs=1e-14)
    # A = 1, mu_cm = -1 exactly cannot be drawn (xi > 0) but the limit must stay finite
    E1, o = orc.elastic(1.0, [1, 0, 0], 1.0, 2.0 ** -54, 0.3)
    assert E1 >= 0 and E1 < 1e-15 and np.isfinite(o).all()
    assert abs(np.dot(o, o) - 1) < 1e-12


def test_watt_mean_and_shape(orc):
    """R22: W ~ Maxwellian(T=a), E' = W + a^2 b/4 + (2 xi-1) sqrt(a^2 b W); mean 3a/2 + a^2 b/4 = 2.03084 MeV;
    histogram against C exp(-E/a) sinh sqrt(bE), C = exp(-ab/4)/sqrt(pi a^3 b/4)."""
    a, b = 0.988, 2.249
    rng = np.random.default_rng(5)
    n = 40000
    xi = rng.random((n, 4))
    E = np.array([orc.watt(a, b, *x) for x in xi])
    assert E.min() > 0
    mean = 1.5 * a + a * a * b / 4
    assert mean == pytest.approx(2.03084, abs=2e-5)
    assert abs(E.mean() - mean) < 4 * E.std() / math.sqrt(n)
    edges = np.linspace(0, 12, 25)
    h, _ = np.histogram(E, edges)
    xs = np.linspace(0, 40, 80001)
    C = math.exp(-a * b / 4) / math.sqrt(math.pi * a ** 3 * b / 4)
    pdf = C * np.exp(-xs / a) * np.sinh(np.sqrt(b * xs))
    cdf = np.concatenate([[0], np.cumsum(0.5 * (pdf[1:] + pdf[:-1]) * np.diff(xs))])
    assert cdf[-1] == pytest.approx(1.0, abs=2e-4)  # the quoted normalisation constant is right
    exp = n * np.diff(np.interp(edges, xs, cdf))
    keep = exp > 20
    chi2 = ((h[keep] - exp[keep]) ** 2 / exp[keep]).sum()
    assert chi2 < keep.sum() + 5 * math.sqrt(2 * keep.sum())


def _ce_problem(jitter):
    P = inputs.config5(n_particles=10, n_grid=3000, jitter=jitter)
    return P


@pytest.mark.parametrize("jitter", [False, True])
def test_grid_search_matches_linear_scan(orc, jitter):
    """R19: index i with grid[i] <= E < grid[i+1], clamped to [0, n-2] -- against numpy's searchsorted
    (a library routine) and a brute-force linear scan, incl. exact nodes, ends and out-of-range."""
    P = _ce_problem(jitter)
    o = orc.Oracle(P)
    g = P["grid"]
    rng = np.random.default_rng(3)
    E = np.concatenate([np.exp(rng.uniform(np.log(1e-6), np.log(1e8), 3000)), g[::37], g[:3], g[-3:],
                        np.nextafter(g[::91], 0), np.nextafter(g[::91], np.inf), [1e-7, 5e7]])
    ref = np.clip(np.searchsorted(g, E, side="right") - 1, 0, len(g) - 2)
    got = np.array([o.grid_index(e) for e in E])
    assert (got == ref).all()
    for e in E[:200]:
        i = 0
        while i + 1 < len(g) - 1 and g[i + 1] <= e:
            i += 1
        assert o.grid_index(e) == i


def test_ce_interpolation_nodes_and_midpoints(orc):
    """R19: table values are the definition; lin-lin between nodes; cumulative order [el_1..el_n, fission, capture]."""
    P = _ce_problem(True)
    o = orc.Oracle(P)
    g = P["grid"]
    for m in range(2):
        n0, n1 = P["mat_nuc_off"][m], P["mat_nuc_off"][m + 1]
        ids, dens = P["mat_nuc_id"][n0:n1], P["mat_nuc_dens"][n0:n1]

        def cols(i):
            el = [d * P["nuc_el"][k, i] for k, d in zip(ids, dens)]
            f = sum(d * P["nuc_f"][k, i] for k, d in zip(ids, dens))
            c = sum(d * P["nuc_c"][k, i] for k, d in zip(ids, dens))
            return np.array(el + [f, c])

        for i in (0, 1, 777, 1500, len(g) - 2):
            got = o.ce_xs(m, g[i])
            assert np.allclose(got[1:], np.cumsum(cols(i)), rtol=1e-13)
            assert got[0] == got[-1]
            Em = 0.25 * g[i] + 0.75 * g[i + 1]
            got = o.ce_xs(m, Em)
            assert np.allclose(got[1:], np.cumsum(0.25 * cols(i) + 0.75 * cols(i + 1)), rtol=1e-12)
        # outside the grid: linear extrapolation is never used after clamping (R19); the index clamps
        assert o.grid_index(1e-9) == 0 and o.grid_index(1e9) == len(g) - 2
