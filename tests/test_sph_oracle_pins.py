"""Pins of the short-range (SPH) oracle functions (oracle/sph_oracle.c) and of the
neighbour-list builder of the harness, against what the mathematics fixes: textbook values of the cubic spline, its
unit volume integral, finite differences, brute force, symmetry and conservation, the analytic Plummer density.
None of these values comes from the CUDA path; none retypes the oracle's piecewise polynomial.
"""
import math

import numpy as np
import pytest

import oracle
from oracle import bhtree_ref
from paper_1907_02290_b200.workload import SPH_CONFIGS, build_tree_and_lists, make_particles, make_sph_fields, make_workload


def all_pairs_lists(n):
    """One group holding every particle, whose list is every particle."""
    return (np.array([0], np.int32), np.array([n], np.int32), np.array([0, n], np.int64), np.arange(n, dtype=np.int32))


def sph4(h, u=1.0, rho=0.0, pr2=0.0, n=None):
    h = np.atleast_1d(np.asarray(h, np.float64))
    n = h.shape[0] if n is None else n
    out = np.zeros((n, 4), np.float32)
    out[:, 0], out[:, 1], out[:, 2], out[:, 3] = h, u, rho, pr2
    return out


# ---------------------------------------------------------------- the kernel itself
def test_kernel_textbook_values():
    """Monaghan & Lattanzio's M4 spline in 3-D: W(0) = 1/(pi h^3), W(h) = 1/(4 pi h^3), W(3h/2) = 1/(32 pi h^3),
    W(>= 2h) = 0; dW/dr(h) = -3/(4 pi h^4), dW/dr(0) = 0.  Catches a wrong normalisation (2-D's 10/7pi, 1-D's 2/3),
    a wrong power of h and swapped branches."""
    for h in (1.0, 0.5, 3.0):
        s = 1.0 / (math.pi * h ** 3)
        assert oracle.sph_w(0.0, h) == pytest.approx(s, rel=1e-15)
        assert oracle.sph_w(h, h) == pytest.approx(s / 4, rel=1e-15)
        assert oracle.sph_w(1.5 * h, h) == pytest.approx(s / 32, rel=1e-14)
        assert oracle.sph_w(2.0 * h, h) == 0.0 and oracle.sph_w(2.5 * h, h) == 0.0
        assert oracle.sph_dwdr(h, h) == pytest.approx(-0.75 * s / h, rel=1e-15)
        assert oracle.sph_dwdr(0.0, h) == 0.0 and oracle.sph_dwdr(2.0 * h, h) == 0.0


def test_kernel_is_normalised_and_smooth():
    """int W dV = 1 by quadrature; W is continuous with continuous first derivative at q = 1 and q = 2."""
    h = 0.7
    r = (np.arange(200000) + 0.5) * (2 * h / 200000)
    w = np.array([oracle.sph_w(x, h) for x in r[::100]])
    integral = np.sum(4 * math.pi * r[::100] ** 2 * w) * (2 * h / 2000)
    assert integral == pytest.approx(1.0, abs=2e-6)
    for q in (1.0, 2.0):
        e = 1e-7
        assert oracle.sph_w((q - e) * h, h) == pytest.approx(oracle.sph_w((q + e) * h, h), abs=1e-6)
        assert oracle.sph_dwdr((q - e) * h, h) == pytest.approx(oracle.sph_dwdr((q + e) * h, h), abs=1e-5)


def test_dwdr_is_the_derivative_of_w():
    """Central differences of W at points in both branches (catches a sign or factor in the printed dW/dr)."""
    h = 1.3
    for q in (0.1, 0.5, 0.99, 1.01, 1.5, 1.9):
        r, e = q * h, 1e-6
        fd = (oracle.sph_w(r + e, h) - oracle.sph_w(r - e, h)) / (2 * e)
        assert oracle.sph_dwdr(r, h) == pytest.approx(fd, rel=1e-6, abs=1e-10)


# ---------------------------------------------------------------- density
def test_density_of_two_particles():
    """rho_1 = m_1 W(0, h_1) + m_2 W(r, h_1): the i-particle's OWN h (gather), self term included, m_k not m_i."""
    posm = np.array([[0, 0, 0, 2.0], [0.5, 0, 0, 3.0]], np.float32)     # r = 0.5
    s = sph4([0.5, 1.0], u=[1.5, 0.25])                                # q = 1 for particle 0, q = 1/2 for particle 1
    rho, pr2 = oracle.sph_density(posm, s, *all_pairs_lists(2), gamma=1.4)
    w0 = 1.0 / (math.pi * 0.125)
    assert rho[0] == pytest.approx(2.0 * w0 + 3.0 * w0 / 4, rel=1e-14)
    w1 = 1.0 / math.pi                                                  # W(q = 1/2) = (1 - 3/8 + 3/32) / (pi h^3)
    assert rho[1] == pytest.approx(3.0 * w1 + 2.0 * w1 * (1 - 0.375 + 0.09375), rel=1e-14)
    np.testing.assert_allclose(pr2, 0.4 * np.array([1.5, 0.25]) / rho, rtol=1e-14)   # ideal gas, P/rho^2 = (gamma-1) u / rho


def test_density_of_a_lattice_is_the_mass_density():
    """A cubic lattice of spacing d with unit mass density seen with h = 2.5 d: the kernel sum is a quadrature of
    int W dV = 1, so rho = 1 to ~1e-4 (the lattice quadrature error of a C2 kernel)
    away from the faces.  Catches normalisation and polynomial errors globally."""
    k = 13
    d = 0.1
    g = (np.arange(k) - k // 2) * d
    pos = np.stack(np.meshgrid(g, g, g, indexing="ij"), -1).reshape(-1, 3)
    posm = np.concatenate([pos, np.full((len(pos), 1), d ** 3)], 1).astype(np.float32)
    s = sph4(np.full(len(pos), 2.5 * d))
    rho = oracle.sph_density_direct(posm, s)
    centre = np.argmin(np.sum(pos ** 2, 1))
    assert rho[centre] == pytest.approx(1.0, abs=3e-4)


def test_lists_give_exactly_the_all_pairs_sums():
    """Compact support: over a COMPLETE neighbour list the density and the acceleration equal the sums over all
    particles (to rounding).  Pins the list evaluation and the neighbour search of the harness together, with
    particle-dependent h so that both the gather and the scatter reach matter."""
    cfg = SPH_CONFIGS[0]
    w = make_workload(cfg, n=3000)
    rho, pr2 = oracle.sph_density(w.posm, w.sph, w.grp_first, w.grp_n, w.epj_off, w.epj_id, cfg.gamma)
    np.testing.assert_allclose(rho, oracle.sph_density_direct(w.posm, w.sph), rtol=1e-13)
    s = w.sph.copy()
    s[:, 2], s[:, 3] = rho, pr2
    acc, scale = oracle.sph_hydro(w.posm, s, w.grp_first, w.grp_n, w.epj_off, w.epj_id)
    acc_d, scale_d = oracle.sph_hydro_direct(w.posm, s)
    lone = scale_d == 0                                                  # halo particles with nobody inside 2h
    assert np.max(np.abs(acc - acc_d)[~lone] / scale_d[~lone, None]) < 1e-13
    assert np.all(acc[lone] == 0) and np.all(scale[lone] == 0)
    np.testing.assert_allclose(scale, scale_d, rtol=1e-12)
    assert np.mean(~lone) > 0.7


# ---------------------------------------------------------------- pressure-gradient acceleration
def test_hydro_pair_matches_finite_difference_of_density():
    """Two particles, equal h: a_1 = -m_2 (P_1/rho_1^2 + P_2/rho_2^2) dW/dx_1, and m_2 dW/dx_1 is the derivative of
    rho_1 with respect to x_1 -- taken by central differences of the DENSITY function.  Pins sign and direction of
    the gradient and the (P_i/rho_i^2 + P_k/rho_k^2) factor without retyping dW/dr."""
    h, m2 = 0.8, 3.0
    x1 = np.array([0.3, -0.2, 0.4])
    p1, p2 = 0.7, 1.9

    def rho1(x):
        posm = np.array([[*x, 2.0], [0, 0, 0, m2]], np.float32).astype(np.float32)
        return oracle.sph_density_direct(posm, sph4([h, h]))[0]

    posm = np.array([[*x1, 2.0], [0, 0, 0, m2]], np.float32)
    s = sph4([h, h], pr2=[p1, p2])
    acc, scale = oracle.sph_hydro_direct(posm, s)
    x1f = posm[0, :3].astype(np.float64)
    for d in range(3):
        e = np.zeros(3)
        e[d] = 2.0 ** -9                                                 # exactly representable step
        grad = (rho1(x1f + e) - rho1(x1f - e)) / (2 * e[d])
        assert acc[0, d] == pytest.approx(-(p1 + p2) * grad, rel=2e-4)
    # Newton's third law for the pair
    np.testing.assert_allclose(2.0 * acc[0], -m2 * acc[1], rtol=1e-14)
    assert scale[0] == pytest.approx(np.linalg.norm(acc[0]), rel=1e-14)


def test_hydro_symmetrised_gradient_uses_both_smoothing_lengths():
    """r between 2 h_1 and 2 h_2: only the scatter half (gradW with h_2) acts, with weight 1/2."""
    posm = np.array([[1.0, 0, 0, 1.0], [0, 0, 0, 1.0]], np.float32)
    s = sph4([0.25, 1.0], pr2=[1.0, 1.0])                                # r = 1 = q_2 h_2, beyond 2 h_1
    acc, _ = oracle.sph_hydro_direct(posm, s)
    want = -1.0 * 2.0 * 0.5 * (-0.75 / math.pi)                          # -m (P1+P2) 1/2 dW/dr(q = 1, h = 1), along +x
    np.testing.assert_allclose(acc[0], [want, 0, 0], rtol=1e-14, atol=1e-18)


def test_hydro_conserves_momentum_and_vanishes_in_a_uniform_lattice():
    rng = np.random.default_rng(11)
    n = 400
    posm = np.concatenate([rng.uniform(0, 1, (n, 3)), rng.uniform(0.5, 2.0, (n, 1))], 1).astype(np.float32)
    s = sph4(rng.uniform(0.08, 0.25, n), pr2=rng.uniform(0.5, 2.0, n))
    acc, scale = oracle.sph_hydro_direct(posm, s)
    mom = np.sum(posm[:, 3:4].astype(np.float64) * acc, 0)
    assert np.linalg.norm(mom) < 1e-13 * np.sum(posm[:, 3].astype(np.float64) * scale)
    # uniform lattice, uniform pressure: every interior particle sits at a centre of symmetry
    k, d = 9, 0.125
    g = (np.arange(k) - k // 2) * d
    pos = np.stack(np.meshgrid(g, g, g, indexing="ij"), -1).reshape(-1, 3)
    posm = np.concatenate([pos, np.full((len(pos), 1), 1.0)], 1).astype(np.float32)
    acc, scale = oracle.sph_hydro_direct(posm, sph4(np.full(len(pos), 1.5 * d), pr2=1.0))
    centre = np.argmin(np.sum(pos ** 2, 1))
    assert np.linalg.norm(acc[centre]) < 1e-14 * scale[centre]


def test_hydro_reproduces_a_linear_pressure_gradient():
    """Lattice of unit density with P/rho^2 = p0 + g x: the SPH estimate of -grad(P)/rho at the centre is -g along x
    (second-order consistent on a symmetric lattice).  Catches a missing factor 1/2 or m."""
    k, d = 13, 0.1
    g_ = (np.arange(k) - k // 2) * d
    pos = np.stack(np.meshgrid(g_, g_, g_, indexing="ij"), -1).reshape(-1, 3)
    posm = np.concatenate([pos, np.full((len(pos), 1), d ** 3)], 1).astype(np.float32)
    grad = 0.3
    s = sph4(np.full(len(pos), 2.5 * d), pr2=1.0 + grad * pos[:, 0])
    acc, _ = oracle.sph_hydro_direct(posm, s)
    centre = np.argmin(np.sum(pos ** 2, 1))
    np.testing.assert_allclose(acc[centre], [-grad, 0, 0], rtol=5e-3, atol=1e-6)   # lattice discretisation: 0.24 %


def test_coincident_particles_exert_no_pressure_force():
    posm = np.array([[0.5, 0.5, 0.5, 1.0], [0.5, 0.5, 0.5, 2.0], [0.6, 0.5, 0.5, 1.0]], np.float32)
    s = sph4([0.2, 0.2, 0.2], pr2=1.0)
    acc, _ = oracle.sph_hydro_direct(posm, s)
    assert np.all(np.isfinite(acc))
    np.testing.assert_allclose(acc[0], acc[1], rtol=1e-15)             # both feel only particle 2


# ---------------------------------------------------------------- generator + density together
def test_sph_density_of_the_plummer_gas_sphere():
    """Particles drawn independently from the analytic Plummer density rho(r) = 3/(4 pi) (1 + r^2)^(-5/2) that the
    smoothing lengths were derived from: by Campbell's theorem the expected kernel sum over the OTHER particles at a
    particle's position is the (smoothed) analytic density, so mean[(rho_i - m_i W(0, h_i)) / rho(r_i)] = 1 up to the
    O(h^2) smoothing bias, with a per-particle scatter of ~ 1/sqrt(58 neighbours); with the self term the mean is
    1 + 1/(pi eta^3).  Pins generator, smoothing lengths and density together (cf. pin P6 for gravity)."""
    cfg = SPH_CONFIGS[0]
    w = make_workload(cfg)
    rho, _ = oracle.sph_density(w.posm, w.sph, w.grp_first, w.grp_n, w.epj_off, w.epj_id, cfg.gamma)
    r2 = np.sum(w.posm[:, :3].astype(np.float64) ** 2, 1)
    ana = 3.0 / (4.0 * math.pi) * (1.0 + r2) ** -2.5
    inner = r2 < 4.0
    h, m = w.sph[:, 0].astype(np.float64), w.posm[:, 3].astype(np.float64)
    others = (rho - m / (math.pi * h ** 3)) / ana
    assert abs(np.mean(others[inner]) - 1.0) < 0.03
    assert np.std(others[inner]) < 0.4
    assert np.mean(rho[inner] / ana[inner]) == pytest.approx(1.0 + 1.0 / (math.pi * cfg.eta ** 3), abs=0.03)


# ---------------------------------------------------------------- neighbour lists of the harness
def test_neighbour_builder_matches_plain_restatement():
    cfg = SPH_CONFIGS[0]
    for n, n_leaf, n_grp, skin in ((700, 8, 32, 0.0), (1500, 16, 64, 0.2), (64, 4, 8, 0.0)):
        posm, _ = make_particles(cfg, n)
        s = make_sph_fields(cfg, posm)
        w = build_tree_and_lists(posm, n_leaf, n_grp, 0.0, sph=s, skin=skin)
        ref = bhtree_ref.build(posm, n_leaf, n_grp, 0.0, h=s[:, 0], skin=skin)
        np.testing.assert_array_equal(w.perm, ref["perm"])
        np.testing.assert_array_equal(w.grp_cell, ref["groups"])
        assert w.spj_off[-1] == 0
        for g in range(w.n_group):
            np.testing.assert_array_equal(w.epj_id[w.epj_off[g]:w.epj_off[g + 1]], np.array(ref["epj"][g], np.int32))


def test_neighbour_lists_are_complete_and_stay_complete_within_the_skin():
    """Every pair with r < 2 max(h_i, h_k) is in the list of i's group (brute force), without duplicates; with a skin
    the lists still cover all interacting pairs after the particles have moved by less than skin * h_min / ... ."""
    cfg = SPH_CONFIGS[0]
    n = 2500
    posm, _ = make_particles(cfg, n)
    s = make_sph_fields(cfg, posm)
    for skin, move in ((0.0, 0.0), (0.15, 0.07)):
        w = build_tree_and_lists(posm, 16, 48, 0.0, sph=s, skin=skin)
        pos = w.posm[:, :3].astype(np.float64)
        h = w.sph[:, 0].astype(np.float64)
        if move:
            rng = np.random.default_rng(3)
            step = rng.normal(size=(n, 3))
            pos = pos + move * h[:, None] * step / np.linalg.norm(step, axis=1)[:, None]   # each by 0.07 h_i: pairs close by < 0.15 max(h)
        d = np.linalg.norm(pos[:, None, :] - pos[None, :, :], axis=2)
        need = d < 2.0 * np.maximum(h[:, None], h[None, :])
        for g in range(w.n_group):
            ids = w.epj_id[w.epj_off[g]:w.epj_off[g + 1]]
            assert len(np.unique(ids)) == len(ids)
            have = np.zeros(n, bool)
            have[ids] = True
            f, c = w.grp_first[g], w.grp_n[g]
            assert not np.any(need[f:f + c] & ~have[None, :])
