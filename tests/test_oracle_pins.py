"""Pins of the fp64 oracle (oracle/) against closed forms, invariants and brute force.

Each test names the SURVEY.md section 8(c) pin (P1..P8) it implements and the mistake it is meant to
catch.  None of these values comes from the CUDA path.
"""
import math

import numpy as np
import pytest

import oracle
from paper_1907_02290_b200.workload import CONFIGS, build_tree_and_lists, make_particles, make_workload


def one_group_lists(n, i_first, n_i, epj, spj=()):
    grp_first = np.array([i_first], np.int32)
    grp_n = np.array([n_i], np.int32)
    epj_off = np.array([0, len(epj)], np.int64)
    spj_off = np.array([0, len(spj)], np.int64)
    return grp_first, grp_n, epj_off, np.array(epj, np.int32), spj_off, np.array(spj, np.int32)


def eval_lists(posm, mom, lists, eps, G=1.0):
    gf, gn, eo, ei, so, si = lists
    return oracle.forces(posm, mom, gf, gn, eo, ei, so, si, eps, G)


# ---------------------------------------------------------------- P1: closed forms
def test_single_source_is_a_plummer_sphere():
    """One source of mass M with eps = a IS a Plummer sphere: phi = -GM/sqrt(r^2+a^2),
    |a| = GM r/(r^2+a^2)^(3/2), pointing at the source.  Catches sign, exponent, eps and G errors."""
    M, a, G = 2.0, 0.5, 3.0
    src = np.array([1.0, -2.0, 0.5])
    d = np.array([3.0, 4.0, 12.0])            # |d| = 13, all exactly representable in fp32
    posm = np.array([[*src, M], [*(src + d), 0.25]], np.float32)
    r2 = 169.0 + a * a
    want_acc = -G * M * d / r2 ** 1.5         # test particle is pulled back toward the source
    want_pot = -G * M / math.sqrt(r2)
    acc, pot = oracle.direct(posm, a, G)
    np.testing.assert_allclose(acc[1], want_acc, rtol=1e-14)
    assert pot[1] == pytest.approx(want_pot, rel=1e-14)
    # the same through the list path, source as an EPJ
    mom = np.zeros((1, 4))
    acc, pot = eval_lists(posm, mom, one_group_lists(2, 1, 1, [0, 1]), a, G)
    np.testing.assert_allclose(acc[1], want_acc, rtol=1e-14)
    assert pot[1] == pytest.approx(want_pot, rel=1e-14)
    # and with the source given as an SPJ (cell 0 = a monopole at src with mass M)
    mom = np.array([[*src, M]])
    acc, pot = eval_lists(posm, mom, one_group_lists(2, 1, 1, [1], [0]), a, G)
    np.testing.assert_allclose(acc[1], want_acc, rtol=1e-14)
    assert pot[1] == pytest.approx(want_pot, rel=1e-14)


def test_two_unequal_bodies():
    """a_1 = G m_2 d/(..), a_2 = -G m_1 d/(..): catches using m_i where m_j belongs and a flipped d."""
    posm = np.array([[0, 0, 0, 3.0], [1, 2, 2, 0.5]], np.float32)   # |d| = 3
    eps = 4.0                                                      # r2 = 25
    acc, pot = oracle.direct(posm, eps, 1.0)
    d = np.array([1.0, 2.0, 2.0])
    np.testing.assert_allclose(acc[0], 0.5 * d / 125.0, rtol=1e-15)
    np.testing.assert_allclose(acc[1], -3.0 * d / 125.0, rtol=1e-15)
    assert pot[0] == pytest.approx(-0.5 / 5.0, rel=1e-15)
    assert pot[1] == pytest.approx(-3.0 / 5.0, rel=1e-15)


def test_ring_on_axis():
    """n equal masses on a ring of radius R: on the axis at height z,
    a_z = -G n m z/(R^2+z^2+eps^2)^(3/2), a_x = a_y = 0, phi = -G n m/sqrt(R^2+z^2+eps^2).
    Catches per-component mix-ups (a transposed coordinate breaks the cancellation)."""
    n, R, z, m, eps = 16, 2.0, 1.5, 0.125, 0.25
    ang = 2 * np.pi * np.arange(n) / n
    ring = np.stack([R * np.cos(ang), R * np.sin(ang), np.zeros(n), np.full(n, m)], axis=1)
    posm = np.concatenate([ring, [[0, 0, z, 1.0]]]).astype(np.float32)
    acc, pot = oracle.direct(posm, eps, 1.0)
    s = R * R + z * z + eps * eps
    assert acc[n, 2] == pytest.approx(-n * m * z / s ** 1.5, rel=1e-6)   # fp32 rounding of the ring
    assert abs(acc[n, 0]) < 1e-8 and abs(acc[n, 1]) < 1e-8
    assert pot[n] == pytest.approx(-n * m / math.sqrt(s), rel=1e-6)


def test_exact_scaling_laws():
    """x -> 2x, eps -> 2eps gives acc/4 and pot/2; m -> 4m gives 4x both.  Powers of two are exact in
    fp32, so this pins the -3/2 and -1/2 exponents to rounding."""
    posm, _ = make_particles(CONFIGS[0], 256)
    a1, p1 = oracle.direct(posm, 1 / 64, 1.0)
    q = posm.copy()
    q[:, :3] *= 2
    a2, p2 = oracle.direct(q, 2 / 64, 1.0)
    np.testing.assert_allclose(a2, a1 / 4, rtol=1e-13)
    np.testing.assert_allclose(p2, p1 / 2, rtol=1e-13)
    q = posm.copy()
    q[:, 3] *= 4
    a3, p3 = oracle.direct(q, 1 / 64, 0.5)
    np.testing.assert_allclose(a3, a1 * 2, rtol=1e-13)
    np.testing.assert_allclose(p3, p1 * 2, rtol=1e-13)


def test_coincident_distinct_particles_are_a_real_pair():
    """Reading S4: only the entry whose INDEX equals i is skipped; another particle at the same
    position adds 0 to acc and -G m/eps to pot."""
    posm = np.array([[1, 1, 1, 2.0], [1, 1, 1, 5.0]], np.float32)
    acc, pot = oracle.direct(posm, 0.5, 1.0)
    assert np.all(acc == 0)
    assert pot[0] == -5.0 / 0.5 and pot[1] == -2.0 / 0.5


# ---------------------------------------------------------------- P2, P3: brute force / theta -> 0
def brute_force(posm, eps, G):
    """Test-local O(N^2) numpy evaluation (fp64), j != i."""
    x = posm[:, :3].astype(np.float64)
    m = posm[:, 3].astype(np.float64)
    d = x[None, :, :] - x[:, None, :]
    r2 = (d ** 2).sum(-1) + eps * eps
    np.fill_diagonal(r2, np.inf)
    w = m[None, :] / r2 ** 1.5
    return G * (w[:, :, None] * d).sum(1), -G * (m[None, :] / np.sqrt(r2)).sum(1)


@pytest.mark.parametrize("n", [1, 2, 37, 700])
def test_direct_equals_brute_force(n):
    posm, _ = make_particles(CONFIGS[0], n)
    a, p = oracle.direct(posm, 1 / 64, 1.5)
    ab, pb = brute_force(posm, 1 / 64, 1.5)
    np.testing.assert_allclose(a, ab, rtol=1e-12, atol=1e-15)
    np.testing.assert_allclose(p, pb, rtol=1e-12, atol=1e-15)


@pytest.mark.parametrize("theta", [0.0, 1e-3])
def test_theta_to_zero_reproduces_direct_summation(theta):
    """north_star pin: with theta -> 0 every list is all particles and the list path equals direct
    summation (checks CSR offsets, group ranges and index-based self exclusion)."""
    posm, _ = make_particles(CONFIGS[0], 1500)
    w = build_tree_and_lists(posm, 8, 64, theta)
    assert w.spj_off[-1] == 0
    mom = oracle.monopoles(w.cells, w.posm)
    acc, pot = oracle.forces(w.posm, mom, w.grp_first, w.grp_n, w.epj_off, w.epj_id, w.spj_off, w.spj_id, 1 / 64)
    ab, pb = brute_force(w.posm, 1 / 64, 1.0)
    np.testing.assert_allclose(acc, ab, rtol=1e-12, atol=1e-14)
    np.testing.assert_allclose(pot, pb, rtol=1e-12)


def test_group_subset_selection():
    w = make_workload(CONFIGS[0], 2000)
    mom = oracle.monopoles(w.cells, w.posm)
    args = (w.posm, mom, w.grp_first, w.grp_n, w.epj_off, w.epj_id, w.spj_off, w.spj_id, 1 / 64)
    acc, pot = oracle.forces(*args)
    sel = np.arange(1, w.n_group, 3)
    acc_s, pot_s = oracle.forces(*args, groups=sel)
    mask = np.zeros(w.n, bool)
    for g in sel:
        mask[w.grp_first[g]:w.grp_first[g] + w.grp_n[g]] = True
    assert np.array_equal(acc_s[mask], acc[mask]) and np.array_equal(pot_s[mask], pot[mask])
    assert np.all(np.isnan(acc_s[~mask])) and np.all(np.isnan(pot_s[~mask]))


# ---------------------------------------------------------------- P5: momentum conservation
def test_direct_sum_conserves_momentum():
    """Newton's third law holds term by term for direct summation: |sum m a| <= 1e-13 sum m|a|."""
    posm, _ = make_particles(CONFIGS[2], 1024)      # unequal masses (disk + halo)
    acc, _ = oracle.direct(posm, 0.005)
    m = posm[:, 3].astype(np.float64)
    resid = np.linalg.norm((m[:, None] * acc).sum(0))
    assert resid <= 1e-13 * (m * np.linalg.norm(acc, axis=1)).sum()


# ---------------------------------------------------------------- P6: Plummer potential energy
def truncated_plummer_W(rc):
    """W of a unit-mass Plummer sphere (G = a = 1) cut at r < rc and renormalised to unit mass:
    W = -4 pi int_0^rc rho(r) M(r) r dr / M(rc)^2, by quadrature."""
    from scipy.integrate import quad
    rho = lambda r: 3.0 / (4 * np.pi) * (1 + r * r) ** -2.5
    mass = lambda r: r ** 3 * (1 + r * r) ** -1.5
    val, _ = quad(lambda r: rho(r) * mass(r) * r, 0, rc, epsabs=1e-13, epsrel=1e-12)
    return -4 * np.pi * val / mass(rc) ** 2


def test_plummer_potential_energy(golden):
    """north_star pin: W = -3 pi G M^2/(32 a); with the cut at 22.8a the exact value is 1.0055x that.
    Ties the generator, the pair sum and the sign/scale of pot (reading S3) together."""
    w_inf = golden["plummer_W_coeff"]
    assert w_inf == pytest.approx(-3 * math.pi / 32, rel=1e-15)
    assert truncated_plummer_W(1e4) == pytest.approx(w_inf, rel=1e-6)
    want = truncated_plummer_W(22.8)
    assert want / w_inf == pytest.approx(1.0055, abs=5e-4)
    posm, _ = make_particles(CONFIGS[0], 16384)
    _, pot = oracle.direct(posm, 1 / 64)
    W = 0.5 * np.sum(posm[:, 3].astype(np.float64) * pot)
    assert W == pytest.approx(want, rel=0.02)       # sampling scatter ~0.4 % at N = 16384; eps shifts -0.05 %


# ---------------------------------------------------------------- P7: Barnes-Hut quality of tree lists
def test_tree_forces_converge_to_direct_sum():
    """The list path with SPJ monopoles approximates direct summation, better as theta falls.
    A wrong SPJ index, a missing list segment or a bad monopole gives O(1) errors here."""
    posm, _ = make_particles(CONFIGS[0], 4096)
    eps = 1 / 64
    rms = []
    for theta in (0.8, 0.5, 0.3):
        w = build_tree_and_lists(posm, 8, 64, theta)
        mom = oracle.monopoles(w.cells, w.posm)
        acc, pot = oracle.forces(w.posm, mom, w.grp_first, w.grp_n, w.epj_off, w.epj_id, w.spj_off, w.spj_id, eps)
        ad, pd = oracle.direct(w.posm, eps)
        e = np.linalg.norm(acc - ad, axis=1) / np.linalg.norm(ad, axis=1)
        rms.append(np.sqrt(np.mean(e ** 2)))
        if theta == 0.5:
            assert 5e-5 < rms[-1] < 3e-3 and e.max() < 5e-2
            assert np.sqrt(np.mean(((pot - pd) / pd) ** 2)) < 5e-4
            m = w.posm[:, 3].astype(np.float64)
            assert 0.5 * np.sum(m * pot) == pytest.approx(0.5 * np.sum(m * pd), rel=3e-4)
    assert rms[0] > rms[1] > rms[2]


# ---------------------------------------------------------------- P8: monopoles
def test_monopole_invariants():
    w = make_workload(CONFIGS[2], 3000)              # unequal masses
    mom = oracle.monopoles(w.cells, w.posm)
    x = w.posm[:, :3].astype(np.float64)
    m = w.posm[:, 3].astype(np.float64)
    # root = whole system
    assert mom[0, 3] == pytest.approx(m.sum(), rel=1e-13)
    np.testing.assert_allclose(mom[0, :3], (m[:, None] * x).sum(0) / m.sum(), rtol=1e-12, atol=1e-15)
    # parent = mass-weighted combination of its children (the paper's bottom-up pass)
    for c in range(w.n_cell):
        fc, nc = w.cells[c, 2], w.cells[c, 3]
        if nc:
            ch = mom[fc:fc + nc]
            assert ch[:, 3].sum() == pytest.approx(mom[c, 3], rel=1e-13)
            np.testing.assert_allclose((ch[:, 3:4] * ch[:, :3]).sum(0) / ch[:, 3].sum(), mom[c, :3], rtol=1e-11, atol=1e-14)
    # centre of mass lies inside the cell cube
    half = 0.5 * w.geom[:, 3:4] * (1 + 1e-12)
    assert np.all(np.abs(mom[:, :3] - w.geom[:, :3]) <= half)
    # translating all particles by t moves every X_c by t and leaves M_c alone; positions are first put
    # on a 2^-12 grid so that the translated fp32 values are exact
    t = np.array([64.0, -32.0, 16.0])
    q0 = w.posm.copy()
    q0[:, :3] = np.clip(np.round(q0[:, :3].astype(np.float64) * 4096) / 4096, -1000, 1000)
    q1 = q0.copy()
    q1[:, :3] = (q0[:, :3].astype(np.float64) + t).astype(np.float32)
    assert np.all(q1[:, :3].astype(np.float64) - t == q0[:, :3])
    mom0, mom1 = oracle.monopoles(w.cells, q0), oracle.monopoles(w.cells, q1)
    assert np.array_equal(mom1[:, 3], mom0[:, 3])
    np.testing.assert_allclose(mom1[:, :3] - t, mom0[:, :3], atol=1e-12)


# ---------------------------------------------------------------- leapfrog (NEXT-1): closed forms
def _kdk(x, v, acc_of, dt, steps):
    """Drive oracle.kick_drift / oracle.kick; the accelerations come from the test (acc_of), fp32 state."""
    x = x.astype(np.float32); v = v.astype(np.float32)
    a = acc_of(x.astype(np.float64)).astype(np.float32)
    for _ in range(steps):
        posm = np.concatenate([x, np.ones((len(x), 1), np.float32)], axis=1)
        v4 = np.concatenate([v, np.zeros((len(x), 1), np.float32)], axis=1)
        a4 = np.concatenate([a, np.zeros((len(x), 1), np.float32)], axis=1)
        xn, vh = oracle.kick_drift(posm, v4, a4, dt)
        x = xn.astype(np.float32); vh = vh.astype(np.float32)
        a = acc_of(x.astype(np.float64)).astype(np.float32)
        v4 = np.concatenate([vh, np.zeros((len(x), 1), np.float32)], axis=1)
        a4 = np.concatenate([a, np.zeros((len(x), 1), np.float32)], axis=1)
        v = oracle.kick(v4, a4, dt).astype(np.float32)
    return x.astype(np.float64), v.astype(np.float64)


def test_leapfrog_constant_acceleration_is_exact():
    """Uniform acceleration g: one kick-drift-kick step gives x0 + v0 dt + g dt^2/2 and v0 + g dt exactly
    (catches a missing 1/2, a drift that uses the old velocity, a kick applied twice).  Dyadic values:
    every operation is exact in fp32, so equality is bitwise."""
    x0 = np.array([[1.0, -2.0, 0.5], [0.25, 4.0, -8.0]])
    v0 = np.array([[0.5, 0.25, -1.0], [2.0, -0.5, 0.125]])
    g = np.array([0.5, -2.0, 4.0])
    dt = 0.25
    x, v = _kdk(x0, v0, lambda x: np.broadcast_to(g, x.shape), dt, 1)
    assert np.array_equal(x, x0 + v0 * dt + 0.5 * g * dt * dt)
    assert np.array_equal(v, v0 + g * dt)
    x, v = _kdk(x0, v0, lambda x: np.broadcast_to(g, x.shape), dt, 4)
    assert np.array_equal(x, x0 + v0 * (4 * dt) + 0.5 * g * (4 * dt) ** 2)
    assert np.array_equal(v, v0 + g * (4 * dt))


def test_leapfrog_harmonic_oscillator_second_order_and_reversible():
    """a = -x: the exact solution is (cos t, -sin t).  The scheme must converge with order 2 (halving dt
    quarters the error) and be time-reversible: running back with -dt returns to the start."""
    x0 = np.array([[1.0, 0.0, 0.0]]); v0 = np.array([[0.0, 0.0, 0.0]])
    errs = []
    for steps in (16, 32, 64):
        dt = 1.0 / steps
        x, v = _kdk(x0, v0, lambda x: -x, dt, steps)
        errs.append(math.hypot(x[0, 0] - math.cos(1.0), v[0, 0] + math.sin(1.0)))
    assert 3.5 < errs[0] / errs[1] < 4.5 and 3.5 < errs[1] / errs[2] < 4.5
    x, v = _kdk(x0, v0, lambda x: -x, 1.0 / 64, 64)
    xb, vb = _kdk(x, v, lambda x: -x, -1.0 / 64, 64)
    assert abs(xb[0, 0] - 1.0) < 1e-5 and abs(vb[0, 0]) < 1e-5


# ---------------------------------------------------------------- NEXT-3: quadrupole SPJ (reading S22)
def _cell_on_points(src_posm, test_points, eps, G=1.0, quad=True):
    """Sources = one cell (cell 0, particles [0, n)); every test point is its own one-particle group whose
    list is that single SPJ entry.  Returns (acc, pot) at the test points."""
    n, k = src_posm.shape[0], test_points.shape[0]
    posm = np.concatenate([src_posm, np.concatenate([test_points, np.zeros((k, 1))], axis=1)]).astype(np.float32)
    cells = np.array([[0, n, 0, 0]], np.int32)
    mom = oracle.monopoles(cells, posm)
    q = oracle.quadrupoles(cells, posm, mom) if quad else None
    gf = np.arange(n, n + k, dtype=np.int32)
    gn = np.ones(k, np.int32)
    eo = np.zeros(k + 1, np.int64)
    so = np.arange(k + 1, dtype=np.int64)
    acc, pot = oracle.forces(posm, mom, gf, gn, eo, np.zeros(0, np.int32), so, np.zeros(k, np.int32), eps, G, quad=q)
    return acc[n:], pot[n:], posm


def test_quadrupole_two_masses_closed_form():
    """Two masses m at (0,0,+-a), eps = 0.  Taylor series of the exact potential to order a^2 (textbook):
    on the x axis  phi = -G (2m/d - m a^2/d^3), on the z axis  phi = -G (2m/d + 2 m a^2/d^3).  Values typed from the
    series, not from the oracle's formula; catches a wrong coefficient or sign of either quadrupole term."""
    m, a, d, G = 0.75, 0.5, 8.0, 2.0
    src = np.array([[0, 0, a, m], [0, 0, -a, m]], np.float64)
    pts = np.array([[d, 0, 0], [0, 0, d], [0, -d, 0]], np.float64)
    acc, pot, _ = _cell_on_points(src, pts, 0.0, G)
    assert pot[0] == pytest.approx(-G * (2 * m / d - m * a * a / d ** 3), rel=1e-14)
    assert pot[1] == pytest.approx(-G * (2 * m / d + 2 * m * a * a / d ** 3), rel=1e-14)
    assert pot[2] == pytest.approx(pot[0], rel=1e-14)
    # radial derivative of the same series: a_x = -d phi/dx on the x axis, a_z = -d phi/dz on the z axis
    np.testing.assert_allclose(acc[0], [-G * (2 * m / d ** 2 - 3 * m * a * a / d ** 4), 0, 0], rtol=1e-13, atol=1e-16)
    np.testing.assert_allclose(acc[1], [0, 0, -G * (2 * m / d ** 2 + 6 * m * a * a / d ** 4)], rtol=1e-13, atol=1e-16)


def test_quadrupole_of_an_octahedron_vanishes():
    """Six equal masses at +-a on the axes have Q = 2 m a^2 * identity: no quadrupole field for eps = 0, so the
    quadrupole evaluation equals the monopole one.  Catches a wrong trace term."""
    a, m = 0.3, 1.5
    src = np.array([[a, 0, 0, m], [-a, 0, 0, m], [0, a, 0, m], [0, -a, 0, m], [0, 0, a, m], [0, 0, -a, m]], np.float64)
    pts = np.array([[3.0, 1.0, -2.0], [0.5, 4.0, 0.25]])
    acc_q, pot_q, _ = _cell_on_points(src, pts, 0.0)
    acc_m, pot_m, _ = _cell_on_points(src, pts, 0.0, quad=False)
    np.testing.assert_allclose(acc_q, acc_m, rtol=1e-13)
    np.testing.assert_allclose(pot_q, pot_m, rtol=1e-13)


@pytest.mark.parametrize("eps", [0.0, 0.7])
def test_quadrupole_convergence_order(eps):
    """Against direct summation over the cluster, the error of the monopole evaluation falls as d^-3 (potential) and
    d^-4 (acceleration) with distance d, that of the quadrupole evaluation one power faster -- also with softening,
    because the expansion is of the softened kernel itself.  A dropped term or a wrong coefficient anywhere leaves a
    residual of the lower order and fails the ratio."""
    rng = np.random.default_rng(5)
    n = 60
    src = np.concatenate([rng.uniform(-0.5, 0.5, size=(n, 3)), rng.uniform(0.5, 1.5, size=(n, 1))], axis=1)
    u = np.array([0.36, -0.48, 0.8])
    dist = np.array([8.0, 16.0, 32.0, 64.0])
    err = {}
    for quad in (False, True):
        acc, pot, posm = _cell_on_points(src, dist[:, None] * u[None, :], eps, quad=quad)
        # direct sum over the (fp32-rounded) sources at the (fp32-rounded) test points
        ea, ep = [], []
        for k in range(len(dist)):
            d = posm[:n, :3].astype(np.float64) - posm[n + k, :3].astype(np.float64)
            r2 = (d * d).sum(1) + eps * eps
            mk = posm[:n, 3].astype(np.float64)
            ep.append(abs(pot[k] - (-(mk / np.sqrt(r2)).sum())))
            ea.append(np.linalg.norm(acc[k] - (mk[:, None] * d / r2[:, None] ** 1.5).sum(0)))
        err[quad] = (np.array(ea), np.array(ep))
    for quad, p_pot in ((False, 3), (True, 4)):
        ea, ep = err[quad]
        # the source centre of mass is the expansion centre, so the dipole vanishes; ratios per doubling of d
        assert np.all(np.abs(np.log2(ep[:-1] / ep[1:]) - p_pot) < 0.35), (quad, ep)
        assert np.all(np.abs(np.log2(ea[:-1] / ea[1:]) - (p_pot + 1)) < 0.35), (quad, ea)
    assert np.all(err[True][1] < 0.2 * err[False][1])


def test_quadrupole_acc_is_minus_grad_pot():
    """acc = -grad(pot) by central differences of the oracle's own potential at displaced test points (positions
    chosen exactly representable in fp32): ties the acceleration formula to the potential that the pins above fix."""
    rng = np.random.default_rng(9)
    src = np.concatenate([rng.uniform(-0.5, 0.5, size=(20, 3)), rng.uniform(0.5, 1.5, size=(20, 1))], axis=1)
    x0 = np.array([3.0, -2.5, 4.25])
    h = 2.0 ** -10
    pts = [x0]
    for ax in range(3):
        for sgn in (+1, -1):
            p = x0.copy()
            p[ax] += sgn * h
            pts.append(p)
    acc, pot, _ = _cell_on_points(src, np.array(pts), 0.3)
    grad = np.array([(pot[1 + 2 * ax] - pot[2 + 2 * ax]) / (2 * h) for ax in range(3)])
    np.testing.assert_allclose(acc[0], -grad, rtol=3e-6)


def test_quadrupole_moment_invariants():
    """Q_c on a real tree: parallel-axis theorem (parent = sum over children of Q_child + M_child dd^T, d = X_child - X),
    trace = sum m |x - X|^2 >= 0, translation invariance, and the root equals the numpy definition."""
    cfg = CONFIGS[0]
    w = make_workload(cfg, 3000)
    mom = oracle.monopoles(w.cells, w.posm)
    q = oracle.quadrupoles(w.cells, w.posm, mom)

    def full(v):
        return np.array([[v[0], v[3], v[4]], [v[3], v[1], v[5]], [v[4], v[5], v[2]]])

    x = w.posm[:, :3].astype(np.float64)
    m = w.posm[:, 3].astype(np.float64)
    y = x - mom[0, :3]
    np.testing.assert_allclose(full(q[0]), np.einsum("p,pa,pb->ab", m, y, y), rtol=1e-12, atol=1e-15)
    assert np.all(q[:, :3].sum(1) >= 0)
    for c in range(w.n_cell):
        fc, nc = w.cells[c, 2], w.cells[c, 3]
        if nc == 0:
            continue
        tot = np.zeros((3, 3))
        for ch in range(fc, fc + nc):
            d = mom[ch, :3] - mom[c, :3]
            tot += full(q[ch]) + mom[ch, 3] * np.outer(d, d)
        np.testing.assert_allclose(full(q[c]), tot, rtol=1e-9, atol=1e-14)
    shifted = w.posm.copy()
    shifted[:, :3] += np.array([0.5, -0.25, 2.0], np.float32)        # exact in fp32 for these magnitudes? compare loosely
    mom2 = oracle.monopoles(w.cells, shifted)
    q2 = oracle.quadrupoles(w.cells, shifted, mom2)
    np.testing.assert_allclose(q2, q, rtol=2e-4, atol=1e-9)


def test_quadrupole_tree_forces_beat_monopole():
    """On Barnes-Hut lists the quadrupole evaluation is closer to direct summation than the monopole one (by more
    than 2x in RMS at theta = 0.7 and 0.4), and both converge as theta falls."""
    cfg = CONFIGS[0]
    posm, _ = make_particles(cfg, 4096)
    rms = {}
    for theta in (0.7, 0.4):
        w = build_tree_and_lists(posm, cfg.n_leaf, cfg.n_grp, theta)
        acc_d, _ = oracle.direct(w.posm, cfg.eps)
        mom = oracle.monopoles(w.cells, w.posm)
        q = oracle.quadrupoles(w.cells, w.posm, mom)
        lists = (w.grp_first, w.grp_n, w.epj_off, w.epj_id, w.spj_off, w.spj_id)
        for name, quad in (("mono", None), ("quad", q)):
            acc, _ = oracle.forces(w.posm, mom, *lists, cfg.eps, quad=quad)
            e = np.linalg.norm(acc - acc_d, axis=1) / np.linalg.norm(acc_d, axis=1)
            rms[(name, theta)] = np.sqrt(np.mean(e ** 2))
    assert rms[("quad", 0.7)] < rms[("mono", 0.7)] / 2
    assert rms[("quad", 0.4)] < rms[("mono", 0.4)] / 2
    assert rms[("quad", 0.4)] < rms[("quad", 0.7)]
    print(rms)
