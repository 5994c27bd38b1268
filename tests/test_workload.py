"""Pins of the host-side input builder (paper_1907_02290_b200/workload): the fast C++ tree / group /
list builder against the plain Python restatement in oracle/bhtree_ref.py, the structural
invariants P3 / P4 of SURVEY.md section 8(c), and sanity checks of the seeded generators."""
import numpy as np
import pytest

from oracle import bhtree_ref
from paper_1907_02290_b200.workload import CONFIGS, build_tree_and_lists, make_particles, make_workload
from paper_1907_02290_b200.workload.generators import clumpy_box, disk_halo, plummer


@pytest.mark.parametrize("cfg_idx,n,theta", [(0, 700, 0.5), (2, 1500, 0.4), (3, 1200, 0.5), (0, 300, 0.0), (0, 900, 1.0)])
def test_fast_builder_matches_plain_restatement(cfg_idx, n, theta):
    cfg = CONFIGS[cfg_idx]
    posm, _ = make_particles(cfg, n)
    n_leaf, n_grp = 8, 64
    w = build_tree_and_lists(posm, n_leaf, n_grp, theta)
    ref = bhtree_ref.build(posm, n_leaf, n_grp, theta)
    assert np.array_equal(w.perm, ref["perm"])
    assert np.array_equal(w.cells, ref["cells"])
    assert np.array_equal(w.geom, ref["geom"])
    assert np.array_equal(w.level, ref["level"])
    assert np.array_equal(w.root, ref["root"])
    assert np.array_equal(w.grp_cell, ref["groups"])
    for g in range(w.n_group):
        assert list(w.epj_id[w.epj_off[g]:w.epj_off[g + 1]]) == ref["epj"][g]
        assert list(w.spj_id[w.spj_off[g]:w.spj_off[g + 1]]) == ref["spj"][g]


def check_structure(w, n_leaf, n_grp):
    n = w.n
    cells = w.cells
    # cells: level order, children contiguous and partition the parent's range, leaves small
    assert cells[0, 0] == 0 and cells[0, 1] == n
    assert np.all(np.diff(w.level) >= 0)
    assert np.array_equal(np.searchsorted(w.level, np.arange(len(w.level_first) - 1)), w.level_first[:-1])
    internal = np.nonzero(cells[:, 3] > 0)[0]
    for c in internal[:: max(1, len(internal) // 500)]:
        fc, nc = cells[c, 2], cells[c, 3]
        ch = cells[fc:fc + nc]
        assert ch[0, 0] == cells[c, 0] and ch[:, 1].sum() == cells[c, 1]
        assert np.array_equal(ch[1:, 0], ch[:-1, 0] + ch[:-1, 1])
        assert np.all(w.level[fc:fc + nc] == w.level[c] + 1)
    leaves = cells[:, 3] == 0
    assert np.all(cells[leaves & (w.level < 21), 1] <= n_leaf)
    assert cells[leaves, 1].sum() == n                      # leaves partition the particles
    # groups partition [0, N) in Morton order
    assert w.grp_first[0] == 0 and w.grp_first[-1] + w.grp_n[-1] == n
    assert np.array_equal(w.grp_first[1:], w.grp_first[:-1] + w.grp_n[:-1])
    assert np.all((w.grp_n <= n_grp) | (cells[w.grp_cell, 3] == 0))
    # particles sit inside their leaf cube
    x = w.posm[:, :3].astype(np.float64)
    for c in np.nonzero(leaves)[0][:: max(1, leaves.sum() // 300)]:
        f, k = cells[c, 0], cells[c, 1]
        assert np.all(np.abs(x[f:f + k] - w.geom[c, :3]) <= 0.5 * w.geom[c, 3] * (1 + 1e-9))


def check_coverage(w, groups):
    """P4: for every group, EPJ particles and the particle ranges of the SPJ cells partition [0, N)."""
    n = w.n
    for g in groups:
        cover = np.zeros(n + 1, np.int64)
        e = w.epj_id[w.epj_off[g]:w.epj_off[g + 1]]
        s = w.spj_id[w.spj_off[g]:w.spj_off[g + 1]]
        np.add.at(cover, e, 1)
        np.add.at(cover, e + 1, -1)
        np.add.at(cover, w.cells[s, 0], 1)
        np.add.at(cover, w.cells[s, 0] + w.cells[s, 1], -1)
        assert np.all(np.cumsum(cover)[:n] == 1)
        # the group's own particles are EPJ entries (self term handled by index)
        own = np.arange(w.grp_first[g], w.grp_first[g] + w.grp_n[g])
        assert np.all(np.isin(own, e))


def check_mac(w, groups):
    """Every SPJ cell satisfies l <= theta d for its group; every ancestor of a list entry was opened."""
    x = w.posm[:, :3].astype(np.float64)
    for g in groups:
        f, k = w.grp_first[g], w.grp_n[g]
        lo, hi = x[f:f + k].min(0), x[f:f + k].max(0)
        s = w.spj_id[w.spj_off[g]:w.spj_off[g + 1]]
        c = w.geom[s, :3]
        d = np.maximum(0, np.maximum(lo - c, c - hi))
        assert np.all(w.geom[s, 3] ** 2 <= w.theta ** 2 * (d ** 2).sum(1))


@pytest.mark.parametrize("cfg_idx,n", [(0, None), (1, 40000), (2, 50000), (3, 60000), (4, 30000)])
def test_structural_invariants(cfg_idx, n):
    cfg = CONFIGS[cfg_idx]
    w = make_workload(cfg, n)
    check_structure(w, cfg.n_leaf, cfg.n_grp)
    rng = np.random.default_rng(0)
    groups = rng.choice(w.n_group, size=min(40, w.n_group), replace=False)
    check_coverage(w, groups)
    check_mac(w, groups)
    # sanity bands (not pins): n_cell ~ n/4 at leaf <= 16; lists are several times the group size
    if cfg.n_leaf == 16:
        assert w.n / 6 < w.n_cell < w.n / 2.5
    assert w.n_list.mean() > 4 * w.grp_n.mean()


def test_theta_zero_lists_are_everything():
    """P3: theta = 0 opens every cell: EPJ is a permutation of [0, N), SPJ is empty."""
    posm, _ = make_particles(CONFIGS[0], 1000)
    w = build_tree_and_lists(posm, 8, 64, 0.0)
    assert w.spj_id.size == 0
    for g in range(w.n_group):
        assert np.array_equal(np.sort(w.epj_id[w.epj_off[g]:w.epj_off[g + 1]]), np.arange(w.n))


def test_degenerate_inputs():
    # one particle; all particles at one point (depth cap makes one big leaf = one big group)
    w = build_tree_and_lists(np.array([[1, 2, 3, 1]], np.float32), 8, 64, 0.5)
    assert w.n_cell == 1 and w.n_group == 1 and list(w.epj_id) == [0] and w.spj_id.size == 0
    same = np.tile(np.array([[0.5, 0.5, 0.5, 1.0]], np.float32), (100, 1))
    w = build_tree_and_lists(same, 8, 64, 0.5)
    assert w.grp_n.sum() == 100 and np.array_equal(np.sort(w.epj_id[: w.epj_off[1]]), np.arange(100))
    # two tight clusters far apart: each sees the other as one SPJ
    rng = np.random.default_rng(1)
    a = rng.normal(0, 1e-3, (50, 3))
    b = rng.normal(0, 1e-3, (50, 3)) + 100.0
    posm = np.concatenate([np.concatenate([a, b]), np.ones((100, 1))], axis=1).astype(np.float32)
    w = build_tree_and_lists(posm, 8, 64, 0.5)
    assert w.n_group == 2 and np.all(np.diff(w.spj_off) == 1) and np.all(np.diff(w.epj_off) == 50)


def test_generators_are_seeded_and_shaped():
    p1, v1, m1 = plummer(20000, 7)
    p2, v2, m2 = plummer(20000, 7)
    assert np.array_equal(p1, p2) and np.array_equal(v1, v2)
    assert not np.array_equal(p1, plummer(20000, 8)[0])
    r = np.linalg.norm(p1, axis=1)
    assert r.max() < 22.8 + 0.1
    assert np.median(r) == pytest.approx(1.0 / np.sqrt(2 ** (2 / 3) - 1), rel=0.03)   # half-mass radius 1.305 a
    assert np.allclose(p1.mean(0), 0, atol=1e-12) and np.allclose(v1.mean(0), 0, atol=1e-12)
    T = 0.5 * np.sum(m1[:, None] * v1 ** 2)
    assert T == pytest.approx(3 * np.pi / 64, rel=0.03)                               # virial: T = -W/2
    pd, _, md = disk_halo(20000, 3)
    assert md.sum() == pytest.approx(1.0) and md[:18000].sum() == pytest.approx(0.1)
    assert md[-1] / md[0] == pytest.approx(81.0)
    Rd = np.hypot(pd[:18000, 0], pd[:18000, 1])
    assert Rd.mean() == pytest.approx(2.0, rel=0.03)                                   # Gamma(2,1) mean
    assert np.abs(pd[:18000, 2]).mean() == pytest.approx(0.1 * np.log(2), rel=0.05)   # sech^2: <|z|> = h ln 2
    assert np.linalg.norm(pd[18000:], axis=1).max() <= 100.0 * (1 + 1e-9)
    pc, _, mc = clumpy_box(20000, 4)
    assert mc.sum() == pytest.approx(1.0)
    assert np.all((pc[:6000] >= 0) & (pc[:6000] < 1))
    assert pc.min() > -0.25 and pc.max() < 1.25


def test_config_table_matches_baseline_json():
    import json, os
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    text = json.load(open(os.path.join(root, "BASELINE.json")))["configs"]
    assert len(text) == len(CONFIGS) == 5
    assert [c.n for c in CONFIGS] == [4096, 1 << 20, 1 << 22, 1 << 23, 1 << 22]
    assert [c.seed for c in CONFIGS] == [1, 2, 3, 4, 5]
    assert [c.theta for c in CONFIGS] == [0.5, 0.5, 0.4, 0.5, 0.5]
    assert [c.n_grp for c in CONFIGS] == [64, 256, 512, 256, 256]
    assert [c.n_leaf for c in CONFIGS] == [8, 16, 16, 16, 16]
    assert [c.eps for c in CONFIGS] == [1 / 64, 1 / 256, 0.005, 1e-4, 1 / 512]
    assert CONFIGS[4].n_reuse == 8 and CONFIGS[4].dt == 1 / 1024


def test_pack_data_lists_is_a_plain_gather():
    """Method G1's host packing: EPJ records then SPJ records per group, contiguous, with run offsets."""
    from paper_1907_02290_b200.workload import pack_data_lists
    cfg = CONFIGS[0]
    w = make_workload(cfg, 3000)
    rng = np.random.default_rng(3)
    spj = rng.normal(size=(w.n_cell, 4)).astype(np.float32)
    g0, g1 = 5, min(w.n_group, 41)
    rec, joff = pack_data_lists(w, g0, g1, w.posm, spj)
    assert joff[0] == 0 and rec.shape[0] == joff[-1]
    for g in range(g0, g1):
        e = w.epj_id[w.epj_off[g]:w.epj_off[g + 1]]
        c = w.spj_id[w.spj_off[g]:w.spj_off[g + 1]]
        want = np.concatenate([w.posm[e], spj[c]])
        assert np.array_equal(rec[joff[g - g0]:joff[g - g0 + 1]], want)


@pytest.mark.parametrize("kind,n,lo,hi", [("uniform", 60000, 0.45, 1.2), ("plummer", 65536, 0.8, 1.9)])
def test_list_length_follows_the_papers_model(golden, kind, n, lo, hi):
    """Sanity band P10: the particle-weighted mean list length of the harness against the paper's
    geometric model, eq. 30, evaluated at the group-mean <n_i>.  The model counts cube surfaces in a uniform
    medium, so a uniform sphere sits somewhat below it and a centrally concentrated one above; a band, not a pin."""
    theta, n_grp = 0.5, 256
    if kind == "uniform":
        rng = np.random.default_rng(9)
        p = rng.normal(size=(n, 3))
        p *= (rng.uniform(0, 1, n) ** (1 / 3) / np.linalg.norm(p, axis=1))[:, None]
        posm = np.concatenate([p, np.full((n, 1), 1.0 / n)], axis=1).astype(np.float32)
    else:
        posm, _ = make_particles(CONFIGS[1], n)
    w = build_tree_and_lists(posm, 16, n_grp, theta)
    ni = n / w.n_group
    model = (ni + golden["nlist_c1"] * ni ** (2 / 3) / theta + golden["nlist_c2"] * np.pi * ni ** (1 / 3) / theta ** 2
             + golden["nlist_c3"] * np.pi / (3 * theta ** 3) * np.log2(theta / golden["nlist_c4"] * (n ** (1 / 3) - ni ** (1 / 3))))
    measured = w.interactions / n                      # sum n_i n_list / n
    print("%s: <n_i> %.1f, <n_list> measured %.0f, eq. 30 %.0f, ratio %.2f" % (kind, ni, measured, model, measured / model))
    assert lo < measured / model < hi
