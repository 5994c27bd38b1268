"""GPU parity of the short-range workload (paper P:79): SPH density and
pressure-gradient acceleration through the index lists, CUDA path (through the C ABI) against the fp64 oracle on the
same seeded inputs.

Tolerances (DESIGN.md section 9d derives them from the arithmetic; north_star states none for this workload):
  density   |rho_gpu - rho_or| / rho_or <= 1e-5 max, 2e-6 RMS      (a sum of non-negative terms, each good to a few ulp)
  P/rho^2   same bar
  hydro     |a_gpu - a_or| <= 1e-5 max, 2e-6 RMS in units of max(scale_i, one_i): scale_i = sum_k |term_k| (the sum
            cancels, so the error is measured against the magnitude of what is summed, which the oracle returns), and
            one_i = the size of ONE pair term at q = 1 with an equal partner, 3 m_i (P/rho^2)_i / (2 pi h_i^4): a particle
            whose only neighbours sit at the edge of the support (q -> 2) sums terms ~ (2-q)^2 whose ABSOLUTE error is a few
            ulp of q ~ 2 times the slope -- negligible against one_i, unbounded against their own vanishing size
No oracle input comes from the CUDA path: the hydro pass is checked on records whose rho and P/rho^2 were made by the
ORACLE's density pass (rounded to fp32); the chained GPU pass (density then hydro) is checked against the chained oracle
pass with the bar widened by the density error it inherits.
"""
import numpy as np
import pytest

import oracle
from paper_1907_02290_b200 import binding
from paper_1907_02290_b200.workload import SPH_CONFIGS, build_tree_and_lists, make_workload

pytestmark = pytest.mark.gpu

RHO_MAX, RHO_RMS = 1e-5, 2e-6
ACC_MAX, ACC_RMS = 1e-5, 2e-6


def make_ctx(w, n_tag=4, mode=binding.MAKE_LIST_FOR_REUSE):
    f = binding.MultiWalkForce.for_workload(w, n_tag=n_tag)
    f.upload_workload(w, mode)
    return f


def gpu_density(f, w, gamma):
    f.dispatch_density(0, 0, w.n_group, gamma)
    out = np.full((w.n, 4), np.nan, np.float32)
    f.retrieve(0, out)
    return out


def gpu_hydro(f, w):
    f.dispatch_hydro(0, 0, w.n_group)
    out = np.full((w.n, 4), np.nan, np.float32)
    f.retrieve(0, out)
    return out


def check_density(rec, rho, pr2, mask=None, label=""):
    r, p = rec[:, 2].astype(np.float64), rec[:, 3].astype(np.float64)
    if mask is not None:
        r, p, rho, pr2 = r[mask], p[mask], rho[mask], pr2[mask]
    er, ep = np.abs(r - rho) / rho, np.abs(p - pr2) / pr2
    msg = "%s: rho max %.2e rms %.2e | P/rho^2 max %.2e rms %.2e" % (label, er.max(), np.sqrt(np.mean(er ** 2)), ep.max(), np.sqrt(np.mean(ep ** 2)))
    print(msg)
    assert np.all(np.isfinite(er)) and np.all(np.isfinite(ep)), msg
    assert er.max() <= RHO_MAX and np.sqrt(np.mean(er ** 2)) <= RHO_RMS, msg
    assert ep.max() <= RHO_MAX and np.sqrt(np.mean(ep ** 2)) <= RHO_RMS, msg


def check_hydro(out, acc, scale, posm, rec, mask=None, label="", widen=1.0):
    a = out[:, :3].astype(np.float64)
    one = 1.5 * posm[:, 3].astype(np.float64) * rec[:, 3].astype(np.float64) / (np.pi * rec[:, 0].astype(np.float64) ** 4)
    if mask is not None:
        a, acc, scale, one = a[mask], acc[mask], scale[mask], one[mask]
    lone = scale == 0
    assert np.all(a[lone] == 0)                                         # nobody inside 2h: exactly nothing
    e = np.linalg.norm(a - acc, axis=1)[~lone] / np.maximum(scale, one)[~lone]
    if e.size == 0:
        e = np.zeros(1)
    msg = "%s: acc error / scale max %.2e rms %.2e (%d particles, %d without neighbours)" % (label, e.max(), np.sqrt(np.mean(e ** 2)), len(scale), lone.sum())
    print(msg)
    assert np.all(np.isfinite(a)), msg
    assert e.max() <= widen * ACC_MAX and np.sqrt(np.mean(e ** 2)) <= widen * ACC_RMS, msg
    if mask is None:
        assert np.all(out[:, 3] == 0)


def oracle_records(w, gamma, groups=None):
    rho, pr2 = oracle.sph_density(w.posm, w.sph, w.grp_first, w.grp_n, w.epj_off, w.epj_id, gamma, groups)
    rec = w.sph.copy()
    rec[:, 2], rec[:, 3] = rho, pr2
    return rho, pr2, rec


def group_mask(w, groups):
    m = np.zeros(w.n, bool)
    for g in groups:
        m[w.grp_first[g]:w.grp_first[g] + w.grp_n[g]] = True
    return m


# ------------------------------------------------------------------ the small config in full
def test_sph_small_config_full():
    cfg = SPH_CONFIGS[0]
    w = make_workload(cfg)
    f = make_ctx(w)
    rec = gpu_density(f, w, cfg.gamma)
    np.testing.assert_array_equal(rec[:, :2], w.sph[:, :2])              # h and u travel untouched
    rho, pr2, orec = oracle_records(w, cfg.gamma)
    check_density(rec, rho, pr2, label=cfg.name)
    # chained on the GPU: hydro on the densities the GPU just made
    acc, scale = oracle.sph_hydro(w.posm, orec, w.grp_first, w.grp_n, w.epj_off, w.epj_id)
    check_hydro(gpu_hydro(f, w), acc, scale, w.posm, orec, label=cfg.name + " chained", widen=3.0)
    # hydro alone, on records made by the oracle
    f.set_sph(orec)
    check_hydro(gpu_hydro(f, w), acc, scale, w.posm, orec, label=cfg.name + " hydro on oracle records")
    # the densities are still what the upload said (hydro writes no record)
    np.testing.assert_array_equal(f.get_sph(0, w.n), orec)
    f.close()


@pytest.mark.parametrize("n", [1, 2, 3, 63, 64, 65, 129, 1000])
def test_sph_every_width_and_tail_against_all_pairs(n):
    """One group of n particles whose list is all n particles (every remainder width, ragged list tail), random h:
    equals the oracle's all-pairs sums."""
    rng = np.random.default_rng(100 + n)
    posm = np.concatenate([rng.uniform(0, 1, (n, 3)), rng.uniform(0.5, 2.0, (n, 1))], 1).astype(np.float32)
    rec = np.zeros((n, 4), np.float32)
    rec[:, 0] = rng.uniform(0.15, 0.6, n)
    rec[:, 1] = rng.uniform(0.5, 2.0, n)
    w = build_tree_and_lists(posm, max(n, 1), max(n, 1), 0.0, sph=rec, skin=10.0)   # one leaf = one group; skin 10: list = everything
    assert w.n_group == 1 and w.epj_off[-1] == n
    f = binding.MultiWalkForce(1.0, max_ptcl=n, max_cell=w.n_cell, max_group=1, max_entry=n, n_tag=1)
    f.upload_workload(w)
    got = gpu_density(f, w, 1.4)
    rho = oracle.sph_density_direct(w.posm, w.sph)
    check_density(got, rho, 0.4 * w.sph[:, 1].astype(np.float64) / rho, label="n=%d" % n)
    orec = w.sph.copy()
    orec[:, 2], orec[:, 3] = rho, rng.uniform(0.5, 2.0, n)
    f.set_sph(orec)
    acc, scale = oracle.sph_hydro_direct(w.posm, orec)
    check_hydro(gpu_hydro(f, w), acc, scale, w.posm, orec, label="n=%d" % n)
    f.close()


def test_sph_coincident_and_isolated_particles():
    """Two distinct particles at one position (finite, no pressure force between them), and one particle far from all
    others (density = its own term m W(0, h) = m / (pi h^3), no acceleration)."""
    posm = np.array([[0.5, 0.5, 0.5, 1.0], [0.5, 0.5, 0.5, 2.0], [0.6, 0.5, 0.5, 1.0], [5.0, 5.0, 5.0, 3.0]], np.float32)
    rec = np.array([[0.2, 1, 0, 1.0], [0.2, 1, 0, 1.5], [0.2, 1, 0, 0.5], [0.25, 1, 0, 1.0]], np.float32)
    w = build_tree_and_lists(posm, 4, 4, 0.0, sph=rec, skin=100.0)
    f = binding.MultiWalkForce(1.0, max_ptcl=4, max_cell=w.n_cell, max_group=1, max_entry=4, n_tag=1)
    f.upload_workload(w)
    got = gpu_density(f, w, 5.0 / 3.0)
    rho = oracle.sph_density_direct(w.posm, w.sph)
    check_density(got, rho, (2.0 / 3.0) * w.sph[:, 1].astype(np.float64) / rho)
    lone = int(np.argmax(w.posm[:, 0]))
    assert got[lone, 2] == pytest.approx(3.0 / (np.pi * 0.25 ** 3), rel=1e-6)
    f.set_sph(w.sph)
    out = gpu_hydro(f, w)
    acc, scale = oracle.sph_hydro_direct(w.posm, w.sph)
    check_hydro(out, acc, scale, w.posm, w.sph)
    assert np.all(out[lone] == 0)
    f.close()


def test_sph_batched_dispatch_is_bitwise_the_single_dispatch_and_state_machine():
    cfg = SPH_CONFIGS[0]
    w = make_workload(cfg, n=20011)
    f = binding.MultiWalkForce.for_workload(w, n_tag=3)
    f.begin_step(binding.MAKE_LIST_FOR_REUSE)
    f.set_particles(w.posm)
    f.set_tree(w.cells)
    f.set_lists(w.grp_first, w.grp_n, w.epj_off, w.epj_id, w.spj_off, w.spj_id)
    with pytest.raises(binding.MwfError) as e:
        f.dispatch_density(0, 0, w.n_group, cfg.gamma)                    # no records yet
    assert e.value.code == binding.ESTATE
    f.set_sph(w.sph)
    with pytest.raises(binding.MwfError) as e:
        f.dispatch_density(0, 0, w.n_group, 1.0)                          # gamma must exceed 1
    assert e.value.code == binding.EINVAL
    one = gpu_density(f, w, cfg.gamma)
    f.set_sph(w.sph)
    out = np.full((w.n, 4), np.nan, np.float32)
    step = 97
    tags = []
    for k, gb in enumerate(range(0, w.n_group, step)):
        t = k % 3
        if t in tags:
            f.retrieve(t, out)
            tags.remove(t)
        f.dispatch_density(t, gb, min(w.n_group, gb + step), cfg.gamma)
        tags.append(t)
    with pytest.raises(binding.MwfError) as e:
        f.dispatch_hydro(tags[0], 0, 1)                                   # that tag still holds density records
    assert e.value.code == binding.ESTATE
    for t in tags:
        f.retrieve(t, out)
    np.testing.assert_array_equal(out, one)
    one_h = gpu_hydro(f, w)
    out_h = np.full((w.n, 4), np.nan, np.float32)
    for k, gb in enumerate(range(0, w.n_group, 4 * step)):
        f.dispatch_hydro(k % 3, gb, min(w.n_group, gb + 4 * step))
        f.retrieve(k % 3, out_h)
    np.testing.assert_array_equal(out_h, one_h)
    f.close()


# ------------------------------------------------------------------ full size, bench launch configuration, with list reuse
def test_sph_full_size_sampled_groups_with_reuse():
    """sph_plummer_1m as bench.py launches it (one dispatch over all groups per pass), on seeded group samples that include
    the longest list, the largest and the smallest group; then the particles drift (each by less than skin * h / 2) and the
    SAME lists are reused (REUSE_LIST) -- parity again, on the moved particles."""
    cfg = SPH_CONFIGS[1]
    w = make_workload(cfg)
    f = make_ctx(w, n_tag=2)
    rng = np.random.default_rng(42)
    n_list = w.n_list
    sample = set(rng.choice(w.n_group, 300, replace=False).tolist())
    sample |= {int(np.argmax(n_list)), int(np.argmax(w.grp_n)), int(np.argmin(w.grp_n)), 0, w.n_group - 1}
    sample = np.array(sorted(sample), np.int64)
    mask = group_mask(w, sample)
    posm = w.posm.copy()
    for step in range(2):
        if step:
            f.begin_step(binding.REUSE_LIST)
            d = rng.normal(size=(w.n, 3))
            d *= (0.04 * w.sph[:, 0].astype(np.float64) / np.linalg.norm(d, axis=1))[:, None]
            posm = posm.copy()
            posm[:, :3] = (posm[:, :3].astype(np.float64) + d).astype(np.float32)
            f.set_particles(posm)
            f.set_sph(w.sph)
        rec = gpu_density(f, w, cfg.gamma)
        rho, pr2 = oracle.sph_density(posm, w.sph, w.grp_first, w.grp_n, w.epj_off, w.epj_id, cfg.gamma, sample)
        check_density(rec, rho, pr2, mask, label="%s step %d" % (cfg.name, step))
        # hydro needs P/rho^2 of every listed particle: take the oracle's density on ALL groups for the records
        rho_all, pr2_all = oracle.sph_density(posm, w.sph, w.grp_first, w.grp_n, w.epj_off, w.epj_id, cfg.gamma)
        orec = w.sph.copy()
        orec[:, 2], orec[:, 3] = rho_all, pr2_all
        f.set_sph(orec)
        out = gpu_hydro(f, w)
        acc, scale = oracle.sph_hydro(posm, orec, w.grp_first, w.grp_n, w.epj_off, w.epj_id, sample)
        check_hydro(out, acc, scale, posm, orec, mask, label="%s step %d" % (cfg.name, step))
        # any-size property: the symmetrised gradient conserves momentum
        m = posm[:, 3].astype(np.float64)
        assert np.linalg.norm(np.sum(m[:, None] * out[:, :3].astype(np.float64), 0)) < 1e-5 * np.sum(m[mask] * scale[mask]) * w.n / mask.sum()
    f.close()


def test_calc_sph_all_host_buffers_equals_the_single_dispatches():
    """mwf_calc_sph_all through pinned host buffers (groups split over the tags, copies overlapped) gives bitwise what one
    density dispatch and one hydro dispatch give."""
    cfg = SPH_CONFIGS[0]
    w = make_workload(cfg, n=30001)
    f = make_ctx(w, n_tag=4)
    rec1 = gpu_density(f, w, cfg.gamma)
    acc1 = gpu_hydro(f, w)
    src, rec, dst = f.pinned(w.n), f.pinned(w.n), f.pinned(w.n)
    src.numpy()[:] = w.posm
    rec.numpy()[:] = w.sph
    dst.numpy()[:] = np.nan
    f.begin_step(binding.REUSE_LIST)
    f.calc_sph_all(src, rec, dst, cfg.gamma)
    np.testing.assert_array_equal(rec.numpy(), rec1)
    np.testing.assert_array_equal(dst.numpy(), acc1)
    f.close()


# ------------------------------------------------------------------ device-side construction of the neighbour lists
def device_neighbour_build(posm, rec, n_leaf, n_grp, skin, max_entry=None):
    n = posm.shape[0]
    f = binding.MultiWalkForce(1.0, 1.0, max_ptcl=n, max_cell=2 * n + 64, max_group=n + 8,
                               max_entry=max_entry or max(64, min(n * n + 64 * n, 3000 * n + 4096)), n_tag=2)
    f.begin_step(binding.MAKE_LIST_FOR_REUSE)
    f.set_particles(posm)                      # caller order, NOT tree order
    with pytest.raises(binding.MwfError) as e:
        f.build_neighbours(n, n_leaf, n_grp, skin)
    assert e.value.code == binding.ESTATE      # no smoothing lengths yet
    f.set_sph(rec)
    f.build_neighbours(n, n_leaf, n_grp, skin)
    sz = f.get_build_sizes()
    out = dict(sizes=sz, perm=f.get_permutation(n), posm=f.get_particles(0, n), sph=f.get_sph(0, n))
    out["grp_first"], out["grp_n"] = f.get_groups(sz["n_group"])
    out["epj_off"], out["epj_id"], out["spj_off"], out["spj_id"] = f.get_lists(sz["n_group"], sz["n_epj"], sz["n_spj"])
    return out, f


@pytest.mark.parametrize("n,n_leaf,n_grp,skin", [(700, 8, 32, 0.0), (1500, 16, 64, 0.2), (64, 4, 8, 0.0), (3000, 8, 48, 10.0), (1, 8, 8, 0.0)])
def test_device_neighbour_build_matches_plain_restatement(n, n_leaf, n_grp, skin):
    """mwf_build_neighbours against oracle/bhtree_ref.py (reading S24 step by step): permutation, records carried along,
    groups, and per-group EPJ sets; there are no SPJ."""
    from oracle import bhtree_ref
    from paper_1907_02290_b200.workload import make_particles, make_sph_fields
    cfg = SPH_CONFIGS[0]
    posm, _ = make_particles(cfg, n)
    rec = make_sph_fields(cfg, posm)
    ref = bhtree_ref.build(posm, n_leaf, n_grp, 0.0, h=rec[:, 0], skin=skin)
    got, f = device_neighbour_build(posm, rec, n_leaf, n_grp, skin)
    f.close()
    assert np.array_equal(got["perm"], ref["perm"])
    assert np.array_equal(got["posm"], posm[ref["perm"]])
    assert np.array_equal(got["sph"], rec[ref["perm"]])
    assert np.array_equal(got["grp_first"], ref["cells"][ref["groups"], 0])
    assert got["sizes"]["n_spj"] == 0
    for g in range(len(ref["groups"])):
        e = got["epj_id"][got["epj_off"][g]:got["epj_off"][g + 1]]
        assert np.array_equal(np.sort(e), np.sort(np.array(ref["epj"][g], np.int32))), "EPJ set of group %d" % g


def test_device_neighbour_build_full_size_then_both_passes():
    """sph_plummer_1m built on the device from particles in generator order: every list offset and 300 sampled lists equal
    the independent host builder's; then density and hydro on the device-built lists against the oracle on sampled groups."""
    from paper_1907_02290_b200.workload import make_particles, make_sph_fields
    cfg = SPH_CONFIGS[1]
    posm, _ = make_particles(cfg)
    rec = make_sph_fields(cfg, posm)
    w = build_tree_and_lists(posm, cfg.n_leaf, cfg.n_grp, 0.0, cfg=cfg, sph=rec, skin=cfg.skin)
    got, f = device_neighbour_build(posm, rec, cfg.n_leaf, cfg.n_grp, cfg.skin, max_entry=w.n_entry + 1024)
    assert np.array_equal(got["perm"], w.perm)
    assert np.array_equal(got["grp_first"], w.grp_first) and np.array_equal(got["grp_n"], w.grp_n)
    assert np.array_equal(got["epj_off"], w.epj_off) and got["sizes"]["n_spj"] == 0
    rng = np.random.default_rng(5)
    sample = np.sort(rng.choice(w.n_group, 300, replace=False)).astype(np.int64)
    for g in sample:
        a = got["epj_id"][got["epj_off"][g]:got["epj_off"][g + 1]]
        b = w.epj_id[w.epj_off[g]:w.epj_off[g + 1]]
        assert np.array_equal(np.sort(a), np.sort(b))
    mask = group_mask(w, sample)
    out = gpu_density(f, w, cfg.gamma)
    rho, pr2 = oracle.sph_density(w.posm, w.sph, got["grp_first"], got["grp_n"], got["epj_off"], got["epj_id"], cfg.gamma, sample)
    check_density(out, rho, pr2, mask, label="device-built lists")
    rho_all, pr2_all = oracle.sph_density(w.posm, w.sph, got["grp_first"], got["grp_n"], got["epj_off"], got["epj_id"], cfg.gamma)
    orec = w.sph.copy()
    orec[:, 2], orec[:, 3] = rho_all, pr2_all
    f.set_sph(orec)
    acc, scale = oracle.sph_hydro(w.posm, orec, got["grp_first"], got["grp_n"], got["epj_off"], got["epj_id"], sample)
    check_hydro(gpu_hydro(f, w), acc, scale, w.posm, orec, mask, label="device-built lists")
    f.close()
