"""GPU parity of the device-side construction step (mwf_build; paper P:149-172):
sort order, cells, cell geometry, groups and index lists must be exactly those of the plain Python restatement of
readings O1-O4 (oracle/bhtree_ref.py, small N) and of the independent host builder (full sizes); lists are
compared per group as sorted sets (the walk order is free, reading S10).  Then the forces evaluated on the
device-built lists must match the fp64 oracle run on those same lists (north_star tolerances)."""
import numpy as np
import pytest

import oracle
from oracle import bhtree_ref
from paper_1907_02290_b200 import binding
from paper_1907_02290_b200.workload import CONFIGS, build_tree_and_lists, make_particles, make_workload

pytestmark = pytest.mark.gpu

ACC_MAX, ACC_RMS, POT_RMS = 1e-4, 2e-5, 1e-5


def device_build(posm, n_leaf, n_grp, theta, eps=1 / 64, max_cell=None, max_group=None, max_entry=None, vel=None, keep=False):
    n = posm.shape[0]
    f = binding.MultiWalkForce(eps, 1.0, max_ptcl=n, max_cell=max_cell or 2 * n + 64, max_group=max_group or n + 8,
                               max_entry=max_entry or max(64, min(n * n + 64 * n, 400 * n + 4096)), n_tag=2)
    f.begin_step(binding.MAKE_LIST_FOR_REUSE)
    f.set_particles(posm)                      # caller order, NOT tree order
    if vel is not None:
        v4 = np.zeros((n, 4), np.float32)
        v4[:, :3] = vel
        f.set_velocities(v4)
    f.build(n, n_leaf, n_grp, theta, binding.MAKE_LIST_FOR_REUSE)
    sz = f.get_build_sizes()
    out = dict(sizes=sz, perm=f.get_permutation(n))
    out["cells"], out["geom"] = f.get_tree(sz["n_cell"])
    out["grp_first"], out["grp_n"] = f.get_groups(sz["n_group"])
    out["epj_off"], out["epj_id"], out["spj_off"], out["spj_id"] = f.get_lists(sz["n_group"], sz["n_epj"], sz["n_spj"])
    out["posm"] = f.get_particles(0, n)
    if keep:
        return out, f
    f.close()
    return out


@pytest.mark.parametrize("cfg_idx,n,theta,n_leaf,n_grp", [(0, 700, 0.5, 8, 64), (2, 1500, 0.4, 8, 64), (3, 1200, 0.5, 8, 64),
                                                             (0, 300, 0.0, 8, 64), (0, 900, 1.0, 4, 16), (1, 2049, 0.5, 16, 256), (0, 5000, 0.7, 1, 1)])
def test_device_build_matches_plain_restatement(cfg_idx, n, theta, n_leaf, n_grp):
    posm, _ = make_particles(CONFIGS[cfg_idx], n)
    ref = bhtree_ref.build(posm, n_leaf, n_grp, theta)
    got = device_build(posm, n_leaf, n_grp, theta)
    assert np.array_equal(got["perm"], ref["perm"])
    assert np.array_equal(got["posm"], posm[ref["perm"]])
    assert np.array_equal(got["cells"], ref["cells"])
    assert np.array_equal(got["geom"], ref["geom"])            # bitwise: same fp64 operations in the same order
    assert np.array_equal(got["grp_first"], ref["cells"][ref["groups"], 0])
    assert np.array_equal(got["grp_n"], ref["cells"][ref["groups"], 1])
    for g in range(len(ref["groups"])):
        e = got["epj_id"][got["epj_off"][g]:got["epj_off"][g + 1]]
        s = got["spj_id"][got["spj_off"][g]:got["spj_off"][g + 1]]
        assert np.array_equal(np.sort(e), np.sort(np.array(ref["epj"][g], np.int32))), "EPJ set of group %d" % g
        assert np.array_equal(np.sort(s), np.sort(np.array(ref["spj"][g], np.int32))), "SPJ set of group %d" % g


def test_device_build_degenerate_inputs():
    # one particle; two particles; many coincident particles (a depth-21 leaf with more than n_leaf particles)
    for posm in (np.array([[0.5, 0.25, -1.0, 1.0]], np.float32),
                 np.array([[0, 0, 0, 1.0], [1, 1, 1, 2.0]], np.float32),
                 np.concatenate([np.tile(np.array([[0.3, 0.3, 0.3, 1.0]], np.float32), (40, 1)), np.array([[1, 2, 3, 1.0]], np.float32)])):
        ref = bhtree_ref.build(posm, 8, 16, 0.5)
        got = device_build(posm, 8, 16, 0.5)
        assert np.array_equal(got["perm"], ref["perm"])
        assert np.array_equal(got["cells"], ref["cells"])
        assert np.array_equal(got["geom"], ref["geom"])
        for g in range(len(ref["groups"])):
            assert sorted(got["epj_id"][got["epj_off"][g]:got["epj_off"][g + 1]]) == sorted(ref["epj"][g])
            assert sorted(got["spj_id"][got["spj_off"][g]:got["spj_off"][g + 1]]) == sorted(ref["spj"][g])


def test_device_build_errors():
    posm, _ = make_particles(CONFIGS[0], 3000)
    f = binding.MultiWalkForce(1 / 64, 1.0, max_ptcl=3000, max_cell=100, max_group=3000, max_entry=10 ** 6, n_tag=1)
    with pytest.raises(binding.MwfError) as e:
        f.build(3000, 8, 64, 0.5)
    assert e.value.code == binding.ESTATE                       # no particles uploaded
    f.set_particles(posm)
    for bad in ((0, 8, 64, 0.5), (3000, 0, 64, 0.5), (3000, 8, 0, 0.5), (3000, 8, 64, -0.1), (3000, 8, 64, 1.5), (3000, 8, 64, float("nan"))):
        with pytest.raises(binding.MwfError) as e:
            f.build(*bad)
        assert e.value.code == binding.EINVAL
    with pytest.raises(binding.MwfError) as e:
        f.build(3000, 8, 64, 0.5)
    assert e.value.code == binding.ENOMEM                       # max_cell = 100
    f.close()
    f = binding.MultiWalkForce(1 / 64, 1.0, max_ptcl=3000, max_cell=6000, max_group=3000, max_entry=1000, n_tag=1)
    f.set_particles(posm)
    with pytest.raises(binding.MwfError) as e:
        f.build(3000, 8, 64, 0.5)
    assert e.value.code == binding.ENOMEM                       # max_entry = 1000
    with pytest.raises(binding.MwfError) as e:
        f.dispatch(0, 0, 1)
    assert e.value.code == binding.ESTATE                       # a failed build leaves no lists
    with pytest.raises(binding.MwfError) as e:
        f.build(3000, 8, 64, 0.5)
    assert e.value.code == binding.ESTATE                       # ... and the particles in an order nobody knows: upload again
    f.close()


def check_forces(out, acc, pot, label):
    a = out[:, :3].astype(np.float64)
    p = out[:, 3].astype(np.float64)
    ea = np.linalg.norm(a - acc, axis=1) / np.linalg.norm(acc, axis=1)
    ep = np.abs(p - pot) / np.abs(pot)
    msg = "%s: acc max %.2e rms %.2e | pot rms %.2e" % (label, ea.max(), np.sqrt(np.mean(ea ** 2)), np.sqrt(np.mean(ep ** 2)))
    print(msg)
    assert ea.max() <= ACC_MAX and np.sqrt(np.mean(ea ** 2)) <= ACC_RMS and np.sqrt(np.mean(ep ** 2)) <= POT_RMS, msg


@pytest.mark.parametrize("cfg_idx,n", [(0, None), (2, 50000), (3, 60000)])
def test_forces_on_device_built_lists(cfg_idx, n):
    """Whole construction step on the device, then the usual evaluation; the oracle evaluates the lists the
    device built (read back), on the particles in the device's tree order."""
    cfg = CONFIGS[cfg_idx]
    posm, vel = make_particles(cfg, n)
    got, f = device_build(posm, cfg.n_leaf, cfg.n_grp, cfg.theta, eps=cfg.eps, vel=vel, keep=True)
    f.refresh_monopoles()
    ng = got["sizes"]["n_group"]
    f.dispatch(0, 0, ng)
    out = np.zeros((posm.shape[0], 4), np.float32)
    f.retrieve(0, out)
    if vel is not None:                                         # velocities travel with their particles
        v = f.get_velocities(0, posm.shape[0])
        assert np.array_equal(v[:, :3], vel.astype(np.float32)[got["perm"]])
    f.close()
    mom = oracle.monopoles(got["cells"], got["posm"])
    acc, pot = oracle.forces(got["posm"], mom, got["grp_first"], got["grp_n"], got["epj_off"], got["epj_id"], got["spj_off"], got["spj_id"], cfg.eps)
    check_forces(out, acc, pot, "device-built %s" % cfg.name)


@pytest.mark.parametrize("cfg_idx", [1, 4])
def test_device_build_full_size_against_host_builder(cfg_idx):
    """Full-size configs: the device-built tree equals the host builder's (itself pinned by the plain
    restatement) cell for cell; list lengths equal for every group; list contents equal on sampled groups."""
    cfg = CONFIGS[cfg_idx]
    posm, _ = make_particles(cfg)
    w = build_tree_and_lists(posm, cfg.n_leaf, cfg.n_grp, cfg.theta)
    got = device_build(posm, cfg.n_leaf, cfg.n_grp, cfg.theta, eps=cfg.eps, max_cell=w.n_cell + 10, max_group=w.n_group + 10,
                       max_entry=w.n_entry + 10)
    assert np.array_equal(got["perm"], w.perm)
    assert np.array_equal(got["cells"], w.cells)
    assert np.array_equal(got["geom"], w.geom)
    assert np.array_equal(got["grp_first"], w.grp_first) and np.array_equal(got["grp_n"], w.grp_n)
    assert np.array_equal(got["epj_off"], w.epj_off) and np.array_equal(got["spj_off"], w.spj_off)
    rng = np.random.default_rng(7)
    for g in rng.choice(w.n_group, 300, replace=False):
        assert np.array_equal(np.sort(got["epj_id"][w.epj_off[g]:w.epj_off[g + 1]]), np.sort(w.epj_id[w.epj_off[g]:w.epj_off[g + 1]]))
        assert np.array_equal(np.sort(got["spj_id"][w.spj_off[g]:w.spj_off[g + 1]]), np.sort(w.spj_id[w.spj_off[g]:w.spj_off[g + 1]]))


def test_whole_loop_on_the_device():
    """Construction on the device, 3 device-resident reuse steps, construction again from the moved particles
    (now in the previous tree order), evaluation: nothing but the initial upload and the final read-back crosses
    the host link.  The second tree must be the one the plain restatement builds from the moved particles, and
    its forces must match the oracle."""
    cfg = CONFIGS[4]
    posm, vel = make_particles(cfg, 6000)
    got, f = device_build(posm, cfg.n_leaf, cfg.n_grp, cfg.theta, eps=cfg.eps, vel=vel, keep=True)
    n = posm.shape[0]
    ng = got["sizes"]["n_group"]
    f.refresh_monopoles()
    f.dispatch(0, 0, ng)
    f.retrieve(0, None)                                        # wait, keep the forces on the device
    for _ in range(3):
        f.step_reuse(cfg.dt)
    with pytest.raises(binding.MwfError) as e:
        f.build(n, cfg.n_leaf, cfg.n_grp, cfg.theta)
    assert e.value.code == binding.ESTATE                      # results of the last step neither retrieved nor discarded
    f.retrieve(0, None)
    moved = f.get_particles(0, n)                              # tree order of the FIRST build
    v_before = f.get_velocities(0, n)
    f.begin_step(binding.MAKE_LIST_FOR_REUSE)
    f.build(n, cfg.n_leaf, cfg.n_grp, cfg.theta)
    sz = f.get_build_sizes()
    perm2 = f.get_permutation(n)
    ref = bhtree_ref.build(moved, cfg.n_leaf, cfg.n_grp, cfg.theta)
    assert np.array_equal(perm2, ref["perm"])
    cells, geom = f.get_tree(sz["n_cell"])
    assert np.array_equal(cells, ref["cells"]) and np.array_equal(geom, ref["geom"])
    assert np.array_equal(f.get_particles(0, n), moved[perm2])
    assert np.array_equal(f.get_velocities(0, n), v_before[perm2])
    with pytest.raises(binding.MwfError) as e:
        f.kick_drift(cfg.dt)
    assert e.value.code == binding.ESTATE                      # new lists: forces must be evaluated first
    f.refresh_monopoles()
    f.dispatch(0, 0, sz["n_group"])
    out = np.zeros((n, 4), np.float32)
    f.retrieve(0, out)
    gf, gn = f.get_groups(sz["n_group"])
    eo, ei, so, si = f.get_lists(sz["n_group"], sz["n_epj"], sz["n_spj"])
    f.step_reuse(cfg.dt)                                       # and the loop goes on
    f.retrieve(0, None)
    f.close()
    p2 = moved[perm2]
    mom = oracle.monopoles(cells, p2)
    acc, pot = oracle.forces(p2, mom, gf, gn, eo, ei, so, si, cfg.eps)
    check_forces(out, acc, pot, "second construction")


def test_more_than_2_31_list_entries():
    """Maximum sizes: a construction whose lists hold more than 2^31 entries, so every list offset past the first
    2^31 (merged-list offsets, SPJ offsets, the walk's output cursors) needs the 64-bit path (SURVEY.md 8(a) row a2:
    "int32 ids, int64 offsets"; the paper's per-batch `int` offsets, would wrap here).  N = 2^21 with small
    groups and a small opening angle; the forces of sampled groups from both ends of the list are compared with the
    oracle run on the lists read back; then the same lists go through the host path of a second context."""
    cfg = CONFIGS[1]
    n, n_leaf, n_grp, theta = 1 << 21, 8, 32, 0.27
    posm, _ = make_particles(cfg, n)
    f = binding.MultiWalkForce(cfg.eps, 1.0, max_ptcl=n, max_cell=n, max_group=n // 2, max_entry=3_500_000_000, n_tag=2)
    f.begin_step(binding.MAKE_LIST_FOR_REUSE)
    f.set_particles(posm)
    f.build(n, n_leaf, n_grp, theta, binding.MAKE_LIST_FOR_REUSE)
    sz = f.get_build_sizes()
    assert sz["n_spj"] > 2 ** 31 and sz["n_epj"] + sz["n_spj"] < 3_500_000_000, sz
    ng = sz["n_group"]
    f.refresh_monopoles()
    f.dispatch(0, 0, ng)
    out = np.zeros((n, 4), np.float32)
    f.retrieve(0, out)
    cells, _ = f.get_tree(sz["n_cell"], with_geom=False)
    grp_first, grp_n = f.get_groups(ng)
    epj_off, epj_id, spj_off, spj_id = f.get_lists(ng, sz["n_epj"], sz["n_spj"])
    tree_posm = f.get_particles(0, n)
    f.close()
    assert epj_off[-1] == sz["n_epj"] and spj_off[-1] == sz["n_spj"]
    assert np.all(np.diff(epj_off) >= 0) and np.all(np.diff(spj_off) > 0)
    first_past = int(np.searchsorted(spj_off, 2 ** 31))           # first group whose SPJ list starts past 2^31
    assert 0 < first_past < ng
    rng = np.random.default_rng(11)
    sample = np.unique(np.concatenate([rng.choice(first_past, 60, replace=False), [first_past - 1, first_past, ng - 1],
                                       first_past + rng.choice(ng - first_past, 120, replace=False)])).astype(np.int64)
    mom = oracle.monopoles(cells, tree_posm)
    acc, pot = oracle.forces(tree_posm, mom, grp_first, grp_n, epj_off, epj_id, spj_off, spj_id, cfg.eps, 1.0, sample)
    mask = np.zeros(n, bool)
    for g in sample:
        mask[grp_first[g]:grp_first[g] + grp_n[g]] = True
    check_forces(out[mask], acc[mask], pot[mask], "E = %.2e entries, %d sampled groups" % (sz["n_epj"] + sz["n_spj"], len(sample)))
    # the same lists through the host path (mwf_set_tree / mwf_set_lists: validation and merge kernels with 64-bit offsets)
    f2 = binding.MultiWalkForce(cfg.eps, 1.0, max_ptcl=n, max_cell=sz["n_cell"], max_group=ng, max_entry=sz["n_epj"] + sz["n_spj"], n_tag=2)
    f2.begin_step(binding.MAKE_LIST_FOR_REUSE)
    f2.set_particles(tree_posm)
    f2.set_tree(cells)
    f2.set_lists(grp_first, grp_n, epj_off, epj_id, spj_off, spj_id, binding.MAKE_LIST_FOR_REUSE)
    f2.refresh_monopoles()
    f2.dispatch(0, 0, ng)
    out2 = np.zeros((n, 4), np.float32)
    f2.retrieve(0, out2)
    f2.close()
    check_forces(out2[mask], acc[mask], pot[mask], "host path, same lists")
    # same lists in the same order; which SPJ entries count as far (swept like particles) is decided from the cell geometry by
    # the device builder and from the particles by the upload path, so the two sums agree to rounding, not bit for bit
    da = np.linalg.norm(out2[:, :3].astype(np.float64) - out[:, :3], axis=1) / np.linalg.norm(out[:, :3].astype(np.float64), axis=1)
    assert da.max() <= 2e-5 and np.sqrt(np.mean(da ** 2)) <= 1e-6


def test_shadow_store_after_a_device_build():
    """mwf_set_particles_next / mwf_swap_store on a tree and lists built on the device: the evaluation on the swapped-in
    particles is bitwise the one mwf_set_particles gives, and the dummy record the padded list entries point at exists
    in both stores (no NaN from the padding)."""
    cfg = CONFIGS[4]
    posm, _ = make_particles(cfg, 30000)
    got, f = device_build(posm, cfg.n_leaf, cfg.n_grp, cfg.theta, eps=cfg.eps, keep=True)
    n, ng = posm.shape[0], got["sizes"]["n_group"]
    moved = got["posm"].copy()
    moved[:, :3] += np.float32(1e-3) * np.random.default_rng(5).standard_normal((n, 3)).astype(np.float32)
    out_a, out_b = np.zeros((n, 4), np.float32), np.zeros((n, 4), np.float32)
    f.begin_step(binding.REUSE_LIST)
    f.set_particles(moved)
    f.refresh_monopoles()
    f.dispatch(0, 0, ng)
    f.retrieve(0, out_a)
    f.set_particles(got["posm"])                                # back to the built positions in the current store
    half = n // 2
    f.set_particles_next(moved[:half], 0, half)
    with pytest.raises(binding.MwfError) as e:
        f.swap_store()
    assert e.value.code == binding.ESTATE                       # only half of the particles written
    f.set_particles_next(moved[half:], half, n - half)
    f.swap_store()
    assert np.array_equal(f.get_particles(0, n), moved)
    f.refresh_monopoles()
    f.dispatch(0, 0, ng)
    f.retrieve(0, out_b)
    f.close()
    assert np.all(np.isfinite(out_b)) and np.array_equal(out_a, out_b)
