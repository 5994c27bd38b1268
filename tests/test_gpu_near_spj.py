"""Edge cases of the two-run list layout (reading S11b of DESIGN.md): run 1 = EPJ + FAR SPJ entries swept from 16-byte
records, run 2 = NEAR SPJ entries swept in item-centred coordinates with the remainder of their centre of mass.  Every case
is compared with the fp64 oracle on the same lists at the north_star's tolerances (S18); what the library decided
(far / near) is read from the list buffer it hands out (mwf_get_list_buffer)."""
import numpy as np
import pytest

import oracle
from paper_1907_02290_b200 import binding
from paper_1907_02290_b200.workload import CONFIGS, build_tree_and_lists, make_particles, make_workload

pytestmark = pytest.mark.gpu

ACC_MAX, ACC_RMS, POT_RMS = 1e-4, 2e-5, 1e-5


def far_away(posm):
    """The particles moved to coordinates of more than 40 diameters of the system: no separation inside it reaches 1/32 of
    a coordinate, so every SPJ entry has to be near (SPJ_FAR_KAPPA = 32)."""
    diam = float(np.linalg.norm(posm[:, :3].max(0) - posm[:, :3].min(0)))
    shift = np.float32(2.0 ** np.ceil(np.log2(40.0 * diam)))
    out = posm.copy()
    out[:, :3] += shift
    return out


def expect_code(fn, *a):
    with pytest.raises(binding.MwfError) as e:
        fn(*a)
    return e.value.code


def check(out, acc, pot, label):
    a, p = out[:, :3].astype(np.float64), out[:, 3].astype(np.float64)
    ea = np.linalg.norm(a - acc, axis=1) / np.linalg.norm(acc, axis=1)
    ep = np.abs(p - pot) / np.abs(pot)
    msg = "%s: acc max %.2e rms %.2e | pot rms %.2e" % (label, ea.max(), np.sqrt(np.mean(ea ** 2)), np.sqrt(np.mean(ep ** 2)))
    print(msg)
    assert ea.max() <= ACC_MAX and np.sqrt(np.mean(ea ** 2)) <= ACC_RMS and np.sqrt(np.mean(ep ** 2)) <= POT_RMS, msg


def lists_of(w):
    return (w.grp_first, w.grp_n, w.epj_off, w.epj_id, w.spj_off, w.spj_id)


def far_near_counts(f, n, n_cell, epj_off, spj_off):
    """(far, near) SPJ entries as the library laid them out: run 1 of a group = its EPJ entries then its far SPJ entries,
    padded to a whole tile with the dummy index n + n_cell; run 2 = its near SPJ entries, padded likewise."""
    off, lst = f.get_list_buffer()
    run1 = f.get_run1_len().astype(np.int64)
    ne, ns = np.diff(epj_off), np.diff(spj_off)
    assert np.all(run1 >= ne) and np.all(run1 - ne <= ns)
    for g in range(len(ne)):                       # the buffer agrees with those lengths
        seg = lst[off[g]:off[g + 1]]
        is_spj = (seg >= n) & (seg < n + n_cell)
        pad1 = -(-run1[g] // 64) * 64
        n_near = ns[g] - (run1[g] - ne[g])
        assert not is_spj[:ne[g]].any() and is_spj[ne[g]:run1[g]].all() and np.all(seg[run1[g]:pad1] == n + n_cell)
        assert is_spj[pad1:pad1 + n_near].all() and np.all(seg[pad1 + n_near:] == n + n_cell)
    return int((run1 - ne).sum()), int((ns - (run1 - ne)).sum())


def evaluate(f, n, n_group, order=1):
    if order == 2:
        f.set_spj_order(2)
    f.refresh_monopoles()
    f.dispatch(0, 0, n_group)
    out = np.full((n, 4), np.nan, np.float32)
    f.retrieve(0, out)
    return out


def oracle_forces(w_or_lists, cells, posm, eps, order=1):
    mom = oracle.monopoles(cells, posm)
    quad = oracle.quadrupoles(cells, posm, mom) if order == 2 else None
    return oracle.forces(posm, mom, *w_or_lists, eps, quad=quad) if order == 2 else oracle.forces(posm, mom, *w_or_lists, eps)


# ------------------------------------------------------------------ every item width x every run-2 tail
def hand_made_lists(w, spj_only, seed):
    """Groups of 1, 3, 7 ... 255 consecutive particles (every item width: 2 i per lane down to 2 lanes x 16 j-slices) over the
    tree of `w`; group g's SPJ list is L cells drawn at random among the cells that hold none of its particles, L cycling
    through 1, 63, 64, 65, 129 (ragged and exact tile tails; 8 sizes x 5 lengths are coprime cycles, so every pair occurs);
    its EPJ list is empty (spj_only) or its own particles."""
    rng = np.random.default_rng(seed)
    sizes, lengths = [1, 3, 7, 15, 31, 63, 127, 255], [1, 63, 64, 65, 129]
    gf, gn, eo, ei, so, si = [], [], [0], [], [0], []
    at, g = 0, 0
    cf, cn = w.cells[:, 0].astype(np.int64), w.cells[:, 1].astype(np.int64)
    while at + sizes[g % 8] <= w.n and g < 40:
        s, L = sizes[g % 8], lengths[g % 5]
        outside = np.nonzero((cf + cn <= at) | (cf >= at + s))[0]
        si.extend(rng.choice(outside, size=L, replace=False).tolist())
        so.append(len(si))
        if not spj_only:
            ei.extend(range(at, at + s))
        eo.append(len(ei))
        gf.append(at); gn.append(s)
        at += s; g += 1
    assert g == 40
    return (np.array(gf, np.int32), np.array(gn, np.int32), np.array(eo, np.int64), np.array(ei, np.int32),
            np.array(so, np.int64), np.array(si, np.int32))


@pytest.mark.parametrize("order", [1, 2])
@pytest.mark.parametrize("spj_only,shifted", [(True, True), (False, True), (False, False), (True, False)])
def test_every_width_times_every_run2_tail(spj_only, shifted, order):
    posm, _ = make_particles(CONFIGS[0], 3000)
    if shifted:
        posm = far_away(posm)
    w = build_tree_and_lists(posm, 4, 64, 0.5)
    lists = hand_made_lists(w, spj_only, seed=7 + order)
    n_used = int(lists[0][-1] + lists[1][-1])
    f = binding.MultiWalkForce(1 / 64, 1.0, max_ptcl=w.n, max_cell=w.n_cell, max_group=40, max_entry=lists[3].size + lists[5].size, n_tag=1)
    f.set_particles(w.posm)
    f.set_tree(w.cells)
    f.set_lists(*lists, binding.MAKE_LIST_FOR_REUSE)
    far, near = far_near_counts(f, w.n, w.n_cell, lists[2], lists[4])
    if shifted:
        assert far == 0 and near == lists[5].size
    else:
        assert far > 0 and near > 0                # a compact system at the origin: touching cells are near, the rest far
    out = evaluate(f, w.n, 40, order)
    f.close()
    acc, pot = oracle_forces(lists, w.cells, w.posm, 1 / 64, order)
    check(out[:n_used], acc[:n_used], pot[:n_used], "hand-made lists spj_only=%s shifted=%s order=%d" % (spj_only, shifted, order))


# ------------------------------------------------------------------ a workload far from the origin: everything is near
@pytest.mark.parametrize("idx,n", [(0, None), (3, 60000)])
def test_translated_workload_is_all_near(idx, n):
    cfg = CONFIGS[idx]
    posm, _ = make_particles(cfg, n)
    posm = far_away(posm)
    w = build_tree_and_lists(posm, cfg.n_leaf, cfg.n_grp, cfg.theta)
    f = binding.MultiWalkForce.for_workload(w, eps=cfg.eps, n_tag=2)
    f.upload_workload(w)
    far, near = far_near_counts(f, w.n, w.n_cell, w.epj_off, w.spj_off)
    assert far == 0 and near == w.spj_id.size
    for order in (1, 2):
        out = evaluate(f, w.n, w.n_group, order)
        acc, pot = oracle_forces(lists_of(w), w.cells, w.posm, cfg.eps, order)
        check(out, acc, pot, "%s far from the origin, order %d" % (cfg.name, order))
    f.close()
    # the same particles through the device-side construction step (its walk classifies from the cells' cubes)
    g = binding.MultiWalkForce(cfg.eps, 1.0, max_ptcl=w.n, max_cell=2 * w.n + 64, max_group=w.n + 8, max_entry=400 * w.n + 4096, n_tag=2)
    g.begin_step(binding.MAKE_LIST_FOR_REUSE)
    g.set_particles(posm)
    g.build(w.n, cfg.n_leaf, cfg.n_grp, cfg.theta, binding.MAKE_LIST_FOR_REUSE)
    sz = g.get_build_sizes()
    cells, _ = g.get_tree(sz["n_cell"])
    gf, gn = g.get_groups(sz["n_group"])
    lists = (gf, gn) + tuple(g.get_lists(sz["n_group"], sz["n_epj"], sz["n_spj"]))
    sorted_posm = g.get_particles(0, w.n)
    far, near = far_near_counts(g, w.n, sz["n_cell"], lists[2], lists[4])
    assert far == 0 and near == sz["n_spj"]
    out = evaluate(g, w.n, sz["n_group"])
    g.close()
    acc, pot = oracle_forces(lists, cells, sorted_posm, cfg.eps)
    check(out, acc, pot, "%s far from the origin, device-built" % cfg.name)


# ------------------------------------------------------------------ call orders (mwf.h: mwf_set_lists, "Call order and accuracy")
@pytest.mark.parametrize("order", [1, 2])
def test_lists_before_particles_are_all_near(order):
    """mwf_set_lists with no particles of this step in the store has nothing to measure distances with: every SPJ entry
    goes to run 2.  Same answer (to the tolerances) as the usual order, which finds far entries."""
    cfg = CONFIGS[3]
    w = make_workload(cfg, 40000)
    f = binding.MultiWalkForce.for_workload(w, eps=cfg.eps, n_tag=2)
    f.set_tree(w.cells)
    f.set_lists(*lists_of(w), binding.MAKE_LIST_FOR_REUSE)
    far, near = far_near_counts(f, w.n, w.n_cell, w.epj_off, w.spj_off)
    assert far == 0 and near == w.spj_id.size
    assert expect_code(f.refresh_monopoles) == binding.ESTATE      # still no particles
    f.set_particles(w.posm)
    out = evaluate(f, w.n, w.n_group, order)
    acc, pot = oracle_forces(lists_of(w), w.cells, w.posm, cfg.eps, order)
    check(out, acc, pot, "lists before particles, order %d" % order)
    f.upload_workload(w)                                           # particles first: now most entries are far
    far, near = far_near_counts(f, w.n, w.n_cell, w.epj_off, w.spj_off)
    assert far > near > 0
    out = evaluate(f, w.n, w.n_group)
    check(out, acc, pot, "particles before lists, order %d" % order)
    f.close()


def test_second_construction_step_does_not_classify_from_the_previous_steps_store():
    """A second construction step in the order tree, lists, particles: at mwf_set_lists the store still holds the previous
    step's particles in the previous tree's order.  They must not be used (the far marks would belong to other cells):
    everything near, and the result right."""
    cfg = CONFIGS[3]
    posm_a, _ = make_particles(cfg, 30000)
    rng = np.random.default_rng(3)
    posm_b = posm_a.copy()
    posm_b[:, :3] = (posm_a[:, :3] + rng.normal(scale=0.05, size=(30000, 3))).astype(np.float32) % np.float32(1.0)
    wa = build_tree_and_lists(posm_a, cfg.n_leaf, cfg.n_grp, cfg.theta)
    wb = build_tree_and_lists(posm_b, cfg.n_leaf, cfg.n_grp, cfg.theta)
    cap = dict(max_ptcl=30000, max_cell=max(wa.n_cell, wb.n_cell), max_group=max(wa.n_group, wb.n_group),
               max_entry=max(wa.epj_id.size + wa.spj_id.size, wb.epj_id.size + wb.spj_id.size))
    f = binding.MultiWalkForce(cfg.eps, 1.0, n_tag=2, **cap)
    f.upload_workload(wa)
    far, _ = far_near_counts(f, wa.n, wa.n_cell, wa.epj_off, wa.spj_off)
    assert far > 0
    evaluate(f, wa.n, wa.n_group)
    f.begin_step(binding.MAKE_LIST_FOR_REUSE)
    f.set_tree(wb.cells)
    f.set_lists(*lists_of(wb), binding.MAKE_LIST_FOR_REUSE)
    far, near = far_near_counts(f, wb.n, wb.n_cell, wb.epj_off, wb.spj_off)
    assert far == 0 and near == wb.spj_id.size
    f.set_particles(wb.posm)
    out = evaluate(f, wb.n, wb.n_group)
    f.close()
    acc, pot = oracle_forces(lists_of(wb), wb.cells, wb.posm, cfg.eps)
    check(out, acc, pot, "second construction step: tree, lists, particles")


def test_uploaded_spj_id_carrying_the_far_mark_is_refused():
    """Bit 30 of a staged SPJ id is the library's own far mark between its two passes; an uploaded id with that bit over a
    valid cell index must be reported as out of range, not taken for a marked entry."""
    cfg = CONFIGS[0]
    w = make_workload(cfg)
    f = binding.MultiWalkForce.for_workload(w, eps=cfg.eps, n_tag=1)
    f.set_particles(w.posm)
    f.set_tree(w.cells)
    for k in (0, 3, w.spj_id.size - 1):
        bad = w.spj_id.copy()
        bad[k] |= 0x40000000
        assert expect_code(f.set_lists, w.grp_first, w.grp_n, w.epj_off, w.epj_id, w.spj_off, bad) == binding.ERANGE
    g = binding.MultiWalkForce.for_workload(w, eps=cfg.eps, n_tag=1)   # and when there are no particles to classify with
    g.set_tree(w.cells)
    bad = w.spj_id.copy()
    bad[5] |= 0x40000000
    assert expect_code(g.set_lists, w.grp_first, w.grp_n, w.epj_off, w.epj_id, w.spj_off, bad) == binding.ERANGE
    g.close()
    f.set_lists(*lists_of(w))                                       # the ctx is still usable
    out = evaluate(f, w.n, w.n_group)
    f.close()
    acc, pot = oracle_forces(lists_of(w), w.cells, w.posm, cfg.eps)
    check(out, acc, pot, "after refused lists")
