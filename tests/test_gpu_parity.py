"""GPU parity: the CUDA path (through the C ABI) against the fp64 oracle, element by element on the
same seeded inputs.  Tolerances are BASELINE.json's north_star: per-particle relative acceleration
error <= 1e-4 max and <= 2e-5 RMS, relative potential error <= 1e-5 RMS."""
import numpy as np
import pytest

import oracle
from paper_1907_02290_b200 import binding
from paper_1907_02290_b200.workload import CONFIGS, build_tree_and_lists, make_particles, make_workload, pack_data_lists

pytestmark = pytest.mark.gpu

ACC_MAX, ACC_RMS, POT_RMS = 1e-4, 2e-5, 1e-5


def gpu_eval(w, eps, G=1.0, n_tag=4, batches=None, mode=binding.MAKE_LIST_FOR_REUSE, keep=False):
    f = binding.MultiWalkForce.for_workload(w, eps=eps, G=G, n_tag=n_tag)
    f.upload_workload(w, mode)
    f.refresh_monopoles()
    out = np.full((w.n, 4), np.nan, np.float32)
    if batches is None:
        f.dispatch(0, 0, w.n_group)
        f.retrieve(0, out)
    else:
        tag = 0
        pending = []
        for gb in range(0, w.n_group, batches):
            if len(pending) == n_tag:
                f.retrieve(pending.pop(0), out)
            f.dispatch(tag, gb, min(w.n_group, gb + batches))
            pending.append(tag)
            tag = (tag + 1) % n_tag
        for t in pending:
            f.retrieve(t, out)
    if keep:
        return out, f
    f.close()
    return out


def oracle_eval(w, eps, G=1.0, groups=None, posm=None):
    posm = w.posm if posm is None else posm
    mom = oracle.monopoles(w.cells, posm)
    acc, pot = oracle.forces(posm, mom, w.grp_first, w.grp_n, w.epj_off, w.epj_id, w.spj_off, w.spj_id, eps, G, groups)
    return acc, pot, mom


def errors(out, acc, pot, mask=None):
    a = out[:, :3].astype(np.float64)
    p = out[:, 3].astype(np.float64)
    if mask is not None:
        a, p, acc, pot = a[mask], p[mask], acc[mask], pot[mask]
    ea = np.linalg.norm(a - acc, axis=1) / np.linalg.norm(acc, axis=1)
    ep = np.abs(p - pot) / np.abs(pot)
    return ea, ep


def check(out, acc, pot, mask=None, label=""):
    ea, ep = errors(out, acc, pot, mask)
    msg = "%s: acc max %.2e rms %.2e | pot max %.2e rms %.2e" % (
        label, ea.max(), np.sqrt(np.mean(ea ** 2)), ep.max(), np.sqrt(np.mean(ep ** 2)))
    print(msg)
    assert np.all(np.isfinite(ea)) and np.all(np.isfinite(ep)), msg
    assert ea.max() <= ACC_MAX, msg
    assert np.sqrt(np.mean(ea ** 2)) <= ACC_RMS, msg
    assert np.sqrt(np.mean(ep ** 2)) <= POT_RMS, msg


def group_mask(w, groups):
    m = np.zeros(w.n, bool)
    for g in groups:
        m[w.grp_first[g]:w.grp_first[g] + w.grp_n[g]] = True
    return m


def expect_code(fn, *a):
    with pytest.raises(binding.MwfError) as e:
        fn(*a)
    return e.value.code


# ------------------------------------------------------------------ config 1 in full, others reduced
def test_config1_full():
    cfg = CONFIGS[0]
    w = make_workload(cfg)
    out = gpu_eval(w, cfg.eps)
    acc, pot, _ = oracle_eval(w, cfg.eps)
    check(out, acc, pot, label=cfg.name)


@pytest.mark.parametrize("idx,n", [(1, 60000), (2, 70001), (3, 65537), (4, 50000)])
def test_reduced_configs_every_particle(idx, n):
    cfg = CONFIGS[idx]
    w = make_workload(cfg, n)
    out = gpu_eval(w, cfg.eps)
    acc, pot, _ = oracle_eval(w, cfg.eps)
    check(out, acc, pot, label="%s n=%d" % (cfg.name, n))


def test_G_and_unequal_masses():
    cfg = CONFIGS[2]
    w = make_workload(cfg, 20000)
    out = gpu_eval(w, cfg.eps, G=6.5)
    acc, pot, _ = oracle_eval(w, cfg.eps, G=6.5)
    check(out, acc, pot, label="G=6.5")


# ------------------------------------------------------------------ full sizes, sampled groups
@pytest.mark.parametrize("idx,n_sample", [(1, 300), (2, 120), (3, 200), (4, 200)])
def test_full_size_sampled_groups(idx, n_sample):
    """BASELINE.json's full sizes in bench.py's launch configuration (one dispatch over all groups);
    the oracle evaluates a seeded sample of groups, every particle of each."""
    cfg = CONFIGS[idx]
    w = make_workload(cfg)
    out = gpu_eval(w, cfg.eps)
    assert np.all(np.isfinite(out))
    rng = np.random.default_rng(100 + idx)
    groups = rng.choice(w.n_group, size=n_sample, replace=False)
    cost = w.grp_n.astype(np.int64) * w.n_list
    # always include the heaviest group, the smallest group and both ends
    groups = np.unique(np.concatenate([groups, [np.argmax(cost), np.argmin(w.grp_n), 0, w.n_group - 1]]))
    acc, pot, _ = oracle_eval(w, cfg.eps, groups=groups)
    check(out, acc, pot, mask=group_mask(w, groups), label="%s full size" % cfg.name)
    # properties that hold at any size: tree forces nearly conserve momentum; W matches the closed form
    m = w.posm[:, 3].astype(np.float64)
    a = out[:, :3].astype(np.float64)
    assert np.linalg.norm((m[:, None] * a).sum(0)) < 1e-3 * (m * np.linalg.norm(a, axis=1)).sum()
    if cfg.kind == "plummer":
        W = 0.5 * np.sum(m * out[:, 3].astype(np.float64))
        assert W == pytest.approx(-3 * np.pi / 32 * 1.0055, rel=0.005)    # pin P6 at N >= 2^20


# ------------------------------------------------------------------ monopole refresh (row a3, reading S11)
@pytest.mark.parametrize("idx,n", [(0, None), (2, 100000), (3, 80000)])
def test_monopole_refresh(idx, n):
    cfg = CONFIGS[idx]
    w = make_workload(cfg, n)
    f = binding.MultiWalkForce.for_workload(w)
    f.upload_workload(w)
    f.refresh_monopoles()
    got = f.get_monopoles(w.n_cell).astype(np.float64)
    f.refresh_monopoles()                      # self-cleaning counters: a second refresh gives the same bits
    again = f.get_monopoles(w.n_cell).astype(np.float64)
    f.close()
    assert np.array_equal(got, again)
    mom = oracle.monopoles(w.cells, w.posm)
    assert np.all(np.abs(got[:, 3] - mom[:, 3]) <= 1e-6 * mom[:, 3])
    dx = np.linalg.norm(got[:, :3] - mom[:, :3], axis=1)
    scale = np.maximum(np.linalg.norm(mom[:, :3], axis=1), w.geom[:, 3])
    assert np.all(dx <= 2.0 ** -22 * scale)


def _check_monopoles(cells, posm, side):
    n_cell = cells.shape[0]
    f = binding.MultiWalkForce(0.01, max_ptcl=posm.shape[0], max_cell=n_cell, max_group=4, max_entry=64, n_tag=1)
    f.set_particles(posm)
    f.set_tree(cells)
    f.refresh_monopoles()
    got = f.get_monopoles(n_cell).astype(np.float64)
    f.refresh_monopoles()
    assert np.array_equal(got, f.get_monopoles(n_cell).astype(np.float64))
    f.close()
    mom = oracle.monopoles(cells, posm)
    assert np.all(np.abs(got[:, 3] - mom[:, 3]) <= 1e-6 * mom[:, 3])
    dx = np.linalg.norm(got[:, :3] - mom[:, :3], axis=1)
    assert np.all(dx <= 2.0 ** -22 * np.maximum(np.linalg.norm(mom[:, :3], axis=1), side))


def test_monopole_refresh_tree_shapes():
    """Tree shapes beyond the configs': very large leaves (n_leaf = 5000), one particle per leaf, a small tree, and a
    hand-made chain 90 levels deep (far deeper than 21-bit keys can make)."""
    posm, _ = make_particles(CONFIGS[0], 30011)
    for n_leaf, n in ((5000, 30011), (16, 2048), (1, 1500), (3, 9000)):
        w = build_tree_and_lists(posm[:n], n_leaf, 64, 0.9)
        _check_monopoles(w.cells, w.posm, w.geom[:, 3])
    # chain: cell 2k (k >= 1) is internal with a one-particle leaf 2k+1 and the next internal cell 2k+2 as children
    depth, rng = 90, np.random.default_rng(11)
    n = depth + 1
    pts = np.concatenate([rng.normal(size=(n, 3)), rng.uniform(0.5, 2.0, size=(n, 1))], axis=1).astype(np.float32)
    cells = [(0, n, 1, 2)]
    for k in range(depth):
        first = k                                   # particles [k, n) are below the k-th chain cell
        cells.append((first, 1, 0, 0))              # leaf with particle k
        last = k == depth - 1
        cells.append((first + 1, n - first - 1, 0 if last else len(cells) + 1, 0 if last else 2))
    cells = np.array(cells, np.int32)
    _check_monopoles(cells, pts, np.full(cells.shape[0], 8.0))


# ------------------------------------------------------------------ dispatch shapes
def test_batched_dispatch_over_tags_is_bitwise_identical():
    """Config 2's pipeline: 64-256 groups per dispatch, tags round-robin over the streams."""
    cfg = CONFIGS[1]
    w = make_workload(cfg, 150000)
    one = gpu_eval(w, cfg.eps)
    for batch in (64, 256):
        many = gpu_eval(w, cfg.eps, n_tag=8, batches=batch)
        assert np.array_equal(one, many)


@pytest.mark.parametrize("sizes", [[64] * 12, [3] * 40, [64, 1, 200, 7, 64, 33, 2, 129, 16, 64, 5, 255]])
def test_arbitrary_group_ranges_equal_one_dispatch(sizes):
    """A dispatch over any group range takes its items widest-first from the class-sorted permutation (five runs per
    range): ranges of one group, ranges in which some width classes are empty, ranges dispatched out of order -- the
    results are bitwise those of the whole-workload dispatch, and match direct summation."""
    n = int(np.sum(sizes))
    posm, _ = make_particles(CONFIGS[0], n)
    gf, gn, eo, ei, so, si = synthetic_groups(n, sizes)
    ng = len(sizes)
    f = binding.MultiWalkForce(1 / 64, 1.0, max_ptcl=n, max_cell=1, max_group=ng, max_entry=ei.size, n_tag=3)
    f.begin_step(binding.MAKE_LIST_FOR_REUSE)
    f.set_particles(posm)
    f.set_tree(np.array([[0, n, 0, 0]], np.int32))
    f.set_lists(gf, gn, eo, ei, so, si, binding.MAKE_LIST_FOR_REUSE)
    f.refresh_monopoles()
    one = np.full((n, 4), np.nan, np.float32)
    f.dispatch(0, 0, ng)
    f.retrieve(0, one)
    cuts = sorted({0, 1, 2, ng // 3, ng // 2, ng - 1, ng})
    ranges = list(zip(cuts[:-1], cuts[1:]))[::-1]                  # last range first
    many = np.full((n, 4), np.nan, np.float32)
    f.begin_step(binding.REUSE_LIST)
    for k, (gb, ge) in enumerate(ranges):
        t = k % 3
        if k >= 3:
            f.retrieve(t, many)
        f.dispatch(t, gb, ge)
    for t in range(min(3, len(ranges))):
        f.retrieve(t, many)
    f.close()
    assert np.array_equal(one, many)
    acc, pot = oracle.direct(posm, 1 / 64)
    check(many, acc, pot, label="arbitrary ranges")


def test_calc_force_all_host_and_device_destinations():
    import torch
    cfg = CONFIGS[1]
    w = make_workload(cfg, 100000)
    ref, f = gpu_eval(w, cfg.eps, n_tag=8, keep=True)
    host = f.pinned(w.n)
    src = f.pinned(w.n)
    src.numpy()[:] = w.posm
    f.begin_step(binding.REUSE_LIST)
    f.calc_force_all(src, host)                                   # split over the 8 tags, one D2H per tag
    assert np.array_equal(host.numpy(), ref)
    dev = torch.zeros((w.n, 4), dtype=torch.float32, device="cuda")
    f.calc_force_all(torch.from_numpy(w.posm).cuda(), dev)        # device source and destination, one dispatch
    assert np.array_equal(dev.cpu().numpy(), ref)
    f.close()


def test_pipelined_host_loop_equals_the_blocking_one():
    """mwf_set_particles_next / mwf_swap_store: the next step's particles go into the shadow store tag
    by tag, right behind the retrieve of that tag's results and while the other tags' kernels still read the current
    store.  Every step must give bitwise the results of the blocking mwf_calc_force_all on the same particles, and the
    oracle's on the last step."""
    import torch
    cfg = CONFIGS[4]
    w = make_workload(cfg, 60000)
    rng = np.random.default_rng(3)
    steps = [w.posm.copy()]
    for _ in range(3):                                           # moved particles, lists reused (tree order unchanged)
        q = steps[-1].copy()
        q[:, :3] += (1e-3 * rng.standard_normal((w.n, 3))).astype(np.float32)
        steps.append(q)
    n_tag = 4
    ref = []
    f = binding.MultiWalkForce.for_workload(w, n_tag=n_tag)
    f.upload_workload(w, binding.MAKE_LIST_FOR_REUSE)
    src, dst = f.pinned(w.n), f.pinned(w.n)
    for q in steps:
        src.numpy()[:] = q
        f.begin_step(binding.REUSE_LIST)
        f.calc_force_all(src, dst)
        ref.append(dst.numpy().copy())
    f.close()

    f = binding.MultiWalkForce.for_workload(w, n_tag=n_tag)
    f.upload_workload(w, binding.MAKE_LIST_FOR_REUSE)
    split = f.get_tag_split()
    assert split[0] == 0 and split[-1] == w.n_group and np.all(np.diff(split) >= 0)
    # shares of the interactions per tag: equal over the first half of the tags, tapering to an eighth for the last one
    per_group = w.grp_n.astype(np.int64) * w.n_list
    share = np.array([per_group[split[t]:split[t + 1]].sum() for t in range(n_tag)], np.float64)
    share /= share[0]
    want = np.minimum(1.0, 2.0 * (n_tag - np.arange(n_tag) - 0.5) / n_tag)
    assert np.all(np.abs(share - want) <= 0.02 + 2.0 * per_group.max() / (per_group.sum() / n_tag))
    first = [int(w.grp_first[split[t]]) if split[t] < w.n_group else w.n for t in range(n_tag)] + [w.n]
    up = torch.cuda.Stream()
    host_in = [f.pinned(w.n) for _ in steps]
    for h, q in zip(host_in, steps):
        h.numpy()[:] = q
    out = f.pinned(w.n)

    def dispatch_all():
        f.refresh_monopoles()
        for t in range(n_tag):
            if split[t + 1] > split[t]:
                f.dispatch(t, int(split[t]), int(split[t + 1]))

    assert expect_code(f.swap_store) == binding.ESTATE            # nothing in the shadow store yet
    assert expect_code(f.set_particles_next, host_in[0], w.n - 1, 2, up) == binding.ERANGE
    dispatch_all()                                               # step 0 on the uploaded particles
    for k in range(len(steps)):
        nxt = host_in[(k + 1) % len(steps)]
        for t in range(n_tag):
            if split[t + 1] == split[t]:
                continue
            f.retrieve(t, out)                                   # results of step k for this tag's particles
            if t == 0:
                assert expect_code(f.swap_store) == binding.ESTATE   # not all N written, tags in flight
            f.set_particles_next(nxt[first[t]:first[t + 1]], first[t], first[t + 1] - first[t], up)
        assert np.array_equal(out.numpy(), ref[k]), "step %d" % k
        f.swap_store()
        assert expect_code(f.dispatch, 0, 0, 1) == binding.ESTATE   # monopoles stale after the swap
        dispatch_all()
    for t in range(n_tag):                                       # the loop wrapped around: step 0 again
        if split[t + 1] > split[t]:
            f.retrieve(t, out)
    assert np.array_equal(out.numpy(), ref[0])
    assert np.array_equal(f.get_particles(0, w.n), steps[0])
    f.close()
    acc, pot, _ = oracle_eval(w, cfg.eps, posm=steps[-1])
    check(ref[-1], acc, pot, label="pipelined loop, last step")


# ------------------------------------------------------------------ edge cases of the kernel mapping
def synthetic_groups(n, sizes):
    """Consecutive groups of the given sizes over n particles with EVERY particle in every list
    (theta = 0): the result must equal direct summation whatever the group sizes are."""
    sizes = np.asarray(sizes, np.int32)
    assert int(sizes.sum()) == n
    first = np.concatenate([[0], np.cumsum(sizes)[:-1]]).astype(np.int32)
    ng = len(sizes)
    epj_off = np.arange(ng + 1, dtype=np.int64) * n
    epj_id = np.tile(np.arange(n, dtype=np.int32), ng)
    return first, sizes, epj_off, epj_id, np.zeros(ng + 1, np.int64), np.zeros(0, np.int32)


@pytest.mark.parametrize("n", [1, 2, 63, 64, 65, 129, 1000])
def test_every_remainder_width_against_direct_summation(n):
    """Group sizes 1, 3, 7, ... 255 hit every item kind (64 = 2 per lane; <= 32, <= 16, <= 8 with 1/2/4
    j-slices); list lengths n = 1, 63, 64, 65 hit the ragged and exact tile tails."""
    posm, _ = make_particles(CONFIGS[0], n)
    sizes, left, k = [], n, 1
    while left > 0:
        s = min(left, k)
        sizes.append(s)
        left -= s
        k = k * 2 + 1 if k < 130 else 1
    gf, gn, eo, ei, so, si = synthetic_groups(n, sizes)
    f = binding.MultiWalkForce(1 / 64, 1.0, max_ptcl=n, max_cell=1, max_group=len(sizes), max_entry=ei.size, n_tag=2)
    f.begin_step(binding.MAKE_LIST)
    f.set_particles(posm)
    f.set_tree(np.array([[0, n, 0, 0]], np.int32))
    f.set_lists(gf, gn, eo, ei, so, si, binding.MAKE_LIST)
    f.refresh_monopoles()
    f.dispatch(1, 0, len(sizes))
    out = np.full((n, 4), np.nan, np.float32)
    f.retrieve(1, out)
    f.close()
    acc, pot = oracle.direct(posm, 1 / 64)
    if n == 1:
        assert np.all(out == 0)          # a lone particle feels nothing (self term excluded, reading S2)
    else:
        check(out, acc, pot, label="direct n=%d" % n)


def test_lists_without_self_and_spj_only():
    """A group whose EPJ list holds none of its own particles gets no self correction; a list may be
    SPJ-only or EPJ-only."""
    posm, _ = make_particles(CONFIGS[0], 300)
    cells = np.array([[0, 300, 1, 2], [0, 100, 0, 0], [100, 200, 0, 0]], np.int32)
    gf = np.array([0, 100], np.int32)
    gn = np.array([100, 200], np.int32)
    # group 0 sees particles 100..299 as EPJ only (no self); group 1 sees cell 1 as one SPJ and no EPJ at all
    eo = np.array([0, 200, 200], np.int64)
    ei = np.arange(100, 300, dtype=np.int32)
    so = np.array([0, 0, 1], np.int64)
    si = np.array([1], np.int32)
    f = binding.MultiWalkForce(1 / 64, 1.0, max_ptcl=300, max_cell=3, max_group=2, max_entry=201, n_tag=1)
    f.set_particles(posm)
    f.set_tree(cells)
    f.set_lists(gf, gn, eo, ei, so, si, binding.MAKE_LIST_FOR_REUSE)
    f.refresh_monopoles()
    f.dispatch(0, 0, 2)
    out = np.full((300, 4), np.nan, np.float32)
    f.retrieve(0, out)
    f.close()
    mom = oracle.monopoles(cells, posm)
    acc, pot = oracle.forces(posm, mom, gf, gn, eo, ei, so, si, 1 / 64)
    check(out, acc, pot, label="no-self / spj-only")


def test_coincident_particles():
    """Reading S4: distinct particles at one position are a real pair (0 to acc, -G m/eps to pot)."""
    posm = np.array([[1, 1, 1, 2.0], [1, 1, 1, 5.0], [2, 1, 1, 1.0]], np.float32)
    gf, gn, eo, ei, so, si = synthetic_groups(3, [3])
    f = binding.MultiWalkForce(0.5, 1.0, max_ptcl=3, max_cell=1, max_group=1, max_entry=3, n_tag=1)
    f.set_particles(posm)
    f.set_tree(np.array([[0, 3, 0, 0]], np.int32))
    f.set_lists(gf, gn, eo, ei, so, si)
    f.refresh_monopoles()
    f.dispatch(0, 0, 1)
    out = np.zeros((3, 4), np.float32)
    f.retrieve(0, out)
    f.close()
    acc, pot = oracle.direct(posm, 0.5)
    np.testing.assert_allclose(out[:, :3], acc, rtol=1e-5, atol=1e-7)
    np.testing.assert_allclose(out[:, 3], pot, rtol=1e-5)


# ------------------------------------------------------------------ method G1: data lists (NEXT-3; Fig. 2)
def test_data_lists_equal_index_lists():
    """The paper's method G1 (the lists carry j records, sent with every dispatch) against its method G2 (indices into
    the device store) on the same lists: same items, sweep and summation order.  The 16-byte records of G1 hold
    the SPJ centres rounded to fp32, the index path also reads their rounding remainders (reading S11b), so the two agree
    bitwise on lists without SPJ entries and to the oracle's tolerance otherwise; G1 is bitwise the same however it is
    batched."""
    cfg = CONFIGS[1]
    w = make_workload(cfg, 60001)
    out_idx, f = gpu_eval(w, cfg.eps, keep=True)
    spj = f.get_monopoles(w.n_cell)
    assert expect_code(f.dispatch_data, 0, 0, 1, np.zeros((4, 4), np.float32), np.zeros(2, np.int64)) == binding.ESTATE   # nothing reserved
    cap = int(w.n_list.max()) * 40
    f.reserve_data_lists(cap)
    out = np.full((w.n, 4), np.nan, np.float32)
    tag, pending, keep_alive = 0, [], {}
    for gb in range(0, w.n_group, 37):
        ge = min(w.n_group, gb + 37)
        if len(pending) == f.n_tag:
            f.retrieve(pending.pop(0), out)
        rec, joff = pack_data_lists(w, gb, ge, w.posm, spj)
        keep_alive[tag] = (rec, joff)                      # host sources stay valid until the tag is retrieved
        f.dispatch_data(tag, gb, ge, rec, joff)
        pending.append(tag)
        tag = (tag + 1) % f.n_tag
    for t in pending:
        f.retrieve(t, out)
    acc, pot, _ = oracle_eval(w, cfg.eps)
    check(out, acc, pot, label="G1 data lists")
    check(out_idx, acc, pot, label="G2 index lists")
    assert np.abs(out - out_idx).max() <= 1e-4 * np.abs(out_idx).max()
    # device-resident records, one dispatch over everything
    import torch
    rec, joff = pack_data_lists(w, 0, w.n_group, w.posm, spj)
    f.reserve_data_lists(rec.shape[0])
    out2 = np.full((w.n, 4), np.nan, np.float32)
    f.dispatch_data(1, 0, w.n_group, torch.from_numpy(rec).cuda(), joff)
    assert expect_code(f.dispatch_data, 1, 0, 1, rec, joff[:2].copy()) == binding.ESTATE              # tag still in flight
    f.retrieve(1, out2)
    assert np.array_equal(out2, out)
    bad = joff.copy()
    bad[1] += 1
    assert expect_code(f.dispatch_data, 0, 0, w.n_group, rec, bad) == binding.ERANGE                  # run length != list length
    f.reserve_data_lists(10)
    assert expect_code(f.dispatch_data, 0, 0, w.n_group, rec, joff) == binding.ENOMEM
    f.close()
    # lists without SPJ entries (theta = 0: every particle is an EPJ of every group): bitwise the index path
    w0 = make_workload(cfg, 3000, theta=0.0)
    assert w0.spj_id.size == 0
    idx0, f = gpu_eval(w0, cfg.eps, keep=True)
    rec, joff = pack_data_lists(w0, 0, w0.n_group, w0.posm, np.zeros((w0.n_cell, 4), np.float32))
    f.reserve_data_lists(rec.shape[0])
    dat0 = np.full((w0.n, 4), np.nan, np.float32)
    f.dispatch_data(0, 0, w0.n_group, rec, joff)
    f.retrieve(0, dat0)
    f.close()
    assert np.array_equal(idx0, dat0)


# ------------------------------------------------------------------ quadrupole SPJ (NEXT-3, reading S22)
@pytest.mark.parametrize("idx,n", [(0, None), (2, 65537), (3, 50000)])
def test_quadrupole_spj(idx, n):
    """order 2: the refresh also makes Q bottom-up, the dispatch evaluates the Q terms of the SPJ entries in the sweep of
    the force kernel.  Moments and forces against the oracle's quadrupole evaluation on the same lists; switching back to order 1
    reproduces the monopole result bit for bit."""
    cfg = CONFIGS[idx]
    w = make_workload(cfg, n)
    out1, f = gpu_eval(w, cfg.eps, keep=True)
    assert expect_code(f.get_quadrupoles, w.n_cell) == binding.ESTATE             # order 1 keeps no quadrupoles
    f.set_spj_order(2)
    assert expect_code(f.dispatch, 0, 0, w.n_group) == binding.ESTATE             # moments of the other order are stale
    f.refresh_monopoles()
    got = f.get_quadrupoles(w.n_cell).astype(np.float64)
    mom = oracle.monopoles(w.cells, w.posm)
    quad = oracle.quadrupoles(w.cells, w.posm, mom)
    tr = quad[:, :3].sum(1)
    assert np.all(np.abs(got[:, :6] - quad) <= 1e-6 * tr[:, None] + 1e-30)
    assert np.all(np.abs(got[:, 6] - 0.5 * tr) <= 1e-6 * tr + 1e-30)
    out2 = np.full((w.n, 4), np.nan, np.float32)
    f.dispatch(0, 0, w.n_group)
    f.retrieve(0, out2)
    lists = (w.grp_first, w.grp_n, w.epj_off, w.epj_id, w.spj_off, w.spj_id)
    acc, pot = oracle.forces(w.posm, mom, *lists, cfg.eps, quad=quad)
    check(out2, acc, pot, label="%s quadrupole" % cfg.name)
    acc1, pot1 = oracle.forces(w.posm, mom, *lists, cfg.eps)
    ea, _ = errors(out2, acc1, pot1)
    assert ea.max() > 10 * ACC_MAX or idx == 0                                     # it is not the monopole answer
    # batched over tags: same bits
    out3 = np.full((w.n, 4), np.nan, np.float32)
    step = max(1, w.n_group // 7)
    tags = []
    for k, gb in enumerate(range(0, w.n_group, step)):
        t = k % f.n_tag
        if t in tags:
            f.retrieve(t, out3)
            tags.remove(t)
        f.dispatch(t, gb, min(w.n_group, gb + step))
        tags.append(t)
    for t in tags:
        f.retrieve(t, out3)
    assert np.array_equal(out2, out3)
    if idx == 0:
        f.reserve_data_lists(64)
        assert expect_code(f.dispatch_data, 0, 0, 1, np.zeros((4, 4), np.float32), np.zeros(2, np.int64)) == binding.ESTATE
    f.set_spj_order(1)
    f.refresh_monopoles()
    out4 = np.full((w.n, 4), np.nan, np.float32)
    f.dispatch(0, 0, w.n_group)
    f.retrieve(0, out4)
    assert np.array_equal(out1, out4)
    f.close()


def test_quadrupole_device_resident_steps():
    """mwf_step_reuse with order 2: kick-drift, refresh (monopoles + quadrupoles), the order-2 force kernel with the closing kick -- per step the
    forces match the oracle's quadrupole evaluation at the positions the device holds."""
    cfg = CONFIGS[4]
    w = make_workload(cfg, 30000)
    f = binding.MultiWalkForce.for_workload(w, n_tag=2)
    f.upload_workload(w)
    f.set_spj_order(2)
    vel4 = np.zeros((w.n, 4), np.float32)
    vel4[:, :3] = w.vel
    f.set_velocities(vel4)
    f.refresh_monopoles()
    out = np.zeros((w.n, 4), np.float32)
    f.dispatch(0, 0, w.n_group)
    f.retrieve(0, out)
    lists = (w.grp_first, w.grp_n, w.epj_off, w.epj_id, w.spj_off, w.spj_id)
    for step in range(3):
        f.step_reuse(cfg.dt)
        f.retrieve(0, out)
        posm = f.get_particles(0, w.n)
        mom = oracle.monopoles(w.cells, posm)
        quad = oracle.quadrupoles(w.cells, posm, mom)
        acc, pot = oracle.forces(posm, mom, *lists, cfg.eps, quad=quad)
        check(out, acc, pot, label="quadrupole reuse step %d" % (step + 1))
    f.close()


# ------------------------------------------------------------------ list-reuse driver (rows a6, a7)
def test_state_machine_and_validation():
    cfg = CONFIGS[0]
    w = make_workload(cfg, 2000)
    lists = (w.grp_first, w.grp_n, w.epj_off, w.epj_id, w.spj_off, w.spj_id)
    f = binding.MultiWalkForce.for_workload(w, n_tag=2)
    out = np.zeros((w.n, 4), np.float32)
    assert expect_code(f.dispatch, 0, 0, 1) == binding.ESTATE                  # nothing uploaded
    assert expect_code(f.begin_step, binding.REUSE_LIST) == binding.ESTATE     # no saved lists
    assert expect_code(f.set_lists, *lists) == binding.ESTATE                  # no tree yet
    assert expect_code(f.refresh_monopoles) == binding.ESTATE
    f.set_particles(w.posm)
    f.set_tree(w.cells)
    f.set_lists(*lists, binding.MAKE_LIST)
    assert expect_code(f.dispatch, 0, 0, w.n_group) == binding.ESTATE          # monopoles stale
    f.refresh_monopoles()
    assert expect_code(f.dispatch, 5, 0, 1) == binding.EINVAL                  # bad tag
    assert expect_code(f.dispatch, 0, 0, w.n_group + 1) == binding.ERANGE
    assert expect_code(f.retrieve, 0, out) == binding.ESTATE                   # idle tag
    f.dispatch(0, 0, w.n_group)
    f.retrieve(0, out)
    # MAKE_LIST keeps nothing: REUSE_LIST afterwards is a user error
    assert expect_code(f.begin_step, binding.REUSE_LIST) == binding.ESTATE
    assert expect_code(f.dispatch, 0, 0, 1) == binding.ESTATE
    # MAKE_LIST_FOR_REUSE keeps them; evaluation 0 is identical under either mode (pin P9)
    f.begin_step(binding.MAKE_LIST_FOR_REUSE)
    f.set_particles(w.posm)        # a construction step brings its particles (mwf.h, mwf_set_lists: without them every SPJ entry is near)
    f.set_tree(w.cells)
    f.set_lists(*lists, binding.MAKE_LIST_FOR_REUSE)
    f.refresh_monopoles()
    f.dispatch(1, 0, w.n_group)
    out2 = np.zeros_like(out)
    f.retrieve(1, out2)
    assert np.array_equal(out, out2)
    f.begin_step(binding.REUSE_LIST)
    f.set_particles(w.posm)
    assert expect_code(f.dispatch, 0, 0, 1) == binding.ESTATE                  # a refresh must follow an upload
    f.refresh_monopoles()
    f.dispatch(0, 0, w.n_group)
    f.retrieve(0, out2)
    assert np.array_equal(out, out2)
    # validation of indices, offsets, self-membership, tree and capacity
    bad = w.epj_id.copy()
    bad[7] = w.n
    assert expect_code(f.set_lists, w.grp_first, w.grp_n, w.epj_off, bad, w.spj_off, w.spj_id) == binding.ERANGE
    bad = w.spj_id.copy()
    bad[3] = -1
    assert expect_code(f.set_lists, w.grp_first, w.grp_n, w.epj_off, w.epj_id, w.spj_off, bad) == binding.ERANGE
    bad = w.epj_off.copy()
    bad[2] = bad[1] - 1
    assert expect_code(f.set_lists, w.grp_first, w.grp_n, bad, w.epj_id, w.spj_off, w.spj_id) == binding.ERANGE
    bad = w.epj_id.copy()
    seg = bad[: w.epj_off[1]]
    own = np.nonzero(seg == w.grp_first[0])[0][0]
    outsider = np.setdiff1d(np.arange(w.n), np.arange(w.grp_first[0], w.grp_first[0] + w.grp_n[0]))[0]
    if w.grp_n[0] > 1:
        bad[own] = outsider                                                    # one own particle missing from the list
        assert expect_code(f.set_lists, w.grp_first, w.grp_n, w.epj_off, bad, w.spj_off, w.spj_id) == binding.EINVAL
    cells = w.cells.copy()
    cells[1, 0] += 1
    assert expect_code(f.set_tree, cells) == binding.ERANGE
    # a cell nobody claims (its parent's child range stops short of it) / a cell claimed by two parents
    par = np.nonzero(w.cells[:, 3] >= 2)[0][-1]
    cells = w.cells.copy()
    last = cells[par, 2] + cells[par, 3] - 1
    cells[par, 3] -= 1                                                         # orphan: `last`
    cells[last - 1, 1] += cells[last, 1]                                       # keep the partition of the parent's range
    assert expect_code(f.set_tree, cells) == binding.ERANGE
    leaves = np.nonzero(w.cells[:, 3] == 0)[0]
    cells = w.cells.copy()
    victim = cells[par, 2]                                                     # first child of `par` ...
    thief = leaves[leaves != victim][0]
    if cells[thief, 1] == cells[victim, 1] and cells[thief, 0] == cells[victim, 0]:
        thief = leaves[leaves != victim][1]
    cells[thief, 2], cells[thief, 3] = victim, 1                               # ... also claimed by a leaf turned parent
    assert expect_code(f.set_tree, cells) == binding.ERANGE
    f.set_tree(w.cells)
    assert expect_code(f.get_particles, w.n - 1, 2) == binding.ERANGE          # behind the particles: the SPJ block
    small = binding.MultiWalkForce(cfg.eps, max_ptcl=w.n, max_cell=w.n_cell, max_group=w.n_group, max_entry=10, n_tag=1)
    small.set_particles(w.posm)
    small.set_tree(w.cells)
    assert expect_code(small.set_lists, *lists) == binding.ENOMEM
    small.close()
    f.close()


def test_reuse_run_per_step():
    """Config 5 at reduced N: lists built once, 8 kick-drift-kick steps reuse them while the monopoles are
    refreshed on the device; every evaluation is compared with the oracle run on exactly the fp32
    positions that were uploaded (reading O7).  The orbit integration is host harness code and uses the
    GPU's forces (the system under test)."""
    cfg = CONFIGS[4]
    w = make_workload(cfg, 40000)
    f = binding.MultiWalkForce.for_workload(w, n_tag=4)
    f.upload_workload(w, binding.MAKE_LIST_FOR_REUSE)
    x = w.posm[:, :3].astype(np.float64)
    v = w.vel.copy()
    posm = w.posm.copy()
    host_in, host_out = f.pinned(w.n), f.pinned(w.n)
    spj_prev, a = None, None
    off0, list0 = f.get_list_buffer()                          # pin P9: the list buffers as the kernel reads them
    for step in range(cfg.n_reuse + 1):
        if step > 0:
            v += 0.5 * cfg.dt * a
            x += cfg.dt * v
            posm[:, :3] = x.astype(np.float32)
            f.begin_step(binding.REUSE_LIST)
        host_in.numpy()[:] = posm
        f.calc_force_all(host_in, host_out)
        out = host_out.numpy().copy()
        acc, pot, mom = oracle_eval(w, cfg.eps, posm=posm)
        check(out, acc, pot, label="step %d" % step)
        spj = f.get_monopoles(w.n_cell)
        assert np.all(np.abs(spj[:, 3] - mom[:, 3]) <= 1e-6 * mom[:, 3])
        assert np.all(np.linalg.norm(spj[:, :3] - mom[:, :3], axis=1)
                      <= 2.0 ** -22 * np.maximum(np.linalg.norm(mom[:, :3], axis=1), w.geom[:, 3]))
        if spj_prev is not None:
            assert not np.array_equal(spj, spj_prev)           # moments follow the particles
        spj_prev = spj
        off1, list1 = f.get_list_buffer()
        assert np.array_equal(off0, off1) and np.array_equal(list0, list1)   # bit-identical on reuse steps
        a = out[:, :3].astype(np.float64)
        if step > 0:
            v += 0.5 * cfg.dt * a
    f.close()


def test_energy_over_the_reuse_run():
    """Sanity band P11: over config 5's 8 kick-drift-kick steps with reused lists the total energy
    E = sum m v^2 / 2 + sum m pot / 2 barely moves, and it moves the same way whether the orbit is driven by the GPU's
    forces or by the oracle's (reduced N; the harness integrates in fp64 and uploads fp32 positions, reading O7)."""
    cfg = CONFIGS[4]
    w = make_workload(cfg, 40000)
    m = w.posm[:, 3].astype(np.float64)
    f = binding.MultiWalkForce.for_workload(w, n_tag=2)
    f.upload_workload(w, binding.MAKE_LIST_FOR_REUSE)
    host_in, host_out = f.pinned(w.n), f.pinned(w.n)

    def gpu_forces(posm):
        host_in.numpy()[:] = posm
        f.begin_step(binding.REUSE_LIST)
        f.calc_force_all(host_in, host_out)
        out = host_out.numpy()
        return out[:, :3].astype(np.float64), out[:, 3].astype(np.float64)

    def oracle_forces(posm):
        acc, pot, _ = oracle_eval(w, cfg.eps, posm=posm)
        return acc, pot

    energies = {}
    for name, forces in (("gpu", gpu_forces), ("oracle", oracle_forces)):
        x, v, posm = w.posm[:, :3].astype(np.float64), w.vel.copy(), w.posm.copy()
        a, pot = forces(posm)
        e = [0.5 * np.sum(m * (v * v).sum(1)) + 0.5 * np.sum(m * pot)]
        for _ in range(cfg.n_reuse):
            v += 0.5 * cfg.dt * a
            x += cfg.dt * v
            posm[:, :3] = x.astype(np.float32)
            a, pot = forces(posm)
            v += 0.5 * cfg.dt * a
            e.append(0.5 * np.sum(m * (v * v).sum(1)) + 0.5 * np.sum(m * pot))
        energies[name] = np.array(e)
    f.close()
    eg, eo = energies["gpu"], energies["oracle"]
    print("energy: E0 %.6f, drift over %d steps gpu %.2e oracle %.2e, |gpu - oracle| max %.2e (relative)" % (
        eo[0], cfg.n_reuse, (eg[-1] - eg[0]) / abs(eg[0]), (eo[-1] - eo[0]) / abs(eo[0]), np.abs(eg - eo).max() / abs(eo[0])))
    assert abs(eo[0] / (0.5 * -3 * np.pi / 32 * 1.0055) - 1) < 0.2   # virial equilibrium: E = W / 2, W of pin P6
    assert abs(eg[-1] - eg[0]) <= 1e-4 * abs(eg[0]) and abs(eo[-1] - eo[0]) <= 1e-4 * abs(eo[0])
    assert np.abs(eg - eo).max() <= 1e-6 * abs(eo[0])


# ------------------------------------------------------------------ NEXT-1: device-resident reuse steps
def _vel4(v):
    out = np.zeros((v.shape[0], 4), np.float32)
    out[:, :3] = v
    return out


def test_device_resident_reuse_run():
    """Config 5 at reduced N with the orbit integration on the device (paper section 7.3):
    lists built once, then 8 x mwf_step_reuse = kick-drift, monopole refresh, force over all groups, kick,
    with no host transfer in the step.  After every step the state is read back and compared with the
    oracle: the leapfrog update in fp64 from the previous fp32 state (within fp32 rounding of one FMA per
    component), and the forces on exactly the fp32 positions the device now holds (north_star tolerances)."""
    cfg = CONFIGS[4]
    w = make_workload(cfg, 30000)
    dt = cfg.dt
    f = binding.MultiWalkForce.for_workload(w, n_tag=2)
    f.upload_workload(w, binding.MAKE_LIST_FOR_REUSE)
    assert expect_code(f.step_reuse, dt) == binding.ESTATE          # no evaluation yet, no velocities
    lists0 = f.get_list_buffer()
    f.refresh_monopoles()
    f.dispatch(0, 0, w.n_group)
    out = np.zeros((w.n, 4), np.float32)
    f.retrieve(0, out)
    assert expect_code(f.kick, dt) == binding.ESTATE                # velocities missing
    f.set_velocities(_vel4(w.vel))
    x_prev, v_prev, a_prev = f.get_particles(0, w.n), f.get_velocities(0, w.n), out.copy()
    assert np.array_equal(x_prev, w.posm)
    for step in range(1, cfg.n_reuse + 1):
        f.step_reuse(dt)
        f.retrieve(0, out)                                          # waits for the step, copies acc + pot
        x_now, v_now = f.get_particles(0, w.n), f.get_velocities(0, w.n)
        # leapfrog parity
        x_or, vh_or = oracle.kick_drift(x_prev, v_prev, a_prev, dt)
        tol_x = 2.0 ** -23 * (np.abs(x_or) + dt * np.abs(vh_or)) + 1e-30
        assert np.all(np.abs(x_now[:, :3] - x_or) <= tol_x), "drift, step %d" % step
        assert np.array_equal(x_now[:, 3], w.posm[:, 3])            # masses untouched
        vh32 = _vel4(vh_or.astype(np.float32))
        v_or = oracle.kick(vh32, out, dt)
        tol_v = 2.0 ** -22 * (np.abs(v_or) + 0.5 * dt * np.abs(out[:, :3])) + 1e-30
        assert np.all(np.abs(v_now[:, :3] - v_or) <= tol_v), "kick, step %d" % step
        # force parity on the positions the device holds
        acc, pot, mom = oracle_eval(w, cfg.eps, posm=x_now)
        check(out, acc, pot, label="device-resident step %d" % step)
        spj = f.get_monopoles(w.n_cell)
        assert np.all(np.abs(spj[:, 3] - mom[:, 3]) <= 1e-6 * mom[:, 3])
        x_prev, v_prev, a_prev = x_now, v_now, out.copy()
    assert np.array_equal(lists0[0], f.get_list_buffer()[0]) and np.array_equal(lists0[1], f.get_list_buffer()[1])   # pin P9
    assert expect_code(f.kick_drift, float("nan")) == binding.EINVAL
    f.set_particles(w.posm)                                         # positions changed: forces are stale
    assert expect_code(f.kick_drift, dt) == binding.ESTATE
    f.close()


def test_device_resident_matches_host_driven_run():
    """The same 4 steps driven from the host in fp32 (upload positions each step) and on the device give
    bitwise identical forces when the host performs the identical fp32 FMAs: the device integrator adds
    nothing but the update itself."""
    cfg = CONFIGS[4]
    w = make_workload(cfg, 20000)
    dt = np.float32(cfg.dt)
    f = binding.MultiWalkForce.for_workload(w, n_tag=2)
    f.upload_workload(w, binding.MAKE_LIST_FOR_REUSE)
    f.refresh_monopoles()
    f.dispatch(0, 0, w.n_group)
    out = np.zeros((w.n, 4), np.float32)
    f.retrieve(0, out)
    f.set_velocities(_vel4(w.vel))
    for _ in range(4):
        f.step_reuse(float(dt))
    f.retrieve(0, out)
    x_dev = f.get_particles(0, w.n)
    g = binding.MultiWalkForce.for_workload(w, n_tag=2)
    g.upload_workload(w, binding.MAKE_LIST_FOR_REUSE)
    g.refresh_monopoles()
    g.dispatch(0, 0, w.n_group)
    ref = np.zeros((w.n, 4), np.float32)
    g.retrieve(0, ref)
    posm = w.posm.copy()
    v = w.vel.astype(np.float32)
    h = np.float32(0.5) * dt
    fma = lambda a, b, c: (a.astype(np.float64) * np.float64(b) + c.astype(np.float64)).astype(np.float32)  # exact product, one rounding
    for _ in range(4):
        v = fma(ref[:, :3], h, v)
        posm[:, :3] = fma(v, dt, posm[:, :3])
        g.begin_step(binding.REUSE_LIST)
        g.calc_force_all(posm, ref)
        v = fma(ref[:, :3], h, v)
    assert np.array_equal(x_dev, posm)
    assert np.array_equal(out, ref)
    f.close()
    g.close()
