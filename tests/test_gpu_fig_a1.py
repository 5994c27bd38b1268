"""The paper's appendix-A experiment as a performance-shape test (Fig. A.1 and eq. A.1):
"the elapsed times are independent of theta (i.e. independent of <n_list>) and depend on <n_i>.  For small <n_i>, the time
decreases as <n_i> increases ... For large <n_i>, the elapsed times are almost constant".  Force-kernel time per interaction
(CUDA events of the library, median of 7 launches) at N = 2^18 against the group size for theta = 1, 0.5, 0.3, lists built on
the device.  What this kernel shows, and what is asserted (measured values in profiles/r03_fig_a1_sweep.md):
  - falling with <n_i>, then flat: asserted for every theta (3 % slack for timing noise; n_grp = 2048 within 10 % of 512);
  - independent of theta: within 10 % between theta = 0.5 and 0.3 from n_grp = 64 on (measured 2-5 %), and within 12 % over
    all three from n_grp = 512 on (measured 5-7 %).  theta = 1 with small groups is NOT on the common curve: its lists are
    under 16 tiles long, so the per-item prologue and epilogue weigh 14 % (n_grp = 256) to 35 % (n_grp = 64) -- the paper's
    GPU model has no such term; this one needs it, and the test says so instead of hiding it."""
import numpy as np
import pytest

from paper_1907_02290_b200 import binding
from paper_1907_02290_b200.workload import CONFIGS, make_particles

pytestmark = pytest.mark.gpu

N = 1 << 18
GROUPS = (32, 64, 128, 256, 512, 1024, 2048)


def test_time_per_interaction_against_group_size_and_theta():
    cfg = CONFIGS[4]
    posm, _ = make_particles(cfg, N)
    f = binding.MultiWalkForce(cfg.eps, 1.0, max_ptcl=N, max_cell=N, max_group=N, max_entry=700 * N, n_tag=2)
    ps, n_i = {}, {}
    for theta in (1.0, 0.5, 0.3):
        for n_grp in GROUPS:
            if theta < 0.4 and n_grp < 64:
                continue                                   # lists beyond the 700 entries per particle this ctx holds
            f.begin_step(binding.MAKE_LIST_FOR_REUSE)
            f.set_particles(posm)
            f.build(N, cfg.n_leaf, n_grp, theta, binding.MAKE_LIST_FOR_REUSE)
            sz = f.get_build_sizes()
            f.refresh_monopoles()
            c0 = f.get_counters()["interactions"]
            ms = []
            for it in range(3 + 7):
                f.dispatch(0, 0, sz["n_group"])
                f.retrieve(0, None)
                if it >= 3:
                    ms.append(f.last_dispatch_ms(0))
            inter = (f.get_counters()["interactions"] - c0) // 10
            ps[theta, n_grp] = 1e9 * float(np.median(ms)) / inter
            n_i[theta, n_grp] = N / sz["n_group"]
    f.close()
    for theta in (1.0, 0.5, 0.3):
        gs = [g for g in GROUPS if (theta, g) in ps]
        print("theta %.1f: " % theta + "  ".join("<n_i> %.0f: %.3f ps" % (n_i[theta, g], ps[theta, g]) for g in gs))
        for a, b in zip(gs, gs[1:]):                       # falls with <n_i> ...
            assert n_i[theta, b] > n_i[theta, a]
            assert ps[theta, b] <= 1.03 * ps[theta, a], (theta, a, b)
        assert ps[theta, 2048] >= 0.90 * ps[theta, 512]    # ... and then is flat
    for g in GROUPS:
        if g >= 64:
            assert abs(ps[0.5, g] / ps[0.3, g] - 1.0) <= 0.10, g
        if g >= 512:
            v = [ps[t, g] for t in (1.0, 0.5, 0.3)]
            assert max(v) / min(v) - 1.0 <= 0.12, g
    assert ps[1.0, 64] > ps[0.5, 64] > 0.0                 # the short lists of theta = 1 pay the per-item overhead
