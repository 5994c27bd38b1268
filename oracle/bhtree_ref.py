"""ORACLE -- TEST INFRASTRUCTURE ONLY.

Plain Python restatement of the construction step the paper describes (P:149 root cell;
P:153-156 Morton keys, sort, cells level by level; P:77 / P:87 one tree walk per group; P:181 index
lists; P:401 theta, n_leaf, n_grp), following readings O1-O4 / S6-S9 of DESIGN.md step by step.
Pure Python loops: small N only.  tests/test_workload.py uses it to pin the fast C++ builder in
paper_1907_02290_b200/workload (which it shares no code with).
"""
from __future__ import annotations

import math

import numpy as np

KEY_BITS = 21


def _key(ix: int, iy: int, iz: int) -> int:
    k = 0
    for b in range(KEY_BITS - 1, -1, -1):
        k = (k << 3) | (((ix >> b) & 1) << 2) | (((iy >> b) & 1) << 1) | ((iz >> b) & 1)
    return k


def build(posm: np.ndarray, n_leaf: int, n_grp: int, theta: float, h=None, skin: float = 0.0):
    """theta-lists (long range, O4).  With `h` (smoothing length per particle, caller's order): the short-range
    neighbour-search criterion instead (reading S24 of DESIGN.md): a cell is opened iff the gap between its
    cube and the group's particle box is <= max(R_g, R_c), R = 2 (1 + skin) x the largest h among the group's / the
    cell's particles; an opened leaf gives its particles as EPJ, anything else is dropped (no SPJ)."""
    pos = np.asarray(posm, dtype=np.float32)[:, :3].astype(np.float64)
    n = pos.shape[0]
    # O1 root cell
    lo, hi = pos.min(axis=0), pos.max(axis=0)
    centre = [0.5 * (lo[a] + hi[a]) for a in range(3)]
    ext = max(hi[a] - lo[a] for a in range(3))
    if not ext > 0:
        ext = 1.0
    side = ext * (1.0 + 1.0 / 1024.0)
    rlo = [centre[a] - 0.5 * side for a in range(3)]
    # O2 keys, stable sort
    keys = []
    for i in range(n):
        g = []
        for a in range(3):
            t = (pos[i, a] - rlo[a]) / side * float(1 << KEY_BITS)
            v = int(math.floor(t))
            g.append(min(max(v, 0), (1 << KEY_BITS) - 1))
        keys.append(_key(*g))
    perm = sorted(range(n), key=lambda i: (keys[i], i))
    skey = [keys[i] for i in perm]
    spos = pos[perm]
    # cells level by level
    cells = [[0, n, 0, 0]]
    geom = [[centre[0], centre[1], centre[2], side]]
    level = [0]
    begin = 0
    for lev in range(KEY_BITS):
        end = len(cells)
        shift = 3 * (KEY_BITS - 1 - lev)
        for c in range(begin, end):
            first, cnt = cells[c][0], cells[c][1]
            if cnt <= n_leaf:
                continue
            cx, cy, cz, s = geom[c]
            first_child, n_child = len(cells), 0
            for octant in range(8):
                members = [p for p in range(first, first + cnt) if ((skey[p] >> shift) & 7) == octant]
                if not members:
                    continue
                qs = 0.25 * s
                cells.append([members[0], len(members), 0, 0])
                geom.append([cx + qs if octant & 4 else cx - qs, cy + qs if octant & 2 else cy - qs,
                             cz + qs if octant & 1 else cz - qs, 0.5 * s])
                level.append(lev + 1)
                n_child += 1
            cells[c][2], cells[c][3] = first_child, n_child
        begin = end
        if len(cells) == end:
            break
    # O3 groups in Morton order
    groups = []

    def descend(c):
        first, cnt, fc, nc = cells[c]
        if cnt <= n_grp or nc == 0:
            groups.append(c)
        else:
            for k in range(nc):
                descend(fc + k)

    descend(0)
    if h is not None:
        hs = np.asarray(h, dtype=np.float32).astype(np.float64)[perm]
        reach = 2.0 * (1.0 + skin)
        epj, spj = [], []
        for gc in groups:
            first, cnt = cells[gc][0], cells[gc][1]
            blo = spos[first:first + cnt].min(axis=0)
            bhi = spos[first:first + cnt].max(axis=0)
            rg = reach * hs[first:first + cnt].max()
            e = []

            def search(c):
                cx, cy, cz, l = geom[c]
                rc = reach * hs[cells[c][0]:cells[c][0] + cells[c][1]].max()
                r = rg if rg > rc else rc
                d2 = 0.0
                for a, sc in enumerate((cx, cy, cz)):
                    d = 0.0
                    if sc + 0.5 * l < blo[a]:
                        d = blo[a] - (sc + 0.5 * l)
                    elif sc - 0.5 * l > bhi[a]:
                        d = (sc - 0.5 * l) - bhi[a]
                    d2 += d * d
                if d2 <= r * r:
                    if cells[c][3] == 0:
                        e.extend(range(cells[c][0], cells[c][0] + cells[c][1]))
                    else:
                        for k in range(cells[c][3]):
                            search(cells[c][2] + k)

            search(0)
            epj.append(e)
            spj.append([])
        return dict(perm=np.array(perm, np.int32), cells=np.array(cells, np.int32), geom=np.array(geom),
                    level=np.array(level, np.int32), groups=np.array(groups, np.int32), epj=epj, spj=spj,
                    root=np.array(centre + [side]))
    # O4 lists
    th2 = theta * theta
    epj, spj = [], []
    for gc in groups:
        first, cnt = cells[gc][0], cells[gc][1]
        blo = spos[first:first + cnt].min(axis=0)
        bhi = spos[first:first + cnt].max(axis=0)
        e, s_ = [], []

        def walk(c):
            cx, cy, cz, l = geom[c]
            d2 = 0.0
            for a, sc in enumerate((cx, cy, cz)):
                d = 0.0
                if sc < blo[a]:
                    d = blo[a] - sc
                elif sc > bhi[a]:
                    d = sc - bhi[a]
                d2 += d * d
            if l * l > th2 * d2:
                if cells[c][3] == 0:
                    e.extend(range(cells[c][0], cells[c][0] + cells[c][1]))
                else:
                    for k in range(cells[c][3]):
                        walk(cells[c][2] + k)
            else:
                s_.append(c)

        walk(0)
        epj.append(e)
        spj.append(s_)
    return dict(perm=np.array(perm, np.int32), cells=np.array(cells, np.int32), geom=np.array(geom),
                level=np.array(level, np.int32), groups=np.array(groups, np.int32), epj=epj, spj=spj,
                root=np.array(centre + [side]))
