#!/usr/bin/env python
"""Writes tests/golden/cfg3_blocks.txt: the fixed AMR hierarchy of BASELINE.json configs[2] built by the
configuration's own criterion ("16^3 patches placed where |grad rho|/rho exceeds 0.1 max"), reading S16 of
SURVEY.md section 8(c) / DESIGN.md section 3.  It calls only oracle/ (the method's arithmetic) and
paper_0910_5547_b200/workloads.py (descriptor-table bookkeeping and the seeded initial state); nothing
here comes from the CUDA path.

Procedure (S16; the criterion is degenerate at t = 0 where rho == 1):
  1. level 0 alone (64^3 = 4^3 patches, outflow), Sedov deposit volume-averaged onto level 0, is advanced
     K = 20 steps by the oracle at CFL 0.3;
  2. per level l = 0 .. 3: ghost fill, per-octant indicator max |grad rho|/rho (S20), octants above
     0.1 x the level's maximum are flagged, every flagged octant and its 26 neighbours become 16^3 patches of
     level l + 1 (clipped to the domain and to octants of existing level-l patches), their interiors are
     prolongated from the parents (S21) and the loop continues on the prolonged field;
  3. the octants that hold the energy deposit (the 32 finest cells at the box centre) are flagged on
     every level, because north_star places the deposit on the finest level;
  4. a level that comes out empty falls back to the nested ball of workloads.ball_hierarchy.
Output: one line "level bx by bz" per patch of levels 1-4 (block coordinates in units of 16 cells of that
level), preceded by comment lines with the recipe and the per-level counts.

  python tests/golden/make_cfg3_hierarchy.py            # rewrites cfg3_blocks.txt
"""
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)

import oracle  # noqa: E402
from paper_0910_5547_b200 import workloads as wl  # noqa: E402

NB, NLEV, K, CFL, GAMMA, FRAC = 4, 5, 20, 0.3, 1.4, 0.1
BC = (1,) * 6


def flagged_blocks(h, ind, l):
    """Octants of level-l patches with indicator > FRAC * max -> set of level-(l+1) block coordinates."""
    ps = wl.level_patches(h, l)
    thr = FRAC * ind.max()
    out = set()
    for n, p in enumerate(ps):
        b = h["blocks"][p]
        for oc in range(8):
            if ind[n, oc] > thr:
                out.add((2 * int(b[0]) + (oc & 1), 2 * int(b[1]) + ((oc >> 1) & 1), 2 * int(b[2]) + (oc >> 2)))
    return out


def grow(blocks, ext, parents):
    """Every block and its 26 neighbours, clipped to the domain [0, ext)^3 and to octants of existing parents."""
    out = set()
    for b in blocks:
        for dz in (-1, 0, 1):
            for dy in (-1, 0, 1):
                for dx in (-1, 0, 1):
                    q = (b[0] + dx, b[1] + dy, b[2] + dz)
                    if all(0 <= c < ext for c in q) and (parents is None or tuple(c >> 1 for c in q) in parents):
                        out.add(q)
    return out


def main():
    threads = os.cpu_count() or 1
    # the t = 0 state of level 0: volume average of the finest-level deposit (workloads.sedov_hierarchy_state
    # computes every level directly from the deposit, so any 5-level hierarchy over the centre serves)
    hb = wl.ball_hierarchy(NB, NLEV, bc=BC)
    U0 = wl.sedov_hierarchy_state(hb, gamma=GAMMA)[: NB ** 3]
    h = wl.uniform_hierarchy(NB, periodic=False)
    assert np.array_equal(h["origin"], hb["origin"][: NB ** 3])
    o = oracle.Oracle(h, GAMMA, 5, threads=threads)
    o.upload(0, U0)
    for _ in range(K):
        o.advance(CFL)
    state = o.download(0)                       # evolved level 0
    refined, notes = [], []
    for l in range(NLEV - 1):
        o.fill_ghosts(l, 0, 0, 0, 0.0)
        ind = o.refine_indicator(l)
        ext = NB << (l + 1)
        centre = {(ext // 2 - a, ext // 2 - b, ext // 2 - c) for a in (0, 1) for b in (0, 1) for c in (0, 1)}
        flags = flagged_blocks(h, ind, l)
        parents = None if l == 0 else set(tuple(int(c) for c in b) for b in h["blocks"][wl.level_patches(h, l)])
        if not flags:
            notes.append("level %d: no octant flagged, nested-ball fall-back" % (l + 1))
            blocks = set(tuple(int(c) for c in b) for b in hb["blocks"][wl.level_patches(hb, l + 1)])
        else:
            blocks = grow(flags | centre, ext, parents)
        notes.append("level %d: indicator max %.6g, %d octants flagged (+%d for the deposit), %d patches after growth"
                     % (l + 1, ind.max(), len(flags), len(centre - flags), len(blocks)))
        refined.append(sorted(blocks))
        h = wl.build_hierarchy((NB,) * 3, refined, BC)
        # the field on the new hierarchy: coarser levels keep their data, the new level is prolongated (S21)
        n_old = state.shape[0]
        U = np.zeros((len(h["level"]), 5, 16, 16, 16))
        U[:n_old] = state
        o = oracle.Oracle(h, GAMMA, 5, threads=threads)
        o.upload(0, U)
        for ll in range(l + 1):
            o.fill_ghosts(ll, 0, 0, 0, 0.0)
        for p in wl.level_patches(h, l + 1):
            o.prolong_interior(int(p))
        state = o.download(0)
    path = os.path.join(HERE, "cfg3_blocks.txt")
    with open(path, "w") as f:
        f.write("# config 3 (BASELINE.json configs[2]) hierarchy by its own criterion, reading S16; written by\n")
        f.write("# tests/golden/make_cfg3_hierarchy.py (oracle only): level 0 = %d^3 patches advanced %d steps at CFL %g,\n" % (NB, K, CFL))
        f.write("# octants with max |grad rho|/rho > %g x level max flagged, grown by 26 neighbours, next level prolongated.\n" % FRAC)
        for s in notes:
            f.write("# " + s + "\n")
        f.write("# columns: level bx by bz (block = 16^3 cells of that level)\n")
        for l, blocks in enumerate(refined):
            for b in blocks:
                f.write("%d %d %d %d\n" % (l + 1, b[0], b[1], b[2]))
    print("\n".join(notes))
    print("wrote", path, "patches per level:", [NB ** 3] + [len(b) for b in refined])


if __name__ == "__main__":
    main()
