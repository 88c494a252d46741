"""Pins P18-P19 of the CPU oracle for the regrid steps around the hot path (NEXT-3, readings S20-S21):
the refinement indicator |grad rho|/rho of BASELINE.json config 3 and the interior prolongation of a
new fine patch.  CPU only."""
import numpy as np
import pytest

import oracle
from paper_0910_5547_b200 import workloads as wl


def centre_hier():
    fine = [(i, j, k) for i in (1, 2) for j in (1, 2) for k in (1, 2)]
    return wl.build_hierarchy((2, 2, 2), [fine], (0,) * 6)


# ---------------------------------------------------------------- P18: indicator against its closed form
@pytest.mark.parametrize("axis", [0, 1, 2])
def test_p18_indicator_closed_form(axis):
    """rho = 2 + sin(2 pi s): the centred difference is cos(2 pi s) sin(2 pi dx)/dx exactly."""
    nb = 2
    n = 16 * nb
    h = wl.uniform_hierarchy(nb, periodic=True, order="linear")
    grids = wl._grid(n)                                    # Z, Y, X cell centres
    s = grids[2 - axis]
    rho = 2 + np.sin(2 * np.pi * s)
    one = np.ones_like(rho)
    G = wl.cons_from_prim(rho, one, (0 * one, 0 * one, 0 * one), 1.4)
    o = oracle.Oracle(h, 1.4, 5)
    o.upload(0, wl.split_global(h, G))
    o.fill_ghosts(0, 0)
    ind = o.refine_indicator(0)
    dx = 1.0 / n
    g = np.abs(np.cos(2 * np.pi * s)) * np.sin(2 * np.pi * dx) / dx / rho
    org = np.asarray(h["origin"])
    for p in range(len(org)):
        ox, oy, oz = org[p]
        for oc in range(8):
            x0, y0, z0 = ox + 8 * (oc & 1), oy + 8 * ((oc >> 1) & 1), oz + 8 * (oc >> 2)
            want = g[z0:z0 + 8, y0:y0 + 8, x0:x0 + 8].max()
            assert abs(ind[p, oc] - want) <= 1e-12 * want, (p, oc)


def test_p18_flags_follow_the_shell_of_a_blob():
    """Gaussian blob: |grad rho|/rho = 2 r / w^2 / (1 + 1/amp e^{...}) peaks on a shell; with the 0.1 max
    threshold of config 3 the octants at the centre of the blob and far outside it stay unflagged."""
    nb = 4
    n = 16 * nb
    h = wl.uniform_hierarchy(nb, periodic=True, order="linear")
    Z, Y, X = wl._grid(n)
    r2 = (X - 0.5) ** 2 + (Y - 0.5) ** 2 + (Z - 0.5) ** 2
    rho = 1 + 5 * np.exp(-r2 / 0.12 ** 2)
    one = np.ones_like(rho)
    o = oracle.Oracle(h, 1.4, 5)
    o.upload(0, wl.split_global(h, wl.cons_from_prim(rho, one, (0 * one, 0 * one, 0 * one), 1.4)))
    o.fill_ghosts(0, 0)
    ind = o.refine_indicator(0)
    flags = ind > 0.1 * ind.max()
    org = np.asarray(h["origin"])
    corner = int(np.where((org == 0).all(axis=1))[0][0])
    assert not flags[corner].any()                          # far field: gradient ~ 0
    assert flags.sum() >= 8 and flags.sum() < flags.size // 2
    # the analytic maximum of 2 r amp e / (w^2 (1 + amp e)) bounds the discrete one from above (centred differences smooth)
    r = np.sqrt(r2); e = np.exp(-r2 / 0.12 ** 2)
    assert ind.max() <= (2 * r / 0.12 ** 2 * 5 * e / (1 + 5 * e)).max() * 1.001


# ---------------------------------------------------------------- P19: interior prolongation
def test_p19_prolongation_is_conservative_exact_on_linear_data_and_monotone():
    h = centre_hier()
    lev = np.asarray(h["level"])
    fine = np.where(lev == 1)[0]
    rng = np.random.default_rng(7)
    n = len(lev)
    U = rng.uniform(0.5, 1.5, (n, 5, 16, 16, 16))
    # coarse level: a linear field with dyadic coefficients in variable 0, random data in the others
    Z, Y, X = np.meshgrid(np.arange(32), np.arange(32), np.arange(32), indexing="ij")
    lin = 3.0 + 0.5 * X - 0.25 * Y + 0.125 * Z
    G = wl.join_global(h, U[lev == 0])
    G[0] = lin
    U[lev == 0] = wl.split_global(h, G)
    o = oracle.Oracle(h, 1.4, 5)
    o.upload(0, U)
    o.fill_ghosts(0, 0)
    for p in fine:
        o.prolong_interior(int(p))
    R = o.download(0)
    Gc = wl.join_global(h, R[lev == 0])
    org = np.asarray(h["origin"])
    for p in fine:
        ox, oy, oz = org[p] // 2                              # coarse cell index of the patch corner
        C = Gc[:, oz:oz + 8, oy:oy + 8, ox:ox + 8]
        F = R[p]
        kids = F.reshape(5, 8, 2, 8, 2, 8, 2)
        assert np.abs(kids.mean(axis=(2, 4, 6)) - C).max() <= 4e-16 * 1.5      # conservative
        fz, fy, fx = np.meshgrid(np.arange(16), np.arange(16), np.arange(16), indexing="ij")
        cc = lambda o, f: (o + f + 0.5) / 2 - 0.5             # fine cell centre in coarse index units
        exact = 3.0 + 0.5 * cc(org[p][0], fx) - 0.25 * cc(org[p][1], fy) + 0.125 * cc(org[p][2], fz)
        assert np.array_equal(F[0], exact)                                       # linear data: exact
        # monotone: every child lies between the extremes of the parent cell and its six face neighbours
        Gp = np.pad(Gc[1:], ((0, 0), (1, 1), (1, 1), (1, 1)), mode="wrap")
        sl = lambda a, d: Gp[:, 1 + oz + a[0]:1 + oz + 8 + a[0], 1 + oy + a[1]:1 + oy + 8 + a[1], 1 + ox + a[2]:1 + ox + 8 + a[2]]
        nbrs = np.stack([sl(a, 0) for a in ((0, 0, 0), (1, 0, 0), (-1, 0, 0), (0, 1, 0), (0, -1, 0), (0, 0, 1), (0, 0, -1))])
        lo, hi = nbrs.min(axis=0), nbrs.max(axis=0)
        k = kids[1:]
        up = lambda a: np.broadcast_to(a[:, :, None, :, None, :, None], k.shape)
        assert (k >= up(lo) - 1e-15).all() and (k <= up(hi) + 1e-15).all()
    with pytest.raises(ValueError):
        o.prolong_interior(0)                                  # a level-0 patch has no parent


# ---------------------------------------------------------------- S16: config 3's hierarchy by its own criterion
def test_cfg3_blocks_golden_is_what_the_script_writes(tmp_path, monkeypatch):
    """tests/golden/cfg3_blocks.txt is reproduced from the oracle alone by the committed script, is properly
    nested (build_hierarchy checks it), holds the deposit on its finest level and has the counts DESIGN.md states."""
    import importlib.util
    import os
    gold = os.path.join(os.path.dirname(__file__), "golden")
    spec = importlib.util.spec_from_file_location("make_cfg3_hierarchy", os.path.join(gold, "make_cfg3_hierarchy.py"))
    m = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(m)
    monkeypatch.setattr(m, "HERE", str(tmp_path))
    m.main()
    body = lambda p: [ln for ln in open(p).read().splitlines() if ln and not ln.startswith("#")]
    assert body(os.path.join(str(tmp_path), "cfg3_blocks.txt")) == body(os.path.join(gold, "cfg3_blocks.txt"))
    h = wl.blocks_hierarchy(os.path.join(gold, "cfg3_blocks.txt"), 4)
    assert [int((h["level"] == l).sum()) for l in range(5)] == [64, 64, 160, 432, 1880]
    U = wl.sedov_hierarchy_state(h)
    l4 = wl.level_patches(h, 4)
    dx4 = h["dx0"] / 16
    assert abs((U[l4, 4] - 1e-5 / 0.4).sum() * dx4 ** 3 - 1.0) <= 1e-12        # E = 1 on the finest level
