"""GPU parity of the regrid steps around the hot path (NEXT-3; S20, S21): the per-octant refinement
indicator and the interior prolongation of new fine patches, and one host-driven regrid cycle
(indicator on the device -> flags and descriptor table on the host -> new hierarchy -> data of the new
patches prolongated on the device -> subcycled steps), each against the oracle doing the same."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from paper_0910_5547_b200 import workloads as wl  # noqa: E402
from util import norm_err  # noqa: E402


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (no CPU fallback exists)")
    from paper_0910_5547_b200 import binding
    binding.load_library()
    return binding


def blob_state(h, nv=5, amp=5.0, w=0.12, seed=0, noise=0.01):
    """rho = 1 + amp exp(-r^2/w^2) plus seeded noise, at rest, p = 1, on every level of h."""
    rng = np.random.default_rng(seed)
    out = []
    for p in range(len(h["level"])):
        x, y, z = wl.cell_centres(h, p)
        Z, Y, X = np.meshgrid(z, y, x, indexing="ij")
        r2 = (X - 0.5) ** 2 + (Y - 0.5) ** 2 + (Z - 0.5) ** 2
        rho = 1 + amp * np.exp(-r2 / w ** 2) + noise * rng.standard_normal(r2.shape)
        one = np.ones_like(rho)
        B = (0.1 * one, 0.2 * one, 0 * one) if nv >= 8 else None
        out.append(wl.cons_from_prim(rho, one, (0.1 * one, 0 * one, -0.1 * one), 1.4, B=B))
    return np.stack(out)


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("periodic", [True, False])
@pytest.mark.parametrize("halo", [0, 1])
def test_refine_indicator_matches_oracle(gpu, dtype, periodic, halo):
    """halo = 1: fill_ghosts leaves the sibling ghosts of the finest level to rk_stage's direct reads; the
    indicator materialises them itself before it differentiates across patch borders."""
    import oracle
    h = wl.uniform_hierarchy(3, periodic=periodic)
    U = blob_state(h)
    if dtype == "f32":
        U = U.astype(np.float32).astype(np.float64)
    g = gpu.AmrHydro(h, 1.4, 5, dtype=dtype, halo=halo)
    o = oracle.Oracle(h, 1.4, 5)
    g.upload(0, U); o.upload(0, U)
    g.fill_ghosts(0, 0); o.fill_ghosts(0, 0)
    G, O = g.refine_indicator(0), o.refine_indicator(0)
    assert G.shape == O.shape == (27, 8) and O.max() > 1.0
    assert np.abs(G - O).max() <= (1e-13 if dtype == "f64" else 1e-13) * O.max()      # both differentiate the same stored rho in double
    assert np.array_equal(G > 0.1 * G.max(), O > 0.1 * O.max())                         # config 3's criterion: same flags
    U[5, 0, 3, 4, 5] = np.nan
    g.upload(0, U); g.fill_ghosts(0, 0)
    assert np.isnan(g.refine_indicator(0)[5]).any()


@pytest.mark.parametrize("halo", [0, 1])
def test_refine_indicator_on_the_finest_level_of_a_hierarchy(gpu, halo):
    """The same on the fine level of a two-level hierarchy (coarse-fine faces prolongated by fill_ghosts,
    sibling faces materialised by the indicator in direct-halo mode) and on its coarse level."""
    import oracle
    fine = [(i, j, k) for i in (2, 3) for j in (2, 3) for k in (2, 3)]
    h = wl.build_hierarchy((3, 3, 3), [fine], (0,) * 6)
    U = blob_state(h, w=0.2)
    g = gpu.AmrHydro(h, 1.4, 5, halo=halo)
    o = oracle.Oracle(h, 1.4, 5)
    g.upload(0, U); o.upload(0, U)
    for lev in (0, 1):
        g.fill_ghosts(lev, 0, 0, 0, 0.0); o.fill_ghosts(lev, 0, 0, 0, 0.0)
    for lev in (0, 1):
        G, O = g.refine_indicator(lev), o.refine_indicator(lev)
        assert G.shape == O.shape and O.max() > 0.5
        assert np.abs(G - O).max() <= 1e-13 * O.max()


@pytest.mark.parametrize("nv,dtype", [(5, "f64"), (8, "f64"), (5, "f32")])
def test_prolong_interior_matches_oracle(gpu, nv, dtype):
    import oracle
    h = wl.ball_hierarchy(2, 3, bc=(1,) * 6)
    U = blob_state(h, nv=nv, seed=3)
    if dtype == "f32":
        U = U.astype(np.float32).astype(np.float64)
    g = gpu.AmrHydro(h, 1.4, nv, dtype=dtype)
    o = oracle.Oracle(h, 1.4, nv)
    g.upload(0, U); o.upload(0, U)
    for lev in (0, 1):
        for x in (g, o):
            x.fill_ghosts(lev, 0, 0, 0, 0.0)
        for p in wl.level_patches(h, lev + 1):
            g.prolong_interior(int(p)); o.prolong_interior(int(p))
    G, O = g.download(0).astype(np.float64), o.download(0)
    assert not np.array_equal(O, U)
    assert norm_err(G, O).max() <= (4e-16 if dtype == "f64" else 1e-6)     # fp32: a few ulp over two nested prolongations
    with pytest.raises(gpu.AmrHydroError):
        g.prolong_interior(0)


def test_one_regrid_cycle_host_driven(gpu):
    """Level 0 only -> indicator (device) -> flagged octants + one octant of buffer (host) -> two-level
    hierarchy -> level-1 data prolongated (device) -> two subcycled coarse steps; oracle alongside."""
    import oracle
    nb = 3
    h0 = wl.uniform_hierarchy(nb, periodic=True)
    U0 = blob_state(h0, seed=5, noise=1e-3)
    g0 = gpu.AmrHydro(h0, 1.4, 5)
    g0.upload(0, U0); g0.fill_ghosts(0, 0)
    ind = g0.refine_indicator(0)
    flags = ind > 0.1 * ind.max()                                   # BASELINE config 3
    org = np.asarray(h0["origin"]) // 16
    marked = np.zeros((2 * nb,) * 3, bool)                          # [bx][by][bz] in level-1 patch units
    for p in range(len(org)):
        for oc in range(8):
            if flags[p, oc]:
                marked[2 * org[p][0] + (oc & 1), 2 * org[p][1] + ((oc >> 1) & 1), 2 * org[p][2] + (oc >> 2)] = True
    grown = marked.copy()                                           # one octant of buffer, periodic
    for ax in range(3):
        for s in (-1, 1):
            grown |= np.roll(marked, s, axis=ax)
    fine = [tuple(int(c) for c in b) for b in np.argwhere(grown)]
    assert 8 <= len(fine) < grown.size
    h1 = wl.build_hierarchy((nb,) * 3, [fine], (0,) * 6)
    n0 = len(h0["level"])
    U1 = np.zeros((len(h1["level"]), 5, 16, 16, 16))
    # level-0 patches keep their data (both hierarchies order level 0 the same way: checked)
    assert np.array_equal(np.asarray(h1["origin"])[:n0], np.asarray(h0["origin"]))
    U1[:n0] = U0
    g = gpu.AmrHydro(h1, 1.4, 5, halo=1)
    o = oracle.Oracle(h1, 1.4, 5, threads=8)
    g.upload(0, U1); o.upload(0, U1)
    for x in (g, o):
        x.fill_ghosts(0, 0)
        for p in wl.level_patches(h1, 1):
            x.prolong_interior(int(p))
    tot0 = o.download(0)[:n0].sum(axis=(0, 2, 3, 4))
    for x in (g, o):
        x.restrict(1)                                               # conservative prolongation: restriction gives level 0 back
    assert np.abs(o.download(0)[:n0].sum(axis=(0, 2, 3, 4)) - tot0).max() <= 1e-12 * np.abs(tot0).max()
    for _ in range(2):
        dt = o.advance(0.3)
        g.advance(0.3, dt)
    G, O = g.download(0), o.download(0)
    assert np.isfinite(G).all() and norm_err(G, O).max() <= 1e-12


# ------------------------------------------------------------------ amrhydro_regrid: the cycle on the live pool
def old_of_new(h_old, h_new):
    """Index in the old table of every patch of the new one (same level and origin), -1 for a new patch."""
    key = {(int(l), tuple(int(c) for c in o)): p for p, (l, o) in enumerate(zip(h_old["level"], h_old["origin"]))}
    return np.array([key.get((int(l), tuple(int(c) for c in o)), -1) for l, o in zip(h_new["level"], h_new["origin"])], np.int32)


def oracle_regrid(o_old, h_old, h_new, gamma, nv):
    """The same cycle with the oracle's primitives and a host copy: restrict, carry the survivors over, fill ghosts level
    by level, prolongate the new patches (S8, S21)."""
    import oracle
    for l in range(h_old["nlevels"] - 1, 0, -1):
        o_old.restrict(l)
    Uo = o_old.download(0)
    m = old_of_new(h_old, h_new)
    U = np.zeros((len(m), nv, 16, 16, 16))
    U[m >= 0] = Uo[m[m >= 0]]
    o = oracle.Oracle(h_new, gamma, nv, threads=8)
    o.upload(0, U)
    for l in range(h_new["nlevels"] - 1):
        o.fill_ghosts(l, 0, 0, 0, 0.0)
        for p in wl.level_patches(h_new, l + 1):
            if m[p] < 0:
                o.prolong_interior(int(p))
    return o, m


def test_regrid_one_level_to_two_on_the_live_pool(gpu):
    """test_one_regrid_cycle_host_driven with the new handle and the re-upload replaced by amrhydro_regrid."""
    import oracle
    nb = 3
    h0 = wl.uniform_hierarchy(nb, periodic=True)
    U0 = blob_state(h0, seed=5, noise=1e-3)
    g = gpu.AmrHydro(h0, 1.4, 5, halo=1, nslots=3, max_patches=400)
    o0 = oracle.Oracle(h0, 1.4, 5, threads=8)
    g.upload(0, U0); o0.upload(0, U0)
    g.fill_ghosts(0, 0)
    ind = g.refine_indicator(0)
    flags = ind > 0.1 * ind.max()
    org = np.asarray(h0["origin"]) // 16
    marked = np.zeros((2 * nb,) * 3, bool)
    for p in range(len(org)):
        for oc in range(8):
            if flags[p, oc]:
                marked[2 * org[p][0] + (oc & 1), 2 * org[p][1] + ((oc >> 1) & 1), 2 * org[p][2] + (oc >> 2)] = True
    fine = [tuple(int(c) for c in b) for b in np.argwhere(marked)]
    h1 = wl.build_hierarchy((nb,) * 3, [fine], (0,) * 6)
    o, m = oracle_regrid(o0, h0, h1, 1.4, 5)
    assert (m >= 0).sum() == len(h0["level"]) and (m < 0).sum() == len(fine)
    launches = g.get_counter(gpu.CNT_LAUNCHES, reset=True)
    g.regrid(h1, m)
    assert g.get_counter(gpu.CNT_LAUNCHES) <= 4            # move, ghost fill of level 0, ONE prolongation launch for all new patches
    G, O = g.download(0), o.download(0)
    assert norm_err(G, O).max() <= 4e-16
    for _ in range(2):
        dt = o.advance(0.3)
        assert abs(g.advance(0.3) - dt) <= 1e-12 * dt
    G, O = g.download(0), o.download(0)
    assert np.isfinite(G).all() and norm_err(G, O).max() <= 1e-12


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_regrid_moves_keeps_removes_and_creates(gpu, dtype):
    """Three levels -> three levels with other blocks: some patches survive at another index, some disappear (their
    parents keep the restricted data), some are new on levels 1 and 2 (a new level-2 patch under a new level-1 patch
    included).  One step before, two after, oracle alongside."""
    import oracle
    nb = 2
    A1 = [(i, j, k) for i in (1, 2) for j in (1, 2) for k in (1, 2)]
    A2 = [(i, j, k) for i in (3, 4) for j in (3, 4) for k in (3, 4)]
    B1 = [(i, j, k) for i in (1, 2, 3) for j in (1, 2) for k in (1, 2)]            # grown along x
    B2 = [(i, j, k) for i in (4, 5, 6) for j in (3, 4) for k in (3, 4)]            # shifted along x: (3,..) removed, (5,..),(6,..) new
    hA = wl.build_hierarchy((nb,) * 3, [A1, A2], (0,) * 6)
    hB = wl.build_hierarchy((nb,) * 3, [B1, B2], (0,) * 6)
    U = blob_state(hA, seed=11, w=0.25)
    if dtype == "f32":
        U = U.astype(np.float32).astype(np.float64)
    g = gpu.AmrHydro(hA, 1.4, 5, dtype=dtype, max_patches=len(hB["level"]) + 8)
    oA = oracle.Oracle(hA, 1.4, 5, threads=8)
    g.upload(0, U); oA.upload(0, U)
    for x in (g, oA):
        x.restrict(2); x.restrict(1)
    dt = oA.advance(0.3)
    g.advance(0.3, dt)
    oB, m = oracle_regrid(oA, hA, hB, 1.4, 5)
    moved = [(int(a), q) for q, a in enumerate(m) if a >= 0 and a != q]
    assert moved and (m < 0).sum() >= 8 and len(set(range(len(hA["level"]))) - set(m.tolist())) >= 4
    g.regrid(hB, m)
    tol = 1e-12 if dtype == "f64" else 1e-5
    # (the state carries the round-off of the step before the regrid: rho v_y is ~0 in this blob, its norm is tiny)
    assert norm_err(g.download(0).astype(np.float64), oB.download(0), vector=(dtype == "f32")).max() <= tol
    for _ in range(2):
        dt = oB.advance(0.3)
        g.advance(0.3, dt)
    G, O = g.download(0).astype(np.float64), oB.download(0)
    assert np.isfinite(G).all() and norm_err(G, O, vector=(dtype == "f32")).max() <= tol


def test_regrid_rejects_bad_maps(gpu):
    h0 = wl.uniform_hierarchy(2, periodic=True)
    fine = [(i, j, k) for i in (1, 2) for j in (1, 2) for k in (1, 2)]
    h1 = wl.build_hierarchy((2, 2, 2), [fine], (0,) * 6)
    g = gpu.AmrHydro(h0, 1.4, 5, nslots=3, max_patches=32)
    U0 = blob_state(h0, seed=2)
    g.upload(0, U0)
    m = old_of_new(h0, h1)
    bad = m.copy(); bad[1] = bad[0]
    with pytest.raises(gpu.AmrHydroError):
        g.regrid(h1, bad)                                   # a patch named twice
    bad = m.copy(); bad[0] = -1
    with pytest.raises(gpu.AmrHydroError):
        g.regrid(h1, bad)                                   # a new level-0 patch has no parent
    bad = m.copy(); bad[0], bad[1] = m[1], m[0]
    with pytest.raises(gpu.AmrHydroError):
        g.regrid(h1, bad)                                   # a survivor must keep its origin
    assert np.array_equal(g.download(0), U0)               # nothing happened
    small = gpu.AmrHydro(h0, 1.4, 5, nslots=3)
    with pytest.raises(gpu.AmrHydroError):
        small.regrid(h1, m)                                 # the pool is too small
    g.regrid(h1, m)
    assert g.npatch == 16
