"""Pins of the oracle's level-wide steps (S5-S10, P12): ghost fill, prolongation, restriction,
flux registers, refluxing and the subcycled advance.  CPU only."""
import numpy as np
import pytest

import oracle
from paper_0910_5547_b200 import workloads as wl

REGIONS = {
    "centre": [(i, j, k) for i in (1, 2) for j in (1, 2) for k in (1, 2)],
    # fine faces coincide with parent faces in x; periodic wrap of fine siblings in z
    "slab": [(i, j, k) for i in (2, 3) for j in (1, 2) for k in (0, 1, 2, 3)],
}


def two_level(region="centre", bc=(0,) * 6):
    return wl.build_hierarchy((2, 2, 2), [REGIONS[region]], bc)


def analytic_state(h, fn, gamma, nv=5):
    U = np.zeros((len(h["level"]), nv, 16, 16, 16))
    for p in range(len(h["level"])):
        x, y, z = wl.cell_centres(h, p)
        Z, Y, X = np.meshgrid(z, y, x, indexing="ij")
        rho, pr, v, B = fn(X, Y, Z)
        U[p] = wl.cons_from_prim(rho, pr, v, gamma, B=B)
    return U


def blast(X, Y, Z):
    r2 = (X - 0.5) ** 2 + (Y - 0.5) ** 2 + (Z - 0.5) ** 2
    rho = 1 + 0.3 * np.sin(2 * np.pi * X) * np.cos(2 * np.pi * Y)
    p = 1 + 20.0 * np.exp(-r2 / 0.01)
    v = (0.3 * np.sin(2 * np.pi * Z), 0.2 * np.cos(2 * np.pi * X), -0.25 + 0 * X)
    return rho, p, v, None


def blast_mhd(X, Y, Z):
    rho, p, v, _ = blast(X, Y, Z)
    return rho, p, v, (0.5 + 0 * X, 0.3 * np.sin(2 * np.pi * X), 0.2 * np.cos(2 * np.pi * Y))


def composite_total(h, U):
    """Sum over level-0 cells times cell volume (covered cells hold the restricted fine data)."""
    l0 = wl.level_patches(h, 0)
    return U[l0].sum(axis=(0, 2, 3, 4)) * h["dx0"] ** 3


# ---------------------------------------------------------------- S5: sibling copy and outflow
def test_sibling_fill_equals_numpy_wrap_pad():
    h = wl.uniform_hierarchy(2, periodic=True)
    rng = np.random.default_rng(1)
    G = rng.uniform(1, 2, (5, 32, 32, 32))
    o = oracle.Oracle(h, 1.4, 5)
    o.upload(0, wl.split_global(h, G))
    o.fill_ghosts(0, 0)
    P = o.download_padded(0)
    Gp = np.pad(G, ((0, 0), (2, 2), (2, 2), (2, 2)), mode="wrap")
    for p in range(8):
        ox, oy, oz = h["origin"][p]
        assert np.array_equal(P[p], Gp[:, oz:oz + 20, oy:oy + 20, ox:ox + 20])


def test_outflow_fill_equals_numpy_edge_pad():
    h = wl.uniform_hierarchy(2, periodic=False)
    rng = np.random.default_rng(2)
    G = rng.uniform(1, 2, (5, 32, 32, 32))
    o = oracle.Oracle(h, 1.4, 5)
    o.upload(0, wl.split_global(h, G))
    o.fill_ghosts(0, 0)
    P = o.download_padded(0)
    Gp = np.pad(G, ((0, 0), (2, 2), (2, 2), (2, 2)), mode="edge")
    for p in range(8):
        ox, oy, oz = h["origin"][p]
        assert np.array_equal(P[p], Gp[:, oz:oz + 20, oy:oy + 20, ox:ox + 20])


# ---------------------------------------------------------------- S6/S7: prolongation
def _fill_fine_from_coarse(h, Ucoarse_fn, alpha=0.0, Unew_fn=None):
    o = oracle.Oracle(h, 1.4, 5)
    U = analytic_state(h, Ucoarse_fn, 1.4)
    o.upload(0, U)
    o.upload(2, U if Unew_fn is None else U)
    if Unew_fn is not None:
        o.upload(0, analytic_state(h, Unew_fn, 1.4))
    o.fill_ghosts(0, 0)
    o.fill_ghosts(0, 2)
    o.fill_ghosts(1, 1, pold=2, pnew=0, alpha=alpha)  # fine slot 1 is empty: only CF ghosts get data
    return o


@pytest.mark.parametrize("region", ["centre", "slab"])
def test_prolongation_reproduces_linear_fields_exactly(region):
    bc = (1,) * 6  # outflow so that the linear field is not wrapped
    h = two_level(region, bc)
    lin = lambda X, Y, Z: (1 + 0.25 * X + 0.5 * Y + 0.125 * Z, 0.4 * (1 + 0.25 * X + 0.5 * Y + 0.125 * Z) * 0 + 0.4, (0 * X, 0 * X, 0 * X), None)
    o = _fill_fine_from_coarse(h, lin)
    P = o.download_padded(1)
    n_cf = 0
    for p in wl.level_patches(h, 1):
        if (h["nbr"][p] == -2).any():
            continue  # next to an outflow boundary the coarse slope is (rightly) limited to zero
        dx = h["dx0"] / 2
        c = [(h["origin"][p, d] + np.arange(-2, 18) + 0.5) * dx for d in range(3)]
        Z, Y, X = np.meshgrid(c[2], c[1], c[0], indexing="ij")
        want = 1 + 0.25 * X + 0.5 * Y + 0.125 * Z
        for r in range(27):
            if r == 13 or h["nbr"][p, r] != -1:
                continue
            off = (r % 3 - 1, (r // 3) % 3 - 1, r // 9 - 1)
            sl = tuple(slice(0, 2) if o_ < 0 else slice(2, 18) if o_ == 0 else slice(18, 20) for o_ in off[::-1])
            got = P[p, 0][sl]
            # linear data: both one-sided differences agree, minmod returns the slope, +-1/4 offsets exact
            assert np.allclose(got, want[sl], rtol=0, atol=4e-16), (p, r)
            n_cf += 1
    assert n_cf > 0


def test_prolongation_children_average_to_parent_and_limit():
    h = two_level("centre")
    rough = lambda X, Y, Z: (1 + 0.3 * np.sin(9 * X) * np.cos(7 * Y + 3 * Z), 1 + 0 * X, (0 * X, 0 * X, 0 * X), None)
    o = _fill_fine_from_coarse(h, rough)
    P1 = o.download_padded(1)
    P0 = o.download_padded(2)
    checked = 0
    for p in wl.level_patches(h, 1):
        Q = h["parent"][p]
        if h["nbr"][p, 12] != -1:
            continue
        # x-lo ghost layer: fine padded i = 0,1 <-> one coarse cell; j,k interior pairs
        oc = (h["origin"][p] - 2 * h["origin"][Q]) // 16
        ci = 2 + 8 * oc[0] - 1
        for ck in range(8):
            for cj in range(8):
                kids = P1[p, 0, 2 + 2 * ck:4 + 2 * ck, 2 + 2 * cj:4 + 2 * cj, 0:2]
                par = P0[Q, 0, 2 + 8 * oc[2] + ck, 2 + 8 * oc[1] + cj, ci]
                assert abs(kids.mean() - par) < 1e-15
                nb = P0[Q, 0, 1 + 8 * oc[2] + ck:4 + 8 * oc[2] + ck, 1 + 8 * oc[1] + cj:4 + 8 * oc[1] + cj, ci - 1:ci + 2]
                assert kids.min() >= nb.min() - 1e-15 and kids.max() <= nb.max() + 1e-15  # limited: no new extrema
                checked += 1
    assert checked > 0


def test_prolongation_time_interpolation_S7():
    h = two_level("centre")
    f0 = lambda X, Y, Z: (1 + 0 * X, 1 + 0 * X, (0 * X, 0 * X, 0 * X), None)
    f1 = lambda X, Y, Z: (3 + 0 * X, 1 + 0 * X, (0 * X, 0 * X, 0 * X), None)
    for alpha in (0.0, 0.5, 1.0):
        o = _fill_fine_from_coarse(h, f0, alpha=alpha, Unew_fn=f1)
        P = o.download_padded(1)
        p = wl.level_patches(h, 1)[0]
        r = [r for r in range(27) if h["nbr"][p, r] == -1][0]
        off = (r % 3 - 1, (r // 3) % 3 - 1, r // 9 - 1)
        sl = tuple(slice(0, 2) if o_ < 0 else slice(2, 18) if o_ == 0 else slice(18, 20) for o_ in off[::-1])
        assert np.all(P[p, 0][sl] == 1 + 2 * alpha)


# ---------------------------------------------------------------- S8: restriction
def test_restriction_is_the_2x2x2_mean():
    h = two_level("centre")
    rng = np.random.default_rng(4)
    U = rng.uniform(1, 2, (len(h["level"]), 5, 16, 16, 16))
    o = oracle.Oracle(h, 1.4, 5)
    o.upload(0, U)
    o.restrict(1)
    R = o.download(0)
    covered = np.zeros((8, 16, 16, 16), bool)
    for p in wl.level_patches(h, 1):
        Q = h["parent"][p]
        oc = (h["origin"][p] - 2 * h["origin"][Q]) // 16
        want = U[p].reshape(5, 8, 2, 8, 2, 8, 2).mean(axis=(2, 4, 6))
        sl = tuple(slice(8 * o_, 8 * o_ + 8) for o_ in oc[::-1])
        assert np.allclose(R[Q][(slice(None),) + sl], want, rtol=0, atol=2e-15)
        covered[(Q,) + sl] = True
    assert covered.sum() == 8 * 512
    for Q in range(8):  # uncovered cells untouched
        assert np.array_equal(R[Q][:, ~covered[Q]], U[Q][:, ~covered[Q]])
    assert np.array_equal(R[8:], U[8:])


# ---------------------------------------------------------------- P12: coarse-fine conservation
def manual_advance(o, h, lev, dt, a1, a2, reflux=True, w=0.5):
    """The S9 recursion written with the primitive calls (also documents the driver order)."""
    kids = lev + 1 < h["nlevels"]
    o.fill_ghosts(lev, 0, 2, 0, a1)
    if kids:
        o.copy_slot(lev, 0, 2)
    o.rk_stage(lev, 0, 0, 1, 0.0, 1.0, dt, w)
    o.fill_ghosts(lev, 1, 2, 0, a2)
    o.rk_stage(lev, 1, 0, 0, 0.5, 0.5, dt, w)
    if kids:
        o.fill_ghosts(lev, 0, 2, 0, a2)
        manual_advance(o, h, lev + 1, 0.5 * dt, 0.0, 0.5, reflux, w)
        manual_advance(o, h, lev + 1, 0.5 * dt, 0.5, 1.0, reflux, w)
        o.restrict(lev + 1)
        if reflux:
            o.reflux(lev)


@pytest.mark.parametrize("region,nv", [("centre", 5), ("slab", 5), ("centre", 8)])
def test_p12_composite_conservation_with_reflux(region, nv, ncpu):
    h = two_level(region)
    g = 1.4
    U = analytic_state(h, blast if nv == 5 else blast_mhd, g, nv)
    o = oracle.Oracle(h, g, nv, threads=ncpu)
    o.upload(0, U)
    o.restrict(1)
    U0 = o.download(0)
    tot0 = composite_total(h, U0)
    scale = np.abs(U0[:8]).sum(axis=(0, 2, 3, 4)) * h["dx0"] ** 3
    for _ in range(4):
        o.advance(0.3)
    R = o.download(0)
    assert np.isfinite(R).all()
    drift = (composite_total(h, R) - tot0) / scale
    assert np.abs(drift).max() < 5e-15, drift
    # the blast has reached the coarse-fine boundary: the correction was not trivially zero
    assert np.abs(R[:8] - U0[:8]).max() > 1e-3


def test_p12_negative_controls_detect_missing_reflux_and_wrong_weights(ncpu):
    h = two_level("centre")
    U = analytic_state(h, blast, 1.4)
    drifts = {}
    for name, kw in (("ok", {}), ("noreflux", dict(reflux=False)), ("w1", dict(w=1.0))):
        o = oracle.Oracle(h, 1.4, 5, threads=ncpu)
        o.upload(0, U)
        o.restrict(1)
        U0 = o.download(0)
        tot0 = composite_total(h, U0)
        for _ in range(3):
            manual_advance(o, h, 0, 2.0e-3, 0.0, 0.0, **kw)
        drifts[name] = np.abs((composite_total(h, o.download(0)) - tot0)[[0, 4]] / tot0[[0, 4]]).max()
    assert drifts["ok"] < 5e-15
    assert drifts["noreflux"] > 1e-7 and drifts["w1"] > 1e-7, drifts


def test_advance_equals_manual_sequence(ncpu):
    h = two_level("slab")
    U = analytic_state(h, blast, 1.4)
    a = oracle.Oracle(h, 1.4, 5, threads=ncpu); a.upload(0, U)
    b = oracle.Oracle(h, 1.4, 5, threads=1); b.upload(0, U)
    for _ in range(2):
        dt = a.advance(0.3)
        manual_advance(b, h, 0, dt, 0.0, 0.0)
    assert np.array_equal(a.download(0), b.download(0))  # threads do not change results either


def test_p12_uniform_state_bitwise_across_coarse_fine():
    h = wl.ball_hierarchy(2, 3, bc=(1,) * 6)
    one = lambda X, Y, Z: (1.3 + 0 * X, 0.7 + 0 * X, (0.3 + 0 * X, -0.2 + 0 * X, 0.9 + 0 * X), None)
    U = analytic_state(h, one, 1.4)
    o = oracle.Oracle(h, 1.4, 5)
    o.upload(0, U)
    for _ in range(2):
        o.advance(0.3)
    assert np.array_equal(o.download(0), U)


def test_two_level_smooth_wave_stays_second_order(ncpu):
    """P12 last clause: fine level over the middle of a smooth advected wave keeps order ~2."""
    errs = []
    for nb in (2, 4):
        fine = [(i, j, k) for i in range(nb, 3 * nb) for j in range(2) for k in range(2)]
        h = wl.build_hierarchy((nb * 2, 1, 1), [fine], (0,) * 6, box=1.0)
        wave = lambda X, Y, Z: (1 + 0.2 * np.sin(2 * np.pi * X), 1 + 0 * X, (1 + 0 * X, 0 * X, 0 * X), None)
        U = analytic_state(h, wave, 1.4)
        o = oracle.Oracle(h, 1.4, 5, threads=ncpu)
        o.upload(0, U)
        o.restrict(1)
        t = 0.0
        while t < 0.5 - 1e-12:
            dt = min(o.cfl_dt(1, 0, 0.4) * 2, 0.5 - t)
            o.advance(0.4, dt=dt)
            t += dt
        R = o.download(0)
        err, n = 0.0, 0
        for p in wl.level_patches(h, 0):
            x, _, _ = wl.cell_centres(h, p)
            err += np.abs(R[p, 0, 3, 5, :] - (1 + 0.2 * np.sin(2 * np.pi * (x - 0.5)))).sum()
            n += 16
        errs.append(err / n)
    assert np.log2(errs[0] / errs[1]) > 1.7, errs
