"""Pins P1-P11 of the CPU oracle: the oracle is checked against what the
paper and the mathematics fix, never against itself or the CUDA path.  CPU only."""
import itertools
import os

import numpy as np
import pytest

import oracle
from paper_0910_5547_b200 import workloads as wl
from util import exact_sod, norm_err, run_to, slab_hierarchy

GOLD = os.path.join(os.path.dirname(__file__), "golden")


# ------------------------------------------------------------------ P1: worked face
def _read_p1():
    cells, rows = [], {}
    for line in open(os.path.join(GOLD, "p1_face.txt")):
        if line.startswith("#") or not line.strip():
            continue
        tok = line.split()
        if tok[0] == "cell":
            cells.append([float(x) for x in tok[1:]])
        else:
            rows[tok[0]] = [float(x) for x in tok[1:]]
    return np.array(cells), rows


def test_p1_worked_face_golden():
    cells, rows = _read_p1()
    WL, WR, lam, F = oracle.face(5, 1.4, 1.5, 0, *cells)
    g = rows["theta1.5"]
    assert np.allclose(WL, g[0:5], rtol=0, atol=1e-15)
    assert np.allclose(WR, g[5:10], rtol=0, atol=1e-15)
    assert abs(lam - g[10]) < 1e-14
    assert np.allclose(F, g[11:16], rtol=1e-13, atol=1e-15)
    for th in ("1.0", "2.0"):
        _, _, lam, F = oracle.face(5, 1.4, float(th), 0, *cells)
        assert abs(lam - rows["theta" + th][0]) < 1e-14
        assert abs(F[0] - rows["theta" + th][1]) < 1e-14


def test_p1_states_by_hand():
    # Eq. 9 with G1, rho: 0.9 + 0.5*minmod(1.5*(-0.1), 1.5*(-0.2), 0.5*(-0.3)) = 0.9 - 0.075
    # Eq. 10 with G1, rho: 0.7 + 0.5*minmod(1.5*(0.05), 1.5*(0.2), 0.5*(0.25)) = 0.7 + 0.0375
    cells, _ = _read_p1()
    WL, WR, lam, F = oracle.face(5, 1.4, 1.5, 0, *cells)
    assert abs(WL[0] - 0.825) < 1e-15 and abs(WR[0] - 0.7375) < 1e-15
    # lambda0 = max(|v|+c) with c = sqrt(gamma (gamma-1) e)   (S2)
    c = lambda e: (1.4 * 0.4 * e) ** 0.5
    assert abs(lam - max(0.175 + c(2.325), 0.2625 + c(2.075))) < 1e-14
    # mass flux by hand: 0.5 (rhoL vL + rhoR vR - lam (rhoR - rhoL))
    f0 = 0.5 * (0.825 * 0.175 + 0.7375 * 0.2625 - lam * (0.7375 - 0.825))
    assert abs(F[0] - f0) < 1e-15


# ------------------------------------------------------------------ Eq. 11 brute force
def test_minmod_equals_casewise_definition():
    vals = [-3.0, -1.5, -0.25, 0.0, 0.25, 1.0, 2.5]
    for a, b, c in itertools.product(vals, repeat=3):
        if a > 0 and b > 0 and c > 0:
            want = min(a, b, c)
        elif a < 0 and b < 0 and c < 0:
            want = max(a, b, c)
        else:
            want = 0.0
        got = oracle.minmod(a, b, c)
        assert got == want, (a, b, c, got, want)
        assert oracle.minmod(-a, -b, -c) == -got  # odd


# ------------------------------------------------------------------ P2: linear data exact (G1)
@pytest.mark.parametrize("theta", [1.0, 1.5, 2.0])
def test_p2_linear_reconstruction_exact(theta):
    q = np.array([1.0, 2.0, 3.0, 4.0])
    cells = [np.array([x, 2.0 + 0.25 * x, 0.5 * x, -0.125 * x, 0.0625 * x]) for x in q]
    WL, WR, _, _ = oracle.face(5, 1.4, theta, 0, *cells)
    face = 2.5
    want = np.array([face, 2.0 + 0.25 * face, 0.5 * face, -0.125 * face, 0.0625 * face])
    assert np.array_equal(WL, want) and np.array_equal(WR, want)


def test_extremum_is_clipped():
    cells = [np.array([x, 1.0, 0, 0, 0]) for x in (1.0, 2.0, 1.0, 2.0)]
    WL, WR, _, _ = oracle.face(5, 1.4, 1.5, 0, *cells)
    assert WL[0] == 2.0 and WR[0] == 1.0  # both cells are extrema -> zero slope


# ------------------------------------------------------------------ P8: special cases
def _rand_state(rng, nv):
    W = np.empty(nv)
    W[0] = rng.uniform(0.2, 2.0); W[1] = rng.uniform(0.5, 3.0)
    W[2:5] = rng.uniform(-1, 1, 3)
    if nv == 8:
        W[5:8] = rng.uniform(-1, 1, 3)
    return W


@pytest.mark.parametrize("nv", [5, 8])
def test_p8_eq12_is_textbook_hll_with_symmetric_speeds(nv):
    rng = np.random.default_rng(7)
    for d in range(3):
        cells = [_rand_state(rng, nv) for _ in range(4)]
        WL, WR, lam, F = oracle.face(nv, 1.4, 1.5, d, *cells)
        UL, FL, _ = oracle.flux(nv, 1.4, d, WL)
        UR, FR, _ = oracle.flux(nv, 1.4, d, WR)
        SL, SR = -lam, lam
        hll = (SR * FL - SL * FR + SL * SR * (UR - UL)) / (SR - SL)  # Harten-Lax-van Leer
        assert np.allclose(F, hll, rtol=1e-13, atol=1e-14)


def test_p8_theta0_first_order_rusanov_by_hand():
    """theta=0 => zero slopes => first-order scheme; one cell update computed here from the
    textbook Rusanov flux of 1-D gas dynamics, written independently in numpy."""
    g = 1.4
    h, _ = slab_hierarchy(1, 0, periodic=True)
    rng = np.random.default_rng(3)
    rho = rng.uniform(0.5, 1.5, 16); p = rng.uniform(0.5, 1.5, 16); u = rng.uniform(-0.5, 0.5, 16)
    shape = (16, 16, 16)
    z = np.zeros(shape)
    U0 = wl.cons_from_prim(np.broadcast_to(rho, shape), np.broadcast_to(p, shape),
                           (np.broadcast_to(u, shape), z, z), g)[None]
    o = oracle.Oracle(h, g, 5, theta=0.0)
    o.upload(0, U0)
    dt, dx = 0.01, 1.0 / 16
    o.fill_ghosts(0, 0)
    o.rk_stage(0, 0, 0, 1, 0.0, 1.0, dt)
    U1 = o.download(1)[0][:, 3, 5, :]

    def F(r, uu, pp):
        E = pp / (g - 1) + 0.5 * r * uu * uu
        return np.array([r * uu, r * uu * uu + pp, (E + pp) * uu]), np.array([r, r * uu, E])

    def rus(i, j):  # face between cells i and j=i+1 (periodic)
        fl, ul = F(rho[i], u[i], p[i]); fr, ur = F(rho[j], u[j], p[j])
        lam = max(abs(u[i]) + np.sqrt(g * p[i] / rho[i]), abs(u[j]) + np.sqrt(g * p[j] / rho[j]))
        return 0.5 * (fl + fr - lam * (ur - ul))

    for i in (0, 7, 15):
        fm, fp = rus((i - 1) % 16, i), rus(i, (i + 1) % 16)
        _, u0 = F(rho[i], u[i], p[i])
        want = u0 - dt / dx * (fp - fm)
        got = U1[[0, 1, 4], i]
        assert np.allclose(got, want, rtol=1e-13, atol=1e-15)


# ------------------------------------------------------------------ flux / speed closed forms
def test_euler_flux_and_sound_speed_closed_form():
    W = np.array([2.0, 1.25, 0.5, -0.25, 0.125])      # rho e vx vy vz, gamma = 1.4
    p = 0.4 * 2.0 * 1.25                               # Eq. 6 = 1.0
    for d in range(3):
        U, F, c = oracle.flux(5, 1.4, d, W)
        vd = W[2 + d]
        E = 2.0 * (0.5 * (0.25 + 0.0625 + 0.015625) + 1.25)
        want = np.array([2.0 * vd, 2.0 * 0.5 * vd, 2.0 * -0.25 * vd, 2.0 * 0.125 * vd, (E + p) * vd])
        want[1 + d] += p
        assert np.allclose(F, want, rtol=1e-15)
        assert np.allclose(U, [2.0, 1.0, -0.5, 0.25, E], rtol=1e-15)
        assert abs(c - np.sqrt(1.4 * p / 2.0)) < 1e-15


def test_mhd_fast_speed_special_cases():
    g = 5.0 / 3.0
    rho, e = 1.5, 0.9
    a2 = g * (g - 1) * e
    # B parallel to d: c_f = max(a, b);  B perpendicular to d: c_f = sqrt(a^2 + b^2)
    for Bmag in (0.3, 2.0):
        W = np.array([rho, e, 0, 0, 0, Bmag, 0.0, 0.0])
        b2 = Bmag ** 2 / rho
        assert abs(oracle.flux(8, g, 0, W)[2] - np.sqrt(max(a2, b2))) < 1e-14
        assert abs(oracle.flux(8, g, 1, W)[2] - np.sqrt(a2 + b2)) < 1e-14
        assert abs(oracle.flux(8, g, 2, W)[2] - np.sqrt(a2 + b2)) < 1e-14


def test_mhd_flux_axis_permutation_G3():
    """F^y and F^z must be the cyclic relabelling of F^x (reading G3): rotating the state
    (x->y->z->x) and the direction together permutes the flux components."""
    rng = np.random.default_rng(11)
    g = 5.0 / 3.0
    for _ in range(5):
        W = _rand_state(rng, 8)
        U0, F0, c0 = oracle.flux(8, g, 0, W)
        for shift in (1, 2):
            perm = [(i - shift) % 3 for i in range(3)]  # new component i = old component perm[i]
            Wr = W.copy()
            Wr[2:5] = W[2:5][perm]; Wr[5:8] = W[5:8][perm]
            U1, F1, c1 = oracle.flux(8, g, shift, Wr)
            want = F0.copy()
            want[1:4] = F0[1:4][perm]; want[5:8] = F0[5:8][perm]
            assert np.allclose(F1, want, rtol=1e-14, atol=1e-15)
            assert abs(c1 - c0) < 1e-14
    # x-flux against the textbook ideal-MHD form for one state written out by hand
    W = np.array([1.0, 1.5, 0.5, 0.25, -0.5, 0.75, 1.0, -0.25])
    p = (g - 1) * 1.5; B2 = 0.75 ** 2 + 1.0 + 0.0625; v2 = 0.25 + 0.0625 + 0.25
    Bv = 0.75 * 0.5 + 1.0 * 0.25 + 0.25 * 0.5
    Etot = 0.5 * v2 + 1.5 + 0.5 * B2
    want = [0.5, 0.25 + p + 0.5 * B2 - 0.75 ** 2, 0.125 - 0.75, -0.25 + 0.75 * 0.25,
            (Etot + p + 0.5 * B2) * 0.5 - 0.75 * Bv, 0.0, 0.5 * 1.0 - 0.75 * 0.25, 0.5 * -0.25 - 0.75 * -0.5]
    assert np.allclose(oracle.flux(8, g, 0, W)[1], want, rtol=1e-14)


# ------------------------------------------------------------------ P5: uniform state bitwise
@pytest.mark.parametrize("nv", [5, 8])
def test_p5_uniform_state_preserved_bitwise(nv):
    h = wl.uniform_hierarchy(2, periodic=True)
    shape = (32, 32, 32)
    one = np.ones(shape)
    B = (0.3 * one, -0.7 * one, 0.2 * one) if nv == 8 else None
    G = wl.cons_from_prim(1.3 * one, 0.7 * one, (0.3 * one, -0.2 * one, 0.9 * one), 1.4, B=B)
    U = wl.split_global(h, G)
    o = oracle.Oracle(h, 1.4, nv)
    o.upload(0, U)
    for _ in range(3):
        o.advance(0.3)
    assert np.array_equal(o.download(0), U)


# ------------------------------------------------------------------ P6: periodic conservation
@pytest.mark.parametrize("nv", [5, 8])
def test_p6_periodic_conservation(nv, ncpu):
    h = wl.uniform_hierarchy(2, periodic=True)
    rng = np.random.default_rng(5)
    shape = (32, 32, 32)
    sm = lambda: 0.2 * np.sin(2 * np.pi * (_X[0] + rng.uniform())) * np.cos(2 * np.pi * (_X[1] + rng.uniform()))
    Z, Y, X = wl._grid(32)
    _X = (X, Y + Z)
    rho, p = 1.0 + sm(), 1.0 + sm()
    v = (sm(), sm(), sm())
    B = (0.5 + sm(), sm(), sm()) if nv == 8 else None
    U = wl.split_global(h, wl.cons_from_prim(rho, p, v, 5 / 3, B=B))
    o = oracle.Oracle(h, 5 / 3, nv, threads=ncpu)
    o.upload(0, U)
    tot0 = U.sum(axis=(0, 2, 3, 4))
    for _ in range(5):
        o.advance(0.3)
    tot1 = o.download(0).sum(axis=(0, 2, 3, 4))
    scale = np.abs(U).sum(axis=(0, 2, 3, 4))
    assert np.all(np.abs(tot1 - tot0) <= 2e-14 * scale), (tot1 - tot0) / scale


# ------------------------------------------------------------------ P7: mirror symmetry
@pytest.mark.parametrize("axis", [0, 1, 2])
def test_p7_mirror_symmetry_bitwise(axis, ncpu):
    h = wl.uniform_hierarchy(2, periodic=True)
    rng = np.random.default_rng(9)
    f = lambda: rng.uniform(0.5, 1.5, (32, 32, 32))
    rho, p = f(), f()
    v = [f() - 1.0 for _ in range(3)]
    G = wl.cons_from_prim(rho, p, v, 1.4)
    ax = 3 - axis  # array axis of [v][z][y][x]
    Gm = np.flip(G, axis=ax).copy()
    Gm[1 + axis] *= -1.0
    res = []
    for g in (G, Gm):
        o = oracle.Oracle(h, 1.4, 5, threads=ncpu)
        o.upload(0, wl.split_global(h, g))
        for _ in range(2):
            o.advance(0.3, dt=2e-3)
        res.append(wl.join_global(h, o.download(0)))
    back = np.flip(res[1], axis=ax).copy()
    back[1 + axis] *= -1.0
    assert np.array_equal(res[0], back)


# ------------------------------------------------------------------ P9: axis permutation (Sod, Brio-Wu)
def _run_1d(nv, gamma, axis, prim_fn, nblk, steps, cfl=0.4, theta=1.5, ncpu=1):
    h, nb = slab_hierarchy(nblk, axis, periodic=False)
    n = 16 * nblk
    s = (np.arange(n) + 0.5) / n
    shape = [16, 16, 16]
    shape[2 - axis] = n
    idx = [None, None, None]
    idx[2 - axis] = slice(None)
    prof = lambda a: np.broadcast_to(np.asarray(a, float)[tuple(idx)], shape)
    rho, p, vpar, Bpar, Bperp = prim_fn(s)
    zero = np.zeros(shape)
    v = [zero, zero, zero]
    v[axis] = prof(vpar)
    B = None
    if nv == 8:
        B = [zero, zero, zero]
        B[axis] = prof(Bpar)
        B[(axis + 1) % 3] = prof(Bperp)
    G = wl.cons_from_prim(prof(rho), prof(p), v, gamma, B=B)
    o = oracle.Oracle(h, gamma, nv, theta=theta, threads=ncpu)
    o.upload(0, wl.split_global(h, G))
    for _ in range(steps):
        o.advance(cfl)
    R = wl.join_global(h, o.download(0))
    # profile along the axis at a fixed transverse position, all variables
    take = [slice(None), 5, 7, 3]
    take[3 - axis] = slice(None)
    return R[tuple(take)], R


def test_p9_sod_axis_permutation_bitwise(ncpu):
    sod = lambda s: (np.where(s < 0.5, 1.0, 0.125), np.where(s < 0.5, 1.0, 0.1), 0 * s, 0 * s, 0 * s)
    px, Rx = _run_1d(5, 1.4, 0, sod, 2, 8, ncpu=ncpu)
    py, _ = _run_1d(5, 1.4, 1, sod, 2, 8, ncpu=ncpu)
    pz, _ = _run_1d(5, 1.4, 2, sod, 2, 8, ncpu=ncpu)
    assert np.array_equal(px[0], py[0]) and np.array_equal(px[0], pz[0])       # rho
    assert np.array_equal(px[4], py[4]) and np.array_equal(px[4], pz[4])       # energy
    assert np.array_equal(px[1], py[2]) and np.array_equal(px[1], pz[3])       # momentum along the axis
    assert not px[2].any() and not px[3].any()
    # every x-line identical across (y, z): the 3-D run reproduces the 1-D profile
    assert np.array_equal(Rx, np.broadcast_to(Rx[:, 5:6, 7:8, :], Rx.shape))


def test_p9_brio_wu_axis_permutation_pins_G3(ncpu):
    # reading G4: left (1,1,0,Bx=.75,By=1), right (.125,.1,0,.75,-1), Gamma=2
    bw = lambda s: (np.where(s < 0.5, 1.0, 0.125), np.where(s < 0.5, 1.0, 0.1), 0 * s,
                    0 * s + 0.75, np.where(s < 0.5, 1.0, -1.0))
    px, _ = _run_1d(8, 2.0, 0, bw, 2, 8, ncpu=ncpu)
    py, _ = _run_1d(8, 2.0, 1, bw, 2, 8, ncpu=ncpu)
    pz, _ = _run_1d(8, 2.0, 2, bw, 2, 8, ncpu=ncpu)
    # x-run: parallel=x(1,5) perp=y(2,6); y-run: parallel=y(2,6) perp=z(3,7); z-run: parallel=z(3,7) perp=x(1,5)
    for a, b, c in ((0, 0, 0), (4, 4, 4), (1, 2, 3), (2, 3, 1), (5, 6, 7), (6, 7, 5)):
        assert np.allclose(px[a], py[b], rtol=0, atol=1e-14), (a, b)
        assert np.allclose(px[a], pz[c], rtol=0, atol=1e-14), (a, c)
    assert np.all(px[5] == 0.75)            # B_parallel stays exactly constant in 1-D
    assert np.abs(px[2]).max() > 0.05       # the transverse field really drives transverse flow


def test_p11prime_brio_wu_profile_qualitative(ncpu):
    bw = lambda s: (np.where(s < 0.5, 1.0, 0.125), np.where(s < 0.5, 1.0, 0.1), 0 * s,
                    0 * s + 0.75, np.where(s < 0.5, 1.0, -1.0))
    h, _ = slab_hierarchy(13, 0, periodic=False)  # N = 208 ~ the paper's 200
    # run to t = 0.1 with CFL 0.4
    n = 208
    s = (np.arange(n) + 0.5) / n
    shape = (16, 16, n)
    b = lambda a: np.broadcast_to(np.asarray(a, float), shape)
    rho, p, _, bx, by = bw(s)
    z = np.zeros(shape)
    G = wl.cons_from_prim(b(rho), b(p), (z, z, z), 2.0, B=(b(bx), b(by), z))
    o = oracle.Oracle(h, 2.0, 8, threads=ncpu)
    o.upload(0, wl.split_global(h, G))
    run_to(o, 0.1, 0.4)
    R = wl.join_global(h, o.download(0))[:, 4, 4, :]
    assert np.isfinite(R).all() and np.all(R[5] == 0.75)
    assert 0.11 < R[0].min() and R[0].max() <= 1.0 + 1e-12
    at = lambda x: np.interp(x, s, R[0])
    # SURVEY P11' scratch values (N=200): 0.666, 0.687, 0.553, 0.117 -- qualitative check only
    assert abs(at(0.45) - 0.666) < 0.03 and abs(at(0.5) - 0.687) < 0.03
    assert abs(at(0.55) - 0.553) < 0.05 and abs(at(0.7) - 0.117) < 0.01


# ------------------------------------------------------------------ P10: MHD with B=0 is Euler
def test_p10_mhd_reduces_to_euler(ncpu):
    h = wl.uniform_hierarchy(2, periodic=True)
    rng = np.random.default_rng(21)
    f = lambda: rng.uniform(0.6, 1.4, (32, 32, 32))
    rho, p = f(), f()
    v = [f() - 1.0 for _ in range(3)]
    zero = np.zeros((32, 32, 32))
    Ue = wl.split_global(h, wl.cons_from_prim(rho, p, v, 1.4))
    Um = wl.split_global(h, wl.cons_from_prim(rho, p, v, 1.4, B=(zero, zero, zero)))
    oe = oracle.Oracle(h, 1.4, 5, threads=ncpu); oe.upload(0, Ue)
    om = oracle.Oracle(h, 1.4, 8, threads=ncpu); om.upload(0, Um)
    for _ in range(3):
        dt = oe.advance(0.3)
        om.advance(0.3, dt=dt)
    Re, Rm = oe.download(0), om.download(0)
    assert not Rm[:, 5:].any()
    assert norm_err(Rm[:, :5], Re).max() < 1e-13


# ------------------------------------------------------------------ CFL closed forms (S4)
def test_cfl_dt_closed_form():
    h = wl.uniform_hierarchy(2, periodic=True)
    one = np.ones((32, 32, 32))
    g = 1.4
    G = wl.cons_from_prim(2.0 * one, 1.0 * one, (0.3 * one, -0.9 * one, 0.1 * one), g)
    o = oracle.Oracle(h, g, 5)
    o.upload(0, wl.split_global(h, G))
    c = np.sqrt(g * 1.0 / 2.0)
    assert abs(o.max_speed(0) - (0.9 + c)) < 1e-14
    assert abs(o.cfl_dt(0, 0, 0.4) - 0.4 * (1 / 32) / (0.9 + c)) < 1e-16
    # one hot cell decides the maximum
    G2 = G.copy()
    G2[:, 7, 20, 3] = wl.cons_from_prim(np.array(2.0), np.array(1.0), (np.array(-2.5), np.array(0.0), np.array(0.0)), g)
    o.upload(0, wl.split_global(h, G2))
    assert abs(o.max_speed(0) - (2.5 + c)) < 1e-14


# ------------------------------------------------------------------ P20: the floors of S11, by hand
def test_p20_primitive_recovery_floors_by_hand():
    """O1 with the floors of reading S11 (`Phys::prim`): a density below the floor is replaced BEFORE the
    velocities are formed, an internal energy below the floor AFTER; states above the floors are untouched.
    Values written out by hand (gamma = 1.4 does not enter O1)."""
    # rho = 0.5 < 0.8 -> rho := 0.8; v = m / 0.8 = (0.5, -0.25, 1.0); e = E/0.8 - v^2/2 = 4/0.8 - 0.65625 = 4.34375
    W, hits = oracle.prim_floors(5, 1.4, 0.8, 2.2, [0.5, 0.4, -0.2, 0.8, 4.0])
    assert hits == 1
    assert np.array_equal(W, [0.8, 4.34375, 0.5, -0.25, 1.0])
    # e = 1.0/1.0 - 0.5 (0.25) = 0.875 < 2.2 -> e := 2.2, density and velocities untouched
    W, hits = oracle.prim_floors(5, 1.4, 0.8, 2.2, [1.0, 0.5, 0.0, 0.0, 1.0])
    assert hits == 1
    assert np.array_equal(W, [1.0, 2.2, 0.5, 0.0, 0.0])
    # both: rho = 0.25 -> 0.8, v = (1, 0, 0), e = 0.4/0.8 - 0.5 = 0 -> 2.2
    W, hits = oracle.prim_floors(5, 1.4, 0.8, 2.2, [0.25, 0.8, 0.0, 0.0, 0.4])
    assert hits == 2 and np.array_equal(W, [0.8, 2.2, 1.0, 0.0, 0.0])
    # negative and NaN densities are floored too (the test is !(rho >= floor)); a state above the floors is untouched
    assert oracle.prim_floors(5, 1.4, 0.8, 2.2, [-1.0, 0.0, 0.0, 0.0, 8.0])[0][0] == 0.8
    assert oracle.prim_floors(5, 1.4, 0.8, 2.2, [np.nan, 0.0, 0.0, 0.0, 8.0])[0][0] == 0.8
    U = [2.0, 1.0, -0.5, 0.25, 12.0]
    W, hits = oracle.prim_floors(5, 1.4, 0.8, 2.2, U)
    assert hits == 0 and np.array_equal(W, oracle.prim(5, 1.4, U))
    assert np.array_equal(W, [2.0, 6.0 - 0.5 * (0.25 + 0.0625 + 0.015625), 0.5, -0.25, 0.125])
    # MHD: the magnetic energy leaves the energy slot before the floor is tested:
    # e = (3.0 - 0.5 * 4) / 1 - 0 = 1.0 < 2.2 -> floored; without B the same E would pass (e = 3.0)
    W, hits = oracle.prim_floors(8, 1.4, 0.8, 2.2, [1.0, 0.0, 0.0, 0.0, 3.0, 2.0, 0.0, 0.0])
    assert hits == 1 and W[1] == 2.2 and W[5] == 2.0
    assert oracle.prim_floors(5, 1.4, 0.8, 2.2, [1.0, 0.0, 0.0, 0.0, 3.0]) [1] == 0


def test_p20_reconstructed_state_floors_by_hand():
    """S11 on the l and r states of O2 (`Phys::floor_state` inside `plm`), with theta = 2 so that the limited
    slope undershoots nowhere by itself: the floors are set ABOVE reconstructed values on purpose.
    Cells (rho, e, vx, vy, vz): i-2 = (1.0, 3.0), i-1 = (0.9, 2.8), i = (0.7, 2.4), i+1 = (0.6, 2.3), at rest."""
    cells = [np.array([r, e, 0.0, 0.0, 0.0]) for r, e in ((1.0, 3.0), (0.9, 2.8), (0.7, 2.4), (0.6, 2.3))]
    # Eq. 9 (G1), theta = 2: rho_l = 0.9 + 0.5 minmod(2(-0.1), 2(-0.2), 0.5(-0.3)) = 0.9 - 0.075 = 0.825
    #                         e_l  = 2.8 + 0.5 minmod(2(-0.2), 2(-0.4), 0.5(-0.6)) = 2.8 - 0.15  = 2.65
    # Eq. 10:                 rho_r = 0.7 + 0.5 minmod(2(0.1), 2(0.2), 0.5(0.3))   = 0.7 + 0.075 = 0.775
    #                         e_r  = 2.4 + 0.5 minmod(2(0.1), 2(0.4), 0.5(0.5))   = 2.4 + 0.1   = 2.5
    WL, WR, lam, F, hits = oracle.face_floors(5, 1.4, 2.0, 0, 1e-300, 1e-300, *cells)
    assert hits == 0
    assert np.allclose([WL[0], WL[1], WR[0], WR[1]], [0.825, 2.65, 0.775, 2.5], rtol=0, atol=2e-16)
    assert np.array_equal(oracle.face(5, 1.4, 2.0, 0, *cells)[3], F)        # the default helper is the same path
    # floors between the two states: rho floor 0.8 lifts only rho_r, e floor 2.6 lifts only e_r
    WL2, WR2, lam2, F2, hits = oracle.face_floors(5, 1.4, 2.0, 0, 0.8, 2.6, *cells)
    assert hits == 2
    assert np.array_equal(WL2, WL) and WR2[0] == 0.8 and WR2[1] == 2.6 and np.array_equal(WR2[2:], WR[2:])
    # Eq. 12 on the floored states, by hand: at rest F_rho = -lam/2 (rho_r - rho_l), F_mx = (p_l + p_r)/2,
    # lam = max c = sqrt(gamma (gamma - 1) max e) = sqrt(0.56 * 2.65)
    assert abs(lam2 - np.sqrt(0.56 * 2.65)) < 1e-15
    assert abs(F2[0] - (-0.5 * lam2 * (0.8 - 0.825))) < 1e-16
    assert abs(F2[1] - 0.5 * 0.4 * (0.825 * 2.65 + 0.8 * 2.6)) < 1e-15
    # floors above both states: four activations, both sides equal -> the flux of a uniform state at rest
    WL3, WR3, lam3, F3, hits = oracle.face_floors(5, 1.4, 2.0, 0, 0.9, 2.7, *cells)
    assert hits == 4 and WL3[0] == WR3[0] == 0.9 and WL3[1] == WR3[1] == 2.7
    assert F3[0] == 0.0 and abs(F3[1] - 0.4 * 0.9 * 2.7) < 1e-15 and F3[4] == 0.0


def test_p20_floors_fire_inside_a_stage_and_are_counted():
    """The same floors through `rk_stage` of a hierarchy: one cell below the density floor in otherwise uniform data
    changes exactly the cells whose stencil (2 cells per side) sees it, and is counted."""
    h = wl.uniform_hierarchy(1, periodic=True)
    one = np.ones((1, 16, 16, 16))
    rho = 1.0 * one
    rho[0, 8, 8, 8] = 0.5
    U = np.moveaxis(wl.cons_from_prim(rho, 1.0 * one, (0 * one, 0 * one, 0 * one), 1.4), 0, 1).copy()
    res = []
    for fl in (1e-30, 0.8):
        o = oracle.Oracle(h, 1.4, 5, rho_floor=fl)
        o.upload(0, U)
        o.fill_ghosts(0, 0)
        o.rk_stage(0, 0, 0, 1, 0.0, 1.0, 1e-3)
        res.append((o.download(1), o.floor_hits()))
    assert res[0][1] == 0 and res[1][1] > 0
    diff = np.argwhere(np.abs(res[0][0][0, 0] - res[1][0][0, 0]) > 0)
    assert len(diff) > 0 and np.abs(diff - 8).max() <= 2          # only the stencil neighbourhood of the cell


# ------------------------------------------------------------------ P21: the global time step on a hierarchy (S4)
def test_p21_global_dt_on_three_levels_closed_form():
    """`Hier::global_dt` (S4): dt0 = CFL dx0 / max over ALL levels of max(|v_d| + c), and every level l steps with
    dt0 / 2^l.  Uniform gas at rest (c = sqrt(gamma p / rho) = sqrt(1.4)) with ONE hot, moving cell on level 1:
    the returned dt must be CFL dx0 / (|v| + c)_hot -- a min for the max, or a per-level dx in place of dx0,
    would return something else -- and each level's own CFL number dt_l S_l / dx_l stays <= CFL."""
    lvl1 = [(i, j, k) for i in (1, 2) for j in (1, 2) for k in (1, 2)]
    lvl2 = [(i, j, k) for i in (3, 4) for j in (3, 4) for k in (3, 4)]
    h = wl.build_hierarchy((2, 2, 2), [lvl1, lvl2], (0,) * 6)
    assert h["nlevels"] == 3
    n = len(h["level"])
    one = np.ones((n, 16, 16, 16))
    rho, p = 1.0 * one, 1.0 * one
    vx, vy, vz = 0 * one, 0 * one, 0 * one
    hot = int(wl.level_patches(h, 1)[3])
    p[hot, 5, 6, 7] = 9.0
    vy[hot, 5, 6, 7] = -2.0
    U = np.moveaxis(wl.cons_from_prim(rho, p, (vx, vy, vz), 1.4), 0, 1).copy()
    c0, shot = np.sqrt(1.4), 2.0 + np.sqrt(1.4 * 9.0)
    dx0 = 1.0 / 32.0
    for cfl in (0.3, 0.15):
        o = oracle.Oracle(h, 1.4, 5)
        o.upload(0, U)
        assert abs(o.max_speed(0) - c0) < 1e-15 and abs(o.max_speed(2) - c0) < 1e-15
        assert abs(o.max_speed(1) - shot) < 1e-14
        dt = o.advance(cfl)
        assert abs(dt - cfl * dx0 / shot) <= 1e-15 * dt
        for l, s in enumerate((c0, shot, c0)):
            assert (dt / 2 ** l) * s / (dx0 / 2 ** l) <= cfl * (1 + 1e-14)
    # the per-level call uses that level's own dx and maximum (what a single-level run needs)
    o = oracle.Oracle(h, 1.4, 5)
    o.upload(0, U)
    assert abs(o.cfl_dt(2, 0, 0.3) - 0.3 * (dx0 / 4) / c0) < 1e-16
    assert abs(o.cfl_dt(1, 0, 0.3) - 0.3 * (dx0 / 2) / shot) < 1e-16
