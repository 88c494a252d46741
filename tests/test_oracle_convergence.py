"""Pins P3, P4, P11 of the CPU oracle: convergence against closed-form solutions.  CPU only."""
import numpy as np
import pytest

import oracle
from paper_0910_5547_b200 import workloads as wl
from util import exact_sod, norm_err, run_to, slab_hierarchy


def _slab_run(nv, gamma, axis, nblk, prim, t_end, cfl, periodic, theta=1.5, ncpu=1):
    h, _ = slab_hierarchy(nblk, axis, periodic=periodic)
    n = 16 * nblk
    s = (np.arange(n) + 0.5) / n
    shape = [16, 16, 16]
    shape[2 - axis] = n
    idx = [None, None, None]
    idx[2 - axis] = slice(None)
    b = lambda a: np.broadcast_to(np.asarray(a, float)[tuple(idx)], shape)
    rho, p, v, B = prim(s)
    perm = lambda comps: [b(comps[(i - axis) % 3]) for i in range(3)]  # rotate x->axis
    G = wl.cons_from_prim(b(rho), b(p), perm(v), gamma, B=None if B is None else perm(B))
    o = oracle.Oracle(h, gamma, nv, theta=theta, threads=ncpu)
    o.upload(0, wl.split_global(h, G))
    run_to(o, t_end, cfl)
    R = wl.join_global(h, o.download(0))
    take = [slice(None), 5, 7, 3]
    take[3 - axis] = slice(None)
    return s, R[tuple(take)]


# ---------------------------------------------------------------- P3: smooth advected wave, order 2
@pytest.mark.parametrize("axis", [0, 2])
def test_p3_smooth_wave_second_order(axis, ncpu):
    prim = lambda s: (1 + 0.2 * np.sin(2 * np.pi * s), 1 + 0 * s, (1 + 0 * s, 0 * s, 0 * s), None)
    errs = []
    for nblk in (2, 4):
        s, R = _slab_run(5, 1.4, axis, nblk, prim, 1.0, 0.4, True, ncpu=ncpu)
        errs.append(np.abs(R[0] - (1 + 0.2 * np.sin(2 * np.pi * (s - 1.0)))).mean())
    order = np.log2(errs[0] / errs[1])
    # SURVEY P3 scratch, theta=1.5: L1 = 7.43e-3 (N=32), 1.95e-3 (N=64), order 1.93
    assert abs(errs[0] - 7.43e-3) < 0.05 * 7.43e-3, errs
    assert abs(errs[1] - 1.95e-3) < 0.05 * 1.95e-3, errs
    assert 1.8 < order < 2.2, (errs, order)


def test_p3_diagonal_wave_converges(ncpu):
    """3-D: wave advected along the cube diagonal (CFL 0.3, S4) -- exercises all three sweeps."""
    errs = []
    for nb in (1, 2):
        n = 16 * nb
        h = wl.uniform_hierarchy(nb, periodic=True)
        Z, Y, X = wl._grid(n)
        rho = 1 + 0.2 * np.sin(2 * np.pi * (X + Y + Z))
        one = np.ones_like(rho)
        G = wl.cons_from_prim(rho, one, (one, one, one), 1.4)
        o = oracle.Oracle(h, 1.4, 5, threads=ncpu)
        o.upload(0, wl.split_global(h, G))
        run_to(o, 0.25, 0.3)
        R = wl.join_global(h, o.download(0))[0]
        errs.append(np.abs(R - (1 + 0.2 * np.sin(2 * np.pi * (X + Y + Z - 0.75)))).mean())
    assert np.log2(errs[0] / errs[1]) > 1.25 and errs[1] < 9e-3, errs  # N=16->32 is pre-asymptotic (cf. P11: 1.34)


# ---------------------------------------------------------------- P4: Sod vs the exact Riemann solution
def test_p4_exact_star_state_matches_survey():
    _, _, _, st = exact_sod(np.array([0.5]), 0.14)
    assert abs(st["ps"] - 0.303130178) < 1e-8 and abs(st["us"] - 0.927452620) < 1e-8
    assert abs(st["rsl"] - 0.426319428) < 1e-8 and abs(st["rsr"] - 0.265573712) < 1e-8
    assert abs(st["S"] - 1.752155732) < 1e-8


def test_p4_sod_l1_error_falls_at_first_order(ncpu):
    prim = lambda s: (np.where(s < 0.5, 1.0, 0.125), np.where(s < 0.5, 1.0, 0.1), (0 * s, 0 * s, 0 * s), None)
    errs = {}
    for nblk in (6, 12):  # N = 96, 192 (the paper uses N = 100)
        s, R = _slab_run(5, 1.4, 0, nblk, prim, 0.14, 0.4, False, ncpu=ncpu)
        rho, u, p, _ = exact_sod(s, 0.14)
        errs[16 * nblk] = np.abs(R[0] - rho).mean()
        assert np.abs(R[1] / R[0] - u).mean() < 0.02
    order = np.log2(errs[96] / errs[192])
    # SURVEY P4 scratch: 6.77e-3 at N=100, 3.63e-3 at N=200, order 0.85-0.93
    assert 6.0e-3 < errs[96] < 7.8e-3 and 3.2e-3 < errs[192] < 4.2e-3, errs
    assert 0.75 < order < 1.1, (errs, order)


# ---------------------------------------------------------------- P11: circularly polarised Alfven wave
@pytest.mark.parametrize("axis", [0, 1])
def test_p11_alfven_wave_second_order(axis, ncpu):
    def prim(s):
        by, bz = 0.1 * np.sin(2 * np.pi * s), 0.1 * np.cos(2 * np.pi * s)
        return 1 + 0 * s, 0.1 + 0 * s, (0 * s, -by, -bz), (1 + 0 * s, by, bz)
    errs = []
    for nblk in (1, 2, 4):
        s, R = _slab_run(8, 5.0 / 3.0, axis, nblk, prim, 1.0, 0.4, True, ncpu=ncpu)
        comp = 5 + (axis + 1) % 3  # the rotated By slot
        errs.append(np.abs(R[comp] - 0.1 * np.sin(2 * np.pi * s)).mean())
    o1, o2 = np.log2(errs[0] / errs[1]), np.log2(errs[1] / errs[2])
    # SURVEY P11 scratch: 8.73e-3 (N=16), 3.45e-3 (32), 9.38e-4 (64): orders 1.34, 1.88
    assert abs(errs[0] - 8.73e-3) < 0.06 * 8.73e-3, errs
    assert abs(errs[2] - 9.38e-4) < 0.06 * 9.38e-4, errs
    assert o1 > 1.2 and o2 > 1.75, (errs, o1, o2)


def test_fp32_arithmetic_bounds_the_strict_per_variable_norm(ncpu):
    """Why fp32 whole-run parity uses reading S14' for small vector components: the oracle's own fp32 instantiation
    (same scheme, same operation order, plain fp32) against its fp64 self on config 2 at 64^3, 10 steps, same data
    and time steps.  rho, rho v_x and E agree to a few 1e-7; rho v_y (3 % of |rho v|_max) and rho v_z (0.7 %) do not
    reach 1e-5 of their OWN maximum, because the rounding of the O(1) fluxes is absolute.  Measured against the
    maximum of the momentum vector they are below 1e-6 like everything else."""
    h = wl.uniform_hierarchy(4, periodic=True)
    U = wl.split_global(h, wl.kelvin_helmholtz_global(64)).astype(np.float32).astype(np.float64)
    o64, o32 = oracle.Oracle(h, 5.0 / 3.0, 5, threads=ncpu), oracle.Oracle(h, 5.0 / 3.0, 5, bits=32, threads=ncpu)
    o64.upload(0, U); o32.upload(0, U)
    for _ in range(10):
        o32.advance(0.3, o64.advance(0.3))
    A, B = o32.download(0), o64.download(0)
    strict = norm_err(A, B)
    assert (strict[[0, 1, 4]] < 1e-6).all()
    assert strict[2] > 5e-6 and strict[3] > 1e-5            # the plain-fp32 scheme itself misses 1e-5 here
    assert (norm_err(A, B, vector=True) < 1e-6).all()       # S14'
