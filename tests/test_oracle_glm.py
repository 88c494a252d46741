"""Pins P13-P17 of the CPU oracle for the 9-variable GLM-MHD system (Eq. 14-15; readings
S17-S19 of DESIGN.md: c_h a caller-given constant that also enters lambda0 and the time step, the mixed-GLM
damping of Dedner et al. 2002 applied as an exact exponential after each step).  CPU only."""
import numpy as np
import pytest

import oracle
from paper_0910_5547_b200 import workloads as wl
from util import run_to, slab_hierarchy


def _slab(nblk, axis, prim9, gamma, ch, cr, t_end, cfl=0.4, ncpu=1, nv=9):
    """1-D problem along `axis` (components rotated with it).  prim9(s) -> rho, p, v[3], B[3], psi."""
    h, _ = slab_hierarchy(nblk, axis, periodic=True)
    n = 16 * nblk
    s = (np.arange(n) + 0.5) / n
    shape = [16, 16, 16]
    shape[2 - axis] = n
    idx = [None, None, None]
    idx[2 - axis] = slice(None)
    b = lambda a: np.broadcast_to(np.asarray(a, float)[tuple(idx)], shape)
    rho, p, v, B, psi = prim9(s)
    perm = lambda comps: [b(comps[(i - axis) % 3]) for i in range(3)]  # rotate x -> axis
    G = wl.cons_from_prim(b(rho), b(p), perm(v), gamma, B=perm(B), psi=b(psi) if nv == 9 else None)
    o = oracle.Oracle(h, gamma, nv, threads=ncpu, ch=ch, cr=cr)
    o.upload(0, wl.split_global(h, G))
    nsteps = run_to(o, t_end, cfl)
    R = wl.join_global(h, o.download(0))
    take = [slice(None), 5, 7, 3]
    take[3 - axis] = slice(None)
    return s, R[tuple(take)], nsteps


# ---------------------------------------------------------------- P13: the printed F^x of Eq. 15, and its rotations
def test_p13_flux_rows_of_eq15():
    g, ch = 1.4, 2.0
    rho, e, vx, vy, vz, Bx, By, Bz, psi = W = np.array([1.1, 2.0, 0.3, -0.2, 0.1, 0.5, -0.4, 0.7, 0.05])
    p = (g - 1) * rho * e
    h = e + p / rho
    v2, B2, Bv = vx * vx + vy * vy + vz * vz, Bx * Bx + By * By + Bz * Bz, Bx * vx + By * vy + Bz * vz
    # F^x exactly as printed
    Fx = np.array([rho * vx, rho * vx * vx + p + B2 / 2 - Bx * Bx, rho * vy * vx - By * Bx, rho * vz * vx - Bz * Bx,
                   rho * (v2 / 2 + h) * vx + B2 * vx - Bx * Bv, psi, vx * By - vy * Bx, -vz * Bx + vx * Bz, ch * ch * Bx])
    U, F = oracle.flux_glm(g, ch, 0, W)
    assert np.allclose(F, Fx, rtol=1e-15, atol=1e-16)
    assert np.allclose(U, [rho, rho * vx, rho * vy, rho * vz, rho * (v2 / 2 + e) + B2 / 2, Bx, By, Bz, psi], rtol=1e-15)
    # F^y, F^z are F^x with the axes relabelled (reading G3): rotate the state, rotate the flux back
    for d in (1, 2):
        rot = lambda a: np.roll(a, -d)                                     # component i <- component i+d
        Wr = np.concatenate([W[:2], rot(W[2:5]), rot(W[5:8]), W[8:]])
        _, Fr = oracle.flux_glm(g, ch, 0, Wr)
        _, Fd = oracle.flux_glm(g, ch, d, W)
        back = lambda a: np.roll(a, d)
        assert np.allclose(Fd, np.concatenate([Fr[:1], back(Fr[1:4]), Fr[4:5], back(Fr[5:8]), Fr[8:]]), rtol=1e-15, atol=1e-16)
    # psi == 0, and the first eight rows are the 8-variable flux
    W0 = W.copy(); W0[8] = 0.0
    _, F9 = oracle.flux_glm(g, ch, 1, W0)
    _, F8, _ = oracle.flux(8, g, 1, W[:8])
    assert np.array_equal(F9[:8], F8)


def test_p13_lambda0_includes_ch():
    g = 5.0 / 3.0
    W = np.array([1.0, 0.9, 0.1, 0.0, 0.0, 0.3, 0.2, 0.1, 0.0])
    lam_small, _ = oracle.riemann_glm(g, 0.01, 0, W, W)
    lam_big, F = oracle.riemann_glm(g, 7.5, 0, W, W)
    assert lam_big == 7.5 and 1.0 < lam_small < 2.0
    _, Fx = oracle.flux_glm(g, 7.5, 0, W)
    assert np.allclose(F, Fx, rtol=1e-15, atol=1e-16)                        # consistency: F(W, W) = F^x(W)


# ---------------------------------------------------------------- P14: the (B_d, psi) pair is a wave equation at c_h
@pytest.mark.parametrize("axis", [0, 1, 2])
def test_p14_glm_wave_closed_form_second_order(axis, ncpu):
    """B_d = eps sin(kx) cos(c_h k t), psi = -eps c_h cos(kx) sin(c_h k t) solves B_t + psi_x = 0,
    psi_t + c_h^2 B_x = 0 exactly; with B = O(eps) the coupling to the gas is O(eps^2)."""
    eps, ch, t_end = 1e-6, 2.0, 0.2
    k = 2 * np.pi

    def prim9(s):
        z = 0 * s
        return 1 + z, 1 + z, (z, z, z), (eps * np.sin(k * s), z, z), z
    errs = []
    for nblk in (1, 2, 4):
        s, R, _ = _slab(nblk, axis, prim9, 1.4, ch, 0.0, t_end, ncpu=ncpu)
        Bd = R[5 + axis]
        errs.append((np.abs(Bd - eps * np.sin(k * s) * np.cos(ch * k * t_end)).mean() / eps,
                     np.abs(R[8] + eps * ch * np.cos(k * s) * np.sin(ch * k * t_end)).mean() / (eps * ch)))
        assert np.abs(R[0] - 1).max() < 1e-10 and np.abs(R[1:4]).max() < 1e-10   # the gas does not notice
    (b0, p0), (b1, p1), (b2, p2) = errs
    # same pre-asymptotic behaviour as P11 (extrema clipping of the limiter): 1.59, 1.76 for B_d; 2.17, 2.20 for psi
    assert np.log2(b0 / b1) > 1.4 and np.log2(b1 / b2) > 1.65 and np.log2(p1 / p2) > 1.9, errs
    assert b2 < 1.2e-3 and p2 < 2e-3, errs


# ---------------------------------------------------------------- P15: damping is the exact exponential
def test_p15_damping_exact_exponential():
    h = wl.uniform_hierarchy(1, periodic=True)
    one = np.ones((16, 16, 16))
    G = wl.cons_from_prim(one, one, (0 * one, 0 * one, 0 * one), 1.4, B=(0 * one, 0 * one, 0 * one), psi=0.3 * one)
    ch, cr = 1.5, 0.18
    o = oracle.Oracle(h, 1.4, 9, ch=ch, cr=cr)
    o.upload(0, wl.split_global(h, G))
    dts = [o.advance(0.3) for _ in range(3)]
    R = o.download(0)
    expect = 0.3 * np.prod([np.exp(-dt * ch / cr) for dt in dts])
    assert np.abs(R[:, 8] - expect).max() <= 4e-16 * 0.3            # uniform psi: all fluxes cancel exactly
    assert np.array_equal(R[:, :8], wl.split_global(h, G)[:, :8])
    o2 = oracle.Oracle(h, 1.4, 9, ch=ch, cr=0.0)                    # cr = 0: no damping
    o2.upload(0, wl.split_global(h, G))
    o2.advance(0.3)
    assert np.array_equal(o2.download(0)[:, 8], 0.3 * np.ones((1, 16, 16, 16)))
    # the time step sees c_h (S17): gas at rest with c_s = sqrt(1.4) < c_h
    assert abs(dts[0] - 0.3 * (1.0 / 16) / ch) <= 1e-15


# ---------------------------------------------------------------- P16: psi = 0, div B = 0, small c_h  ==  the 8-variable solver
def test_p16_reduces_to_ideal_mhd(ncpu):
    def brio_wu(s):                                                  # reading G4; smooth enough in 12 steps
        z = 0 * s
        L = np.abs(s - 0.5) < 0.25
        return (np.where(L, 1.0, 0.125), np.where(L, 1.0, 0.1), (z, z, z),
                (0.75 + z, np.where(L, 1.0, -1.0), z), z)
    s, R9, n9 = _slab(4, 0, brio_wu, 2.0, 0.05, 0.0, 0.02, ncpu=ncpu, nv=9)
    s, R8, n8 = _slab(4, 0, brio_wu, 2.0, 0.05, 0.0, 0.02, ncpu=ncpu, nv=8)
    assert n9 == n8 and n9 >= 5
    assert np.array_equal(R9[:8], R8)                                # c_h below every lambda0: bitwise
    assert np.array_equal(R9[8], 0 * s)                              # B_x uniform: psi is never generated


# ---------------------------------------------------------------- P17: psi generated by a monopole, and cleaned
def test_p17_monopole_is_transported_away(ncpu):
    """A localised div B error (B_x bump along x) splits into two pulses moving at +-c_h; with damping
    its L1 norm decays.  Qualitative invariant: total B_x and total psi are conserved (periodic)."""
    eps, ch = 1e-3, 2.0

    def prim9(s):
        z = 0 * s
        return 1 + z, 1 + z, (z, z, z), (eps * np.exp(-((s - 0.5) / 0.05) ** 2), z, z), z
    s, R0, _ = _slab(4, 0, prim9, 1.4, ch, 0.0, 1e-9, ncpu=ncpu)
    s, R1, _ = _slab(4, 0, prim9, 1.4, ch, 0.0, 0.1, ncpu=ncpu)
    s, R2, _ = _slab(4, 0, prim9, 1.4, ch, 0.18, 0.1, ncpu=ncpu)
    assert abs(R1[5].sum() - R0[5].sum()) < 1e-12 * eps * len(s) + 1e-18 and abs(R1[8].sum()) < 1e-15 * len(s)
    i_l, i_r = np.argmin(np.abs(s - 0.3)), np.argmin(np.abs(s - 0.7))
    assert R1[5][i_l] > 0.3 * eps and R1[5][i_r] > 0.3 * eps and R1[5][len(s) // 2] < 0.1 * eps   # two pulses at 0.5 -+ c_h t
    assert np.abs(R2[8]).sum() < 0.8 * np.abs(R1[8]).sum()          # damping removes psi
