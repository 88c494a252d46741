"""CPU oracle for the AMR finite-volume hot path -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Thin ctypes wrapper over ``oracle/amr_oracle.cpp`` (plain single-file C++17, compiled with
``-O2 -ffp-contract=off``).  Only ``tests/``, ``__graft_entry__.smoke()`` and the
``cpu_baseline`` / ``--impl reference`` legs of ``bench.py`` may import this package.
It imports nothing from ``paper_0910_5547_b200`` and shares no code with the CUDA path.

Method source: /root/reference/PAPER.md (Wang, Abel & Kaehler, arXiv:0910.5547), Eq. 1-15;
readings G1-G6 / S1-S16 are listed in DESIGN.md.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_DIR = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_DIR, "liboracle.so")
_SRC = os.path.join(_DIR, "amr_oracle.cpp")

NI, NG, NP = 16, 2, 20


def build(force=False):
    """Compile the oracle with g++ (no CUDA involved)."""
    if (not force and os.path.exists(_SO)
            and os.path.getmtime(_SO) >= os.path.getmtime(_SRC)):
        return _SO
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fPIC", "-shared", "-pthread",
           "-o", _SO, _SRC]
    subprocess.check_call(cmd)
    return _SO


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_SO)
        dp = C.POINTER(C.c_double)
        ip = C.POINTER(C.c_int)
        L.orc_create.restype = C.c_void_p
        L.orc_create.argtypes = [C.c_int, C.c_double, C.c_int, C.c_double, C.c_double, C.c_double]
        L.orc_destroy.argtypes = [C.c_void_p]
        L.orc_set_threads.argtypes = [C.c_void_p, C.c_int]
        L.orc_set_theta.argtypes = [C.c_void_p, C.c_double]
        L.orc_floor_hits.restype = C.c_long
        L.orc_floor_hits.argtypes = [C.c_void_p]
        L.orc_set_hierarchy.argtypes = [C.c_void_p, C.c_int, C.c_int, ip, ip, ip, ip, C.c_double, ip, C.c_int]
        for name in ("orc_upload", "orc_download", "orc_upload_padded", "orc_download_padded"):
            getattr(L, name).argtypes = [C.c_void_p, C.c_int, C.c_int, dp]
        L.orc_download_registers.argtypes = [C.c_void_p, C.c_int, dp, dp]
        L.orc_max_speed.restype = C.c_double
        L.orc_max_speed.argtypes = [C.c_void_p, C.c_int, C.c_int]
        L.orc_cfl_dt.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_double, dp]
        L.orc_fill_ghosts.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_double]
        L.orc_rk_stage.argtypes = [C.c_void_p] + [C.c_int] * 4 + [C.c_double] * 4
        L.orc_restrict.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int]
        L.orc_reflux.argtypes = [C.c_void_p, C.c_int, C.c_int]
        L.orc_copy_slot.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int]
        L.orc_advance.argtypes = [C.c_void_p, C.c_double, C.c_double, dp]
        L.orc_minmod.restype = C.c_double
        L.orc_minmod.argtypes = [C.c_double] * 3
        L.orc_face.restype = C.c_double
        L.orc_face.argtypes = [C.c_int, C.c_double, C.c_double, C.c_int] + [dp] * 7
        L.orc_prim.argtypes = [C.c_int, C.c_double, dp, dp]
        L.orc_flux.argtypes = [C.c_int, C.c_double, C.c_int, dp, dp, dp, dp]
        L.orc_refine_indicator.argtypes = [C.c_void_p, C.c_int, C.c_int, dp]
        L.orc_prolong_interior.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int]
        L.orc_set_glm.argtypes = [C.c_void_p, C.c_double, C.c_double]
        L.orc_set_glm.restype = None
        L.orc_glm_damp.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_double]
        L.orc_flux_glm.argtypes = [C.c_double, C.c_double, C.c_int, dp, dp, dp]
        L.orc_flux_glm.restype = None
        L.orc_riemann_glm.argtypes = [C.c_double, C.c_double, C.c_int, dp, dp, dp]
        L.orc_riemann_glm.restype = C.c_double
        _lib = L
    return _lib


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _ip(a):
    return a.ctypes.data_as(C.POINTER(C.c_int))


def minmod(a, b, c):
    return lib().orc_minmod(a, b, c)


def face(nvars, gamma, theta, direction, Wm2, Wm1, W0, Wp1):
    """PLM states + Eq. 12 flux at one face.  Returns (WL, WR, lambda0, F)."""
    arrs = [np.ascontiguousarray(x, dtype=np.float64) for x in (Wm2, Wm1, W0, Wp1)]
    WL, WR, F = (np.zeros(nvars) for _ in range(3))
    lam = lib().orc_face(nvars, gamma, theta, direction, *[_dp(a) for a in arrs], _dp(WL), _dp(WR), _dp(F))
    return WL, WR, lam, F


def prim(nvars, gamma, U):
    U = np.ascontiguousarray(U, dtype=np.float64)
    W = np.zeros(nvars)
    lib().orc_prim(nvars, gamma, _dp(U), _dp(W))
    return W


def face_floors(nvars, gamma, theta, direction, rho_floor, e_floor, Wm2, Wm1, W0, Wp1):
    """face() with the floors of S11 given explicitly.  Returns (WL, WR, lambda0, F, floor activations)."""
    arrs = [np.ascontiguousarray(x, dtype=np.float64) for x in (Wm2, Wm1, W0, Wp1)]
    WL, WR, F = (np.zeros(nvars) for _ in range(3))
    hits = C.c_long(0)
    f = lib().orc_face_floors
    f.restype = C.c_double
    lam = f(C.c_int(nvars), C.c_double(gamma), C.c_double(theta), C.c_int(direction), C.c_double(rho_floor),
            C.c_double(e_floor), *[_dp(a) for a in arrs], _dp(WL), _dp(WR), _dp(F), C.byref(hits))
    return WL, WR, lam, F, hits.value


def prim_floors(nvars, gamma, rho_floor, e_floor, U):
    """prim() with the floors of S11 given explicitly.  Returns (W, floor activations)."""
    U = np.ascontiguousarray(U, dtype=np.float64)
    W = np.zeros(nvars)
    hits = C.c_long(0)
    lib().orc_prim_floors(C.c_int(nvars), C.c_double(gamma), C.c_double(rho_floor), C.c_double(e_floor), _dp(U), _dp(W),
                          C.byref(hits))
    return W, hits.value


def flux(nvars, gamma, direction, W):
    """(U(W), F^d(W), signal speed along d) of one primitive state."""
    W = np.ascontiguousarray(W, dtype=np.float64)
    U, F = np.zeros(nvars), np.zeros(nvars)
    c = C.c_double(0)
    lib().orc_flux(nvars, gamma, direction, _dp(W), _dp(U), _dp(F), C.byref(c))
    return U, F, c.value


def flux_glm(gamma, ch, direction, W):
    """(U(W), F^d(W)) of one 9-variable GLM-MHD primitive state (Eq. 14-15)."""
    W = np.ascontiguousarray(W, dtype=np.float64)
    U, F = np.zeros(9), np.zeros(9)
    lib().orc_flux_glm(gamma, ch, direction, _dp(W), _dp(U), _dp(F))
    return U, F


def riemann_glm(gamma, ch, direction, WL, WR):
    """Eq. 12 between two given 9-variable states.  Returns (lambda0, F)."""
    WL, WR = (np.ascontiguousarray(x, dtype=np.float64) for x in (WL, WR))
    F = np.zeros(9)
    lam = lib().orc_riemann_glm(gamma, ch, direction, _dp(WL), _dp(WR), _dp(F))
    return lam, F


class Oracle:
    """One hierarchy + pool held by the C++ oracle.  Slots: 0=A, 1=B, 2=C.
    nvars = 9: GLM-MHD with wave speed ch and damping ratio cr = c_p^2/c_h (0 = no damping)."""

    def __init__(self, hier, gamma, nvars, bits=64, theta=1.5, rho_floor=1e-30, e_floor=1e-30,
                 nslots=3, threads=1, ch=1.0, cr=0.18):
        L = lib()
        self.h = L.orc_create(bits, gamma, nvars, theta, rho_floor, e_floor)
        if not self.h:
            raise ValueError("orc_create failed")
        self.nv, self.bits, self.hier = nvars, bits, hier
        self.np = hier["level"].shape[0]
        arrs = [np.ascontiguousarray(hier[k], dtype=np.int32) for k in ("level", "origin", "parent", "nbr")]
        bc = np.ascontiguousarray(hier["bc"], dtype=np.int32)
        r = L.orc_set_hierarchy(self.h, self.np, int(hier["nlevels"]), *[_ip(a) for a in arrs],
                                float(hier["dx0"]), _ip(bc), nslots)
        if r:
            raise ValueError("orc_set_hierarchy failed: %d" % r)
        L.orc_set_threads(self.h, threads)
        if nvars == 9:
            L.orc_set_glm(self.h, ch, cr)

    def __del__(self):
        if getattr(self, "h", None):
            lib().orc_destroy(self.h)
            self.h = None

    def set_threads(self, n):
        lib().orc_set_threads(self.h, n)

    def upload(self, slot, U):
        """U: [npatch][nv][16][16][16] float64."""
        U = np.ascontiguousarray(U, dtype=np.float64)
        for p in range(self.np):
            lib().orc_upload(self.h, slot, p, _dp(U[p]))

    def download(self, slot):
        out = np.zeros((self.np, self.nv, NI, NI, NI))
        for p in range(self.np):
            lib().orc_download(self.h, slot, p, _dp(out[p]))
        return out

    def upload_padded(self, slot, U):
        U = np.ascontiguousarray(U, dtype=np.float64)
        for p in range(self.np):
            lib().orc_upload_padded(self.h, slot, p, _dp(U[p]))

    def download_padded(self, slot):
        out = np.zeros((self.np, self.nv, NP, NP, NP))
        for p in range(self.np):
            lib().orc_download_padded(self.h, slot, p, _dp(out[p]))
        return out

    def registers(self, p):
        rf = np.zeros((6, self.nv, 8, 8))
        rc = np.zeros((6, self.nv, 8, 8))
        lib().orc_download_registers(self.h, p, _dp(rf), _dp(rc))
        return rf, rc

    def max_speed(self, level, slot=0):
        return lib().orc_max_speed(self.h, level, slot)

    def cfl_dt(self, level, slot, cfl):
        dt = C.c_double(0)
        r = lib().orc_cfl_dt(self.h, level, slot, cfl, C.byref(dt))
        if r:
            raise FloatingPointError("cfl_dt: non-finite or zero signal speed")
        return dt.value

    def fill_ghosts(self, level, slot, pold=2, pnew=0, alpha=0.0):
        lib().orc_fill_ghosts(self.h, level, slot, pold, pnew, alpha)

    def rk_stage(self, level, sin, sbase, sout, a, b, dt, w=0.0):
        if lib().orc_rk_stage(self.h, level, sin, sbase, sout, a, b, dt, w):
            raise ValueError("rk_stage: slot_out must differ from slot_in")

    def restrict(self, fine_level, fslot=0, cslot=0):
        lib().orc_restrict(self.h, fine_level, fslot, cslot)

    def reflux(self, coarse_level, slot=0):
        if lib().orc_reflux(self.h, coarse_level, slot):
            raise ValueError("reflux: improper nesting")

    def refine_indicator(self, level, slot=0):
        """S20: max of |grad rho|/rho over each octant of each patch of the level -> [npatch_level][8]."""
        n = int((np.asarray(self.hier["level"]) == level).sum())
        out = np.zeros((n, 8))
        lib().orc_refine_indicator(self.h, level, slot, _dp(out))
        return out

    def prolong_interior(self, patch, slot=0, parent_slot=0):
        if lib().orc_prolong_interior(self.h, patch, slot, parent_slot):
            raise ValueError("prolong_interior: bad patch")

    def glm_damp(self, level, slot, factor):
        lib().orc_glm_damp(self.h, level, slot, factor)

    def copy_slot(self, level, src, dst):
        lib().orc_copy_slot(self.h, level, src, dst)

    def advance(self, cfl, dt=0.0):
        """One coarse step of the whole hierarchy (S9).  Returns the dt0 used."""
        out = C.c_double(0)
        r = lib().orc_advance(self.h, cfl, dt, C.byref(out))
        if r:
            raise FloatingPointError("advance failed: %d" % r)
        return out.value

    def floor_hits(self):
        return lib().orc_floor_hits(self.h)
