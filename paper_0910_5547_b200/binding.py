"""Thin ctypes binding over libamrhydro.so (include/amrhydro.h): argument marshalling only.

Every step of the path runs in the library's CUDA kernels; PyTorch is used here for the
device allocation of the pool and for the stream.  There is no CPU fallback: if the shared
library is missing or no CUDA device is present, construction raises.
"""
import ctypes as C
import os

import numpy as np

_DIR = os.path.dirname(os.path.abspath(__file__))
# AMRHYDRO_LIB: an alternative build of the same library (kernel tuning variants)
_SO = os.environ.get("AMRHYDRO_LIB") or os.path.join(_DIR, "libamrhydro.so")

OPT_DTYPE, OPT_THETA, OPT_RHO_FLOOR, OPT_EINT_FLOOR, OPT_KERNEL, OPT_HALO, OPT_FUSE_CFL, OPT_GLM_CH, OPT_GLM_CR, OPT_ZSPLIT, OPT_GRAPH = 1, 2, 3, 4, 5, 6, 7, 8, 9, 10, 11
CNT_LAUNCHES, CNT_FLOOR_HITS, CNT_GRAPH_REPLAYS = 1, 2, 3

EXPORTS = [
    "amrhydro_create", "amrhydro_destroy", "amrhydro_last_error", "amrhydro_set_option",
    "amrhydro_get_counter", "amrhydro_pool_bytes", "amrhydro_bind_pool", "amrhydro_set_hierarchy",
    "amrhydro_upload", "amrhydro_download", "amrhydro_download_padded", "amrhydro_download_registers",
    "amrhydro_cfl_dt", "amrhydro_cfl_dt_device", "amrhydro_fill_ghosts", "amrhydro_rk_stage", "amrhydro_restrict",
    "amrhydro_reflux", "amrhydro_copy_slot", "amrhydro_glm_damp", "amrhydro_refine_indicator",
    "amrhydro_prolong_interior", "amrhydro_regrid", "amrhydro_set_owned", "amrhydro_set_halo_plan",
    "amrhydro_halo_bytes", "amrhydro_halo_pack", "amrhydro_halo_unpack", "amrhydro_advance", "amrhydro_advance_host", "amrhydro_sync",
    "amrhydro_noalloc_setup", "amrhydro_cfl_dt_noalloc", "amrhydro_noalloc_last_error",
]
NOALLOC_MAX_PATCHES = 32768          # AMRHYDRO_NOALLOC_MAX_PATCHES


class PatchDesc(C.Structure):
    _fields_ = [("level", C.c_int), ("origin", C.c_int * 3), ("parent", C.c_int), ("nbr", C.c_int * 27)]


_lib = None


def load_library():
    """dlopen libamrhydro.so and declare the prototypes.  Raises if it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_SO):
        raise RuntimeError("libamrhydro.so is not built: run `python -m paper_0910_5547_b200.build` "
                           "(or __graft_entry__.build()); there is no CPU fallback")
    L = C.CDLL(_SO)
    vp, dp, i, d = C.c_void_p, C.POINTER(C.c_double), C.c_int, C.c_double
    L.amrhydro_create.restype = vp
    L.amrhydro_create.argtypes = [d, i, i, i]
    L.amrhydro_destroy.argtypes = [vp]
    L.amrhydro_destroy.restype = None
    L.amrhydro_last_error.restype = C.c_char_p
    L.amrhydro_last_error.argtypes = [vp]
    L.amrhydro_set_option.argtypes = [vp, i, d]
    L.amrhydro_get_counter.argtypes = [vp, i, C.POINTER(C.c_longlong), i]
    L.amrhydro_pool_bytes.restype = C.c_size_t
    L.amrhydro_pool_bytes.argtypes = [vp, i, i]
    L.amrhydro_bind_pool.argtypes = [vp, vp, C.c_size_t, i, i, vp]
    L.amrhydro_set_hierarchy.argtypes = [vp, C.POINTER(PatchDesc), i, i, d, C.POINTER(C.c_int)]
    L.amrhydro_upload.argtypes = [vp, i, i, i, vp]
    L.amrhydro_download.argtypes = [vp, i, i, i, vp]
    L.amrhydro_download_padded.argtypes = [vp, i, i, dp]
    L.amrhydro_download_registers.argtypes = [vp, i, dp, dp]
    L.amrhydro_cfl_dt.argtypes = [vp, i, i, d, dp, dp]
    L.amrhydro_cfl_dt_device.argtypes = [vp, i, i, i, d, C.POINTER(vp)]
    L.amrhydro_fill_ghosts.argtypes = [vp, i, i, i, i, d]
    L.amrhydro_rk_stage.argtypes = [vp, i, i, i, i, d, d, d, d]
    L.amrhydro_restrict.argtypes = [vp, i, i, i]
    L.amrhydro_reflux.argtypes = [vp, i, i]
    L.amrhydro_copy_slot.argtypes = [vp, i, i, i]
    L.amrhydro_glm_damp.argtypes = [vp, i, i, d]
    L.amrhydro_refine_indicator.argtypes = [vp, i, i, dp]
    L.amrhydro_prolong_interior.argtypes = [vp, i, i, i]
    L.amrhydro_regrid.argtypes = [vp, C.POINTER(PatchDesc), i, i, C.POINTER(C.c_int), i]
    L.amrhydro_set_owned.argtypes = [vp, i]
    L.amrhydro_set_halo_plan.argtypes = [vp, C.POINTER(C.c_int), i, C.POINTER(C.c_int), i]
    L.amrhydro_halo_bytes.restype = C.c_size_t
    L.amrhydro_halo_bytes.argtypes = [vp, i]
    L.amrhydro_halo_pack.argtypes = [vp, i, vp]
    L.amrhydro_halo_unpack.argtypes = [vp, i, vp]
    L.amrhydro_advance.argtypes = [vp, d, d, dp]
    L.amrhydro_advance_host.argtypes = [vp, d, d, i, vp, vp, dp]
    L.amrhydro_sync.argtypes = [vp]
    L.amrhydro_noalloc_setup.argtypes = []
    L.amrhydro_cfl_dt_noalloc.argtypes = [vp, i, i, i, d, d, d, d, d, vp, vp]
    L.amrhydro_noalloc_last_error.restype = C.c_char_p
    L.amrhydro_noalloc_last_error.argtypes = []
    _lib = L
    return L


class AmrHydroError(RuntimeError):
    pass


def _ok_noalloc(L, r):
    if r != 0:
        raise AmrHydroError("amrhydro error %d: %s" % (r, L.amrhydro_noalloc_last_error().decode()))


def noalloc_setup():
    """amrhydro_noalloc_setup: once per device, with that device current, outside stream capture."""
    L = load_library()
    _ok_noalloc(L, L.amrhydro_noalloc_setup())


def cfl_dt_noalloc(dev_patches, npatches, nvars, dtype_bits, gamma, cfl_dx, dev_out, stream=0,
                   rho_floor=1e-30, e_floor=1e-30, ch=1.0):
    """amrhydro_cfl_dt_noalloc: the CFL reduction over `npatches` consecutive patches at device address `dev_patches`
    (pool layout) with its scratch in a static device array -- no handle, no allocation.  dev_out: device address of
    three doubles (max signal speed, dt = cfl_dx / max, non-finite flag).  Nothing is synchronised."""
    L = load_library()
    _ok_noalloc(L, L.amrhydro_cfl_dt_noalloc(dev_patches, int(npatches), int(nvars), int(dtype_bits), float(gamma),
                                             float(rho_floor), float(e_floor), float(ch), float(cfl_dx), stream, dev_out))


class AmrHydro:
    """One solver context + pool.  Method names mirror the C ABI (amrhydro_<name>)."""

    def __init__(self, hier, gamma, nvars, dtype="f64", theta=1.5, nslots=None, kernel=3, halo=1,
                 rho_floor=1e-30, e_floor=1e-30, device="cuda:0", stream=None, fuse_cfl=2, ch=1.0, cr=0.18, zsplit=2, graph=0, max_patches=None, patch_dim=None):
        import torch  # device memory + streams only
        if not torch.cuda.is_available():
            raise AmrHydroError("no CUDA device: the amrhydro path has no CPU fallback")
        self.L = load_library()
        self.torch = torch
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.pdim = int(patch_dim or hier.get("ni", 16))          # 16, or 32 / 48 / 64 (held as 16^3 sub-patches by the library)
        self.h = self.L.amrhydro_create(gamma, nvars, self.pdim, 2)
        if not self.h:
            raise AmrHydroError("amrhydro_create failed (bad arguments or no device)")
        self.nv = nvars
        self.np_dtype = {"f64": np.float64, "f32": np.float32}[dtype]
        self._ok(self.L.amrhydro_set_option(self.h, OPT_DTYPE, 64.0 if dtype == "f64" else 32.0))
        for k, v in ((OPT_THETA, theta), (OPT_RHO_FLOOR, rho_floor), (OPT_EINT_FLOOR, e_floor),
                     (OPT_KERNEL, kernel), (OPT_HALO, halo), (OPT_FUSE_CFL, fuse_cfl), (OPT_ZSPLIT, zsplit), (OPT_GRAPH, graph)) + \
                (((OPT_GLM_CH, ch), (OPT_GLM_CR, cr)) if nvars == 9 else ()):
            self._ok(self.L.amrhydro_set_option(self.h, k, float(v)))
        self.hier = hier
        self.npatch = int(hier["level"].shape[0])
        nlev = int(hier["nlevels"])
        self.nslots = nslots or (3 if nlev > 1 else 2)
        self.max_patches = max(self.npatch, int(max_patches or 0))     # room for a later regrid
        nbytes = self.L.amrhydro_pool_bytes(self.h, self.max_patches, self.nslots)
        self.pool = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        self._ok(self.L.amrhydro_bind_pool(self.h, self.pool.data_ptr(), nbytes, self.max_patches, self.nslots,
                                           self.stream.cuda_stream))
        tbl = self._table(hier)
        bc = (C.c_int * 6)(*[int(x) for x in hier["bc"]])
        self._ok(self.L.amrhydro_set_hierarchy(self.h, tbl, self.npatch, nlev, float(hier["dx0"]), bc))

    @staticmethod
    def _table(hier):
        n = int(hier["level"].shape[0])
        tbl = (PatchDesc * n)()
        lv, org, par, nbr = (np.ascontiguousarray(hier[k], dtype=np.int32) for k in ("level", "origin", "parent", "nbr"))
        view = np.frombuffer(tbl, dtype=np.int32).reshape(n, 32)
        view[:, 0] = lv
        view[:, 1:4] = org
        view[:, 4] = par
        view[:, 5:32] = nbr
        return tbl

    # ---- patch sharding (one shard per handle)
    def set_owned(self, owned):
        self._ok(self.L.amrhydro_set_owned(self.h, int(owned)))
        self.owned = int(owned)

    def set_halo_plan(self, send_pairs, recv_pairs):
        sp = np.ascontiguousarray(send_pairs, dtype=np.int32).reshape(-1, 2)
        rp = np.ascontiguousarray(recv_pairs, dtype=np.int32).reshape(-1, 2)
        ip = C.POINTER(C.c_int)
        self._ok(self.L.amrhydro_set_halo_plan(self.h, sp.ctypes.data_as(ip), len(sp), rp.ctypes.data_as(ip), len(rp)))

    def halo_bytes(self, which):
        return int(self.L.amrhydro_halo_bytes(self.h, which))

    def halo_pack(self, slot, dev_ptr):
        self._ok(self.L.amrhydro_halo_pack(self.h, slot, dev_ptr))

    def halo_unpack(self, slot, dev_ptr):
        self._ok(self.L.amrhydro_halo_unpack(self.h, slot, dev_ptr))

    def regrid(self, hier, old_of_new, slot=0):
        """amrhydro_regrid: the new table on the live pool (needs max_patches >= the new patch count)."""
        n = int(hier["level"].shape[0])
        m = np.ascontiguousarray(old_of_new, dtype=np.int32)
        assert m.shape == (n,)
        self._ok(self.L.amrhydro_regrid(self.h, self._table(hier), n, int(hier["nlevels"]),
                                        m.ctypes.data_as(C.POINTER(C.c_int)), slot))
        self.hier, self.npatch = hier, n

    def _ok(self, r):
        if r != 0:
            raise AmrHydroError("amrhydro error %d: %s" % (r, self.L.amrhydro_last_error(self.h).decode()))

    def close(self):
        if getattr(self, "h", None):
            self.L.amrhydro_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def patch_ptr(self, slot, patch):
        """Device address of 16^3 patch `patch` of `slot` in the pool (the layout amrhydro_cfl_dt_noalloc reads)."""
        if self.pdim != 16:
            raise AmrHydroError("patch_ptr is defined for 16^3 patches")
        return self.pool.data_ptr() + (slot * self.max_patches + patch) * int(self.L.amrhydro_pool_bytes(self.h, 1, 1))

    # ---- options / counters
    def set_option(self, key, value):
        self._ok(self.L.amrhydro_set_option(self.h, key, float(value)))

    def get_counter(self, key, reset=False):
        v = C.c_longlong(0)
        self._ok(self.L.amrhydro_get_counter(self.h, key, C.byref(v), int(reset)))
        return v.value

    # ---- data movement (host arrays in interior layout [npatch][nv][16][16][16])
    def upload(self, slot, U, first=0):
        U = np.ascontiguousarray(U, dtype=self.np_dtype)
        self._ok(self.L.amrhydro_upload(self.h, slot, first, U.shape[0], U.ctypes.data))

    def upload_ptr(self, slot, first, count, host_ptr):
        self._ok(self.L.amrhydro_upload(self.h, slot, first, count, host_ptr))

    def download(self, slot, first=0, count=None):
        count = self.npatch - first if count is None else count
        out = np.empty((count, self.nv, self.pdim, self.pdim, self.pdim), dtype=self.np_dtype)
        self._ok(self.L.amrhydro_download(self.h, slot, first, count, out.ctypes.data))
        return out

    def download_padded(self, slot, patch):
        out = np.empty((self.nv, 20, 20, 20), dtype=np.float64)
        self._ok(self.L.amrhydro_download_padded(self.h, slot, patch, out.ctypes.data_as(C.POINTER(C.c_double))))
        return out

    def download_registers(self, patch):
        rf = np.empty((6, self.nv, 8, 8)); rc = np.empty((6, self.nv, 8, 8))
        dp = C.POINTER(C.c_double)
        self._ok(self.L.amrhydro_download_registers(self.h, patch, rf.ctypes.data_as(dp), rc.ctypes.data_as(dp)))
        return rf, rc

    # ---- the hot-path calls
    def cfl_dt(self, level, slot, cfl):
        dt, s = C.c_double(0), C.c_double(0)
        self._ok(self.L.amrhydro_cfl_dt(self.h, level, slot, cfl, C.byref(dt), C.byref(s)))
        return dt.value

    def cfl_dt_device(self, level_first, level_last, slot, cfl):
        """Device address of (dt, non-finite flag); nothing is synchronised."""
        out = C.c_void_p(0)
        self._ok(self.L.amrhydro_cfl_dt_device(self.h, level_first, level_last, slot, cfl, C.byref(out)))
        return out.value

    def max_speed(self, level, slot=0):
        dt, s = C.c_double(0), C.c_double(0)
        self._ok(self.L.amrhydro_cfl_dt(self.h, level, slot, 1.0, C.byref(dt), C.byref(s)))
        return s.value

    def fill_ghosts(self, level, slot, pold=2, pnew=0, alpha=0.0):
        self._ok(self.L.amrhydro_fill_ghosts(self.h, level, slot, pold, pnew, alpha))

    def rk_stage(self, level, sin, sbase, sout, a, b, dt, w=0.0):
        self._ok(self.L.amrhydro_rk_stage(self.h, level, sin, sbase, sout, a, b, dt, w))

    def restrict(self, fine_level, fslot=0, cslot=0):
        self._ok(self.L.amrhydro_restrict(self.h, fine_level, fslot, cslot))

    def reflux(self, coarse_level, slot=0):
        self._ok(self.L.amrhydro_reflux(self.h, coarse_level, slot))

    def refine_indicator(self, level, slot=0):
        n = int((np.asarray(self.hier["level"]) == level).sum())
        out = np.zeros((n, 8))
        self._ok(self.L.amrhydro_refine_indicator(self.h, level, slot, out.ctypes.data_as(C.POINTER(C.c_double))))
        return out

    def prolong_interior(self, patch, slot=0, parent_slot=0):
        self._ok(self.L.amrhydro_prolong_interior(self.h, patch, slot, parent_slot))

    def glm_damp(self, level, slot, factor):
        self._ok(self.L.amrhydro_glm_damp(self.h, level, slot, factor))

    def copy_slot(self, level, src, dst):
        self._ok(self.L.amrhydro_copy_slot(self.h, level, src, dst))

    def advance(self, cfl, dt=0.0, want_dt=True):
        """want_dt=False passes dt_out = NULL: with graph=1 the call then does not synchronise."""
        if not want_dt:
            self._ok(self.L.amrhydro_advance(self.h, cfl, dt, None))
            return None
        out = C.c_double(0)
        self._ok(self.L.amrhydro_advance(self.h, cfl, dt, C.byref(out)))
        return out.value

    def advance_host(self, cfl, dt, nsteps, host_in_ptr, host_out_ptr):
        out = C.c_double(0)
        self._ok(self.L.amrhydro_advance_host(self.h, cfl, dt, nsteps, host_in_ptr, host_out_ptr, C.byref(out)))
        return out.value

    def sync(self):
        self._ok(self.L.amrhydro_sync(self.h))
