"""amrhydro_cfl_dt_noalloc (include/amrhydro.h): the CFL reduction a1 (S2-S4) for callers that cannot allocate -- its
scratch is a file-scope `static __device__` array of the library, no handle, no cudaMalloc.  The bar is the existing
path, amrhydro_cfl_dt (k_cfl + handle-owned scratch), on the same pool: the maximum of the same per-cell values, so the
tolerance of the other GPU tests (1e-12 fp64, 1e-5 fp32) is asserted and bitwise equality is what is expected.

The file is named so that pytest collects it last (the suite runs with `pytest -x`).  Every test makes two or more
calls in a row: all calls share the one static array, which keeps the last call's contents, and a later call on fewer
patches and slower states would show a stale partial maximum or ticket."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from paper_0910_5547_b200 import workloads as wl  # noqa: E402

TOL = {"f64": 1e-12, "f32": 1e-5}
BITS = {"f64": 64, "f32": 32}
GAMMA = 1.4


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (no CPU fallback exists)")
    from paper_0910_5547_b200 import binding
    binding.load_library()
    return binding


def state(npatch, nv, seed, vmax):
    rng = np.random.default_rng(seed)
    shp = (npatch, 16, 16, 16)
    rho, p = rng.uniform(0.5, 1.5, shp), rng.uniform(0.5, 1.5, shp)
    v = [rng.uniform(-vmax, vmax, shp) for _ in range(3)]
    B = [rng.uniform(-0.3, 0.3, shp) for _ in range(3)] if nv >= 8 else None
    psi = rng.uniform(-0.2, 0.2, shp) if nv == 9 else None
    return np.moveaxis(wl.cons_from_prim(rho, p, v, GAMMA, B=B, psi=psi), 0, 1).copy()


def existing(g, level, slot, cfl):
    """The existing path: (dt, max signal speed) of amrhydro_cfl_dt."""
    import ctypes as C
    dt, s = C.c_double(0), C.c_double(0)
    g._ok(g.L.amrhydro_cfl_dt(g.h, level, slot, cfl, C.byref(dt), C.byref(s)))
    return dt.value, s.value


def noalloc(gpu, g, slot, first, count, dtype, cfl_dx, out, **kw):
    import torch
    g.sync()
    out.fill_(-7.0)                                   # a call must write all three outputs
    gpu.cfl_dt_noalloc(g.patch_ptr(slot, first), count, g.nv, BITS[dtype], GAMMA, cfl_dx, out.data_ptr(),
                       stream=torch.cuda.current_stream().cuda_stream, **kw)
    torch.cuda.synchronize()
    s, dt, flag = out.cpu().numpy()
    return dt, s, flag


def close(a, b, tol):
    return abs(a - b) <= tol * abs(b)


CASES = [(5, "f64"), (5, "f32"), (8, "f64"), (9, "f64"), (9, "f32")]


@pytest.mark.parametrize("nv,dtype", CASES, ids=["nv%d-%s" % c for c in CASES])
def test_noalloc_cfl_matches_existing_path_on_calls_in_a_row(gpu, nv, dtype):
    import torch
    cfl = 0.3
    kw = dict(ch=1.7) if nv == 9 else {}
    big = wl.uniform_hierarchy(3, periodic=True)                    # 27 patches
    small = wl.uniform_hierarchy(2, periodic=True)                  # 8 patches
    gb = gpu.AmrHydro(big, GAMMA, nv, dtype=dtype, **kw)
    gs = gpu.AmrHydro(small, GAMMA, nv, dtype=dtype, **kw)
    gb.upload(0, state(27, nv, 11, 0.9))                            # fast
    gb.upload(1, state(27, nv, 12, 0.4))                            # slower
    gs.upload(0, state(8, nv, 13, 0.05))                            # slowest, fewest patches
    want = [existing(gb, 0, 0, cfl), existing(gb, 0, 1, cfl), existing(gs, 0, 0, cfl)]
    assert want[0][1] > want[1][1] > want[2][1] > 0
    gpu.noalloc_setup()
    out = torch.zeros(3, dtype=torch.float64, device="cuda:0")
    got = [noalloc(gpu, gb, 0, 0, 27, dtype, cfl * big["dx0"], out, **kw),
           noalloc(gpu, gb, 1, 0, 27, dtype, cfl * big["dx0"], out, **kw),
           noalloc(gpu, gs, 0, 0, 8, dtype, cfl * small["dx0"], out, **kw),
           noalloc(gpu, gb, 0, 0, 27, dtype, cfl * big["dx0"], out, **kw)]
    for (dt, s, flag), (dt0, s0) in zip(got, want + want[:1]):
        assert flag == 0.0
        assert close(s, s0, TOL[dtype]) and close(dt, dt0, TOL[dtype]), (s, s0, dt, dt0)
        assert s == s0                                              # max is exact in any order: expected bitwise
    # a sub-range of the pool: the maximum over patches 5..15 alone, against the maximum over the whole level
    dt, s, flag = noalloc(gpu, gb, 1, 5, 11, dtype, cfl * big["dx0"], out, **kw)
    assert flag == 0.0 and 0 < s <= want[1][1]


def test_noalloc_cfl_flags_non_finite_input_and_recovers(gpu):
    import torch
    h = wl.uniform_hierarchy(2, periodic=True)
    g = gpu.AmrHydro(h, GAMMA, 5)
    U = state(8, 5, 3, 0.4)
    g.upload(0, U)
    dt0, s0 = existing(g, 0, 0, 0.3)
    Ubad = U.copy()
    Ubad[6, 2, 3, 4, 5] = np.nan
    g.upload(1, Ubad)
    with pytest.raises(gpu.AmrHydroError):                          # the existing path: AMRHYDRO_ENONFINITE
        existing(g, 0, 1, 0.3)
    out = torch.zeros(3, dtype=torch.float64, device="cuda:0")
    dt, s, flag = noalloc(gpu, g, 1, 0, 8, "f64", 0.3 * h["dx0"], out)
    assert flag == 1.0 and np.isinf(s) and dt == 0.0
    dt, s, flag = noalloc(gpu, g, 0, 0, 8, "f64", 0.3 * h["dx0"], out)     # the next call is clean again
    assert flag == 0.0 and s == s0 and close(dt, dt0, 1e-12)


def test_noalloc_cfl_rejects_bad_arguments_without_launching(gpu):
    import torch
    h = wl.uniform_hierarchy(1, periodic=True)
    g = gpu.AmrHydro(h, GAMMA, 5)
    g.upload(0, state(1, 5, 5, 0.4))
    out = torch.full((3,), -7.0, dtype=torch.float64, device="cuda:0")
    ptr, o = g.patch_ptr(0, 0), out.data_ptr()
    with pytest.raises(gpu.AmrHydroError, match="exceeds AMRHYDRO_NOALLOC_MAX_PATCHES"):
        gpu.cfl_dt_noalloc(ptr, gpu.NOALLOC_MAX_PATCHES + 1, 5, 64, GAMMA, 0.1, o)
    for bad in (dict(npatches=0), dict(nvars=6), dict(dtype_bits=16), dict(gamma=1.0), dict(dev_patches=None),
                dict(dev_out=None), dict(rho_floor=0.0), dict(dev_patches=ptr + 4)):
        a = dict(dev_patches=ptr, npatches=1, nvars=5, dtype_bits=64, gamma=GAMMA, cfl_dx=0.1, dev_out=o)
        a.update(bad)
        with pytest.raises(gpu.AmrHydroError):
            gpu.cfl_dt_noalloc(**a)
    torch.cuda.synchronize()
    assert (out.cpu().numpy() == -7.0).all()                        # nothing ran
    dt, s, flag = noalloc(gpu, g, 0, 0, 1, "f64", 0.1, out)
    assert flag == 0.0 and s == existing(g, 0, 0, 0.3)[1]


def test_noalloc_cfl_at_the_maximum_size(gpu):
    """AMRHYDRO_NOALLOC_MAX_PATCHES = 32768 patches (512^3 cells, fp32: a 6.3 GB slot), inputs written into the pool in
    its own layout on the device, twice in a row, and a smaller call after it."""
    import torch
    n = gpu.NOALLOC_MAX_PATCHES
    h = wl.uniform_hierarchy(32, periodic=True)
    assert len(h["level"]) == n
    g = gpu.AmrHydro(h, GAMMA, 5, dtype="f32", nslots=1)
    per = int(g.L.amrhydro_pool_bytes(g.h, 1, 1)) // 4              # elements per patch
    pool = g.pool.view(torch.float32).view(n, 5, per // 5)
    gen = torch.Generator(device="cuda:0").manual_seed(2024)
    chunk = 4096
    for a in range(0, n, chunk):                                    # rho, momenta, total energy with e > 0 everywhere
        shp = (chunk, per // 5)
        pool[a:a + chunk, 0] = 0.5 + torch.rand(shp, generator=gen, device="cuda:0")
        for v in (1, 2, 3):
            pool[a:a + chunk, v] = 0.6 * torch.rand(shp, generator=gen, device="cuda:0") - 0.3
        pool[a:a + chunk, 4] = 2.0 + torch.rand(shp, generator=gen, device="cuda:0")
    torch.cuda.synchronize()
    dt0, s0 = existing(g, 0, 0, 0.3)
    out = torch.zeros(3, dtype=torch.float64, device="cuda:0")
    for _ in range(2):
        dt, s, flag = noalloc(gpu, g, 0, 0, n, "f32", 0.3 * h["dx0"], out)
        assert flag == 0.0 and s == s0 and close(dt, dt0, TOL["f32"])
    dt, s, flag = noalloc(gpu, g, 0, 100, 7, "f32", 0.3 * h["dx0"], out)
    assert flag == 0.0 and 0 < s <= s0
