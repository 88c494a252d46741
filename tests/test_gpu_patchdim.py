"""Patches of 32^3, 48^3 and 64^3 cells: amrhydro_create(patch_dim = 16 s) holds
each as s^3 patches of 16^3.  The scheme is defined on cells, so the bar is the oracle on the equivalent 16^3
hierarchy (1e-12) and bitwise equality with the GPU's own 16^3 run."""
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


def to16(hD, h16, UD):
    """Data of a hierarchy of D^3 patches re-cut into the equivalent 16^3 hierarchy's patches."""
    D = hD["ni"]
    where = {(int(l), tuple(int(c) for c in o)): p for p, (l, o) in enumerate(zip(hD["level"], hD["origin"]))}
    out = np.zeros((len(h16["level"]), UD.shape[1], 16, 16, 16), UD.dtype)
    for q, (l, o) in enumerate(zip(h16["level"], h16["origin"])):
        base = tuple(int(c) // D * D for c in o)
        p = where[(int(l), base)]
        x, y, z = (int(o[d]) - base[d] for d in range(3))
        out[q] = UD[p][:, z:z + 16, y:y + 16, x:x + 16]
    return out


def blob(h, nv=5, seed=0):
    rng = np.random.default_rng(seed)
    out = []
    for p in range(len(h["level"])):
        x, y, z = wl.cell_centres(h, p)
        Z, Y, X = np.meshgrid(z, y, x, indexing="ij")
        r2 = (X - 0.5) ** 2 + (Y - 0.45) ** 2 + (Z - 0.55) ** 2
        rho = 1 + 3 * np.exp(-r2 / 0.04)
        p_ = 1 + 2 * np.exp(-r2 / 0.02)
        B = (0.3 + 0 * rho, 0.2 * np.sin(2 * np.pi * X), 0.1 * np.cos(2 * np.pi * Y)) if nv >= 8 else None
        out.append(wl.cons_from_prim(rho, p_, (0.2 * np.sin(2 * np.pi * Y), 0.1 + 0 * rho, -0.2 * np.cos(2 * np.pi * X)), 1.4, B=B))
    return np.stack(out)


@pytest.mark.parametrize("D,dtype", [(32, "f64"), (32, "f32"), (48, "f64"), (64, "f64")])
def test_uniform_level_of_large_patches(gpu, D, dtype):
    import oracle
    nb = 2
    n = nb * D
    hD = wl.build_hierarchy((nb,) * 3, (), (0,) * 6, ni=D)
    h16 = wl.uniform_hierarchy(n // 16, periodic=True)
    G = wl.stress_global(n, seed=7)
    UD, U16 = wl.split_global(hD, G), wl.split_global(h16, G)
    assert UD.shape[-1] == D and np.array_equal(to16(hD, h16, UD), U16)
    if dtype == "f32":
        UD, U16 = (x.astype(np.float32).astype(np.float64) for x in (UD, U16))
    g = gpu.AmrHydro(hD, 1.4, 5, dtype=dtype)
    g16 = gpu.AmrHydro(h16, 1.4, 5, dtype=dtype)
    o = oracle.Oracle(h16, 1.4, 5, threads=8)
    g.upload(0, UD); g16.upload(0, U16); o.upload(0, U16)
    for _ in range(3):
        dt = o.advance(0.3)
        assert abs(g.advance(0.3) - dt) <= (1e-12 if dtype == "f64" else 2e-6) * dt
        g16.advance(0.3)
    out = g.download(0)
    assert out.shape == (nb ** 3, 5, D, D, D)
    assert np.array_equal(to16(hD, h16, out), g16.download(0))                 # the decomposition changes no bit
    assert norm_err(to16(hD, h16, out).astype(np.float64), o.download(0), vector=(dtype == "f32")).max() <= (1e-12 if dtype == "f64" else 1e-5)


@pytest.mark.parametrize("nv", [5, 8])
def test_refined_hierarchy_of_32_cubed_patches(gpu, nv):
    """Two levels of 32^3 patches (subcycling, prolongation, restriction, refluxing through the sub-patch tables)."""
    import oracle
    fine32 = [(i, j, k) for i in (1, 2) for j in (1, 2) for k in (1, 2)]
    fine16 = [(i, j, k) for i in range(2, 6) for j in range(2, 6) for k in range(2, 6)]
    h32 = wl.build_hierarchy((2, 2, 2), [fine32], (0,) * 6, ni=32)
    h16 = wl.build_hierarchy((4, 4, 4), [fine16], (0,) * 6)
    U32, U16 = blob(h32, nv), blob(h16, nv)
    assert np.array_equal(to16(h32, h16, U32), U16)
    g = gpu.AmrHydro(h32, 1.4, nv)
    o = oracle.Oracle(h16, 1.4, nv, threads=8)
    g.upload(0, U32); o.upload(0, U16)
    g.restrict(1); o.restrict(1)
    for _ in range(2):
        dt = o.advance(0.3)
        assert abs(g.advance(0.3) - dt) <= 1e-12 * dt
    out = to16(h32, h16, g.download(0))
    assert np.isfinite(out).all() and norm_err(out, o.download(0)).max() <= 1e-12
    # partial ranges of the caller's patches
    part = g.download(0, 3, 4)
    assert part.shape == (4, nv, 32, 32, 32) and np.array_equal(part, g.download(0)[3:7])
    g.upload(0, U32[5:7], first=5)
    assert np.array_equal(g.download(0, 5, 2), U32[5:7])


def test_patch_dim_error_behaviour(gpu):
    h16 = wl.uniform_hierarchy(2, periodic=True)
    for bad in (8, 24, 80):
        with pytest.raises(gpu.AmrHydroError):
            gpu.AmrHydro(h16, 1.4, 5, patch_dim=bad)
    h32 = wl.build_hierarchy((2, 2, 2), (), (0,) * 6, ni=32)
    g = gpu.AmrHydro(h32, 1.4, 5)
    assert g.npatch == 8
    for call in (lambda: g.refine_indicator(0), lambda: g.prolong_interior(1), lambda: g.download_padded(0, 0),
                 lambda: g.download_registers(0), lambda: g.set_owned(4)):
        with pytest.raises(gpu.AmrHydroError):
            call()
    with pytest.raises(gpu.AmrHydroError):
        g.download(0, 7, 2)                                                  # ranges count the caller's patches
    bad = dict(h32); bad["origin"] = h32["origin"] + 16                      # origins must be multiples of patch_dim
    with pytest.raises(gpu.AmrHydroError):
        gpu.AmrHydro(bad, 1.4, 5)
