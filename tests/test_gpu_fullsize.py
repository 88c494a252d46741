"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times
(direct sibling halos, default stage kernel), on sampled patches the oracle can compute one by one.

One RK2 step of a patch depends on data within 4 cells of it (2 per stage), so the oracle run on
the 3x3x3 block of patches around a sampled patch (48^3 cells, made periodic: its outer wrap is
more than 4 cells away from the centre patch) reproduces that patch of the full-size run exactly.
The time step is the GPU's own cfl_dt of the full level, checked against the oracle's max wave
speed on the sampled blocks (which can only be smaller or equal).
"""
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


def block_around(G, bx, by, bz, nb):
    """48^3 cells (3x3x3 patches) of the periodic global array G[nv][z][y][x] centred on patch (bx,by,bz)."""
    idx = lambda b: np.arange((b - 1) * 16, (b + 2) * 16) % (nb * 16)
    return G[:, idx(bz)][:, :, idx(by)][:, :, :, idx(bx)]


def check_fullsize(gpu, G, gamma, nv, dtype, nsample, seed, tol, cfl=0.3):
    import oracle
    n = G.shape[-1]
    nb = n // 16
    h = wl.uniform_hierarchy(nb, periodic=True)
    U = wl.split_global(h, G)
    if dtype == "f32":
        U = U.astype(np.float32)
        G = G.astype(np.float32).astype(np.float64)      # S15: the oracle starts from the rounded data
    g = gpu.AmrHydro(h, gamma, nv, dtype=dtype, halo=1)
    g.upload(0, U)
    del U
    dt = g.cfl_dt(0, 0, cfl)
    g.fill_ghosts(0, 0)
    g.rk_stage(0, 0, 0, 1, 0.0, 1.0, dt)
    g.fill_ghosts(0, 1)
    g.rk_stage(0, 1, 0, 0, 0.5, 0.5, dt)
    assert g.get_counter(gpu.CNT_FLOOR_HITS) == 0
    org = np.asarray(h["origin"]) // 16
    rng = np.random.default_rng(seed)
    picks = list(rng.choice(len(org), size=nsample - 2, replace=False)) + [0, len(org) - 1]   # incl. wrap-around patches
    hb = wl.build_hierarchy((3, 3, 3), (), (0,) * 6, box=48.0 / n, order="linear")   # periodic, same cell size as the full level
    assert abs(hb["dx0"] - 1.0 / n) < 1e-15 / n
    ob = np.asarray(hb["origin"]) // 16
    centre = int(np.where((ob == 1).all(axis=1))[0][0])
    smax, worst = 0.0, 0.0
    for p in picks:
        bx, by, bz = (int(x) for x in org[p])
        o = oracle.Oracle(hb, gamma, nv, threads=8)
        o.upload(0, wl.split_global(hb, np.ascontiguousarray(block_around(G, bx, by, bz, nb))))
        smax = max(smax, o.max_speed(0))
        o.fill_ghosts(0, 0)
        o.rk_stage(0, 0, 0, 1, 0.0, 1.0, dt)
        o.fill_ghosts(0, 1)
        o.rk_stage(0, 1, 0, 0, 0.5, 0.5, dt)
        O = o.download(0)[centre:centre + 1]
        Gp = g.download(0, int(p), 1).astype(np.float64)
        worst = max(worst, norm_err(Gp, O, vector=(dtype == "f32")).max())
    dx = 1.0 / n
    assert dt <= cfl * dx / smax * (1 + 1e-6)            # the level-wide maximum bounds every sampled block
    assert worst <= tol, worst


@pytest.mark.parametrize("dtype,tol", [("f64", 1e-12), ("f32", 1e-5)])
def test_config5_stress_512_sampled(gpu, dtype, tol):
    G = wl.stress_global(512, gamma=1.4, seed=20005)
    check_fullsize(gpu, G, 1.4, 5, dtype, nsample=8, seed=5, tol=tol)


@pytest.mark.parametrize("dtype,tol", [("f64", 1e-12), ("f32", 1e-5)])
def test_config2_kelvin_helmholtz_256_sampled(gpu, dtype, tol):
    G = wl.kelvin_helmholtz_global(256, gamma=5.0 / 3.0, seed=20002)
    check_fullsize(gpu, G, 5.0 / 3.0, 5, dtype, nsample=8, seed=2, tol=tol)


def test_config4_mhd_128_sampled(gpu):
    G = wl.mhd_turbulence_global(128, gamma=5.0 / 3.0, seed=20004)
    check_fullsize(gpu, G, 5.0 / 3.0, 8, "f64", nsample=8, seed=4, tol=1e-12)
