"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times
(library defaults: direct sibling halos, default stage kernel, fused CFL reduction), on sampled patches
the oracle can compute one by one, over the run lengths of SURVEY.md 8(d): 10 steps (configs 2 and 4),
3 steps (config 5).

One RK2 step of a patch depends on data within 4 cells of it (2 per stage), k steps on 4k cells.  The oracle
run on the (2r+1)^3 block of patches around a sampled patch, r = ceil(4k/16), made periodic, reproduces that
patch of the full-size run exactly: the block's wrap-around is more than 4k cells from the centre patch
(r = 1: the 3^3 block up to 4 steps; r = 3: 7^3 patches for 10 steps).  Every step uses the GPU's own time
step of the full level (its fused / stand-alone CFL reduction), handed to the oracle, and checked against the
oracle's max wave speed on the sampled blocks (which can only be smaller or equal).
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


def block_around(G, bx, by, bz, nb, r):
    """(2r+1)^3 patches of the periodic global array G[nv][z][y][x] centred on patch (bx,by,bz)."""
    idx = lambda b: np.arange((b - r) * 16, (b + r + 1) * 16) % (nb * 16)
    return G[:, idx(bz)][:, :, idx(by)][:, :, :, idx(bx)]


def check_fullsize(gpu, G, gamma, nv, dtype, nsample, seed, tol, steps, label, cfl=0.3):
    import oracle
    n = G.shape[-1]
    nb = n // 16
    r = -(-4 * steps // 16)
    assert 2 * r + 1 <= nb
    h = wl.uniform_hierarchy(nb, periodic=True, order="zstrip")     # the table order bench.py launches
    U = wl.split_global(h, G)
    if dtype == "f32":
        U = U.astype(np.float32)
        G = G.astype(np.float32).astype(np.float64)      # S15: the oracle starts from the rounded data
    g = gpu.AmrHydro(h, gamma, nv, dtype=dtype)          # library defaults = what bench.py times
    g.upload(0, U)
    del U
    dts = [g.advance(cfl) for _ in range(steps)]         # the GPU's own dt of the full level, every step
    assert g.get_counter(gpu.CNT_FLOOR_HITS) == 0
    org = np.asarray(h["origin"]) // 16
    rng = np.random.default_rng(seed)
    picks = list(rng.choice(len(org), size=max(0, nsample - 2), replace=False)) + [0, len(org) - 1]   # incl. wrap-around patches
    m = 2 * r + 1
    hb = wl.build_hierarchy((m, m, m), (), (0,) * 6, box=16.0 * m / n, order="linear")   # periodic, same cell size as the full level
    assert abs(hb["dx0"] - 1.0 / n) < 1e-15 / n
    ob = np.asarray(hb["origin"]) // 16
    centre = int(np.where((ob == r).all(axis=1))[0][0])
    worst = 0.0
    for p in picks[:nsample]:
        bx, by, bz = (int(x) for x in org[p])
        o = oracle.Oracle(hb, gamma, nv, threads=16)
        o.upload(0, wl.split_global(hb, np.ascontiguousarray(block_around(G, bx, by, bz, nb, r))))
        for dt in dts:
            assert dt <= cfl * (1.0 / n) / o.max_speed(0) * (1 + 1e-6)   # the level-wide maximum bounds every sampled block
            o.advance(cfl, dt)
        O = o.download(0)[centre:centre + 1]
        Gp = g.download(0, int(p), 1).astype(np.float64)
        worst = max(worst, norm_err(Gp, O, vector=(dtype == "f32"), label=label).max())
    assert worst <= tol, worst


@pytest.mark.parametrize("dtype,tol", [("f64", 1e-12), ("f32", 1e-5)])
def test_config5_stress_512_sampled_3_steps(gpu, dtype, tol):
    G = wl.stress_global(512, gamma=1.4, seed=20005)
    check_fullsize(gpu, G, 1.4, 5, dtype, nsample=6, seed=5, tol=tol, steps=3, label="cfg5 512^3 3 steps")


@pytest.mark.parametrize("dtype,tol", [("f64", 1e-12), ("f32", 1e-5)])
def test_config2_kelvin_helmholtz_256_sampled_10_steps(gpu, dtype, tol):
    G = wl.kelvin_helmholtz_global(256, gamma=5.0 / 3.0, seed=20002)
    check_fullsize(gpu, G, 5.0 / 3.0, 5, dtype, nsample=3, seed=2, tol=tol, steps=10, label="cfg2 256^3 10 steps")


def test_config4_mhd_128_sampled_10_steps(gpu):
    G = wl.mhd_turbulence_global(128, gamma=5.0 / 3.0, seed=20004)
    check_fullsize(gpu, G, 5.0 / 3.0, 8, "f64", nsample=2, seed=4, tol=1e-12, steps=10, label="cfg4 128^3 10 steps")


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_large_run_is_bitwise_reproducible(gpu, dtype):
    """A timing-dependent hazard in the stage kernel (its CTA barriers are split mbarrier halves, its rings are refilled by
    TMA while other warps still compute) would show as run-to-run differences once thousands of CTAs compete for the SMs:
    config 5 at 256^3 (4096 patches, 14 waves), 12 steps, twice, on two pools -- every bit of the state and every dt equal."""
    G = wl.stress_global(256, seed=20005)
    h = wl.uniform_hierarchy(16, periodic=True)
    U = wl.split_global(h, G).astype(np.float64 if dtype == "f64" else np.float32)
    del G
    runs = []
    for rep in range(2):
        g = gpu.AmrHydro(h, 1.4, 5, dtype=dtype)
        g.upload(0, U)
        dts = [g.advance(0.3) for _ in range(12)]
        runs.append((dts, g.download(0)))
        del g
    assert runs[0][0] == runs[1][0]
    assert np.isfinite(runs[0][1]).all() and np.array_equal(runs[0][1], runs[1][1])
    assert not np.array_equal(runs[0][1], U)


def test_patch_order_does_not_change_a_bit(gpu):
    """bench.py launches the single-level workloads in "zstrip" table order (strips of 8 rows of patches, z outermost:
    sibling halos then hit in L2).  The order of the table is bookkeeping: the same field in Morton,
    linear and zstrip order gives bitwise the same patches and step sizes (config 5 at 128^3, 3 steps)."""
    G = wl.stress_global(128, seed=20005)
    res = {}
    for order in ("morton", "linear", "zstrip"):
        h = wl.uniform_hierarchy(8, periodic=True, order=order)
        g = gpu.AmrHydro(h, 1.4, 5)
        g.upload(0, wl.split_global(h, G))
        dts = [g.advance(0.3) for _ in range(3)]
        out = g.download(0)
        key = {tuple(int(c) for c in b): i for i, b in enumerate(np.asarray(h["blocks"]))}
        res[order] = (dts, out, key)
    assert [tuple(b) for b in np.asarray(wl.uniform_hierarchy(8, order="zstrip")["blocks"])[:3]] == [(0, 0, 0), (1, 0, 0), (2, 0, 0)]
    d0, o0, k0 = res["morton"]
    assert np.isfinite(o0).all()
    for order in ("linear", "zstrip"):
        d, o, k = res[order]
        assert d == d0
        perm = np.array([k[b] for b in sorted(k0, key=k0.get)])
        assert np.array_equal(o[perm], o0)


@pytest.mark.parametrize("nv", [8, 9])
def test_mhd_run_is_bitwise_reproducible(gpu, nv):
    """The same check for the 8- / 9-variable kernel (TMA rings of three or four slots refilled while other warps compute,
    primitives handed from pass to pass through shared memory, half-patch CTAs in the thin last wave): 216 patches = 1.46
    waves, 8 steps, twice on two pools -- every bit of the state and every dt equal."""
    h = wl.uniform_hierarchy(6, periodic=True, order="zstrip")
    G = wl.mhd_turbulence_global(96, gamma=5.0 / 3.0, seed=20004)
    if nv == 9:
        G = np.concatenate([G, np.zeros_like(G[:1])])
    U = wl.split_global(h, G)
    runs = []
    for rep in range(2):
        g = gpu.AmrHydro(h, 5.0 / 3.0, nv)
        g.upload(0, U)
        dts = [g.advance(0.3) for _ in range(8)]
        runs.append((dts, g.download(0)))
        del g
    assert runs[0][0] == runs[1][0]
    assert np.isfinite(runs[0][1]).all() and np.array_equal(runs[0][1], runs[1][1])
    assert not np.array_equal(runs[0][1], U)
