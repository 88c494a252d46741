"""Patch sharding on one GPU: the level cut into Morton ranges, one pool per shard, face slabs
packed by k_halo_slabs, copied pool to pool (the stand-in for the NVLink peer copy) and unpacked into mirror patches
before every stage; dt from the maximum over shards.  Same kernels on the same data: the bar is bitwise equality with the
unsharded run, step sizes included."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from paper_0910_5547_b200 import sharding, workloads as wl  # noqa: E402


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (no CPU fallback exists)")
    from paper_0910_5547_b200 import binding
    binding.load_library()
    return binding


def single_run(gpu, h, U, gamma, nv, dtype, steps, cfl):
    g = gpu.AmrHydro(h, gamma, nv, dtype=dtype, halo=1)
    g.upload(0, U)
    dts = [g.advance(cfl) for _ in range(steps)]
    return g.download(0), dts


@pytest.mark.parametrize("nshards", [2, 3, 8])
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_config2_64_sharded_is_bitwise_the_single_pool_run(gpu, nshards, dtype):
    h = wl.uniform_hierarchy(4, periodic=True)
    U = wl.split_global(h, wl.kelvin_helmholtz_global(64))
    ref, dts = single_run(gpu, h, U, 5.0 / 3.0, 5, dtype, 3, 0.3)
    run = sharding.ShardedRun(gpu, h, nshards, 5.0 / 3.0, 5, dtype=dtype)
    run.upload(U)
    got = [run.step(0.3) for _ in range(3)]
    assert got == dts
    out = run.download()
    assert np.isfinite(out).all() and np.array_equal(out, ref)
    assert not np.array_equal(out, U.astype(out.dtype))


def test_sharded_mhd_and_outflow(gpu):
    """The 8-variable system (k_rk_stage_march) on two shards, and the Sod tube of config 1 with outflow boundaries
    (physical faces stay physical in a shard's table)."""
    h = wl.uniform_hierarchy(2, periodic=True)
    U = wl.split_global(h, wl.mhd_turbulence_global(32))
    ref, dts = single_run(gpu, h, U, 5.0 / 3.0, 8, "f64", 3, 0.3)
    run = sharding.ShardedRun(gpu, h, 2, 5.0 / 3.0, 8)
    run.upload(U)
    assert [run.step(0.3) for _ in range(3)] == dts
    assert np.array_equal(run.download(), ref)
    h = wl.uniform_hierarchy(2, periodic=False)
    U = wl.split_global(h, wl.sod_global(32))
    g = gpu.AmrHydro(h, 1.4, 5, halo=1)
    g.upload(0, U)
    run = sharding.ShardedRun(gpu, h, 2, 1.4, 5)
    run.upload(U)
    for _ in range(5):
        dt = g.cfl_dt(0, 0, 0.4)
        g.fill_ghosts(0, 0); g.rk_stage(0, 0, 0, 1, 0.0, 1.0, dt)
        g.fill_ghosts(0, 1); g.rk_stage(0, 1, 0, 0, 0.5, 0.5, dt)
        for s in run.g:
            s.fill_ghosts(0, 0)
        smax = max(s.max_speed(0, 0) for s in run.g)
        assert 0.4 * run.dx0 / smax == dt
        run.exchange(0)
        for s in run.g:
            s.rk_stage(0, 0, 0, 1, 0.0, 1.0, dt)
        for s in run.g:
            s.fill_ghosts(0, 1)
        run.exchange(1)
        for s in run.g:
            s.rk_stage(0, 1, 0, 0, 0.5, 0.5, dt)
    assert np.array_equal(run.download(), g.download(0))


def test_sharding_error_behaviour(gpu):
    h = wl.uniform_hierarchy(4, periodic=True)
    sh = sharding.build_shard(h, sharding.partition_morton(h, 8), 0)
    g = gpu.AmrHydro(sh["hier"], 1.4, 5)
    with pytest.raises(gpu.AmrHydroError):
        g.set_owned(0)
    with pytest.raises(gpu.AmrHydroError):
        g.set_owned(len(sh["glob"]))                      # a mirror patch has REMOTE faces: it cannot be owned
    g.set_owned(sh["owned"])
    with pytest.raises(gpu.AmrHydroError):
        g.set_halo_plan([(sh["owned"], 0)], [])           # sends owned patches only
    with pytest.raises(gpu.AmrHydroError):
        g.set_halo_plan([], [(0, 0)])                     # receives into mirrors only
    with pytest.raises(gpu.AmrHydroError):
        g.set_halo_plan([(0, 6)], [])
    g.set_halo_plan(sh["send"][1], sh["recv"][1])
    assert g.halo_bytes(0) == len(sh["send"][1]) * 5 * 512 * 8 and g.halo_bytes(1) == len(sh["recv"][1]) * 5 * 512 * 8
    amr = gpu.AmrHydro(wl.ball_hierarchy(2, 2, bc=(1,) * 6), 1.4, 5)
    with pytest.raises(gpu.AmrHydroError):
        amr.set_owned(4)                                  # refined hierarchies are not sharded in this build
