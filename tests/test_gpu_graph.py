"""amrhydro_advance as a CUDA-graph replay (AMRHYDRO_OPT_GRAPH; "a _device variant that leaves dt in
device memory is allowed for graph capture"): the S9 recursion captured once, dt0 formed on the device.  The bar is
bitwise equality with the eager path (same kernels, same arguments, same order), step sizes included."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from paper_0910_5547_b200 import workloads as wl  # noqa: E402


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (no CPU fallback exists)")
    from paper_0910_5547_b200 import binding
    binding.load_library()
    return binding


def state(h, nv, seed):
    rng = np.random.default_rng(seed)
    shp = (len(h["level"]), 16, 16, 16)
    rho, p = rng.uniform(0.5, 1.5, shp), rng.uniform(0.5, 1.5, shp)
    v = [rng.uniform(-0.4, 0.4, shp) for _ in range(3)]
    B = [rng.uniform(-0.3, 0.3, shp) for _ in range(3)] if nv >= 8 else None
    return np.moveaxis(wl.cons_from_prim(rho, p, v, 1.4, B=B), 0, 1).copy()


CASES = [("uniform periodic 3^3", lambda: wl.uniform_hierarchy(3, periodic=True), 5, "f64"),
         ("uniform periodic 2^3 fp32", lambda: wl.uniform_hierarchy(2, periodic=True), 5, "f32"),
         ("three nested levels, outflow", lambda: wl.ball_hierarchy(2, 3, bc=(1,) * 6), 5, "f64"),
         ("three nested levels, MHD", lambda: wl.ball_hierarchy(2, 3, bc=(1,) * 6), 8, "f64"),
         ("two levels periodic fp32", lambda: wl.build_hierarchy((2, 2, 2), [[(i, j, k) for i in (1, 2) for j in (1, 2) for k in (1, 2)]], (0,) * 6), 5, "f32")]


@pytest.mark.parametrize("name,mk,nv,dtype", CASES, ids=[c[0] for c in CASES])
def test_graph_replay_is_bitwise_the_eager_step(gpu, name, mk, nv, dtype):
    h = mk()
    U = state(h, nv, 7)
    ge = gpu.AmrHydro(h, 1.4, nv, dtype=dtype, graph=0)
    gg = gpu.AmrHydro(h, 1.4, nv, dtype=dtype, graph=1)
    for g in (ge, gg):
        g.upload(0, U)
        for l in range(h["nlevels"] - 1, 0, -1):
            g.restrict(l)
    nsteps = 5
    dte = [ge.advance(0.3) for _ in range(nsteps)]
    dtg = [gg.advance(0.3) for _ in range(nsteps)]
    assert dte == dtg                                                   # bitwise the same step sizes
    assert gg.get_counter(gpu.CNT_GRAPH_REPLAYS) == nsteps - 1         # the first step configures the kernels eagerly
    assert ge.get_counter(gpu.CNT_GRAPH_REPLAYS) == 0
    assert ge.get_counter(gpu.CNT_LAUNCHES) > 0
    E, G = ge.download(0), gg.download(0)
    assert np.isfinite(E).all() and not np.array_equal(E, U.astype(E.dtype))
    assert np.array_equal(E, G)
    # without the host read of dt the replay does not synchronise; same bits again
    for _ in range(3):
        ge.advance(0.3)
        gg.advance(0.3, want_dt=False)
    assert np.array_equal(ge.download(0), gg.download(0))
    # a fixed step and a changed option (re-capture) stay bitwise too
    for g in (ge, gg):
        g.set_option(gpu.OPT_THETA, 1.0)
    a, b = ge.advance(0.3, 1e-4), gg.advance(0.3, 1e-4)
    assert a == b == 1e-4
    assert np.array_equal(ge.download(0), gg.download(0))


def test_graph_reports_non_finite_speed(gpu):
    h = wl.uniform_hierarchy(2, periodic=True)
    U = state(h, 5, 3)
    g = gpu.AmrHydro(h, 1.4, 5, graph=1)
    g.upload(0, U)
    g.advance(0.3)
    g.advance(0.3)
    U[3, 1, 4, 5, 6] = np.nan
    g.upload(0, U)
    with pytest.raises(gpu.AmrHydroError):
        g.advance(0.3)


def test_cfl_dt_device_leaves_dt_on_the_device(gpu):
    """amrhydro_cfl_dt_device: the same number as amrhydro_cfl_dt, bit for bit, without a host read (read back here with
    a plain cudaMemcpy), for one level and as the dt0 of a whole hierarchy (S4); the flag reports a NaN."""
    cudart = pytest.importorskip("cuda.cudart")
    import ctypes

    def read(ptr):
        buf = (ctypes.c_double * 2)()
        err, = cudart.cudaMemcpy(ctypes.addressof(buf), ptr, 16, cudart.cudaMemcpyKind.cudaMemcpyDeviceToHost)
        assert int(err) == 0
        return buf[0], buf[1]

    h = wl.ball_hierarchy(2, 3, bc=(1,) * 6)
    U = state(h, 5, 9)
    g = gpu.AmrHydro(h, 1.4, 5)
    g.upload(0, U)
    for lev in range(3):
        dt, flag = read(g.cfl_dt_device(lev, lev, 0, 0.3))
        assert flag == 0.0 and dt == g.cfl_dt(lev, 0, 0.3)
    dt0, flag = read(g.cfl_dt_device(0, 2, 0, 0.3))
    assert flag == 0.0 and dt0 == g.advance(0.3)                   # the step amrhydro_advance takes
    U[5, 0, 1, 2, 3] = np.nan
    g.upload(0, U)
    assert read(g.cfl_dt_device(0, 2, 0, 0.3))[1] == 1.0
    with pytest.raises(gpu.AmrHydroError):
        g.cfl_dt_device(2, 1, 0, 0.3)
