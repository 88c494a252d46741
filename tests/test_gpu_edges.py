"""GPU edge cases of the C ABI against the oracle: error behaviour, empty ranges, non-cubic and
one-patch-thick base grids, a level with a single patch, AMR in fp32 and with direct sibling halos
(the launch configuration bench.py uses for config 3)."""
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


def rand_state(h, nv, seed, gamma=1.4):
    rng = np.random.default_rng(seed)
    shp = (len(h["level"]), 16, 16, 16)
    rho = rng.uniform(0.5, 1.5, shp); p = rng.uniform(0.5, 1.5, shp)
    v = [rng.uniform(-0.5, 0.5, shp) for _ in range(3)]
    B = [rng.uniform(-0.5, 0.5, shp) for _ in range(3)] if nv >= 8 else None
    return np.moveaxis(wl.cons_from_prim(rho, p, v, gamma, B=B), 0, 1).copy()


def pair(gpu, h, gamma, nv, dtype="f64", **kw):
    import oracle
    return gpu.AmrHydro(h, gamma, nv, dtype=dtype, **kw), oracle.Oracle(h, gamma, nv, threads=8)


def test_errors_are_reported_and_do_not_poison_the_handle(gpu):
    h = wl.uniform_hierarchy(1, periodic=True)
    g = gpu.AmrHydro(h, 1.4, 5)
    U = rand_state(h, 5, 1)
    g.upload(0, U)
    bad = [lambda: g.rk_stage(0, 0, 0, 0, 0.0, 1.0, 1e-3),        # slot_out == slot_in
           lambda: g.rk_stage(0, 0, 0, 7, 0.0, 1.0, 1e-3),        # slot out of range
           lambda: g.rk_stage(3, 0, 0, 1, 0.0, 1.0, 1e-3),        # level out of range
           lambda: g.fill_ghosts(-1, 0),
           lambda: g.cfl_dt(0, 9, 0.3),
           lambda: g.restrict(1),                                  # no fine level
           lambda: g.set_option(gpu.OPT_THETA, 2.5),
           lambda: g.set_option(gpu.OPT_KERNEL, 11),
           lambda: g.set_option(99, 1.0),
           lambda: g.upload(0, np.concatenate([U, U]))]            # more patches than the hierarchy holds
    for f in bad:
        with pytest.raises(gpu.AmrHydroError):
            f()
    g.fill_ghosts(0, 0)
    g.rk_stage(0, 0, 0, 1, 0.0, 1.0, 1e-3)                         # still usable
    assert np.isfinite(g.download(1)).all()
    g.upload(0, U[:0])                                             # empty ranges are no-ops
    assert g.download(0, 0, 0).shape == (0, 5, 16, 16, 16)
    assert np.array_equal(g.download(0), U)
    assert g.L.amrhydro_create(1.0, 5, 16, 2) is None and g.L.amrhydro_create(1.4, 7, 16, 2) is None
    assert g.L.amrhydro_create(1.4, 5, 24, 2) is None and g.L.amrhydro_create(1.4, 5, 16, 3) is None    # (32, 48, 64 are valid: NEXT-4)


def test_set_hierarchy_rejects_tables_no_kernel_can_fill(gpu):
    """A physical-boundary entry on a periodic side (nothing would fill that ghost zone), a physical entry on an
    interior face, an interior entry on a boundary face, and a level-0 patch with a parent."""
    import copy
    h = wl.uniform_hierarchy(2, periodic=True)
    bad = copy.deepcopy(h); bad["nbr"] = h["nbr"].copy(); bad["nbr"][0, 12] = -2
    with pytest.raises(gpu.AmrHydroError):
        gpu.AmrHydro(bad, 1.4, 5)
    h = wl.uniform_hierarchy(2, periodic=False)
    gpu.AmrHydro(h, 1.4, 5)                                         # the generator's own table is accepted
    bad = copy.deepcopy(h); bad["nbr"] = h["nbr"].copy()
    p = int(np.argmax((h["origin"] == 0).all(axis=1)))              # the corner patch: its x-hi face is interior
    bad["nbr"][p, 14] = -2
    with pytest.raises(gpu.AmrHydroError):
        gpu.AmrHydro(bad, 1.4, 5)
    bad = copy.deepcopy(h); bad["nbr"] = h["nbr"].copy(); bad["nbr"][p, 12] = int(h["nbr"][p, 14])   # x-lo is on the boundary
    with pytest.raises(gpu.AmrHydroError):
        gpu.AmrHydro(bad, 1.4, 5)
    bad = copy.deepcopy(h); bad["parent"] = h["parent"].copy(); bad["parent"][0] = 1
    with pytest.raises(gpu.AmrHydroError):
        gpu.AmrHydro(bad, 1.4, 5)


@pytest.mark.parametrize("nb,periodic", [((3, 1, 2), True), ((1, 1, 1), False), ((1, 4, 1), False)])
@pytest.mark.parametrize("halo", [0, 1])
def test_non_cubic_and_one_patch_thick_grids(gpu, nb, periodic, halo):
    h = wl.uniform_hierarchy(nb, periodic=periodic)
    g, o = pair(gpu, h, 1.4, 5, halo=halo)
    U = rand_state(h, 5, 2)
    g.upload(0, U); o.upload(0, U)
    for _ in range(3):
        dt = o.advance(0.3)
        assert abs(g.advance(0.3) - dt) <= 1e-13 * dt
    assert norm_err(g.download(0), o.download(0)).max() <= 1e-12


def single_child_hierarchy():
    return wl.build_hierarchy((2, 2, 2), [[(1, 2, 1)]], (0,) * 6)     # one fine patch = one octant of one coarse patch


@pytest.mark.parametrize("halo", [0, 1])
def test_level_with_a_single_patch(gpu, halo):
    h = single_child_hierarchy()
    assert int((np.asarray(h["level"]) == 1).sum()) == 1
    g, o = pair(gpu, h, 1.4, 5, halo=halo)
    U = rand_state(h, 5, 3)
    g.upload(0, U); o.upload(0, U)
    for x in (g, o):
        x.restrict(1)
    for _ in range(2):
        dt = o.advance(0.3)
        g.advance(0.3, dt)
    assert norm_err(g.download(0), o.download(0)).max() <= 1e-12


@pytest.mark.parametrize("dtype,halo", [("f64", 1), ("f32", 0), ("f32", 1)])
def test_sedov_amr_fp32_and_direct_halos(gpu, dtype, halo):
    """config 3 reduced (32^3 base + 3 levels), in the bench's launch configuration (halo = 1) and in fp32."""
    h = wl.ball_hierarchy(2, 4, bc=(1,) * 6)
    g, o = pair(gpu, h, 1.4, 5, dtype, halo=halo)
    U = wl.sedov_hierarchy_state(h)
    if dtype == "f32":
        U = U.astype(np.float32).astype(np.float64)
    g.upload(0, U); o.upload(0, U)
    for _ in range(2):
        dt = o.advance(0.3)
        g.advance(0.3, dt)
    G, O = g.download(0).astype(np.float64), o.download(0)
    assert np.isfinite(G).all()
    assert norm_err(G, O, vector=(dtype == "f32"), label="Sedov AMR 32^3+2 halo=%d" % halo).max() <= (1e-12 if dtype == "f64" else 1e-5)


@pytest.mark.parametrize("dtype,nv", [("f64", 5), ("f32", 5), ("f64", 8), ("f64", 9)])
def test_whole_path_is_bitwise_reproducible(gpu, dtype, nv):
    """Race detector of last resort (compute-sanitizer is closed on this pool): the same inputs through the
    whole path three times, on a grid of several waves of CTAs and on an AMR hierarchy, give the same bits."""
    cases = [(wl.uniform_hierarchy(4, periodic=True), dict(halo=1)), (wl.ball_hierarchy(2, 4, bc=(1,) * 6), dict(halo=1)),
             (wl.ball_hierarchy(2, 3, bc=(1,) * 6), dict(halo=0))]
    for h, kw in cases:
        U = rand_state(h, nv, 17)
        if nv == 9:
            U = np.concatenate([U, 0.05 * np.random.default_rng(18).standard_normal(U[:, :1].shape)], axis=1)
        outs = []
        for rep in range(3):
            g = gpu.AmrHydro(h, 1.4, nv, dtype=dtype, **kw)
            g.upload(0, U)
            if h["nlevels"] > 1:
                for lev in range(h["nlevels"] - 1, 0, -1):
                    g.restrict(lev)
            for _ in range(3):
                g.advance(0.3)
            outs.append(g.download(0))
            assert np.isfinite(outs[-1]).all()
        assert np.array_equal(outs[0], outs[1]) and np.array_equal(outs[0], outs[2])


def test_periodic_conservation_on_the_gpu_over_many_steps(gpu):
    """P6 on the device path: mass, momentum and energy of a periodic box (config 5 recipe, 128^3, 512 patches) are
    conserved to round-off over 20 steps (each face flux is computed by both neighbouring patches and must be the
    same bits for this to hold), and the state stays finite at CFL 0.3 (S4)."""
    n = 128
    h = wl.uniform_hierarchy(n // 16, periodic=True)
    U = wl.split_global(h, wl.stress_global(n, gamma=1.4, seed=20005))
    g = gpu.AmrHydro(h, 1.4, 5, halo=1)
    g.upload(0, U)
    t0 = U.sum(axis=(0, 2, 3, 4))
    scale = np.abs(U).sum(axis=(0, 2, 3, 4))
    for _ in range(20):
        g.advance(0.3)
    R = g.download(0)
    assert np.isfinite(R).all() and g.get_counter(gpu.CNT_FLOOR_HITS) == 0
    assert (np.abs(R.sum(axis=(0, 2, 3, 4)) - t0) <= 2e-14 * scale).all()
    assert np.abs(R - U).max() > 1e-2                    # it did evolve


def test_upload_download_round_trip_over_several_staging_chunks(gpu):
    """Ranges larger than the 256 MB staging chunk go through two alternating halves of the staging buffer (host copy of one
    chunk beside k_pack / k_unpack of the other): 4096 fp64 patches = 3 chunks, 5000 fp32 patches = 2, bit for bit, also
    for a sub-range that starts inside the second chunk."""
    for dtype, nb in (("f64", (16, 16, 16)), ("f32", (20, 25, 10))):
        h = wl.build_hierarchy(nb, (), (0,) * 6)
        n = len(h["level"])
        rng = np.random.default_rng(5)
        U = rng.standard_normal((n, 5, 16, 16, 16)).astype(np.float64 if dtype == "f64" else np.float32)
        g = gpu.AmrHydro(h, 1.4, 5, dtype=dtype, nslots=1)
        g.upload(0, U)
        assert np.array_equal(g.download(0), U)
        V = rng.standard_normal((1900, 5, 16, 16, 16)).astype(U.dtype)
        g.upload(0, V, first=1700)
        U[1700:3600] = V
        assert np.array_equal(g.download(0, 1650, 2000), U[1650:3650])
        del g
