"""Seeded synthetic inputs shared by the CUDA path and the oracle's tests.

This module builds patch-descriptor tables (host-side hierarchy bookkeeping) and initial
conserved-variable arrays.  It contains none of the method's arithmetic (no reconstruction,
flux, update, ghost fill, prolongation, restriction or refluxing) and imports neither the
CUDA binding nor the oracle.  The only physics here is the definition of the conserved
variables (Eq. 2, Eq. 14) needed to state an initial condition
that the paper / BASELINE.json give in primitive form.

Recipes ("Input recipe"): BASELINE.json configs 1-5; Sod PAPER.md:260; Sedov
PAPER.md:266-272; Brio-Wu PAPER.md:341 (reading G4); spectrum P(k)~k^-2 PAPER.md:361.
None of these is a public benchmark dataset: every field is generated here from a seed.
"""
import numpy as np

NI = 16  # interior cells per patch side
FACE_REGION = (12, 14, 10, 16, 4, 22)  # x-lo x-hi y-lo y-hi z-lo z-hi in the 27-entry table
BC_PERIODIC, BC_OUTFLOW = 0, 1


# --------------------------------------------------------------------------- hierarchy
ZSTRIP_ROWS = 8      # 32 x 8 patches per z-layer of a strip at 512^3: one wave of the fp64 stage kernel (296 CTAs)


def _morton(b):
    key = 0
    for bit in range(10):
        for d in range(3):
            key |= ((int(b[d]) >> bit) & 1) << (3 * bit + d)
    return key


def build_hierarchy(base_blocks, refined=(), bc=(0,) * 6, box=1.0, order="morton", ni=NI):
    """Flat descriptor table of a block-structured hierarchy (refinement ratio 2).

    base_blocks: (nbx, nby, nbz) level-0 patches per axis (all exist).
    refined: for level 1, 2, ...: iterable of block coordinates (bx, by, bz) on that level
             (block b covers cells [16 b, 16 b + 16) of the level); each must be an octant
             of an existing patch one level down.
    bc: per face (x-lo, x-hi, y-lo, y-hi, z-lo, z-hi): 0 periodic, 1 outflow.
    ni: cells per patch side (16; 32, 48, 64 for amrhydro_create's larger patch_dim).
    Returns dict(level, origin, parent, nbr, nlevels, dx0, bc, blocks).
    nbr[p][r], r=(dz+1)*9+(dy+1)*3+(dx+1): >=0 same-level patch, -1 coarse-fine, -2 physical.
    """
    base_blocks = tuple(int(x) for x in base_blocks)
    levels = [[(i, j, k) for k in range(base_blocks[2]) for j in range(base_blocks[1])
               for i in range(base_blocks[0])]]
    for blocks in refined:
        levels.append(sorted(set(tuple(int(x) for x in b) for b in blocks)))
    if order == "morton":
        levels = [sorted(lv, key=_morton) for lv in levels]
    elif order == "zstrip":
        # launch order for large single-level runs (any order is a valid table): strips of ZSTRIP_ROWS rows of patches in
        # y; inside a strip z outermost, then y, then x.  One wave of CTAs is then about one z-layer of a strip: x and y
        # neighbours march in step and a patch starts roughly one wave after the patch below it, when that one has just
        # read the planes the two share -- the sibling-halo reads hit in L2 instead of DRAM
        def key(b, l):
            nx, nz = base_blocks[0] << l, base_blocks[2] << l
            return ((b[1] // ZSTRIP_ROWS) * nz + b[2]) * (ZSTRIP_ROWS * nx) + (b[1] % ZSTRIP_ROWS) * nx + b[0]
        levels = [sorted(lv, key=lambda b, l=l: key(b, l)) for l, lv in enumerate(levels)]
    elif order != "linear":
        raise ValueError("order must be morton, zstrip or linear")
    ids, pid = [], 0
    for lv in levels:
        m = {}
        for b in lv:
            m[b] = pid
            pid += 1
        ids.append(m)
    n = pid
    level = np.zeros(n, np.int32)
    origin = np.zeros((n, 3), np.int32)
    parent = np.full(n, -1, np.int32)
    nbr = np.full((n, 27), -1, np.int32)
    blocks = np.zeros((n, 3), np.int32)
    for l, lv in enumerate(levels):
        ext = [base_blocks[d] << l for d in range(3)]
        for b in lv:
            p = ids[l][b]
            level[p] = l
            blocks[p] = b
            origin[p] = [ni * x for x in b]
            if l > 0:
                pb = tuple(x >> 1 for x in b)
                if pb not in ids[l - 1]:
                    raise ValueError("patch %s on level %d has no parent" % (b, l))
                parent[p] = ids[l - 1][pb]
            for r in range(27):
                off = (r % 3 - 1, (r // 3) % 3 - 1, r // 9 - 1)
                q = [b[d] + off[d] for d in range(3)]
                outside = False
                for d in range(3):
                    if q[d] < 0 or q[d] >= ext[d]:
                        side = 2 * d + (1 if q[d] >= ext[d] else 0)
                        if bc[side] == BC_PERIODIC:
                            q[d] %= ext[d]
                        else:
                            outside = True
                nbr[p, r] = -2 if outside else ids[l].get(tuple(q), -1)
    h = dict(level=level, origin=origin, parent=parent, nbr=nbr, nlevels=len(levels),
             dx0=float(box) / (ni * base_blocks[0]), bc=np.asarray(bc, np.int32), blocks=blocks,
             base_blocks=base_blocks, ni=ni)
    _check_nesting(h)
    return h


def _check_nesting(h):
    """Every coarse cell touching a fine patch face must belong to a level-(l-1) patch."""
    for p in range(len(h["level"])):
        if h["level"][p] == 0:
            continue
        Q = h["parent"][p]
        for f in range(6):
            if h["nbr"][p, FACE_REGION[f]] != -1:
                continue
            d, hi = f // 2, f & 1
            rel = (h["origin"][p, d] - 2 * h["origin"][Q, d]) // h.get("ni", NI)  # octant bit along d
            on_parent_face = (rel == 1) if hi else (rel == 0)
            if on_parent_face and h["nbr"][Q, FACE_REGION[f]] < 0:
                raise ValueError("improper nesting at patch %d face %d" % (p, f))


def uniform_hierarchy(nblocks, periodic=True, order="morton"):
    nb = (nblocks,) * 3 if np.isscalar(nblocks) else tuple(nblocks)
    bc = (BC_PERIODIC,) * 6 if periodic else (BC_OUTFLOW,) * 6
    return build_hierarchy(nb, (), bc, order=order)


def ball_hierarchy(base_blocks, nlevels, radius_in_patches=1.5, centre=(0.5, 0.5, 0.5),
                   bc=(1,) * 6, order="morton"):
    """Fixed nested hierarchy: level l+1 holds the 16^3 blocks whose nearest point is closer
    than `radius_in_patches` level-(l+1) patch widths to `centre` (unit box).  Stand-in for
    config 3's "|grad rho|/rho > 0.1 max" criterion, which is degenerate at t=0 (S16)."""
    nb = (base_blocks,) * 3 if np.isscalar(base_blocks) else tuple(base_blocks)
    refined = []
    for l in range(1, nlevels):
        s = 1.0 / (nb[0] << l)  # patch width on level l
        ext = [x << l for x in nb]
        sel = []
        for bz in range(ext[2]):
            for by in range(ext[1]):
                for bx in range(ext[0]):
                    d2 = 0.0
                    for d, b in enumerate((bx, by, bz)):
                        lo, hi = b * s, (b + 1) * s
                        t = 0.0 if lo <= centre[d] <= hi else min(abs(centre[d] - lo), abs(centre[d] - hi))
                        d2 += t * t
                    if d2 < (radius_in_patches * s) ** 2 * (1 - 1e-12):
                        sel.append((bx, by, bz))
        refined.append(sel)
    return build_hierarchy(nb, refined, bc, order=order)


def blocks_hierarchy(path, base_blocks, bc=(1,) * 6, order="morton"):
    """Hierarchy from a block list written as text lines "level bx by bz" (levels >= 1; '#' comments).
    Config 3's criterion-built table (reading S16) is stored this way: tests/golden/cfg3_blocks.txt,
    written by tests/golden/make_cfg3_hierarchy.py."""
    nb = (base_blocks,) * 3 if np.isscalar(base_blocks) else tuple(base_blocks)
    per_level = {}
    with open(path) as f:
        for line in f:
            line = line.split("#")[0].split()
            if not line:
                continue
            l, bx, by, bz = (int(x) for x in line)
            per_level.setdefault(l, []).append((bx, by, bz))
    nlev = max(per_level) if per_level else 0
    refined = [per_level.get(l, []) for l in range(1, nlev + 1)]
    return build_hierarchy(nb, refined, bc, order=order)


def level_patches(h, l):
    return np.nonzero(h["level"] == l)[0]


def cell_centres(h, p):
    """(x, y, z) 1-D arrays of the interior cell centres of patch p (unit box)."""
    dx = h["dx0"] / (1 << int(h["level"][p]))
    return tuple((h["origin"][p, d] + np.arange(h.get("ni", NI)) + 0.5) * dx for d in range(3))


def split_global(h, G, l=0):
    """Cut a global [nv][nz][ny][nx] array of level l into [npatch_l][nv][ni][ni][ni] (ni = 16 unless the hierarchy says otherwise)."""
    ps = level_patches(h, l)
    ni = h.get("ni", NI)
    out = np.empty((len(ps), G.shape[0], ni, ni, ni), G.dtype)
    for n, p in enumerate(ps):
        ox, oy, oz = h["origin"][p]
        out[n] = G[:, oz:oz + ni, oy:oy + ni, ox:ox + ni]
    return out


def join_global(h, U, l=0):
    """Inverse of split_global for a fully covered level."""
    ps = level_patches(h, l)
    ext = [NI * (h["base_blocks"][d] << l) for d in range(3)]
    G = np.zeros((U.shape[1], ext[2], ext[1], ext[0]), U.dtype)
    for n, p in enumerate(ps):
        ox, oy, oz = h["origin"][p]
        G[:, oz:oz + NI, oy:oy + NI, ox:ox + NI] = U[n]
    return G


# --------------------------------------------------------------------------- initial data
def cons_from_prim(rho, p, v, gamma, B=None, psi=None):
    """U of Eq. 2 (Eq. 14 when B is given; its ninth slot when psi is given too) from primitive fields."""
    ke = 0.5 * rho * (v[0] ** 2 + v[1] ** 2 + v[2] ** 2)
    E = p / (gamma - 1.0) + ke
    comps = [rho, rho * v[0], rho * v[1], rho * v[2], E]
    if B is not None:
        comps[4] = E + 0.5 * (B[0] ** 2 + B[1] ** 2 + B[2] ** 2)
        comps += [B[0], B[1], B[2]]
        if psi is not None:
            comps.append(psi)
    return np.stack([np.broadcast_to(c, np.shape(rho)).astype(np.float64) for c in comps])


def _grid(n):
    x = (np.arange(n) + 0.5) / n
    return np.meshgrid(x, x, x, indexing="ij")  # returns Z, Y, X for [z][y][x] arrays


def sod_global(n=32, gamma=1.4, axis=0, x0=0.5):
    """Config 1 / PAPER.md:260.  axis: 0 x, 1 y, 2 z (P9 permutations)."""
    Z, Y, X = _grid(n)
    s = (X, Y, Z)[axis]
    left = s < x0
    rho = np.where(left, 1.0, 0.125)
    p = np.where(left, 1.0, 0.1)
    z = np.zeros_like(rho)
    return cons_from_prim(rho, p, (z, z, z), gamma)


def kelvin_helmholtz_global(n=256, gamma=5.0 / 3.0, seed=20002):
    """Config 2 (BASELINE.json): shear layer |y-0.5|<0.25, vy = 0.01 N(0,1) per cell."""
    rng = np.random.Generator(np.random.PCG64(seed))
    Z, Y, X = _grid(n)
    inner = np.abs(Y - 0.5) < 0.25
    rho = np.where(inner, 2.0, 1.0)
    vx = np.where(inner, 0.5, -0.5)
    vy = 0.01 * rng.standard_normal((n, n, n))
    p = np.full_like(rho, 2.5)
    return cons_from_prim(rho, p, (vx, vy, np.zeros_like(rho)), gamma)


def _kgrid(n):
    k1 = np.fft.fftfreq(n, 1.0 / n)
    kz, ky, kx = np.meshgrid(k1, k1, np.fft.rfftfreq(n, 1.0 / n), indexing="ij")
    return kz, ky, kx


def _irfftn(a, n):
    try:
        import scipy.fft as sf
        return sf.irfftn(a, s=(n, n, n), workers=-1)
    except Exception:  # pragma: no cover
        return np.fft.irfftn(a, s=(n, n, n))


def _rfftn(a):
    try:
        import scipy.fft as sf
        return sf.rfftn(a, workers=-1)
    except Exception:  # pragma: no cover
        return np.fft.rfftn(a)


def stress_global(n=512, gamma=1.4, seed=20005, mach=0.5, dtype=np.float64):
    """Config 5: rho, p = 1 + 0.1 N(0,1) (clipped at 0.1); velocity = Gaussian random field with
    E(k) ~ k^-2 (|v_k| ~ k^-2) rescaled to rms Mach `mach` w.r.t. c = sqrt(gamma)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    rho = np.maximum(1.0 + 0.1 * rng.standard_normal((n, n, n)), 0.1)
    p = np.maximum(1.0 + 0.1 * rng.standard_normal((n, n, n)), 0.1)
    kz, ky, kx = _kgrid(n)
    k2 = kx * kx + ky * ky + kz * kz
    k2[0, 0, 0] = 1.0
    amp = 1.0 / k2  # |v_k| ~ k^-2
    amp[0, 0, 0] = 0.0
    v = []
    for _ in range(3):
        w = _rfftn(rng.standard_normal((n, n, n)))
        v.append(_irfftn(w * amp, n))
        del w
    rms = np.sqrt(np.mean(v[0] ** 2 + v[1] ** 2 + v[2] ** 2))
    scale = mach * np.sqrt(gamma) / rms
    v = [c * scale for c in v]
    return cons_from_prim(rho, p, v, gamma).astype(dtype, copy=False)


def mhd_turbulence_global(n=128, gamma=5.0 / 3.0, seed=20004, rms=0.1):
    """Config 4: rho=1, p=1, B0=(1,0,0) + solenoidal random-phase dv, dB at 1<=|k|<=4, rms 0.1."""
    rng = np.random.Generator(np.random.PCG64(seed))
    kz, ky, kx = _kgrid(n)
    k2 = kx * kx + ky * ky + kz * kz
    mask = (k2 >= 1.0) & (k2 <= 16.0)
    k2s = np.where(k2 > 0, k2, 1.0)

    def field():
        comps = []
        for _ in range(3):
            ph = rng.uniform(0.0, 2.0 * np.pi, k2.shape)
            comps.append(np.where(mask, np.exp(1j * ph), 0.0))
        div = (kx * comps[0] + ky * comps[1] + kz * comps[2]) / k2s  # k (k.a)/k^2
        comps = [comps[0] - kx * div, comps[1] - ky * div, comps[2] - kz * div]
        real = [_irfftn(c, n) for c in comps]
        r = np.sqrt(np.mean(real[0] ** 2 + real[1] ** 2 + real[2] ** 2))
        return [c * (rms / r) for c in real]

    dv = field()
    dB = field()
    one = np.ones((n, n, n))
    return cons_from_prim(one, one, dv, gamma, B=(1.0 + dB[0], dB[1], dB[2]))


def sedov_hierarchy_state(h, gamma=1.4, E0=1.0, p_amb=1e-5):
    """Config 3: rho=1, p=1e-5, energy E0 spread over the finest-level cells whose centres lie
    within 2 finest cells of the box centre (32 cells when the centre is a cell corner);
    coarser levels hold the volume average of the finest data (S16).
    Returns U [npatch][5][16][16][16]."""
    n = len(h["level"])
    U = np.zeros((n, 5, NI, NI, NI))
    U[:, 0] = 1.0
    U[:, 4] = p_amb / (gamma - 1.0)
    lf = h["nlevels"] - 1
    dxf = h["dx0"] / (1 << lf)
    # finest-level deposit, expressed as a function of position so every level can average it
    ps = level_patches(h, lf)
    cells = []
    for p in ps:
        x, y, z = cell_centres(h, p)
        r2 = (z[:, None, None] - 0.5) ** 2 + (y[None, :, None] - 0.5) ** 2 + (x[None, None, :] - 0.5) ** 2
        cells.append(r2 < (2.0 * dxf) ** 2)
    ncell = int(sum(c.sum() for c in cells))
    if ncell == 0:
        raise ValueError("no finest-level cell inside the deposit radius")
    e_dep = E0 / (ncell * dxf ** 3)  # energy density so that the discrete total is E0
    for p, c in zip(ps, cells):
        U[p, 4][c] += e_dep
    # coarser levels: average of the (up to 2^(3k)) finest cells they cover, computed directly
    for l in range(lf - 1, -1, -1):
        ratio = 1 << (lf - l)
        dxl = h["dx0"] / (1 << l)
        for p in level_patches(h, l):
            x, y, z = cell_centres(h, p)
            # count deposit cells (finest index space) under each coarse cell: deposit cells are
            # those with |c - 0.5| < 2 dxf per the ball test; enumerate the 4^3 candidates
            cand = (np.arange(-2, 2) + 0.5) * dxf + 0.5
            for cz in cand:
                for cy in cand:
                    for cx in cand:
                        if (cx - 0.5) ** 2 + (cy - 0.5) ** 2 + (cz - 0.5) ** 2 >= (2.0 * dxf) ** 2:
                            continue
                        i = int(np.floor(cx / dxl)) - h["origin"][p, 0]
                        j = int(np.floor(cy / dxl)) - h["origin"][p, 1]
                        k = int(np.floor(cz / dxl)) - h["origin"][p, 2]
                        if 0 <= i < NI and 0 <= j < NI and 0 <= k < NI:
                            U[p, 4, k, j, i] += e_dep / ratio ** 3
    return U


def to_patches(h, G):
    """Global single-level array -> per-patch array in table order."""
    return split_global(h, G, 0)
