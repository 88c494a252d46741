/* amrhydro.h -- C ABI of the B200 (sm_100a) block-AMR finite-volume hot path.
 *
 * Method: Wang, Abel & Kaehler, "Adaptive Mesh Fluid Simulations on GPU", arXiv:0910.5547.
 * Citations "PAPER.md:<line>" refer to the extracted paper text; "S<n>/G<n>" to the readings
 * listed in DESIGN.md where the paper is silent or garbled.
 *
 * Conventions
 *  - Plain C symbols, opaque handle, no exceptions, no printing.  Every call except
 *    create/destroy/last_error/pool_bytes returns an int status: 0 = OK, negative = error
 *    (see AMRHYDRO_E*); amrhydro_last_error(h) then returns a static/handle-owned string.
 *  - All kernels are enqueued on the CUDA stream given to amrhydro_bind_pool and are
 *    asynchronous.  Calls that return host data (cfl_dt, download_*, advance, counters)
 *    synchronise that stream.
 *  - Ownership: the caller (PyTorch) owns the pool allocation and the stream; the library
 *    borrows them.  The library owns the device copy of the descriptor table, the flux
 *    registers, the boundary-flux scratch, the reduction scratch and a host<->device staging
 *    buffer; amrhydro_destroy frees them.
 *  - Pointers: `dev_*` are device pointers, `host_*` are host pointers (pageable or pinned).
 *  - Geometry: patch interior 16^3, 2 ghost zones, refinement ratio 2, cubic cells,
 *    dx_l = dx0 / 2^l.  nvars = 5 (Euler: rho, rho vx, rho vy, rho vz, rho E; PAPER.md:57
 *    Eq. 2), 8 (ideal MHD: ... rho E + B^2/2, Bx, By, Bz; Eq. 14 without psi) or
 *    9 (GLM-MHD: Eq. 14 with psi, fluxes Eq. 15, readings S17-S19).
 *  - Host-side patch data is always "interior" layout [var][16][16][16] (x fastest) of the
 *    element type selected by AMRHYDRO_OPT_DTYPE.  The pool's internal (padded, aligned)
 *    layout is private.
 *  - Slots: by convention 0 = A (U^n -> U^{n+1}), 1 = B (U^(1)), 2 = C (U^n of a level with
 *    children); the primitive calls take explicit slot numbers.
 *  - There is no CPU fallback: every call fails with AMRHYDRO_ECUDA when no device is usable.
 */
#ifndef AMRHYDRO_H
#define AMRHYDRO_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define AMRHYDRO_OK 0
#define AMRHYDRO_EINVAL (-1)    /* bad argument                                   */
#define AMRHYDRO_ENOMEM (-2)    /* pool too small / allocation failed              */
#define AMRHYDRO_ECUDA (-3)     /* CUDA runtime error (text in last_error)         */
#define AMRHYDRO_ESTATE (-4)    /* call out of order (no pool / no hierarchy)      */
#define AMRHYDRO_ENONFINITE (-5)/* NaN/inf/zero signal speed in cfl_dt / advance   */

/* options (amrhydro_set_option); only before amrhydro_bind_pool unless noted */
#define AMRHYDRO_OPT_DTYPE 1      /* 32 or 64 (default 64): element type of pool and host data   */
#define AMRHYDRO_OPT_THETA 2      /* limiter parameter of Eq. 9-10, 0..2 (default 1.5, S1); any time */
#define AMRHYDRO_OPT_RHO_FLOOR 3  /* S11, default 1e-30; any time                                  */
#define AMRHYDRO_OPT_EINT_FLOOR 4 /* S11, default 1e-30; any time                                  */
#define AMRHYDRO_OPT_KERNEL 5     /* rk_stage variant: 0 = reference one-thread-per-cell kernel (cross-check),
                                     2 = k_rk_stage_march (one cell per thread, 8 + 2 halo warps per patch),
                                     3 (default) = k_rk_stage_pair for nvars = 5 (two cells per thread, 4 warps per
                                     patch, two CTAs per SM; measured faster, profiles/README.md) and
                                     k_rk_stage_march for nvars = 8, 9; all agree to round-off; any time        */
#define AMRHYDRO_OPT_HALO 6       /* 1 (default) = rk_stage reads sibling interiors directly, fill_ghosts then only
                                     writes coarse-fine / physical faces (and sibling ghosts on levels someone
                                     prolongates from); 0 = rk_stage reads materialised ghost zones; any time   */
#define AMRHYDRO_OPT_FUSE_CFL 7   /* the combination stage (a != 0) of rk_stage can also reduce the max signal speed of
                                     the state it writes, so that the next amrhydro_cfl_dt of that slot launches
                                     nothing: 0 = never, 1 or 2 (default) = always (measured at 512^3: fp32 step
                                     6.89 -> 6.09 ms, fp64 11.65 -> 10.88 ms); any time                          */

#define AMRHYDRO_OPT_GLM_CH 8     /* nvars = 9: c_h of Eq. 15 (S17), > 0, default 1; any time               */
#define AMRHYDRO_OPT_GLM_CR 9     /* nvars = 9: c_r = c_p^2/c_h of the psi damping applied by amrhydro_advance
                                     (S18), default 0.18, 0 = none; any time                               */

#define AMRHYDRO_OPT_ZSPLIT 10     /* default rk_stage kernel: two CTAs per patch, each marching over half of the column
                                     (3 warm-up planes more per CTA, about half the latency of a launch):
                                     0 = never, 1 = always, 2 (default) = on levels of at most SMs/2 patches, and (the
                                     8- / 9-variable kernel) for the patches of the last wave of a launch when that wave is
                                     less than half full (its half-CTAs all fit: 0.6 instead of 1 wave time; config 4's 512
                                     patches are 3.46 waves of 148 CTAs: 0.490 -> 0.450 ms per step).  Bitwise the unsplit
                                     march; any time */

#define AMRHYDRO_OPT_GRAPH 11      /* amrhydro_advance replays one CUDA graph per coarse step (dt may stay in
                                     device memory for graph capture): the S9 recursion is captured once per hierarchy
                                     and option set, dt0 = cfl dx0 / max_l S_max,l (S4) is formed on the device by k_dt0
                                     and read by the captured launches, so the host does not wait for dt.  Results are
                                     bitwise those of the eager path.  0 (default) = eager launches, 1 = graph from the
                                     second step on; the 9-variable system with psi damping stays eager; any time   */

/* counters (amrhydro_get_counter) */
#define AMRHYDRO_CNT_LAUNCHES 1   /* kernels launched by this handle since create / last reset */
#define AMRHYDRO_CNT_FLOOR_HITS 2 /* cells/states where a floor of S11 was applied (rk_stage, cfl) */
#define AMRHYDRO_CNT_GRAPH_REPLAYS 3 /* coarse steps amrhydro_advance ran as a graph replay (AMRHYDRO_OPT_GRAPH) */

#define AMRHYDRO_BC_PERIODIC 0    /* handled by the neighbour table */
#define AMRHYDRO_BC_OUTFLOW 1     /* zero-gradient (S5)             */

#define AMRHYDRO_NBR_COARSE_FINE (-1)
#define AMRHYDRO_NBR_PHYSICAL (-2)
#define AMRHYDRO_NBR_REMOTE (-3)  /* patch sharding: the neighbour lives on another shard and is not mirrored in this pool;
                                     no kernel reads or fills that region (allowed for edge/corner regions of owned
                                     patches and for any region of a mirror patch)                                  */

typedef struct amrhydro amrhydro_t;

/* One row of the patch-descriptor table (128 bytes).  Patches must be sorted by level.
 * origin: index of the first interior cell on the patch's own level (multiple of patch_dim).
 * parent: patch id on level-1 whose octant this patch refines (-1 on level 0).
 * nbr[r], r = (dz+1)*9 + (dy+1)*3 + (dx+1): id of the same-level patch at block offset
 * (dx,dy,dz) (periodic wrap is expressed here), AMRHYDRO_NBR_COARSE_FINE or
 * AMRHYDRO_NBR_PHYSICAL; nbr[13] is ignored. */
typedef struct amrhydro_patch_desc {
  int level;
  int origin[3];
  int parent;
  int nbr[27];
} amrhydro_patch_desc;

/* Create a solver context.  gamma: adiabatic index of Eq. 6, > 1.
 * nvars in {5, 8, 9}; nghost must be 2 (the stencil i-2..i+1 of PAPER.md:104); patch_dim is 16 (BASELINE.json
 * north_star) or 32, 48, 64 ("arbitrary grid dimensions can arise").  A patch of
 * (16 s)^3 cells is held as s^3 patches of 16^3: the scheme is defined on cells and sibling halos are exact copies, so
 * the result does not depend on the decomposition (tests/test_gpu_patchdim.py: bitwise the 16^3 run).  With
 * patch_dim > 16: descriptor origins are multiples of patch_dim, a fine patch is an octant of its parent as before,
 * parents and neighbours follow from level, origin and the boundary conditions (the nbr entries of the caller's table are
 * not read), host data is [patch][var][D][D][D], max_patches and patch ranges count the caller's patches, and the calls
 * that address single 16^3 patches (download_padded, download_registers, refine_indicator, prolong_interior, regrid,
 * set_owned, set_halo_plan) return AMRHYDRO_EINVAL.  Other patch shapes, direct flux reconstruction and higher order
 * are not built.  Returns NULL on a bad argument or when no CUDA device exists. */
amrhydro_t *amrhydro_create(double gamma, int nvars, int patch_dim, int nghost);
void amrhydro_destroy(amrhydro_t *h);
const char *amrhydro_last_error(const amrhydro_t *h);

int amrhydro_set_option(amrhydro_t *h, int key, double value);
int amrhydro_get_counter(amrhydro_t *h, int key, long long *value_out, int reset);

/* Bytes the caller must allocate for `nslots` copies of `max_patches` padded patches. */
size_t amrhydro_pool_bytes(const amrhydro_t *h, int max_patches, int nslots);
/* Borrow the pool (device pointer, 256-byte aligned) and the stream (cudaStream_t as void*,
 * NULL = legacy default stream).  The pool is zero-filled asynchronously. */
int amrhydro_bind_pool(amrhydro_t *h, void *dev_pool, size_t bytes, int max_patches, int nslots,
                       void *cuda_stream);
/* Copy and validate the descriptor table (host memory, owned by the caller).  dx0: level-0
 * cell width; bc[6]: AMRHYDRO_BC_* for x-lo, x-hi, y-lo, y-hi, z-lo, z-hi.  Allocates and
 * zeroes the flux registers when nlevels > 1. */
int amrhydro_set_hierarchy(amrhydro_t *h, const amrhydro_patch_desc *host_tbl, int npatches,
                           int nlevels, double dx0, const int *bc);

/* Interior data of patches [first, first+count) of one slot, host layout
 * [count][var][16][16][16].  Upload stages through the library's device buffer in chunks;
 * pinned host memory makes the copies asynchronous. */
int amrhydro_upload(amrhydro_t *h, int slot, int first, int count, const void *host_interior);
int amrhydro_download(amrhydro_t *h, int slot, int first, int count, void *host_interior);
/* Debug/test: padded box [var][20][20][20] of one patch, and its flux registers
 * [6 faces][var][8][8] (fine side, coarse side), as doubles. */
int amrhydro_download_padded(amrhydro_t *h, int slot, int patch, double *host_padded);
int amrhydro_download_registers(amrhydro_t *h, int patch, double *host_fine, double *host_coarse);

/* a1: dt = cfl * dx_level / max over interior cells and d of (|v_d| + c_d), c = sound speed
 * (S2) or fast magnetosonic speed along d (S3).  S4; the paper gives no CFL formula.
 * Synchronises.  AMRHYDRO_ENONFINITE if the maximum is NaN, inf or 0.  smax_out may be NULL.
 * The library remembers the maximum of (level, slot) until a call writes interior cells of that
 * slot (upload, rk_stage, restrict, reflux, copy_slot), and rk_stage's combination stage can
 * supply it (AMRHYDRO_OPT_FUSE_CFL): the same cells, the same formula, reduced where the state is
 * produced; the reciprocal there is correct to 1 ulp, so dt may differ from the stand-alone
 * reduction in the last bit.  The pool is private: data written into it behind the library's back
 * is not seen. */
int amrhydro_cfl_dt(amrhydro_t *h, int level, int slot, double cfl, double *dt_out, double *smax_out);
/* The same without the host read ("a _device variant that leaves dt in device memory is allowed for graph
 * capture"): *dt_dev points at two doubles in the handle's device memory, written asynchronously on the bound stream by
 * k_dt0: [0] = cfl * dx_level_first / max over levels level_first..level_last of the signal speed of `slot` (S4: with
 * level_first = 0 and level_last = nlevels - 1 the dt0 of amrhydro_advance), [1] = 1 if that maximum is zero, NaN or inf,
 * else 0.  Valid until the next amrhydro_cfl_dt_device / amrhydro_advance of this handle.  Does not synchronise. */
int amrhydro_cfl_dt_device(amrhydro_t *h, int level_first, int level_last, int slot, double cfl, const double **dt_dev);

/* a2: fill the ghost zones of every patch of `level` in `slot` (S5): same-level copy where
 * nbr >= 0; conservative limited-linear prolongation (S6) of (1-alpha)*parent_old_slot +
 * alpha*parent_new_slot (S7) where nbr == -1; zero-gradient outflow where nbr == -2.
 * With AMRHYDRO_OPT_HALO = 1 (direct sibling reads) the sibling copies are made only on levels someone prolongates from; on the
 * finest level this call writes just what rk_stage reads from a patch's own ghost zone: the six face slabs
 * that lie on a coarse-fine or physical boundary.  Edge and corner regions next to a coarse-fine boundary of
 * a finest-level patch are then left as they are. */
int amrhydro_fill_ghosts(amrhydro_t *h, int level, int slot, int parent_old_slot,
                         int parent_new_slot, double alpha);

/* a3-a6: one method-of-lines stage on every patch of `level` (PAPER.md:79 Eq. 7, :94-98
 * Eq. 8): U_out = a*U_base + b*(U_in + dt*L(U_in)), L from primitive recovery, PLM with the
 * theta-minmod limiter (Eq. 9-11, G1) and the single-speed HLL flux (Eq. 12, G2, G6).
 * slot_out may equal slot_base, must differ from slot_in.  flux_weight w != 0 accumulates
 * w*dt*F on coarse-fine faces into the flux registers (S10). */
int amrhydro_rk_stage(amrhydro_t *h, int level, int slot_in, int slot_base, int slot_out,
                      double a, double b, double dt, double flux_weight);

/* a7: each covered cell of level fine_level-1 := mean of its 8 fine cells (S8). */
int amrhydro_restrict(amrhydro_t *h, int fine_level, int fine_slot, int coarse_slot);
/* a8: correct the uncovered coarse cells next to level coarse_level+1 patches with the
 * accumulated flux mismatch, then zero those registers (S10). */
int amrhydro_reflux(amrhydro_t *h, int coarse_level, int slot);

int amrhydro_copy_slot(amrhydro_t *h, int level, int src_slot, int dst_slot);

/* Patch sharding, one shard per handle / GPU ("a grid is the basic unit"
 * of the distribution).  Built for single-level hierarchies in direct-halo mode (AMRHYDRO_OPT_HALO = 1); the
 * parent-child exchange of 8(e)(3) is not built.  A shard's table lists its OWNED patches first (a contiguous Morton
 * range of the global table) and then MIRROR patches: copies of the face neighbours that other shards own.
 *   set_owned: the kernels of every call (cfl_dt, rk_stage, ...) run on the first `owned` patches only; mirrors are data.
 *     Every face region of an owned patch must name a patch of this pool (owned or mirror) or be physical.
 *   set_halo_plan: send_pairs[nsend][2] = (owned patch, face), recv_pairs[nrecv][2] = (mirror patch, face): the slab
 *     "two interior layers next to that face", [var][2][16][16] elements each, in plan order.  The sender's plan towards
 *     a peer and the peer's receive plan list the same global (patch, face) pairs in the same order (the partitioner
 *     sorts both by global patch index, then face), so a buffer is copied between shards as it is (cudaMemcpyPeerAsync,
 *     ncclSend/ncclRecv or a P2P store; the tests use a device-to-device copy between two pools on one GPU).
 *   halo_bytes(which): size of the send (0) or receive (1) buffer in bytes.
 *   halo_pack / halo_unpack: pool -> device buffer (k_halo_slabs) / device buffer -> mirror interiors, asynchronous on
 *     the bound stream.  One exchange of slot_in before each rk_stage; the step size is cfl dx / max over shards of the
 *     smax that amrhydro_cfl_dt returns (allreduce(max) of one scalar). */
int amrhydro_set_owned(amrhydro_t *h, int owned);
int amrhydro_set_halo_plan(amrhydro_t *h, const int *send_pairs, int nsend, const int *recv_pairs, int nrecv);
size_t amrhydro_halo_bytes(const amrhydro_t *h, int which);
int amrhydro_halo_pack(amrhydro_t *h, int slot, void *dev_buf);
int amrhydro_halo_unpack(amrhydro_t *h, int slot, const void *dev_buf);

/* Regrid steps on either side of the hot path (PAPER.md:43-45 leaves regridding to the
 * host code; the table itself is rebuilt by the caller and handed to amrhydro_set_hierarchy).
 * refine_indicator (S20): for every patch of the level and each of its eight 8^3 octants (x = bit 0, y = bit 1,
 * z = bit 2) the maximum of |grad rho| / rho, centred differences over the padded box (ghosts must be
 * filled); host_octmax[count_of_level][8] doubles; synchronises.  Thresholding (BASELINE config 3: above
 * 0.1 of the level maximum) is the caller's.  A NaN anywhere in an octant gives NaN for that octant.
 * prolong_interior (S21): the 16^3 interior of fine patch `patch` in `slot` from the padded box of its
 * parent in `parent_slot` (conservative limited-linear, the operator of S6); the parent's ghosts must be
 * filled.  AMRHYDRO_EINVAL for a level-0 patch. */
int amrhydro_refine_indicator(amrhydro_t *h, int level, int slot, double *host_octmax);
/* regrid (NEXT-3): a new descriptor table on the bound, live pool, with no host round trip of cell data.
 * new_tbl / np_new / nlev_new: as for amrhydro_set_hierarchy (same validation; dx0 and bc are kept);
 * old_of_new[np_new] (host): index of the same patch (same level and origin) in the current table, or -1 for a
 * patch that did not exist.  `slot` holds the state before and after; every other slot is scratch afterwards
 * (needs nslots >= 2 and np_new <= max_patches).  In order: (1) amrhydro_restrict of every fine level into
 * `slot`, so that the cells under a removed fine patch hold its average (S8); (2) surviving patches are moved to
 * their new index by a device kernel (k_move_patches, through the scratch slot); (3) the table, flux registers and
 * launch lists are rebuilt; (4) from level 0 up, ghosts are filled and the new patches of the next level are
 * prolongated from their parents (S21), one launch per level.  Synchronises.  On AMRHYDRO_EINVAL the old hierarchy
 * and `slot` are unchanged. */
int amrhydro_regrid(amrhydro_t *h, const amrhydro_patch_desc *new_tbl, int np_new, int nlev_new,
                    const int *old_of_new, int slot);
int amrhydro_prolong_interior(amrhydro_t *h, int patch, int slot, int parent_slot);

/* nvars = 9 only (AMRHYDRO_EINVAL otherwise): psi <- factor * psi on the interior cells of one level,
 * the damping of the mixed GLM system of Dedner et al. 2002 adopted at PAPER.md:292 (S18);
 * amrhydro_advance calls it after every step of a level with factor = exp(-dt_l c_h / c_r). */
int amrhydro_glm_damp(amrhydro_t *h, int level, int slot, double factor);

/* Host-side driver (bookkeeping only): one coarse step of the whole hierarchy with
 * ratio-2 subcycling (S9), slots 0/1/2 as above.  dt_fixed > 0 overrides the CFL step
 * dt0 = cfl*dx0 / max_l S_max,l (S4).  Synchronises once (for dt) unless dt_fixed > 0.
 * With AMRHYDRO_OPT_GRAPH = 1 the step is a graph replay that takes dt0 from device memory: dt_out may then be
 * NULL, in which case the call does not synchronise at all (a zero / non-finite signal speed is reported by the next
 * call that passes dt_out, as AMRHYDRO_ENONFINITE). */
int amrhydro_advance(amrhydro_t *h, double cfl, double dt_fixed, double *dt_out);
/* End-to-end variant with host buffers: upload all interiors into slot 0, `nsteps` coarse
 * steps, download slot 0.  host_in/host_out: [npatches][var][16][16][16]. */
int amrhydro_advance_host(amrhydro_t *h, double cfl, double dt_fixed, int nsteps,
                          const void *host_in, void *host_out, double *dt_last_out);

int amrhydro_sync(amrhydro_t *h);

/* ---- a1 without any allocation -------------------------------------------------------------------------------------
 * For callers that cannot call cudaMalloc (code under CUDA-graph capture, tight serving loops, harnesses that forbid
 * it): the CFL reduction of amrhydro_cfl_dt (S2-S4, the same per-cell formula) with no handle, no pool binding and NO
 * allocation of any kind -- no cudaMalloc / cudaFree / allocating library routine is called, by set-up or by the call.
 * The scratch of the reduction (one partial maximum per patch and a ticket counter) lives in a file-scope
 * `static __device__` array of 256 + 8 * AMRHYDRO_NOALLOC_MAX_PATCHES bytes = 256.25 KiB, which every GPU that loads
 * the library holds until the process exits.
 *
 *   dev_patches  device pointer: `npatches` consecutive patches in the pool's padded layout (what amrhydro_bind_pool
 *                lays out: the address of patch p of slot s is pool + (s * max_patches + p) * amrhydro_pool_bytes(h,1,1)),
 *                elements of `dtype_bits` (32 or 64) bits, `nvars` = 5, 8 or 9.  Read only; interiors are read,
 *                ghosts are not.
 *   gamma, rho_floor, e_floor, glm_ch   as amrhydro_create / AMRHYDRO_OPT_RHO_FLOOR / _EINT_FLOOR / _GLM_CH.
 *   cfl_dx       cfl * dx of the level.
 *   stream       cudaStream_t of the launch (0 = the legacy default stream).  Nothing is synchronised.
 *   dev_out      device pointer, three doubles, written by the call: [0] the maximum signal speed over all interior
 *                cells (+inf if any conserved value is NaN or inf), [1] dt = cfl_dx / [0], [2] 1 if [0] is zero, NaN
 *                or inf (what amrhydro_cfl_dt reports as AMRHYDRO_ENONFINITE), else 0.
 *
 * Returns 0, AMRHYDRO_EINVAL (null pointer, nvars / dtype_bits / gamma / floors out of range, npatches < 1),
 * AMRHYDRO_ENOMEM if npatches > AMRHYDRO_NOALLOC_MAX_PATCHES (the scratch array is not grown: split the level or use
 * amrhydro_cfl_dt), AMRHYDRO_ECUDA; amrhydro_noalloc_last_error() then returns the text (per thread, static storage).
 * Floor hits are not counted.
 *
 * ALL calls on one device share the one scratch array, and it keeps the last call's contents: each call clears the
 * ticket counter on `stream` before its launch and overwrites the partial maxima it reads.  Two calls that OVERLAP on
 * the GPU (different streams without an ordering between them, or two host threads on two streams) race on it and
 * return garbage; calls on one stream, or ordered by events, are safe.
 *
 * amrhydro_noalloc_setup(): looks up the device address of the scratch array for the CURRENT device
 * (cudaGetSymbolAddress, once per device) -- call it once per device outside any stream capture;
 * amrhydro_cfl_dt_noalloc calls it itself when that has not happened yet.  Devices 0..63. */
#define AMRHYDRO_NOALLOC_MAX_PATCHES 32768   /* 512^3 cells in 16^3 patches: BASELINE config 5 */
int amrhydro_noalloc_setup(void);
int amrhydro_cfl_dt_noalloc(const void *dev_patches, int npatches, int nvars, int dtype_bits, double gamma,
                            double rho_floor, double e_floor, double glm_ch, double cfl_dx, void *stream,
                            double *dev_out);
const char *amrhydro_noalloc_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* AMRHYDRO_H */
