// amrhydro.cu -- host side of the C ABI declared in include/amrhydro.h: handle, descriptor
// table, launches, and the subcycling driver (host bookkeeping only; every arithmetic step of
// the path runs in the kernels).  There is no CPU fallback anywhere in this file.
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <string>
#include <type_traits>
#include <unordered_map>
#include <vector>

#include "../../include/amrhydro.h"
#include "kernels_level.cuh"
#include "layout.cuh"
#include "physics.cuh"
#include "rk_stage_ref.cuh"
#include "rk_stage_march.cuh"
#include "rk_stage_pair.cuh"

using namespace amr;

static_assert(sizeof(amrhydro_patch_desc) == 128 && sizeof(Desc) == 128, "descriptor row is 128 bytes");

struct amrhydro {
  double gamma = 1.4;
  int nv = 5, bits = 64;
  // NEXT-4: patches of 32^3, 48^3, 64^3 cells are held as sub^3 patches of 16^3 (the scheme is defined on cells; sibling
  // halos are exact copies, so the decomposition does not change a bit of the result); np_user counts the caller's patches
  int pdim = NI, sub = 1, nsub = 1, np_user = 0;
  double theta = 1.5, rho_floor = 1e-30, e_floor = 1e-30;
  double glm_ch = 1.0, glm_cr = 0.18;      // S17, S18 (nvars = 9)
  int kernel = 3, halo = 1;                 // rk_stage_pair for nvars = 5 (rk_stage_march otherwise); direct sibling halos
  void *pool = nullptr;
  size_t pool_bytes = 0;
  int maxp = 0, nslots = 0;
  cudaStream_t stream = nullptr;
  bool bound = false;
  int np = 0, nlev = 0;
  double dx0 = 1.0;
  int bc[6] = {0, 0, 0, 0, 0, 0};
  std::vector<amrhydro_patch_desc> tbl;
  std::vector<int> child, octant, lev_first, lev_count;
  std::vector<int> lev_run;                 // patches of a level the kernels run on: all of them, or the owned ones of a shard
  // patch sharding (NEXT-2): slabs this shard sends to / receives from its peers (patch * 8 + face), on the device
  int *d_halo_send = nullptr, *d_halo_recv = nullptr;
  int n_halo_send = 0, n_halo_recv = 0;
  std::vector<char> lev_has_cf, lev_has_phys;   // level has coarse-fine ghost regions / faces on an outflow boundary
  Desc *d_desc = nullptr;
  int *d_child = nullptr, *d_octant = nullptr;
  void *d_Rf = nullptr, *d_Rc = nullptr, *d_bflux = nullptr;
  // found once per hierarchy, so that the per-level launches carry no idle blocks: coarse-fine faces (patch * 8 + face:
  // the tasks of k_fill_cf_faces when sibling copies are skipped), flux-register tasks (local patch * 64 + task of k_flux_registers),
  // and per patch the boundary-flux planes a register reads (bit 3 d + s; rk_stage stores only those)
  int *d_cflist = nullptr, *d_frtasks = nullptr, *d_bneed = nullptr;
  std::vector<int> cf_first, cf_count, fr_first, fr_count;
  size_t bflux_patches = 0;
  unsigned long long *d_scalars = nullptr;  // [0] scratch, [1] floor hits
  unsigned long long *d_smax = nullptr;     // per level: bits of the max signal speed of (level, smax_slot[level])
  std::vector<int> smax_slot;               // slot the cached value belongs to, -1 = stale
  int zsplit = 2;                           // z-split of the stage kernels: 0 never, 1 always, 2 = small levels and the thin last wave of a launch
  int num_sms = 148;
  int fuse_cfl = 2;                         // 0 never, 1 / 2 = the combination stage also reduces the max signal speed
  void *d_stage = nullptr;
  size_t stage_bytes = 0;
  // upload / download move a range in chunks through two halves of the staging buffer: the host copy of one chunk runs on
  // copy_stream while k_pack / k_unpack of the other runs on the bound stream
  cudaStream_t copy_stream = nullptr;
  cudaEvent_t ev_copied[2] = {nullptr, nullptr}, ev_packed[2] = {nullptr, nullptr}, ev_entry = nullptr;
  long long launches = 0;
  // amrhydro_advance as one CUDA graph (AMRHYDRO_OPT_GRAPH): dt0 lives in d_dt, the S9 recursion is captured once per
  // hierarchy / option set and replayed; the host-side bookkeeping a replay skips is restored from the capture
  int use_graph = 0;
  double *d_dt = nullptr;                   // [0] dt0, [1] non-finite flag (k_dt0)
  bool dt_dev = false;                      // launches take dt from d_dt (set while capturing)
  cudaStream_t cap_stream = nullptr;        // capture runs on a stream of the handle's own (the caller's may be the legacy
                                            // default stream, which cannot be captured); replays go to the caller's stream
  cudaGraphExec_t graph_exec = nullptr;
  bool graph_valid = false;
  std::vector<int> graph_smax_slot;
  long long graph_launches = 0;
  long long eager_steps = 0, graph_replays = 0;
  CUtensorMap tmap;            // TMA view of the pool, 16x16 boxes (rk_stage_march, rk_stage_pair)
  bool have_tmap = false;
  std::string err;
};

namespace {

int fail(amrhydro *h, int code, const std::string &msg) {
  if (h) h->err = msg;
  return code;
}
#define CUDA_TRY(h, expr)                                                                   \
  do {                                                                                      \
    cudaError_t e_ = (expr);                                                                \
    if (e_ != cudaSuccess)                                                                  \
      return fail(h, AMRHYDRO_ECUDA, std::string(#expr) + ": " + cudaGetErrorString(e_));   \
  } while (0)
#define LAUNCH_CHECK(h)                                                                     \
  do {                                                                                      \
    ++(h)->launches;                                                                        \
    cudaError_t e_ = cudaGetLastError();                                                    \
    if (e_ != cudaSuccess) return fail(h, AMRHYDRO_ECUDA, std::string("launch: ") + cudaGetErrorString(e_)); \
  } while (0)

template <class F> int dispatch(amrhydro *h, F &&f) {
  if (h->bits == 64) {
    if (h->nv == 5) return f(double(0), std::integral_constant<int, 5>());
    if (h->nv == 8) return f(double(0), std::integral_constant<int, 8>());
    return f(double(0), std::integral_constant<int, 9>());
  }
  if (h->nv == 5) return f(float(0), std::integral_constant<int, 5>());
  if (h->nv == 8) return f(float(0), std::integral_constant<int, 8>());
  return f(float(0), std::integral_constant<int, 9>());
}

template <typename T> Params<T> make_params(const amrhydro *h) {
  Params<T> P;
  P.gamma = T(h->gamma);
  P.gm1 = T(h->gamma - 1.0);
  P.gg1 = T(h->gamma * (h->gamma - 1.0));
  P.theta = T(h->theta);
  P.rho_floor = T(h->rho_floor);
  P.e_floor = T(h->e_floor);
  P.ch = T(h->glm_ch);
  return P;
}
template <typename T> Pool<T> make_pool(const amrhydro *h) { return Pool<T>{(T *)h->pool, h->maxp, h->nv}; }

size_t elem(const amrhydro *h) { return h->bits == 64 ? 8 : 4; }
size_t vs(const amrhydro *h) { return h->bits == 64 ? Layout<double>::VS : Layout<float>::VS; }

int check_ready(amrhydro *h, bool need_hier = true) {
  if (!h) return AMRHYDRO_EINVAL;
  if (!h->bound) return fail(h, AMRHYDRO_ESTATE, "no pool bound");
  if (need_hier && h->np == 0) return fail(h, AMRHYDRO_ESTATE, "no hierarchy set");
  return 0;
}
int check_level(amrhydro *h, int level) {
  if (level < 0 || level >= h->nlev) return fail(h, AMRHYDRO_EINVAL, "level out of range");
  return 0;
}
int check_slot(amrhydro *h, int s) {
  if (s < 0 || s >= h->nslots) return fail(h, AMRHYDRO_EINVAL, "slot out of range");
  return 0;
}

int ensure_stage(amrhydro *h, size_t bytes) {
  if (h->stage_bytes >= bytes) return 0;
  if (h->d_stage) cudaFree(h->d_stage);
  h->d_stage = nullptr;
  h->stage_bytes = 0;
  CUDA_TRY(h, cudaMalloc(&h->d_stage, bytes));
  h->stage_bytes = bytes;
  return 0;
}

int ensure_copy_stream(amrhydro *h) {
  if (h->copy_stream) return 0;
  CUDA_TRY(h, cudaStreamCreateWithFlags(&h->copy_stream, cudaStreamNonBlocking));
  for (int i = 0; i < 2; ++i) {
    CUDA_TRY(h, cudaEventCreateWithFlags(&h->ev_copied[i], cudaEventDisableTiming));
    CUDA_TRY(h, cudaEventCreateWithFlags(&h->ev_packed[i], cudaEventDisableTiming));
  }
  CUDA_TRY(h, cudaEventCreateWithFlags(&h->ev_entry, cudaEventDisableTiming));
  return 0;
}

// cached max signal speed of (level, slot) goes stale when interior cells of the slot are written
void smax_touch(amrhydro *h, int level, int slot) {
  if (level >= 0 && level < (int)h->smax_slot.size() && h->smax_slot[level] == slot) h->smax_slot[level] = -1;
}

void drop_graph(amrhydro *h) {
  if (h->graph_exec) cudaGraphExecDestroy(h->graph_exec);
  h->graph_exec = nullptr;
  h->graph_valid = false;
}

void free_hierarchy(amrhydro *h) {
  drop_graph(h);
  cudaFree(h->d_desc); cudaFree(h->d_child); cudaFree(h->d_octant);
  cudaFree(h->d_Rf); cudaFree(h->d_Rc); cudaFree(h->d_bflux); cudaFree(h->d_smax);
  cudaFree(h->d_cflist); cudaFree(h->d_frtasks); cudaFree(h->d_bneed);
  cudaFree(h->d_halo_send); cudaFree(h->d_halo_recv);
  h->d_halo_send = h->d_halo_recv = nullptr;
  h->n_halo_send = h->n_halo_recv = 0;
  h->d_cflist = h->d_frtasks = h->d_bneed = nullptr;
  h->d_smax = nullptr;
  h->smax_slot.clear();
  h->d_desc = nullptr; h->d_child = h->d_octant = nullptr;
  h->d_Rf = h->d_Rc = h->d_bflux = nullptr;
  h->bflux_patches = 0;
  h->np = 0;
}

}  // namespace

extern "C" {

static int materialise_sibling_ghosts(amrhydro_t *h, int level, int slot);

amrhydro_t *amrhydro_create(double gamma, int nvars, int patch_dim, int nghost) {
  if (!(gamma > 1.0) || (nvars != 5 && nvars != 8 && nvars != 9) || patch_dim < NI || patch_dim > 4 * NI || patch_dim % NI ||
      nghost != NG)
    return nullptr;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return nullptr;   // no CPU fallback
  amrhydro *h = new amrhydro;
  h->gamma = gamma;
  h->nv = nvars;
  h->pdim = patch_dim;
  h->sub = patch_dim / NI;
  h->nsub = h->sub * h->sub * h->sub;
  {
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) == cudaSuccess && cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && sms > 0)
      h->num_sms = sms;
  }
  if (cudaMalloc(&h->d_scalars, 2 * sizeof(unsigned long long)) != cudaSuccess) { delete h; return nullptr; }
  if (cudaMalloc(&h->d_dt, 2 * sizeof(double)) != cudaSuccess) { cudaFree(h->d_scalars); delete h; return nullptr; }
  cudaMemset(h->d_scalars, 0, 2 * sizeof(unsigned long long));
  cudaMemset(h->d_dt, 0, 2 * sizeof(double));
  cudaDeviceSynchronize();                 // (legacy-stream memset; later work runs on the caller's stream)
  return h;
}

void amrhydro_destroy(amrhydro_t *h) {
  if (!h) return;
  if (h->bound) cudaStreamSynchronize(h->stream);
  free_hierarchy(h);
  cudaFree(h->d_scalars);
  cudaFree(h->d_dt);
  if (h->cap_stream) cudaStreamDestroy(h->cap_stream);
  if (h->copy_stream) {
    cudaStreamSynchronize(h->copy_stream);
    cudaStreamDestroy(h->copy_stream);
    for (int i = 0; i < 2; ++i) { cudaEventDestroy(h->ev_copied[i]); cudaEventDestroy(h->ev_packed[i]); }
    cudaEventDestroy(h->ev_entry);
  }
  cudaFree(h->d_stage);
  delete h;
}

const char *amrhydro_last_error(const amrhydro_t *h) { return h ? h->err.c_str() : "null handle"; }

int amrhydro_set_option(amrhydro_t *h, int key, double value) {
  if (!h) return AMRHYDRO_EINVAL;
  if (h->bound && h->graph_valid) cudaStreamSynchronize(h->stream);
  drop_graph(h);                              // every option is baked into the captured launches
  switch (key) {
    case AMRHYDRO_OPT_GRAPH:
      if (value != 0 && value != 1) return fail(h, AMRHYDRO_EINVAL, "graph must be 0 or 1");
      h->use_graph = int(value);
      return 0;
    case AMRHYDRO_OPT_DTYPE:
      if (h->bound) return fail(h, AMRHYDRO_ESTATE, "dtype must be set before bind_pool");
      if (value != 32 && value != 64) return fail(h, AMRHYDRO_EINVAL, "dtype must be 32 or 64");
      h->bits = int(value);
      return 0;
    case AMRHYDRO_OPT_THETA:
      if (!(value >= 0.0 && value <= 2.0)) return fail(h, AMRHYDRO_EINVAL, "theta must lie in [0,2]");
      h->theta = value;
      return 0;
    case AMRHYDRO_OPT_RHO_FLOOR:
    case AMRHYDRO_OPT_EINT_FLOOR:
      if (!(value > 0.0) || !std::isfinite(value)) return fail(h, AMRHYDRO_EINVAL, "floors must be positive and finite");
      (key == AMRHYDRO_OPT_RHO_FLOOR ? h->rho_floor : h->e_floor) = value;
      return 0;
    case AMRHYDRO_OPT_KERNEL:
      if (value != 0 && value != 2 && value != 3) return fail(h, AMRHYDRO_EINVAL, "kernel must be 0, 2 or 3");
      h->kernel = int(value);
      return 0;
    case AMRHYDRO_OPT_HALO:
      if (value != 0 && value != 1) return fail(h, AMRHYDRO_EINVAL, "halo must be 0 or 1");
      h->halo = int(value);
      return 0;
    case AMRHYDRO_OPT_GLM_CH:
      if (!(value > 0.0) || !std::isfinite(value)) return fail(h, AMRHYDRO_EINVAL, "c_h must be positive and finite");
      h->glm_ch = value;
      for (auto &sl : h->smax_slot) sl = -1;          // c_h enters the cached maxima
      return 0;
    case AMRHYDRO_OPT_GLM_CR:
      if (!(value >= 0.0) || !std::isfinite(value)) return fail(h, AMRHYDRO_EINVAL, "c_r must be >= 0 and finite");
      h->glm_cr = value;
      return 0;
    case AMRHYDRO_OPT_ZSPLIT:
      if (value != 0 && value != 1 && value != 2) return fail(h, AMRHYDRO_EINVAL, "zsplit must be 0, 1 or 2");
      h->zsplit = int(value);
      return 0;
    case AMRHYDRO_OPT_FUSE_CFL:
      if (value != 0 && value != 1 && value != 2) return fail(h, AMRHYDRO_EINVAL, "fuse_cfl must be 0, 1 or 2");
      h->fuse_cfl = int(value);
      return 0;
  }
  return fail(h, AMRHYDRO_EINVAL, "unknown option");
}

int amrhydro_get_counter(amrhydro_t *h, int key, long long *out, int reset) {
  if (!h || !out) return AMRHYDRO_EINVAL;
  if (key == AMRHYDRO_CNT_LAUNCHES) {
    *out = h->launches;
    if (reset) h->launches = 0;
    return 0;
  }
  if (key == AMRHYDRO_CNT_GRAPH_REPLAYS) {
    *out = h->graph_replays;
    if (reset) h->graph_replays = 0;
    return 0;
  }
  if (key == AMRHYDRO_CNT_FLOOR_HITS) {
    unsigned long long v = 0;
    CUDA_TRY(h, cudaMemcpyAsync(&v, h->d_scalars + 1, sizeof(v), cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    *out = (long long)v;
    if (reset) CUDA_TRY(h, cudaMemsetAsync(h->d_scalars + 1, 0, sizeof(v), h->stream));
    return 0;
  }
  return fail(h, AMRHYDRO_EINVAL, "unknown counter");
}

size_t amrhydro_pool_bytes(const amrhydro_t *h, int max_patches, int nslots) {
  if (!h || max_patches <= 0 || nslots <= 0) return 0;
  return size_t(nslots) * size_t(max_patches) * size_t(h->nsub) * size_t(h->nv) * vs(h) * elem(h);
}

int amrhydro_bind_pool(amrhydro_t *h, void *dev_pool, size_t bytes, int max_patches, int nslots, void *stream) {
  if (!h || !dev_pool) return AMRHYDRO_EINVAL;
  size_t need = amrhydro_pool_bytes(h, max_patches, nslots);
  if (need == 0) return fail(h, AMRHYDRO_EINVAL, "bad max_patches / nslots");
  if (bytes < need) return fail(h, AMRHYDRO_ENOMEM, "pool smaller than amrhydro_pool_bytes()");
  if ((uintptr_t)dev_pool % 256) return fail(h, AMRHYDRO_EINVAL, "pool must be 256-byte aligned");
  drop_graph(h);
  max_patches *= h->nsub;                    // from here on in 16^3 patches
  h->pool = dev_pool; h->pool_bytes = bytes; h->maxp = max_patches; h->nslots = nslots;
  h->stream = (cudaStream_t)stream;
  h->bound = true;
  std::fill(h->smax_slot.begin(), h->smax_slot.end(), -1);
  {
    int r = dispatch(h, [&](auto t, auto nv) {
      using T = decltype(t);
      return make_tensor_map<T, decltype(nv)::value>(&h->tmap, dev_pool, size_t(max_patches), nslots);
    });
    h->have_tmap = (r == 0);
    if (r) { h->bound = false; return fail(h, AMRHYDRO_ECUDA, "cuTensorMapEncodeTiled failed for the pool"); }
  }
  CUDA_TRY(h, cudaMemsetAsync(dev_pool, 0, need, h->stream));
  return 0;
}

// everything amrhydro_set_hierarchy checks about a table, without touching the handle's state
static int check_table(amrhydro_t *h, const amrhydro_patch_desc *tbl, int np, int nlev, const int *bc, std::vector<int> &first,
                       std::vector<int> &count, std::vector<int> &child, std::vector<int> &octant) {
  for (int p = 0; p < np; ++p) {
    const auto &d = tbl[p];
    if (d.level < 0 || d.level >= nlev) return fail(h, AMRHYDRO_EINVAL, "patch level out of range");
    if (p > 0 && d.level < tbl[p - 1].level) return fail(h, AMRHYDRO_EINVAL, "patches must be sorted by level");
    if (first[d.level] < 0) first[d.level] = p;
    ++count[d.level];
    for (int r = 0; r < 27; ++r)
      if (r != 13 && (d.nbr[r] >= np || d.nbr[r] < AMRHYDRO_NBR_REMOTE || (d.nbr[r] >= 0 && tbl[d.nbr[r]].level != d.level)))
        return fail(h, AMRHYDRO_EINVAL, "bad neighbour entry");
    for (int f = 0; f < 6; ++f)                // no kernel fills a physical ghost zone on a periodic side
      if (d.nbr[face_region(f)] == AMRHYDRO_NBR_PHYSICAL && bc[f] == AMRHYDRO_BC_PERIODIC)
        return fail(h, AMRHYDRO_EINVAL, "physical-boundary neighbour entry on a periodic side");
    if (d.level == 0 && d.parent != -1) return fail(h, AMRHYDRO_EINVAL, "level-0 patches have parent -1");
    if (d.level == 0) {
      for (int r = 0; r < 27; ++r)
        if (r != 13 && d.nbr[r] == -1) return fail(h, AMRHYDRO_EINVAL, "level 0 cannot have coarse-fine faces");
      continue;
    }
    int Q = d.parent;
    if (Q < 0 || Q >= np || tbl[Q].level != d.level - 1) return fail(h, AMRHYDRO_EINVAL, "bad parent");
    int o = 0;
    for (int a = 0; a < 3; ++a) {
      int rel = d.origin[a] - 2 * tbl[Q].origin[a];
      if (rel != 0 && rel != NI) return fail(h, AMRHYDRO_EINVAL, "patch is not an octant of its parent");
      if (rel == NI) o |= 1 << a;
    }
    octant[p] = o;
    if (child[size_t(Q) * 8 + o] >= 0) return fail(h, AMRHYDRO_EINVAL, "two patches refine the same octant");
    child[size_t(Q) * 8 + o] = p;
    for (int f = 0; f < 6; ++f) {              // proper nesting: the uncovered coarse cell must exist
      if (d.nbr[face_region(f)] != -1) continue;
      int a = f >> 1, hi = f & 1, bit = (o >> a) & 1;
      if (((hi && bit == 1) || (!hi && bit == 0)) && tbl[Q].nbr[face_region(f)] < 0)
        return fail(h, AMRHYDRO_EINVAL, "improper nesting: fine face on a coarse-fine/physical parent face");
    }
  }
  for (int l = 0; l < nlev; ++l)
    if (count[l] == 0) return fail(h, AMRHYDRO_EINVAL, "empty level");
  {
    // the domain extent follows from level 0: a face is AMRHYDRO_NBR_PHYSICAL if and only if the patch touches that
    // side of the domain (on non-periodic sides)
    int lo0[3] = {1 << 30, 1 << 30, 1 << 30}, hi0[3] = {-(1 << 30), -(1 << 30), -(1 << 30)};
    for (int p = 0; p < np && tbl[p].level == 0; ++p)
      for (int a = 0; a < 3; ++a) {
        lo0[a] = std::min(lo0[a], tbl[p].origin[a]);
        hi0[a] = std::max(hi0[a], tbl[p].origin[a] + NI);
      }
    bool shard = false;                        // a shard's table (AMRHYDRO_NBR_REMOTE entries) holds part of the domain only
    for (int p = 0; p < np && !shard; ++p)
      for (int r = 0; r < 27; ++r) shard |= (r != 13 && tbl[p].nbr[r] == AMRHYDRO_NBR_REMOTE);
    for (int p = 0; p < np && !shard; ++p)
      for (int f = 0; f < 6; ++f) {
        const int a = f >> 1, l = tbl[p].level;
        const bool touches = (f & 1) ? (tbl[p].origin[a] + NI == (hi0[a] << l)) : (tbl[p].origin[a] == (lo0[a] << l));
        const bool phys = tbl[p].nbr[face_region(f)] == AMRHYDRO_NBR_PHYSICAL;
        if (bc[f] != AMRHYDRO_BC_PERIODIC && phys != touches)
          return fail(h, AMRHYDRO_EINVAL, "physical-boundary face entries must match the faces on the domain boundary");
      }
  }
  return 0;
}

static int install_hierarchy(amrhydro_t *h, const amrhydro_patch_desc *tbl, int np, int nlev, double dx0, const int *bc) {
  if (int r = check_ready(h, false)) return r;
  if (!tbl || !bc || np <= 0 || nlev <= 0 || !(dx0 > 0)) return fail(h, AMRHYDRO_EINVAL, "bad hierarchy arguments");
  if (np > h->maxp) return fail(h, AMRHYDRO_ENOMEM, "more patches than the pool holds");
  std::vector<int> first(nlev, -1), count(nlev, 0), child(size_t(np) * 8, -1), octant(np, 0);
  if (int r = check_table(h, tbl, np, nlev, bc, first, count, child, octant)) return r;
  CUDA_TRY(h, cudaStreamSynchronize(h->stream));
  free_hierarchy(h);
  h->tbl.assign(tbl, tbl + np);
  h->child = child; h->octant = octant; h->lev_first = first; h->lev_count = count;
  h->lev_run = count;
  h->nlev = nlev; h->dx0 = dx0;
  for (int i = 0; i < 6; ++i) h->bc[i] = bc[i];
  h->lev_has_cf.assign(nlev, 0);
  h->lev_has_phys.assign(nlev, 0);
  for (int p = 0; p < np; ++p) {
    for (int r = 0; r < 27; ++r)
      if (r != 13 && tbl[p].nbr[r] == -1) h->lev_has_cf[tbl[p].level] = 1;
    for (int f = 0; f < 6; ++f)
      if (tbl[p].nbr[face_region(f)] == -2 && bc[f] == AMRHYDRO_BC_OUTFLOW) h->lev_has_phys[tbl[p].level] = 1;
  }
  CUDA_TRY(h, cudaMalloc(&h->d_smax, size_t(nlev) * sizeof(unsigned long long)));
  h->smax_slot.assign(nlev, -1);
  CUDA_TRY(h, cudaMalloc(&h->d_desc, size_t(np) * sizeof(Desc)));
  CUDA_TRY(h, cudaMalloc(&h->d_child, size_t(np) * 8 * sizeof(int)));
  CUDA_TRY(h, cudaMalloc(&h->d_octant, size_t(np) * sizeof(int)));
  // (h->tbl / h->child / h->octant are the handle's own copies: they outlive the asynchronous uploads)
  CUDA_TRY(h, cudaMemcpyAsync(h->d_desc, h->tbl.data(), size_t(np) * sizeof(Desc), cudaMemcpyHostToDevice, h->stream));
  CUDA_TRY(h, cudaMemcpyAsync(h->d_child, h->child.data(), size_t(np) * 8 * sizeof(int), cudaMemcpyHostToDevice, h->stream));
  CUDA_TRY(h, cudaMemcpyAsync(h->d_octant, h->octant.data(), size_t(np) * sizeof(int), cudaMemcpyHostToDevice, h->stream));
  {
    std::vector<int> cfl, frt, bneed(np, 0);
    h->cf_first.assign(nlev, 0); h->cf_count.assign(nlev, 0); h->fr_first.assign(nlev, 0); h->fr_count.assign(nlev, 0);
    for (int l = 0; l < nlev; ++l) {
      h->cf_first[l] = int(cfl.size());
      h->fr_first[l] = int(frt.size());
      for (int p = first[l]; p < first[l] + count[l]; ++p) {
        const int pl = p - first[l];
        for (int f = 0; f < 6; ++f)                           // fine side of a coarse-fine face
          if (l > 0 && tbl[p].nbr[face_region(f)] == -1) {
            cfl.push_back(p * 8 + f);
            frt.push_back(pl * 64 + f);
            bneed[p] |= 1 << ((f >> 1) * 3 + ((f & 1) ? 2 : 0));
          }
        for (int o = 0; o < 8; ++o) {                         // coarse side: the face of a child that has no sibling there
          const int ch = child[size_t(p) * 8 + o];
          if (ch < 0) continue;
          for (int f = 0; f < 6; ++f)
            if (tbl[ch].nbr[face_region(f)] == -1) {
              frt.push_back(pl * 64 + 6 + o * 6 + f);
              bneed[p] |= 1 << ((f >> 1) * 3 + ((o >> (f >> 1)) & 1) + (f & 1));
            }
        }
      }
      h->cf_count[l] = int(cfl.size()) - h->cf_first[l];
      h->fr_count[l] = int(frt.size()) - h->fr_first[l];
    }
    CUDA_TRY(h, cudaMalloc(&h->d_cflist, std::max<size_t>(1, cfl.size()) * sizeof(int)));
    CUDA_TRY(h, cudaMalloc(&h->d_frtasks, std::max<size_t>(1, frt.size()) * sizeof(int)));
    CUDA_TRY(h, cudaMalloc(&h->d_bneed, size_t(np) * sizeof(int)));
    // (synchronous copies from these locals; the stream is idle: synchronised above)
    if (!cfl.empty()) CUDA_TRY(h, cudaMemcpy(h->d_cflist, cfl.data(), cfl.size() * sizeof(int), cudaMemcpyHostToDevice));
    if (!frt.empty()) CUDA_TRY(h, cudaMemcpy(h->d_frtasks, frt.data(), frt.size() * sizeof(int), cudaMemcpyHostToDevice));
    CUDA_TRY(h, cudaMemcpy(h->d_bneed, bneed.data(), size_t(np) * sizeof(int), cudaMemcpyHostToDevice));
  }
  if (nlev > 1) {
    size_t rb = size_t(np) * 6 * h->nv * 64 * elem(h);
    CUDA_TRY(h, cudaMalloc(&h->d_Rf, rb));
    CUDA_TRY(h, cudaMalloc(&h->d_Rc, rb));
    CUDA_TRY(h, cudaMemsetAsync(h->d_Rf, 0, rb, h->stream));
    CUDA_TRY(h, cudaMemsetAsync(h->d_Rc, 0, rb, h->stream));
    size_t mx = *std::max_element(count.begin(), count.end());
    CUDA_TRY(h, cudaMalloc(&h->d_bflux, mx * 9 * h->nv * 256 * elem(h)));
    h->bflux_patches = mx;
  }
  h->np = np;
  h->np_user = np / h->nsub;
  CUDA_TRY(h, cudaStreamSynchronize(h->stream));   // the pageable-memory copies above are staged: make them final
  return 0;
}

// patch_dim = 16 s, s > 1 (NEXT-4): the caller's table of (16 s)^3 patches becomes a table of 16^3 patches, s^3 per
// patch in (z, y, x) order right after one another, so that internal patch = user patch * s^3 + sub-index and levels stay
// contiguous.  Parents and the 27 neighbour entries follow from level, origin and the boundary conditions alone (periodic
// wrap over the extent of level 0); the caller's nbr entries are not read.
static int expand_table(amrhydro_t *h, const amrhydro_patch_desc *tbl, int np, int nlev, const int *bc,
                        std::vector<amrhydro_patch_desc> &out) {
  const int D = h->pdim, S = h->sub, NS = h->nsub;
  auto key = [](int l, int x, int y, int z) {
    return (uint64_t(l) << 60) | (uint64_t(x) << 40) | (uint64_t(y) << 20) | uint64_t(z);
  };
  int lo0[3] = {1 << 30, 1 << 30, 1 << 30}, hi0[3] = {-(1 << 30), -(1 << 30), -(1 << 30)};
  for (int p = 0; p < np; ++p) {
    const auto &d = tbl[p];
    if (d.level < 0 || d.level >= nlev) return fail(h, AMRHYDRO_EINVAL, "patch level out of range");
    if (p > 0 && d.level < tbl[p - 1].level) return fail(h, AMRHYDRO_EINVAL, "patches must be sorted by level");
    for (int a = 0; a < 3; ++a) {
      if (d.origin[a] < 0 || d.origin[a] % D || d.origin[a] >= (1 << 20)) return fail(h, AMRHYDRO_EINVAL, "origin must be a multiple of patch_dim");
      if (d.level == 0) { lo0[a] = std::min(lo0[a], d.origin[a]); hi0[a] = std::max(hi0[a], d.origin[a] + D); }
    }
    if (d.level == 0 && d.parent != -1) return fail(h, AMRHYDRO_EINVAL, "level-0 patches have parent -1");
    if (d.level > 0) {
      const int Q = d.parent;
      if (Q < 0 || Q >= np || tbl[Q].level != d.level - 1) return fail(h, AMRHYDRO_EINVAL, "bad parent");
      for (int a = 0; a < 3; ++a) {
        const int rel = d.origin[a] - 2 * tbl[Q].origin[a];
        if (rel != 0 && rel != D) return fail(h, AMRHYDRO_EINVAL, "patch is not an octant of its parent");
      }
    }
  }
  if (tbl[0].level != 0) return fail(h, AMRHYDRO_EINVAL, "empty level");
  std::unordered_map<uint64_t, int> id;
  id.reserve(size_t(np) * NS * 2);
  out.assign(size_t(np) * NS, amrhydro_patch_desc{});
  for (int p = 0; p < np; ++p)
    for (int s = 0; s < NS; ++s) {
      const int sx = s % S, sy = (s / S) % S, sz = s / (S * S), q = p * NS + s;
      out[q].level = tbl[p].level;
      out[q].origin[0] = tbl[p].origin[0] + NI * sx;
      out[q].origin[1] = tbl[p].origin[1] + NI * sy;
      out[q].origin[2] = tbl[p].origin[2] + NI * sz;
      if (!id.emplace(key(out[q].level, out[q].origin[0], out[q].origin[1], out[q].origin[2]), q).second)
        return fail(h, AMRHYDRO_EINVAL, "two patches cover the same cells");
    }
  for (auto &d : out) {
    d.parent = -1;
    if (d.level > 0) {
      auto it = id.find(key(d.level - 1, (d.origin[0] / 2) / NI * NI, (d.origin[1] / 2) / NI * NI, (d.origin[2] / 2) / NI * NI));
      if (it == id.end()) return fail(h, AMRHYDRO_EINVAL, "bad parent");
      d.parent = it->second;
    }
    for (int r = 0; r < 27; ++r) {
      const int off[3] = {r % 3 - 1, (r / 3) % 3 - 1, r / 9 - 1};
      int q[3];
      bool outside = false;
      for (int a = 0; a < 3; ++a) {
        q[a] = d.origin[a] + NI * off[a];
        const int lo = lo0[a] << d.level, hi = hi0[a] << d.level;
        if (q[a] < lo || q[a] >= hi) {
          if (bc[2 * a + (q[a] >= hi ? 1 : 0)] == AMRHYDRO_BC_PERIODIC) q[a] = lo + ((q[a] - lo) % (hi - lo) + (hi - lo)) % (hi - lo);
          else outside = true;
        }
      }
      if (outside) { d.nbr[r] = AMRHYDRO_NBR_PHYSICAL; continue; }
      auto it = id.find(key(d.level, q[0], q[1], q[2]));
      d.nbr[r] = it == id.end() ? AMRHYDRO_NBR_COARSE_FINE : it->second;
    }
  }
  return 0;
}

int amrhydro_set_hierarchy(amrhydro_t *h, const amrhydro_patch_desc *tbl, int np, int nlev, double dx0, const int *bc) {
  if (!h) return AMRHYDRO_EINVAL;
  if (h->sub == 1) return install_hierarchy(h, tbl, np, nlev, dx0, bc);
  if (int r = check_ready(h, false)) return r;
  if (!tbl || !bc || np <= 0 || nlev <= 0 || !(dx0 > 0)) return fail(h, AMRHYDRO_EINVAL, "bad hierarchy arguments");
  if (size_t(np) * h->nsub > size_t(h->maxp)) return fail(h, AMRHYDRO_ENOMEM, "more patches than the pool holds");
  std::vector<amrhydro_patch_desc> sub;
  if (int r = expand_table(h, tbl, np, nlev, bc, sub)) return r;
  return install_hierarchy(h, sub.data(), int(sub.size()), nlev, dx0, bc);
}

int amrhydro_upload(amrhydro_t *h, int slot, int first, int count, const void *host) {
  if (int r = check_ready(h)) return r;
  if (int r = check_slot(h, slot)) return r;
  if (!host || first < 0 || count < 0 || first + count > h->np_user) return fail(h, AMRHYDRO_EINVAL, "bad patch range");
  if (count == 0) return 0;
  const size_t per = size_t(h->nv) * h->pdim * h->pdim * h->pdim * elem(h);        // one of the caller's patches
  const int chunk = int(std::max<size_t>(1, std::min<size_t>(count, (size_t(256) << 20) / per)));
  const int nbuf = count > chunk ? 2 : 1;
  if (int r = ensure_stage(h, size_t(nbuf) * chunk * per)) return r;
  if (int r = ensure_copy_stream(h)) return r;
  for (int l = 0; l < h->nlev; ++l) smax_touch(h, l, slot);
  CUDA_TRY(h, cudaEventRecord(h->ev_entry, h->stream));            // the staging buffer may still be read by earlier work
  CUDA_TRY(h, cudaStreamWaitEvent(h->copy_stream, h->ev_entry, 0));
  int it = 0;
  for (int done = 0; done < count; done += chunk, ++it) {
    const int n = std::min(chunk, count - done), b = it & 1;
    char *buf = (char *)h->d_stage + size_t(b) * chunk * per;
    if (it >= 2) CUDA_TRY(h, cudaStreamWaitEvent(h->copy_stream, h->ev_packed[b], 0));   // k_pack of chunk it-2 has drained this half
    CUDA_TRY(h, cudaMemcpyAsync(buf, (const char *)host + size_t(done) * per, size_t(n) * per, cudaMemcpyHostToDevice, h->copy_stream));
    CUDA_TRY(h, cudaEventRecord(h->ev_copied[b], h->copy_stream));
    CUDA_TRY(h, cudaStreamWaitEvent(h->stream, h->ev_copied[b], 0));
    int r = dispatch(h, [&](auto t, auto nv) {
      using T = decltype(t);
      k_pack<T><<<dim3(n * h->nsub, h->nv), 256, 0, h->stream>>>(make_pool<T>(h), slot, (first + done) * h->nsub, (const T *)buf, h->sub);
      LAUNCH_CHECK(h);
      (void)nv;
      return 0;
    });
    if (r) return r;
    CUDA_TRY(h, cudaEventRecord(h->ev_packed[b], h->stream));
  }
  return 0;
}

int amrhydro_download(amrhydro_t *h, int slot, int first, int count, void *host) {
  if (int r = check_ready(h)) return r;
  if (int r = check_slot(h, slot)) return r;
  if (!host || first < 0 || count < 0 || first + count > h->np_user) return fail(h, AMRHYDRO_EINVAL, "bad patch range");
  if (count == 0) return 0;
  const size_t per = size_t(h->nv) * h->pdim * h->pdim * h->pdim * elem(h);
  const int chunk = int(std::max<size_t>(1, std::min<size_t>(count, (size_t(256) << 20) / per)));
  const int nbuf = count > chunk ? 2 : 1;
  if (int r = ensure_stage(h, size_t(nbuf) * chunk * per)) return r;
  if (int r = ensure_copy_stream(h)) return r;
  int it = 0;
  for (int done = 0; done < count; done += chunk, ++it) {
    const int n = std::min(chunk, count - done), b = it & 1;
    char *buf = (char *)h->d_stage + size_t(b) * chunk * per;
    if (it >= 2) CUDA_TRY(h, cudaStreamWaitEvent(h->stream, h->ev_copied[b], 0));       // the host copy of chunk it-2 has drained this half
    int r = dispatch(h, [&](auto t, auto nv) {
      using T = decltype(t);
      k_unpack<T><<<dim3(n * h->nsub, h->nv), 256, 0, h->stream>>>(make_pool<T>(h), slot, (first + done) * h->nsub, (T *)buf, h->sub);
      LAUNCH_CHECK(h);
      (void)nv;
      return 0;
    });
    if (r) return r;
    CUDA_TRY(h, cudaEventRecord(h->ev_packed[b], h->stream));
    CUDA_TRY(h, cudaStreamWaitEvent(h->copy_stream, h->ev_packed[b], 0));
    CUDA_TRY(h, cudaMemcpyAsync((char *)host + size_t(done) * per, buf, size_t(n) * per, cudaMemcpyDeviceToHost, h->copy_stream));
    CUDA_TRY(h, cudaEventRecord(h->ev_copied[b], h->copy_stream));
  }
  CUDA_TRY(h, cudaStreamSynchronize(h->copy_stream));
  CUDA_TRY(h, cudaStreamSynchronize(h->stream));
  return 0;
}

int amrhydro_download_padded(amrhydro_t *h, int slot, int patch, double *out) {
  if (int r = check_ready(h)) return r;
  if (h->sub != 1) return fail(h, AMRHYDRO_EINVAL, "this call addresses 16^3 patches: patch_dim = 16 only");
  if (int r = check_slot(h, slot)) return r;
  if (!out || patch < 0 || patch >= h->np) return fail(h, AMRHYDRO_EINVAL, "bad patch");
  size_t bytes = size_t(h->nv) * NP * NP * NP * sizeof(double);
  if (int r = ensure_stage(h, bytes)) return r;
  if (int r = materialise_sibling_ghosts(h, h->tbl[patch].level, slot)) return r;
  int r = dispatch(h, [&](auto t, auto nv) {
    using T = decltype(t);
    k_unpack_padded<T><<<64, 256, 0, h->stream>>>(make_pool<T>(h), slot, patch, (double *)h->d_stage);
    LAUNCH_CHECK(h);
    (void)nv;
    return 0;
  });
  if (r) return r;
  CUDA_TRY(h, cudaMemcpyAsync(out, h->d_stage, bytes, cudaMemcpyDeviceToHost, h->stream));
  CUDA_TRY(h, cudaStreamSynchronize(h->stream));
  return 0;
}

int amrhydro_download_registers(amrhydro_t *h, int patch, double *rf, double *rc) {
  if (int r = check_ready(h)) return r;
  if (h->sub != 1) return fail(h, AMRHYDRO_EINVAL, "this call addresses 16^3 patches: patch_dim = 16 only");
  if (!rf || !rc || patch < 0 || patch >= h->np) return fail(h, AMRHYDRO_EINVAL, "bad patch");
  size_t n = size_t(6) * h->nv * 64;
  if (!h->d_Rf) { std::fill(rf, rf + n, 0.0); std::fill(rc, rc + n, 0.0); return 0; }
  std::vector<char> a(n * elem(h)), b(n * elem(h));
  CUDA_TRY(h, cudaStreamSynchronize(h->stream));
  CUDA_TRY(h, cudaMemcpy(a.data(), (char *)h->d_Rf + size_t(patch) * n * elem(h), n * elem(h), cudaMemcpyDeviceToHost));
  CUDA_TRY(h, cudaMemcpy(b.data(), (char *)h->d_Rc + size_t(patch) * n * elem(h), n * elem(h), cudaMemcpyDeviceToHost));
  for (size_t i = 0; i < n; ++i) {
    rf[i] = h->bits == 64 ? ((double *)a.data())[i] : double(((float *)a.data())[i]);
    rc[i] = h->bits == 64 ? ((double *)b.data())[i] : double(((float *)b.data())[i]);
  }
  return 0;
}

// The max signal speed of (level, slot) lives in d_smax[level].  It is produced either by k_cfl or,
// for free, by the combination stage of rk_stage_march that wrote the slot (fused reduction), and it
// goes stale whenever a call writes interior cells of that slot (upload, rk_stage, restrict, reflux,
// copy_slot): smax_slot[level] records which slot the value describes.
static int ensure_smax(amrhydro_t *h, int level, int slot) {
  if (h->smax_slot[level] == slot) return 0;
  CUDA_TRY(h, cudaMemsetAsync(h->d_smax + level, 0, sizeof(unsigned long long), h->stream));
  int r = dispatch(h, [&](auto t, auto nv) {
    using T = decltype(t);
    constexpr int NV = decltype(nv)::value;
    k_cfl<T, NV><<<h->lev_run[level], 256, 0, h->stream>>>(make_pool<T>(h), slot, h->lev_first[level],
                                                              make_params<T>(h), h->d_smax + level, h->d_scalars + 1);
    LAUNCH_CHECK(h);
    return 0;
  });
  if (r == 0) h->smax_slot[level] = slot;
  return r;
}
// max over levels [l0, l1] of the cached values (one small copy, one synchronisation)
static int read_smax(amrhydro_t *h, int l0, int l1, double *smax) {
  std::vector<unsigned long long> bits(h->nlev, 0);
  CUDA_TRY(h, cudaMemcpyAsync(bits.data(), h->d_smax, size_t(h->nlev) * sizeof(unsigned long long), cudaMemcpyDeviceToHost,
                              h->stream));
  CUDA_TRY(h, cudaStreamSynchronize(h->stream));
  double s = 0;
  for (int l = l0; l <= l1; ++l) {
    double v;
    std::memcpy(&v, &bits[l], sizeof(v));
    if (!(v <= s)) s = v;                  // keeps NaN/inf
  }
  *smax = s;
  if (!(s > 0.0) || !std::isfinite(s)) return fail(h, AMRHYDRO_ENONFINITE, "max signal speed is zero or not finite");
  return 0;
}

int amrhydro_cfl_dt(amrhydro_t *h, int level, int slot, double cfl, double *dt_out, double *smax_out) {
  if (int r = check_ready(h)) return r;
  if (int r = check_level(h, level)) return r;
  if (int r = check_slot(h, slot)) return r;
  if (!dt_out) return fail(h, AMRHYDRO_EINVAL, "dt_out is null");
  if (int r = ensure_smax(h, level, slot)) return r;
  double s = 0;
  int r = read_smax(h, level, level, &s);
  if (smax_out) *smax_out = s;
  if (r) return r;
  *dt_out = cfl * (h->dx0 / double(1 << level)) / s;
  return 0;
}

// stage_only: the caller knows that only rk_stage will read these ghosts (the fill of U1 before the combination stage
// inside amrhydro_advance): with direct halos that needs the coarse-fine / physical face slabs and nothing else, on any level
static int fill_ghosts_impl(amrhydro_t *h, int level, int slot, int pold, int pnew, double alpha, bool stage_only);

int amrhydro_cfl_dt_device(amrhydro_t *h, int level_first, int level_last, int slot, double cfl, const double **dt_dev) {
  if (int r = check_ready(h)) return r;
  if (int r = check_level(h, level_first)) return r;
  if (int r = check_level(h, level_last)) return r;
  if (int r = check_slot(h, slot)) return r;
  if (level_last < level_first || !dt_dev) return fail(h, AMRHYDRO_EINVAL, "bad level range or null output");
  for (int l = level_first; l <= level_last; ++l)
    if (int r = ensure_smax(h, l, slot)) return r;
  k_dt0<<<1, 32, 0, h->stream>>>(h->d_smax, level_first, level_last, cfl * (h->dx0 / double(1 << level_first)), 0.0, h->d_dt);
  LAUNCH_CHECK(h);
  *dt_dev = h->d_dt;
  return 0;
}

int amrhydro_fill_ghosts(amrhydro_t *h, int level, int slot, int pold, int pnew, double alpha) {
  return fill_ghosts_impl(h, level, slot, pold, pnew, alpha, false);
}

static int fill_ghosts_impl(amrhydro_t *h, int level, int slot, int pold, int pnew, double alpha, bool stage_only) {
  if (int r = check_ready(h)) return r;
  if (int r = check_level(h, level)) return r;
  if (int r = check_slot(h, slot)) return r;
  if (level > 0) {
    if (int r = check_slot(h, pold)) return r;
    if (int r = check_slot(h, pnew)) return r;
  } else {
    pold = pnew = slot;
  }
  // direct-halo mode: sibling copies are only needed where someone prolongates from this level
  const int skip = (h->halo == 1 && (level + 1 >= h->nlev || stage_only)) ? 1 : 0;   // (mode bit 0 of k_fill_ghosts)
  const bool phase1 = !skip || h->lev_has_cf[level], phase2 = h->lev_has_phys[level];
  if (!phase1 && !phase2) return 0;   // e.g. periodic single level with direct halos: nothing to materialise
  return dispatch(h, [&](auto t, auto nv) {
    using T = decltype(t);
    constexpr int NV = decltype(nv)::value;
    if (phase1 && skip) {
      // sibling copies skipped: all there is to fill is the slab behind every coarse-fine face of the level
      if (h->cf_count[level] > 0) {
        k_fill_cf_faces<T, NV><<<h->cf_count[level], 256, 0, h->stream>>>(
            make_pool<T>(h), slot, pold, pnew, T(alpha), h->d_desc, h->d_octant, h->d_cflist + h->cf_first[level]);
        LAUNCH_CHECK(h);
      }
    } else if (phase1) {
      k_fill_ghosts<T, NV><<<dim3(h->lev_run[level], NP), 256, 0, h->stream>>>(
          make_pool<T>(h), slot, pold, pnew, T(alpha), h->lev_first[level], h->d_desc, h->d_octant, 0);
      LAUNCH_CHECK(h);
    }
    if (phase2) {
      k_fill_outflow<T, NV><<<h->lev_run[level], 256, 0, h->stream>>>(
          make_pool<T>(h), slot, h->lev_first[level], h->d_desc, h->bc[0], h->bc[1], h->bc[2], h->bc[3], h->bc[4], h->bc[5]);
      LAUNCH_CHECK(h);
    }
    return 0;
  });
}

// Calls that read a patch's own padded box (refine_indicator, download_padded) need the sibling ghosts that
// fill_ghosts leaves out in direct-halo mode on the finest level: copy them now (siblings only, no prolongation).
static int materialise_sibling_ghosts(amrhydro_t *h, int level, int slot) {
  if (!(h->halo == 1 && level + 1 >= h->nlev)) return 0;
  return dispatch(h, [&](auto t, auto nv) {
    using T = decltype(t);
    constexpr int NV = decltype(nv)::value;
    k_fill_ghosts<T, NV><<<dim3(h->lev_run[level], NP), 256, 0, h->stream>>>(
        make_pool<T>(h), slot, slot, slot, T(0), h->lev_first[level], h->d_desc, h->d_octant, 2);
    LAUNCH_CHECK(h);
    return 0;
  });
}

int amrhydro_rk_stage(amrhydro_t *h, int level, int sin, int sbase, int sout, double a, double b, double dt, double w) {
  if (int r = check_ready(h)) return r;
  if (int r = check_level(h, level)) return r;
  if (check_slot(h, sin) || check_slot(h, sbase) || check_slot(h, sout)) return AMRHYDRO_EINVAL;
  if (sin == sout) return fail(h, AMRHYDRO_EINVAL, "slot_out must differ from slot_in (halo hazard)");
  const bool regs = (w != 0.0) && h->nlev > 1;
  const double hx = h->dx0 / double(1 << level);
  return dispatch(h, [&](auto t, auto nv) {
    using T = decltype(t);
    constexpr int NV = decltype(nv)::value;
    const int n = h->lev_run[level], first = h->lev_first[level];
    T *bflux = regs ? (T *)h->d_bflux : nullptr;
    // captured step: dt carries the exact factor 2^-level and the launches read dt0 from device memory
    const DtDev dtd = h->dt_dev ? DtDev{h->d_dt, dt, hx} : DtDev{nullptr, 0.0, 0.0};
    smax_touch(h, level, sout);
    // the combination stage can also reduce the max signal speed of what it writes (a1 fused into a6)
    const bool fuse = h->kernel != 0 && h->fuse_cfl != 0 && a != 0.0;
    if (fuse) CUDA_TRY(h, cudaMemsetAsync(h->d_smax + level, 0, sizeof(unsigned long long), h->stream));
    if (h->kernel == 0) {
      k_rk_stage_ref<T, NV><<<dim3(n, NI), 256, 0, h->stream>>>(make_pool<T>(h), sin, sbase, sout, first, T(a), T(b),
                                                                T(dt / hx), make_params<T>(h), bflux, h->d_scalars + 1, dtd);
      LAUNCH_CHECK(h);
    } else if (h->kernel == 3 && NV == 5) {
      if constexpr (NV == 5) {
        int r = launch_rk_stage_pair<T, NV>(h->tmap, make_pool<T>(h), sin, sbase, sout, first, n, T(a), T(b), T(dt / hx),
                                            make_params<T>(h), bflux, h->d_scalars + 1, h->d_desc, h->halo, h->stream,
                                            fuse ? h->d_smax + level : nullptr, h->zsplit, h->num_sms, dtd, h->d_bneed);
        if (r) return fail(h, AMRHYDRO_ECUDA, std::string("rk_stage_pair: ") + cudaGetErrorString((cudaError_t)r));
        LAUNCH_CHECK(h);
      }
    } else {
      int r = launch_rk_stage_march<T, NV>(h->tmap, make_pool<T>(h), sin, sbase, sout, first, n, T(a), T(b), T(dt / hx),
                                           make_params<T>(h), bflux, h->d_scalars + 1, h->d_desc, h->halo, h->stream,
                                           fuse ? h->d_smax + level : nullptr, h->zsplit, h->num_sms, dtd);
      if (r) return fail(h, AMRHYDRO_ECUDA, std::string("rk_stage_march: ") + cudaGetErrorString((cudaError_t)r));
      LAUNCH_CHECK(h);
    }
    if (fuse) h->smax_slot[level] = sout;
    if (regs && h->fr_count[level] > 0) {
      k_flux_registers<T, NV><<<h->fr_count[level], 64, 0, h->stream>>>(first, level, h->d_desc, h->d_child, bflux,
                                                                         (T *)h->d_Rf, (T *)h->d_Rc, T(w * dt), w, dtd,
                                                                         h->d_frtasks + h->fr_first[level]);
      LAUNCH_CHECK(h);
    }
    return 0;
  });
}

int amrhydro_restrict(amrhydro_t *h, int flev, int fslot, int cslot) {
  if (int r = check_ready(h)) return r;
  if (flev < 1 || flev >= h->nlev) return fail(h, AMRHYDRO_EINVAL, "fine_level out of range");
  if (check_slot(h, fslot) || check_slot(h, cslot)) return AMRHYDRO_EINVAL;
  smax_touch(h, flev - 1, cslot);
  return dispatch(h, [&](auto t, auto nv) {
    using T = decltype(t);
    constexpr int NV = decltype(nv)::value;
    k_restrict<T, NV><<<h->lev_run[flev], 256, 0, h->stream>>>(make_pool<T>(h), fslot, cslot, h->lev_first[flev],
                                                                  h->d_desc, h->d_octant);
    LAUNCH_CHECK(h);
    return 0;
  });
}

int amrhydro_reflux(amrhydro_t *h, int clev, int slot) {
  if (int r = check_ready(h)) return r;
  if (int r = check_level(h, clev)) return r;
  if (int r = check_slot(h, slot)) return r;
  if (clev + 1 >= h->nlev) return 0;
  smax_touch(h, clev, slot);
  return dispatch(h, [&](auto t, auto nv) {
    using T = decltype(t);
    constexpr int NV = decltype(nv)::value;
    const int nf = h->lev_run[clev + 1];
    for (int axis = 0; axis < 3; ++axis) {
      k_reflux<T, NV><<<dim3(nf, 2), 64, 0, h->stream>>>(make_pool<T>(h), slot, h->lev_first[clev + 1], 2 * axis,
                                                          h->d_desc, h->d_octant, (T *)h->d_Rf, (T *)h->d_Rc,
                                                          T(h->dx0 / double(1 << clev)));
      LAUNCH_CHECK(h);
    }
    return 0;
  });
}

int amrhydro_glm_damp(amrhydro_t *h, int level, int slot, double factor) {
  if (int r = check_ready(h)) return r;
  if (int r = check_level(h, level)) return r;
  if (int r = check_slot(h, slot)) return r;
  if (h->nv != 9) return fail(h, AMRHYDRO_EINVAL, "glm_damp needs the 9-variable system");
  if (!std::isfinite(factor)) return fail(h, AMRHYDRO_EINVAL, "factor must be finite");
  return dispatch(h, [&](auto t, auto nv) {          // psi does not enter the signal speeds: cached maxima stay valid
    using T = decltype(t);
    k_scale_var<T><<<h->lev_run[level], 256, 0, h->stream>>>(make_pool<T>(h), slot, h->lev_first[level], 8, T(factor));
    LAUNCH_CHECK(h);
    (void)nv;
    return 0;
  });
}

int amrhydro_refine_indicator(amrhydro_t *h, int level, int slot, double *host_octmax) {
  if (int r = check_ready(h)) return r;
  if (h->sub != 1) return fail(h, AMRHYDRO_EINVAL, "this call addresses 16^3 patches: patch_dim = 16 only");
  if (int r = check_level(h, level)) return r;
  if (int r = check_slot(h, slot)) return r;
  if (!host_octmax) return fail(h, AMRHYDRO_EINVAL, "host_octmax is null");
  const int n = h->lev_run[level];
  const size_t bytes = size_t(n) * 8 * sizeof(double);
  if (int r = ensure_stage(h, bytes)) return r;
  const double inv2dx = 0.5 / (h->dx0 / double(1 << level));
  if (int r = materialise_sibling_ghosts(h, level, slot)) return r;
  int r = dispatch(h, [&](auto t, auto nv) {
    using T = decltype(t);
    k_refine_indicator<T><<<n, 256, 0, h->stream>>>(make_pool<T>(h), slot, h->lev_first[level], inv2dx, (double *)h->d_stage);
    LAUNCH_CHECK(h);
    (void)nv;
    return 0;
  });
  if (r) return r;
  CUDA_TRY(h, cudaMemcpyAsync(host_octmax, h->d_stage, bytes, cudaMemcpyDeviceToHost, h->stream));
  CUDA_TRY(h, cudaStreamSynchronize(h->stream));
  return 0;
}

int amrhydro_prolong_interior(amrhydro_t *h, int patch, int slot, int parent_slot) {
  if (int r = check_ready(h)) return r;
  if (h->sub != 1) return fail(h, AMRHYDRO_EINVAL, "this call addresses 16^3 patches: patch_dim = 16 only");
  if (check_slot(h, slot) || check_slot(h, parent_slot)) return AMRHYDRO_EINVAL;
  if (patch < 0 || patch >= h->np || h->tbl[patch].level == 0) return fail(h, AMRHYDRO_EINVAL, "patch has no parent");
  smax_touch(h, h->tbl[patch].level, slot);
  return dispatch(h, [&](auto t, auto nv) {
    using T = decltype(t);
    constexpr int NV = decltype(nv)::value;
    k_prolong_interior<T, NV><<<NI, 256, 0, h->stream>>>(make_pool<T>(h), slot, parent_slot, patch, h->d_desc, nullptr);
    LAUNCH_CHECK(h);
    return 0;
  });
}

int amrhydro_regrid(amrhydro_t *h, const amrhydro_patch_desc *tbl, int np_new, int nlev_new, const int *old_of_new, int slot) {
  if (int r = check_ready(h)) return r;
  if (h->sub != 1) return fail(h, AMRHYDRO_EINVAL, "this call addresses 16^3 patches: patch_dim = 16 only");
  if (int r = check_slot(h, slot)) return r;
  if (!tbl || !old_of_new || np_new <= 0 || nlev_new <= 0) return fail(h, AMRHYDRO_EINVAL, "bad regrid arguments");
  if (h->nslots < 2) return fail(h, AMRHYDRO_ESTATE, "regrid needs a second slot as scratch");
  if (np_new > h->maxp) return fail(h, AMRHYDRO_ENOMEM, "more patches than the pool holds");
  {
    std::vector<char> used(h->np, 0);
    for (int q = 0; q < np_new; ++q) {
      const int o = old_of_new[q];
      if (o < -1 || o >= h->np) return fail(h, AMRHYDRO_EINVAL, "old_of_new out of range");
      if (o < 0) {
        if (tbl[q].level == 0) return fail(h, AMRHYDRO_EINVAL, "a new patch needs a parent to be prolongated from");
        continue;
      }
      if (used[o]) return fail(h, AMRHYDRO_EINVAL, "old_of_new names a patch twice");
      used[o] = 1;
      const auto &a = h->tbl[o];
      if (a.level != tbl[q].level || a.origin[0] != tbl[q].origin[0] || a.origin[1] != tbl[q].origin[1] ||
          a.origin[2] != tbl[q].origin[2])
        return fail(h, AMRHYDRO_EINVAL, "a surviving patch must keep its level and origin");
    }
  }
  {
    std::vector<int> first(nlev_new, -1), count(nlev_new, 0), child(size_t(np_new) * 8, -1), octant(np_new, 0);
    if (int r = check_table(h, tbl, np_new, nlev_new, h->bc, first, count, child, octant)) return r;
  }
  const int scratch = (slot + 1) % h->nslots;
  // (1) the cells under fine patches hold the fine average before any fine patch disappears (S8)
  for (int l = h->nlev - 1; l >= 1; --l)
    if (int r = amrhydro_restrict(h, l, slot, slot)) return r;
  // (2) survivors to their new index, through the scratch slot
  int *d_map = nullptr;
  CUDA_TRY(h, cudaMalloc(&d_map, size_t(np_new) * sizeof(int)));
  cudaError_t e = cudaMemcpyAsync(d_map, old_of_new, size_t(np_new) * sizeof(int), cudaMemcpyHostToDevice, h->stream);
  if (e == cudaSuccess) {
    dispatch(h, [&](auto t, auto nv) {
      using T = decltype(t);
      k_move_patches<T><<<np_new, 256, 0, h->stream>>>(make_pool<T>(h), slot, scratch, d_map);
      (void)nv;
      return 0;
    });
    ++h->launches;
    e = cudaGetLastError();
  }
  if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
  if (e != cudaSuccess) { cudaFree(d_map); return fail(h, AMRHYDRO_ECUDA, std::string("regrid move: ") + cudaGetErrorString(e)); }
  // (3) the new table (validated like any other; on failure the old hierarchy is still in place and `slot` untouched)
  const double dx0 = h->dx0;
  int bc[6];
  for (int i = 0; i < 6; ++i) bc[i] = h->bc[i];
  if (int r = amrhydro_set_hierarchy(h, tbl, np_new, nlev_new, dx0, bc)) { cudaFree(d_map); return r; }
  {
    const size_t per = size_t(h->nv) * vs(h) * elem(h);
    char *base = (char *)h->pool;
    e = cudaMemcpyAsync(base + size_t(slot) * h->maxp * per, base + size_t(scratch) * h->maxp * per, size_t(np_new) * per,
                        cudaMemcpyDeviceToDevice, h->stream);
    if (e != cudaSuccess) { cudaFree(d_map); return fail(h, AMRHYDRO_ECUDA, std::string("regrid copy: ") + cudaGetErrorString(e)); }
  }
  // (4) level by level: ghosts of level l, then the new patches of level l + 1 from their parents (S21), one launch
  std::vector<int> newp;
  std::vector<int> nfirst(nlev_new + 1, 0);
  for (int l = 1; l < nlev_new; ++l) {
    nfirst[l] = int(newp.size());
    for (int q = h->lev_first[l]; q < h->lev_first[l] + h->lev_count[l]; ++q)
      if (old_of_new[q] < 0) newp.push_back(q);
  }
  nfirst[nlev_new] = int(newp.size());
  int rc = 0;
  if (!newp.empty()) {
    e = cudaMemcpyAsync(d_map, newp.data(), newp.size() * sizeof(int), cudaMemcpyHostToDevice, h->stream);
    if (e != cudaSuccess) rc = fail(h, AMRHYDRO_ECUDA, std::string("regrid list: ") + cudaGetErrorString(e));
    int last = 0;                             // the coarsest-to-finest chain of ghost fills ends below the last new patch
    for (int l = 1; l < nlev_new; ++l)
      if (nfirst[l + 1] > nfirst[l]) last = l;
    for (int l = 0; l < last && !rc; ++l) {
      const int cnt = nfirst[l + 2] - nfirst[l + 1];
      if ((rc = amrhydro_fill_ghosts(h, l, slot, slot, slot, 0.0))) break;
      if (cnt <= 0) continue;
      smax_touch(h, l + 1, slot);
      rc = dispatch(h, [&](auto t, auto nv) {
        using T = decltype(t);
        constexpr int NV = decltype(nv)::value;
        k_prolong_interior<T, NV><<<dim3(NI, cnt), 256, 0, h->stream>>>(make_pool<T>(h), slot, slot, 0, h->d_desc,
                                                                        d_map + nfirst[l + 1]);
        LAUNCH_CHECK(h);
        return 0;
      });
    }
  }
  cudaStreamSynchronize(h->stream);          // newp / d_map outlive the asynchronous copies
  cudaFree(d_map);
  return rc;
}

// ---- patch sharding: this handle holds one shard
int amrhydro_set_owned(amrhydro_t *h, int owned) {
  if (int r = check_ready(h)) return r;
  if (h->sub != 1) return fail(h, AMRHYDRO_EINVAL, "this call addresses 16^3 patches: patch_dim = 16 only");
  if (h->nlev != 1) return fail(h, AMRHYDRO_EINVAL, "sharding is built for single-level hierarchies (no parent-child exchange yet)");
  if (owned <= 0 || owned > h->np) return fail(h, AMRHYDRO_EINVAL, "owned patch count out of range");
  for (int p = 0; p < owned; ++p)            // an owned patch must find all six face neighbours in this pool
    for (int f = 0; f < 6; ++f)
      if (h->tbl[p].nbr[face_region(f)] == AMRHYDRO_NBR_COARSE_FINE || h->tbl[p].nbr[face_region(f)] == AMRHYDRO_NBR_REMOTE)
        return fail(h, AMRHYDRO_EINVAL, "owned patch without a face neighbour in this pool (mirror patch missing)");
  CUDA_TRY(h, cudaStreamSynchronize(h->stream));
  drop_graph(h);
  h->lev_run[0] = owned;
  std::fill(h->smax_slot.begin(), h->smax_slot.end(), -1);
  return 0;
}

static int upload_plan(amrhydro_t *h, const int *pairs, int n, int **dev, int *count, bool send) {
  for (int i = 0; i < n; ++i) {
    const int p = pairs[2 * i], f = pairs[2 * i + 1];
    if (p < 0 || p >= h->np || f < 0 || f > 5) return fail(h, AMRHYDRO_EINVAL, "bad (patch, face) pair in the halo plan");
    if (send ? p >= h->lev_run[0] : p < h->lev_run[0])
      return fail(h, AMRHYDRO_EINVAL, send ? "a shard sends slabs of owned patches only" : "a shard receives into mirror patches only");
  }
  cudaFree(*dev);
  *dev = nullptr;
  *count = 0;
  if (n == 0) return 0;
  std::vector<int> code(n);
  for (int i = 0; i < n; ++i) code[i] = pairs[2 * i] * 8 + pairs[2 * i + 1];
  CUDA_TRY(h, cudaMalloc(dev, size_t(n) * sizeof(int)));
  CUDA_TRY(h, cudaMemcpy(*dev, code.data(), size_t(n) * sizeof(int), cudaMemcpyHostToDevice));
  *count = n;
  return 0;
}

int amrhydro_set_halo_plan(amrhydro_t *h, const int *send_pairs, int nsend, const int *recv_pairs, int nrecv) {
  if (int r = check_ready(h)) return r;
  if (h->sub != 1) return fail(h, AMRHYDRO_EINVAL, "this call addresses 16^3 patches: patch_dim = 16 only");
  if (nsend < 0 || nrecv < 0 || (nsend && !send_pairs) || (nrecv && !recv_pairs)) return fail(h, AMRHYDRO_EINVAL, "bad halo plan");
  CUDA_TRY(h, cudaStreamSynchronize(h->stream));
  if (int r = upload_plan(h, send_pairs, nsend, &h->d_halo_send, &h->n_halo_send, true)) return r;
  return upload_plan(h, recv_pairs, nrecv, &h->d_halo_recv, &h->n_halo_recv, false);
}

size_t amrhydro_halo_bytes(const amrhydro_t *h, int which) {
  if (!h) return 0;
  return size_t(which ? h->n_halo_recv : h->n_halo_send) * h->nv * (NG * NI * NI) * elem(h);
}

int amrhydro_halo_pack(amrhydro_t *h, int slot, void *dev_buf) {
  if (int r = check_ready(h)) return r;
  if (int r = check_slot(h, slot)) return r;
  if (h->n_halo_send == 0) return 0;
  if (!dev_buf) return fail(h, AMRHYDRO_EINVAL, "send buffer is null");
  return dispatch(h, [&](auto t, auto nv) {
    using T = decltype(t);
    k_halo_slabs<T, true><<<dim3(h->n_halo_send, h->nv), 256, 0, h->stream>>>(make_pool<T>(h), slot, h->d_halo_send, (T *)dev_buf);
    LAUNCH_CHECK(h);
    (void)nv;
    return 0;
  });
}

int amrhydro_halo_unpack(amrhydro_t *h, int slot, const void *dev_buf) {
  if (int r = check_ready(h)) return r;
  if (int r = check_slot(h, slot)) return r;
  if (h->n_halo_recv == 0) return 0;
  if (!dev_buf) return fail(h, AMRHYDRO_EINVAL, "receive buffer is null");
  return dispatch(h, [&](auto t, auto nv) {
    using T = decltype(t);
    k_halo_slabs<T, false><<<dim3(h->n_halo_recv, h->nv), 256, 0, h->stream>>>(make_pool<T>(h), slot, h->d_halo_recv, (T *)dev_buf);
    LAUNCH_CHECK(h);
    (void)nv;
    return 0;
  });
}

int amrhydro_copy_slot(amrhydro_t *h, int level, int src, int dst) {
  if (int r = check_ready(h)) return r;
  if (int r = check_level(h, level)) return r;
  if (check_slot(h, src) || check_slot(h, dst)) return AMRHYDRO_EINVAL;
  if (src == dst) return 0;
  smax_touch(h, level, dst);
  const size_t per = size_t(h->nv) * vs(h) * elem(h);
  char *base = (char *)h->pool;
  CUDA_TRY(h, cudaMemcpyAsync(base + (size_t(dst) * h->maxp + h->lev_first[level]) * per,
                              base + (size_t(src) * h->maxp + h->lev_first[level]) * per,
                              size_t(h->lev_count[level]) * per, cudaMemcpyDeviceToDevice, h->stream));
  return 0;
}

// S9 recursion; a1/a2 = time-interpolation weights of the parent data for the two ghost fills (S7)
static int advance_level(amrhydro_t *h, int lev, double dt, double a1, double a2) {
  const bool kids = lev + 1 < h->nlev;
  const double w = h->nlev > 1 ? 0.5 : 0.0;
  int r;
  if ((r = amrhydro_fill_ghosts(h, lev, 0, 2, 0, a1))) return r;
  if (kids && (r = amrhydro_copy_slot(h, lev, 0, 2))) return r;
  if ((r = amrhydro_rk_stage(h, lev, 0, 0, 1, 0.0, 1.0, dt, w))) return r;      // U1 = Un + dt L(Un)
  if ((r = fill_ghosts_impl(h, lev, 1, 2, 0, a2, true))) return r;              // (U1's ghosts are read by the next line only)
  if ((r = amrhydro_rk_stage(h, lev, 1, 0, 0, 0.5, 0.5, dt, w))) return r;      // Un+1 = (Un + U1 + dt L(U1))/2
  if (h->nv == 9 && h->glm_cr > 0.0 &&                                           // S18
      (r = amrhydro_glm_damp(h, lev, 0, std::exp(-dt * h->glm_ch / h->glm_cr)))) return r;
  if (kids) {
    if ((r = amrhydro_fill_ghosts(h, lev, 0, 2, 0, a2))) return r;
    if ((r = advance_level(h, lev + 1, 0.5 * dt, 0.0, 0.5))) return r;
    if ((r = advance_level(h, lev + 1, 0.5 * dt, 0.5, 1.0))) return r;
    if ((r = amrhydro_restrict(h, lev + 1, 0, 0))) return r;
    if ((r = amrhydro_reflux(h, lev, 0))) return r;
  }
  return 0;
}

// One coarse step as a graph replay: the per-level maxima are brought up to date eagerly (k_cfl only where no fused
// reduction left a valid value), k_dt0 turns them into dt0 in device memory, and the captured S9 recursion reads it.
static int advance_graph(amrhydro_t *h, double cfl, double dt_fixed, double *dt_out) {
  if (!(dt_fixed > 0.0))
    for (int l = 0; l < h->nlev; ++l)
      if (int r = ensure_smax(h, l, 0)) return r;
  k_dt0<<<1, 32, 0, h->stream>>>(h->d_smax, 0, h->nlev - 1, cfl * h->dx0, dt_fixed, h->d_dt);
  LAUNCH_CHECK(h);
  if (!h->graph_valid) {
    const std::vector<int> keep = h->smax_slot;
    const long long l0 = h->launches;
    cudaGraph_t g = nullptr;
    if (!h->cap_stream) CUDA_TRY(h, cudaStreamCreateWithFlags(&h->cap_stream, cudaStreamNonBlocking));
    cudaStream_t user = h->stream;
    CUDA_TRY(h, cudaStreamBeginCapture(h->cap_stream, cudaStreamCaptureModeThreadLocal));
    h->stream = h->cap_stream;
    h->dt_dev = true;
    const int r = advance_level(h, 0, 1.0, 0.0, 0.0);          // "dt" = the factor 2^-level
    h->dt_dev = false;
    h->stream = user;
    const cudaError_t e = cudaStreamEndCapture(h->cap_stream, &g);
    h->graph_smax_slot = h->smax_slot;
    h->graph_launches = h->launches - l0;
    h->smax_slot = keep;
    h->launches = l0;
    if (r || e != cudaSuccess || !g) {
      if (g) cudaGraphDestroy(g);
      cudaGetLastError();
      return r ? r : fail(h, AMRHYDRO_ECUDA, std::string("graph capture: ") + cudaGetErrorString(e));
    }
    const cudaError_t e2 = cudaGraphInstantiate(&h->graph_exec, g, 0);
    cudaGraphDestroy(g);
    if (e2 != cudaSuccess) { h->graph_exec = nullptr; return fail(h, AMRHYDRO_ECUDA, std::string("graph instantiate: ") + cudaGetErrorString(e2)); }
    h->graph_valid = true;
  }
  CUDA_TRY(h, cudaGraphLaunch(h->graph_exec, h->stream));
  h->smax_slot = h->graph_smax_slot;
  h->launches += h->graph_launches;
  ++h->graph_replays;
  if (dt_out) {
    double v[2] = {0, 0};
    CUDA_TRY(h, cudaMemcpyAsync(v, h->d_dt, sizeof(v), cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    *dt_out = v[0];
    if (v[1] != 0.0) return fail(h, AMRHYDRO_ENONFINITE, "max signal speed is zero or not finite");
  }
  return 0;
}

int amrhydro_advance(amrhydro_t *h, double cfl, double dt_fixed, double *dt_out) {
  if (int r = check_ready(h)) return r;
  if (h->nslots < (h->nlev > 1 ? 3 : 2)) return fail(h, AMRHYDRO_ESTATE, "advance needs 2 slots (3 with refinement)");
  // graph replay from the second step on (the first one runs eagerly: it configures the kernels); the GLM damping factor
  // exp(-dt c_h / c_r) is a host value, so the 9-variable system with damping stays eager
  if (h->use_graph && h->eager_steps > 0 && !(h->nv == 9 && h->glm_cr > 0.0)) return advance_graph(h, cfl, dt_fixed, dt_out);
  double dt = dt_fixed;
  if (!(dt > 0.0)) {
    for (int l = 0; l < h->nlev; ++l)
      if (int r = ensure_smax(h, l, 0)) return r;
    double s = 0;
    if (int r = read_smax(h, 0, h->nlev - 1, &s)) return r;
    dt = cfl * h->dx0 / s;                                  // S4: dt_l = dt0 / 2^l
  }
  if (dt_out) *dt_out = dt;
  ++h->eager_steps;
  return advance_level(h, 0, dt, 0.0, 0.0);
}

int amrhydro_advance_host(amrhydro_t *h, double cfl, double dt_fixed, int nsteps, const void *host_in, void *host_out,
                          double *dt_last) {
  if (int r = check_ready(h)) return r;
  if (!host_in || !host_out || nsteps < 0) return fail(h, AMRHYDRO_EINVAL, "bad host buffers");
  if (int r = amrhydro_upload(h, 0, 0, h->np_user, host_in)) return r;
  for (int s = 0; s < nsteps; ++s)
    if (int r = amrhydro_advance(h, cfl, dt_fixed, dt_last)) return r;
  return amrhydro_download(h, 0, 0, h->np_user, host_out);
}

int amrhydro_sync(amrhydro_t *h) {
  if (!h) return AMRHYDRO_EINVAL;
  CUDA_TRY(h, cudaStreamSynchronize(h->stream));
  return 0;
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------------------------------
// a1 without any allocation (include/amrhydro.h: amrhydro_cfl_dt_noalloc).  A variant of k_cfl whose scratch -- one
// partial maximum per patch and a ticket counter -- is a file-scope __device__ array instead of handle-owned memory:
// block b publishes the bits of its maximum in words 32 + b, takes a ticket, and the block that draws the last ticket
// reduces the partial maxima (max is exact in any order) and writes the three output doubles.
//
// g_noalloc_scratch names DEVICE memory.  In host code the identifier is only a host-side stand-in: its device address
// comes from cudaGetSymbolAddress, once per device with that device current (noalloc_scratch_ptr), and that pointer is
// what the kernel is given.  Word 0: ticket counter (must be zero when a launch starts: cleared by a memset node on the
// launch stream before every launch, and reset by the last block).  Words 1..31: padding to 256 bytes.
#include <cstdarg>
#include <mutex>

namespace {

constexpr int NOALLOC_HDR = 32;                                             // 64-bit words before the partial maxima
constexpr int NOALLOC_MAX_DEVICES = 64;
static __device__ __align__(256) unsigned long long g_noalloc_scratch[NOALLOC_HDR + AMRHYDRO_NOALLOC_MAX_PATCHES];

template <typename T, int NV>
__global__ void __launch_bounds__(256) k_cfl_noalloc(const T *__restrict__ patches, Params<T> P, double cfl_dx,
                                                     unsigned long long *__restrict__ scratch, double *__restrict__ out) {
  const T *Ub = patches + size_t(blockIdx.x) * size_t(NV) * Layout<T>::VS;
  const int i = threadIdx.x & 15, j = threadIdx.x >> 4;
  T best = T(0);
  int hits = 0;
  bool bad = false;
#pragma unroll 4
  for (int k = 0; k < NI; ++k) {                    // the per-cell arithmetic of k_cfl (kernels_level.cuh), S2-S4
    T U[NV], W[NV];
    const int c = cell<T>(k + NG, j + NG, i + NG);
#pragma unroll
    for (int v = 0; v < NV; ++v) U[v] = Ub[size_t(v) * Layout<T>::VS + c];
    cons_to_prim<T, NV>(U, W, P, hits);
    T s = max_signal_speed<T, NV>(W, P);
    T chk = s;
#pragma unroll
    for (int v = 0; v < NV; ++v) chk += U[v];
    bad |= !(chk - chk == T(0));                   // NaN or inf anywhere
    best = tmax(best, s);
  }
  double b = bad ? __longlong_as_double(0x7ff0000000000000LL) : double(best);
  __shared__ double wmax[8];
  __shared__ bool last;
  auto block_max = [&](double x) {                  // result valid in thread 0
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x = fmax(x, __shfl_xor_sync(0xffffffffu, x, o));
    if ((threadIdx.x & 31) == 0) wmax[threadIdx.x >> 5] = x;
    __syncthreads();
    if (threadIdx.x < 32) {
      x = threadIdx.x < 8 ? wmax[threadIdx.x] : 0.0;
#pragma unroll
      for (int o = 4; o > 0; o >>= 1) x = fmax(x, __shfl_xor_sync(0xffffffffu, x, o));
    }
    return x;
  };
  b = block_max(b);
  if (threadIdx.x == 0) {
    __stcg(scratch + NOALLOC_HDR + blockIdx.x, (unsigned long long)__double_as_longlong(b));
    __threadfence();                                // the partial maximum is visible before the ticket is
    last = atomicAdd(scratch, 1ULL) == (unsigned long long)(gridDim.x - 1);
  }
  __syncthreads();                                  // also orders the reads of wmax above before the writes below
  if (!last) return;
  __threadfence();
  double m = 0.0;                                   // non-negative doubles or +inf, never NaN
  for (int q = threadIdx.x; q < (int)gridDim.x; q += 256)
    m = fmax(m, __longlong_as_double((long long)__ldcg(scratch + NOALLOC_HDR + q)));
  m = block_max(m);
  if (threadIdx.x == 0) {
    out[0] = m;
    out[1] = cfl_dx / m;
    out[2] = (m > 0.0 && m < __longlong_as_double(0x7ff0000000000000LL)) ? 0.0 : 1.0;
    scratch[0] = 0ULL;                              // leave the ticket at zero for the next call
  }
}

std::mutex g_noalloc_mu;
unsigned long long *g_noalloc_ptr[NOALLOC_MAX_DEVICES] = {};                // device address of the array, per device
thread_local char g_noalloc_err[320] = "";

int noalloc_fail(int code, const char *fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_noalloc_err, sizeof(g_noalloc_err), fmt, ap);
  va_end(ap);
  return code;
}

// the device address of g_noalloc_scratch on the current device (looked up once per device)
int noalloc_scratch_ptr(unsigned long long **ptr) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return noalloc_fail(AMRHYDRO_ECUDA, "cudaGetDevice: %s", cudaGetErrorString(e));
  if (dev < 0 || dev >= NOALLOC_MAX_DEVICES)
    return noalloc_fail(AMRHYDRO_EINVAL, "device %d is outside 0..%d", dev, NOALLOC_MAX_DEVICES - 1);
  std::lock_guard<std::mutex> lock(g_noalloc_mu);
  if (!g_noalloc_ptr[dev]) {
    void *p = nullptr;
    e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
    if (e != cudaSuccess || !p)
      return noalloc_fail(AMRHYDRO_ECUDA, "cudaGetSymbolAddress(g_noalloc_scratch) on device %d: %s", dev,
                          cudaGetErrorString(e));
    g_noalloc_ptr[dev] = static_cast<unsigned long long *>(p);
  }
  *ptr = g_noalloc_ptr[dev];
  return 0;
}

template <typename T, int NV>
int launch_cfl_noalloc(const void *patches, int np, double gamma, double rho_floor, double e_floor, double ch, double cfl_dx,
                       cudaStream_t st, unsigned long long *scratch, double *out) {
  Params<T> P;
  P.gamma = T(gamma);
  P.gm1 = T(gamma - 1.0);
  P.gg1 = T(gamma * (gamma - 1.0));
  P.theta = T(1.5);                                 // not read by the reduction
  P.rho_floor = T(rho_floor);
  P.e_floor = T(e_floor);
  P.ch = T(ch);
  k_cfl_noalloc<T, NV><<<np, 256, 0, st>>>(static_cast<const T *>(patches), P, cfl_dx, scratch, out);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return noalloc_fail(AMRHYDRO_ECUDA, "launch of k_cfl_noalloc: %s", cudaGetErrorString(e));
  return 0;
}

}  // namespace

extern "C" {

int amrhydro_noalloc_setup(void) {
  unsigned long long *p = nullptr;
  return noalloc_scratch_ptr(&p);
}

const char *amrhydro_noalloc_last_error(void) { return g_noalloc_err; }

int amrhydro_cfl_dt_noalloc(const void *dev_patches, int npatches, int nvars, int dtype_bits, double gamma,
                            double rho_floor, double e_floor, double glm_ch, double cfl_dx, void *stream, double *dev_out) {
  if (!dev_patches || !dev_out) return noalloc_fail(AMRHYDRO_EINVAL, "dev_patches / dev_out is null");
  if (nvars != 5 && nvars != 8 && nvars != 9) return noalloc_fail(AMRHYDRO_EINVAL, "nvars must be 5, 8 or 9 (got %d)", nvars);
  if (dtype_bits != 32 && dtype_bits != 64) return noalloc_fail(AMRHYDRO_EINVAL, "dtype_bits must be 32 or 64 (got %d)", dtype_bits);
  if (!(gamma > 1.0) || !std::isfinite(gamma)) return noalloc_fail(AMRHYDRO_EINVAL, "gamma must be > 1 and finite");
  if (!(rho_floor > 0.0) || !std::isfinite(rho_floor) || !(e_floor > 0.0) || !std::isfinite(e_floor))
    return noalloc_fail(AMRHYDRO_EINVAL, "floors must be positive and finite");
  if (nvars == 9 && (!(glm_ch > 0.0) || !std::isfinite(glm_ch))) return noalloc_fail(AMRHYDRO_EINVAL, "c_h must be positive and finite");
  if (!std::isfinite(cfl_dx)) return noalloc_fail(AMRHYDRO_EINVAL, "cfl_dx must be finite");
  if (npatches < 1) return noalloc_fail(AMRHYDRO_EINVAL, "npatches must be >= 1 (got %d)", npatches);
  if (npatches > AMRHYDRO_NOALLOC_MAX_PATCHES)
    return noalloc_fail(AMRHYDRO_ENOMEM, "npatches = %d exceeds AMRHYDRO_NOALLOC_MAX_PATCHES = %d: the static scratch array holds "
                        "one partial maximum per patch and is not grown (split the level or use amrhydro_cfl_dt)",
                        npatches, AMRHYDRO_NOALLOC_MAX_PATCHES);
  if ((uintptr_t)dev_patches % (dtype_bits / 8) || (uintptr_t)dev_out % 8)
    return noalloc_fail(AMRHYDRO_EINVAL, "dev_patches / dev_out is not aligned to its element size");
  unsigned long long *scratch = nullptr;
  if (int r = noalloc_scratch_ptr(&scratch)) return r;
  cudaStream_t st = (cudaStream_t)stream;
  // the ticket counter must start at zero whatever an earlier (possibly failed) launch left behind
  cudaError_t e = cudaMemsetAsync(scratch, 0, NOALLOC_HDR * sizeof(unsigned long long), st);
  if (e != cudaSuccess) return noalloc_fail(AMRHYDRO_ECUDA, "cudaMemsetAsync(scratch header): %s", cudaGetErrorString(e));
#define NOALLOC_CASE(T, NV)                                                                                              \
  return launch_cfl_noalloc<T, NV>(dev_patches, npatches, gamma, rho_floor, e_floor, glm_ch, cfl_dx, st, scratch, dev_out)
  if (dtype_bits == 64) {
    if (nvars == 5) NOALLOC_CASE(double, 5);
    if (nvars == 8) NOALLOC_CASE(double, 8);
    NOALLOC_CASE(double, 9);
  }
  if (nvars == 5) NOALLOC_CASE(float, 5);
  if (nvars == 8) NOALLOC_CASE(float, 8);
  NOALLOC_CASE(float, 9);
#undef NOALLOC_CASE
}

}  // extern "C"
