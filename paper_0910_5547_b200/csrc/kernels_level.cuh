// kernels_level.cuh -- level-wide kernels around the stage: CFL reduction (a1), ghost fill
// (a2), restriction (a7), flux registers + refluxing (a8), host staging pack/unpack.
// The paper leaves all of these on the CPU inside Enzo; readings S4-S10.
#pragma once
#include "layout.cuh"
#include "physics.cuh"

namespace amr {

// ------------------------------------------------------------------ staging <-> pool
// staging: [count][var][D][D][D] (host interior layout), D = 16 S: the caller's patch.  One block per (16^3 patch, var);
// with S > 1 the block's patch is sub-block (sz, sy, sx) = s of the caller's patch p / S^3 (NEXT-4).
template <typename T> __device__ __forceinline__ size_t stage_base(int p, int v, int nv, int S) {
  const int NS = S * S * S, u = p / NS, s = p % NS, D = NI * S;
  const int sx = s % S, sy = (s / S) % S, sz = s / (S * S);
  return ((size_t(u) * nv + v) * D + sz * NI) * D * D + size_t(sy * NI) * D + sx * NI;
}
template <typename T>
__global__ void __launch_bounds__(256) k_pack(Pool<T> pool, int slot, int first, const T *__restrict__ stage, int S) {
  const int p = blockIdx.x, v = blockIdx.y, D = NI * S;
  T *dst = pool.patch(slot, first + p) + size_t(v) * Layout<T>::VS;
  const T *src = stage + stage_base<T>(p, v, pool.nv, S);
  for (int c = threadIdx.x; c < NI * NI * NI; c += 256) {
    int i = c & 15, j = (c >> 4) & 15, k = c >> 8;
    dst[cell<T>(k + NG, j + NG, i + NG)] = src[(size_t(k) * D + j) * D + i];
  }
}
template <typename T>
__global__ void __launch_bounds__(256) k_unpack(Pool<T> pool, int slot, int first, T *__restrict__ stage, int S) {
  const int p = blockIdx.x, v = blockIdx.y, D = NI * S;
  const T *src = pool.patch(slot, first + p) + size_t(v) * Layout<T>::VS;
  T *dst = stage + stage_base<T>(p, v, pool.nv, S);
  for (int c = threadIdx.x; c < NI * NI * NI; c += 256) {
    int i = c & 15, j = (c >> 4) & 15, k = c >> 8;
    dst[(size_t(k) * D + j) * D + i] = src[cell<T>(k + NG, j + NG, i + NG)];
  }
}
// interior cells of one variable times a factor (S18: psi <- psi exp(-dt c_h / c_r))
template <typename T>
__global__ void __launch_bounds__(256) k_scale_var(Pool<T> pool, int slot, int first, int v, T factor) {
  T *u = pool.patch(slot, first + blockIdx.x) + size_t(v) * Layout<T>::VS;
  for (int c = threadIdx.x; c < NI * NI * NI; c += 256) {
    const int i = c & 15, j = (c >> 4) & 15, k = c >> 8;
    u[cell<T>(k + NG, j + NG, i + NG)] *= factor;
  }
}
// Patch sharding (NEXT-2): the two interior layers of a patch next to one of its faces, [var][2][16][16] per
// (patch, face) entry of the plan (code = patch * 8 + face; the layer index runs along the face normal, low to high).
// PACK: pool -> contiguous buffer on the sending shard; else buffer -> the interior of the mirror patch on the receiver.
// One block per (entry, var).
template <typename T, bool PACK>
__global__ void __launch_bounds__(256) k_halo_slabs(Pool<T> pool, int slot, const int *__restrict__ plan, T *__restrict__ buf) {
  const int code = plan[blockIdx.x], p = code >> 3, f = code & 7, v = blockIdx.y;
  const int d = f >> 1, lo = (f & 1) ? NI - NG : 0;
  T *u = pool.patch(slot, p) + size_t(v) * Layout<T>::VS;
  T *b = buf + (size_t(blockIdx.x) * pool.nv + v) * (NG * NI * NI);
  for (int c = threadIdx.x; c < NG * NI * NI; c += 256) {
    const int t0 = c & 15, t1 = (c >> 4) & 15, a = (c >> 8) + lo;          // two transverse indices (x fastest), layer
    const int i = d == 0 ? a : t0, j = d == 1 ? a : (d == 0 ? t0 : t1), k = d == 2 ? a : t1;
    const int g = cell<T>(k + NG, j + NG, i + NG);
    if (PACK) b[c] = u[g]; else u[g] = b[c];
  }
}

// padded box of one patch as doubles [var][20][20][20] (tests)
template <typename T>
__global__ void k_unpack_padded(Pool<T> pool, int slot, int p, double *__restrict__ out) {
  const T *src = pool.patch(slot, p);
  const int n = pool.nv * NP * NP * NP;
  for (int c = blockIdx.x * blockDim.x + threadIdx.x; c < n; c += gridDim.x * blockDim.x) {
    int v = c / (NP * NP * NP), r = c % (NP * NP * NP);
    int i = r % NP, j = (r / NP) % NP, k = r / (NP * NP);
    out[c] = double(src[size_t(v) * Layout<T>::VS + cell<T>(k, j, i)]);
  }
}

// ------------------------------------------------------------------ a1: CFL reduction (S4)
// One block per patch; thread (j,i) walks k.  Block max by warp shuffles, then one atomicMax
// on the bit pattern of a non-negative double (monotone as an unsigned integer).
template <typename T, int NV>
__global__ void __launch_bounds__(256) k_cfl(Pool<T> pool, int slot, int first, Params<T> P,
                                             unsigned long long *__restrict__ smax_bits,
                                             unsigned long long *__restrict__ floor_hits) {
  const T *Ub = pool.patch(slot, first + blockIdx.x);
  const int i = threadIdx.x & 15, j = threadIdx.x >> 4;
  T best = T(0);
  int hits = 0;
  bool bad = false;
#pragma unroll 4
  for (int k = 0; k < NI; ++k) {
    T U[NV], W[NV];
    const int c = cell<T>(k + NG, j + NG, i + NG);
#pragma unroll
    for (int v = 0; v < NV; ++v) U[v] = Ub[size_t(v) * Layout<T>::VS + c];
    cons_to_prim<T, NV>(U, W, P, hits);
    T s = max_signal_speed<T, NV>(W, P);
    // fmax drops NaNs and the floors replace a NaN density or energy: test the raw conserved inputs and the result
    T chk = s;
#pragma unroll
    for (int v = 0; v < NV; ++v) chk += U[v];
    bad |= !(chk - chk == T(0));                   // NaN or inf anywhere
    best = tmax(best, s);
  }
  double b = bad ? __longlong_as_double(0x7ff0000000000000LL) : double(best);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) b = fmax(b, __shfl_xor_sync(0xffffffffu, b, o));
  __shared__ double wmax[8];
  if ((threadIdx.x & 31) == 0) wmax[threadIdx.x >> 5] = b;
  __syncthreads();
  if (threadIdx.x < 32) {
    b = threadIdx.x < 8 ? wmax[threadIdx.x] : 0.0;
#pragma unroll
    for (int o = 4; o > 0; o >>= 1) b = fmax(b, __shfl_xor_sync(0xffffffffu, b, o));
    if (threadIdx.x == 0) atomicMax(smax_bits, (unsigned long long)__double_as_longlong(b));
  }
  if (hits) atomicAdd(floor_hits, (unsigned long long)hits);
}

// S4 on the device: dt0 = cfl_dx0 / max_l S_max,l from the per-level maxima (bit patterns of non-negative doubles), left
// in device memory for the launches of a captured step.  out[0] = dt0, out[1] = 1 if the maximum is zero, NaN or inf
// (the value amrhydro_cfl_dt reports as AMRHYDRO_ENONFINITE), else 0.  fixed > 0: that step size instead.
__global__ void k_dt0(const unsigned long long *__restrict__ smax_bits, int l0, int l1, double cfl_dx0, double fixed,
                      double *__restrict__ out) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  if (fixed > 0.0) { out[0] = fixed; out[1] = 0.0; return; }
  double s = 0.0;
  for (int l = l0; l <= l1; ++l) {
    const double v = __longlong_as_double((long long)smax_bits[l]);
    if (!(v <= s)) s = v;                        // keeps NaN/inf
  }
  out[0] = cfl_dx0 / s;
  out[1] = (!(s > 0.0) || !(s - s == 0.0)) ? 1.0 : 0.0;
}

// ------------------------------------------------------------------ a2: ghost fill (S5-S7)
template <typename T> __device__ __forceinline__ T minmod2(T a, T b) {
  if (a > T(0) && b > T(0)) return tmin(a, b);
  if (a < T(0) && b < T(0)) return tmax(a, b);
  return T(0);
}

// Phase 1 (k_fill_ghosts): one block per (patch, padded z-plane), so that even a level of a few
// dozen patches fills the machine.  Every ghost cell whose 16^3 neighbour block is a sibling is
// copied from that sibling's interior; where it is a coarse-fine boundary it is prolongated
// from the parent's padded box, conservative limited-linear (S6) in time-interpolated parent
// data (S7; alpha = 0 or 1 reads only the slot that counts, which is the same value bitwise for
// finite data).  mode bit 1: the prolongation is skipped (siblings only: refine_indicator / download_padded in
// direct-halo mode).  Where only rk_stage will read the ghosts and it reads siblings directly (direct halos on the
// finest level, the fill of U1 on any level), k_fill_cf_faces below does the work instead.
// Phase 2 (k_fill_outflow, launched only for levels that touch an outflow boundary): zero-gradient
// outflow, x then y then z over the full padded extent, one block per patch.
template <typename T, int NV>
__global__ void __launch_bounds__(256) k_fill_ghosts(Pool<T> pool, int slot, int pold, int pnew, T alpha,
                                                     int first, const Desc *__restrict__ desc,
                                                     const int *__restrict__ octant, int mode) {
  // Latency is what this kernel costs on small AMR levels, so it is written as two dependent round trips to
  // memory: (1) the patch's descriptor row and octant (every thread reads what it needs, broadcast through
  // L1: no staging, no barrier), (2) all parent cells this plane prolongates from -- 3 coarse planes x 12 x 12
  // per variable, time-interpolated once (S7) into shared memory -- together with the sibling cells to copy.
  // A fine patch is an octant of its parent and origins are multiples of 16, so parent indices follow from
  // the octant bits alone: coarse index of padded fine index t along d = 8 oc_d + floor((t - 2) / 2) + 2.
  const int p = first + blockIdx.x, k = blockIdx.y;
  const Desc &D = desc[p];
  T *U = pool.patch(slot, p);
  constexpr int CT = 12, CTV = 3 * CT * CT;
  __shared__ T s_par[NV * CTV];
  const int Q = D.parent;
  const int oz = k < NG ? -1 : (k >= NG + NI ? 1 : 0);
  const int *nbr = D.nbr + (oz + 1) * 9;             // the nine regions of this plane
  bool cf = false;                                   // block-uniform: does this plane touch a coarse-fine region?
  if (Q >= 0 && !(mode & 2)) {
#pragma unroll
    for (int r = 0; r < 9; ++r) cf |= ((oz + 1) * 9 + r != 13) && nbr[r] == -1;
  }
  int pc0[3] = {0, 0, 0};                            // parent padded index of the tile's first cell
  if (cf) {
    const int o = octant[p];
    pc0[0] = 8 * (o & 1) + NG - 2;                   // covers the fine ghosts and the slope stencil
    pc0[1] = 8 * ((o >> 1) & 1) + NG - 2;
    pc0[2] = 8 * ((o >> 2) & 1) + ((k - NG + 64) / 2 - 32) + NG - 1;
    const T *Co = pool.patch(pold, Q), *Cn = pool.patch(pnew, Q);
    const bool only_old = alpha == T(0), only_new = alpha == T(1);
    // 432 tile cells per variable over 256 threads: two cells per thread, their parent offsets computed once
    const int r0 = threadIdx.x, r1 = threadIdx.x + 256;
    const int c0 = cell<T>(pc0[2] + r0 / (CT * CT), pc0[1] + (r0 / CT) % CT, pc0[0] + r0 % CT);
    const int c1 = r1 < CTV ? cell<T>(pc0[2] + r1 / (CT * CT), pc0[1] + (r1 / CT) % CT, pc0[0] + r1 % CT) : -1;
#pragma unroll
    for (int v = 0; v < NV; ++v) {
      const T *po = Co + size_t(v) * Layout<T>::VS, *pn = Cn + size_t(v) * Layout<T>::VS;
      s_par[v * CTV + r0] = only_old ? po[c0] : (only_new ? pn[c0] : (T(1) - alpha) * po[c0] + alpha * pn[c0]);
      if (c1 >= 0) s_par[v * CTV + r1] = only_old ? po[c1] : (only_new ? pn[c1] : (T(1) - alpha) * po[c1] + alpha * pn[c1]);
    }
  }
  // ghost cells of this plane: all 400 on a z-ghost plane, else the 144 of the frame
  const int ncell = oz != 0 ? NP * NP : NP * NP - NI * NI;
  auto locate = [&](int t, int &i, int &j) {
    if (oz != 0) { i = t % NP; j = t / NP; }
    else if (t < 2 * NG * NP) { i = t % NP; j = t / NP; if (j >= NG) j += NI; }      // rows 0,1,18,19
    else { const int u = t - 2 * NG * NP; j = NG + u / (2 * NG); i = u % (2 * NG); if (i >= NG) i += NI; }
  };
  // sibling copies first: their loads travel with the tile's
  for (int t = threadIdx.x; t < ncell; t += 256) {
    int i, j;
    locate(t, i, j);
    const int ox = i < NG ? -1 : (i >= NG + NI ? 1 : 0), oy = j < NG ? -1 : (j >= NG + NI ? 1 : 0);
    const int nb = nbr[(oy + 1) * 3 + (ox + 1)];
    if (nb < 0) continue;
    const T *S = pool.patch(slot, nb);
    const int me = cell<T>(k, j, i), sc = cell<T>(k - oz * NI, j - oy * NI, i - ox * NI);
#pragma unroll
    for (int v = 0; v < NV; ++v) U[size_t(v) * Layout<T>::VS + me] = S[size_t(v) * Layout<T>::VS + sc];
  }
  if (!cf) return;                                   // block-uniform
  __syncthreads();
  for (int t = threadIdx.x; t < ncell; t += 256) {
    int i, j;
    locate(t, i, j);
    const int ox = i < NG ? -1 : (i >= NG + NI ? 1 : 0), oy = j < NG ? -1 : (j >= NG + NI ? 1 : 0);
    if (nbr[(oy + 1) * 3 + (ox + 1)] != -1) continue;
    const int pad[3] = {i, j, k};
    int c0 = 0;
    T s[3];
    const int st[3] = {1, CT, CT * CT};
    const int o = octant[p];
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      const int f = pad[d] - NG;                     // fine index relative to the patch (>= -2)
      const int fc = (f + 64) / 2 - 32;              // floor(f/2)
      s[d] = (f - 2 * fc == 0) ? T(-0.25) : T(0.25);
      c0 += (8 * ((o >> d) & 1) + fc + NG - pc0[d]) * st[d];
    }
    const int me = cell<T>(k, j, i);
#pragma unroll
    for (int v = 0; v < NV; ++v) {
      const T *c = s_par + v * CTV;
      const T uc = c[c0];
      T val = uc;
#pragma unroll
      for (int d = 0; d < 3; ++d) val = val + s[d] * minmod2(c[c0 + st[d]] - uc, uc - c[c0 - st[d]]);
      U[size_t(v) * Layout<T>::VS + me] = val;
    }
  }
}

// The same prolongation (S6, S7: the expressions of k_fill_ghosts, term by term) for the fills whose only reader is
// rk_stage with direct sibling halos: nobody reads sibling ghosts, edge or corner regions then (the stage
// needs the two layers behind each FACE), so all there is to fill is the 2 x 16 x 16 slab behind every coarse-fine
// face.  One block per (patch, face) task = patch * 8 + face: the slab prolongates from 3 x 10 x 10 parent cells per
// variable (one coarse layer + its two neighbours for the slope, 8 + 2 cells along each tangential direction), staged
// once in shared memory, two fine cells per thread.  A level of thousands of patches launches one block per face
// instead of twenty per patch, and each parent cell is read once instead of up to ten times.
template <typename T, int NV>
__global__ void __launch_bounds__(256) k_fill_cf_faces(Pool<T> pool, int slot, int pold, int pnew, T alpha,
                                                       const Desc *__restrict__ desc, const int *__restrict__ octant,
                                                       const int *__restrict__ tasks) {
  const int task = tasks[blockIdx.x], p = task >> 3, f = task & 7, d = f >> 1, side = f & 1;
  const int Q = desc[p].parent, o = octant[p];
  const int e1 = d == 0 ? 1 : 0, e2 = d == 2 ? 1 : 2;          // the tangential dimensions, ascending
  constexpr int CT = 10, CTV = 3 * CT * CT;
  __shared__ T s_par[NV * CTV];
  int pc0[3], st[3];                                           // parent padded index of the tile's first cell; tile strides
  pc0[d] = 8 * ((o >> d) & 1) + (side ? 8 : -1) + NG - 1;      // the coarse layer behind the face is fc = -1 or 8
  pc0[e1] = 8 * ((o >> e1) & 1) + NG - 1;
  pc0[e2] = 8 * ((o >> e2) & 1) + NG - 1;
  st[d] = CT * CT; st[e1] = 1; st[e2] = CT;
  {
    const T *Co = pool.patch(pold, Q), *Cn = pool.patch(pnew, Q);
    const bool only_old = alpha == T(0), only_new = alpha == T(1);
    for (int r = threadIdx.x; r < CTV; r += 256) {
      int pc[3];
      pc[d] = pc0[d] + r / (CT * CT); pc[e1] = pc0[e1] + r % CT; pc[e2] = pc0[e2] + (r / CT) % CT;
      const int c = cell<T>(pc[2], pc[1], pc[0]);
#pragma unroll
      for (int v = 0; v < NV; ++v) {
        const T *po = Co + size_t(v) * Layout<T>::VS, *pn = Cn + size_t(v) * Layout<T>::VS;
        s_par[v * CTV + r] = only_old ? po[c] : (only_new ? pn[c] : (T(1) - alpha) * po[c] + alpha * pn[c]);
      }
    }
  }
  __syncthreads();
  T *U = pool.patch(slot, p);
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    const int t = threadIdx.x + 256 * h;                       // 512 ghost cells; x fastest among the threads of a warp
    int g, a, b;
    if (d == 0) { g = t & 1; a = (t >> 1) & 15; b = t >> 5; }
    else { a = t & 15; b = (t >> 4) & 15; g = t >> 8; }
    int pad[3];
    pad[d] = side ? NG + NI + g : g; pad[e1] = NG + a; pad[e2] = NG + b;
    int c0 = 0;
    T s[3];
#pragma unroll
    for (int dd = 0; dd < 3; ++dd) {
      const int fr = pad[dd] - NG;                   // fine index relative to the patch (>= -2)
      const int fc = (fr + 64) / 2 - 32;             // floor(fr/2)
      s[dd] = (fr - 2 * fc == 0) ? T(-0.25) : T(0.25);
      c0 += (8 * ((o >> dd) & 1) + fc + NG - pc0[dd]) * st[dd];
    }
    const int me = cell<T>(pad[2], pad[1], pad[0]);
#pragma unroll
    for (int v = 0; v < NV; ++v) {
      const T *c = s_par + v * CTV;
      const T uc = c[c0];
      T val = uc;
#pragma unroll
      for (int dd = 0; dd < 3; ++dd) val = val + s[dd] * minmod2(c[c0 + st[dd]] - uc, uc - c[c0 - st[dd]]);
      U[size_t(v) * Layout<T>::VS + me] = val;
    }
  }
}

template <typename T, int NV>
__global__ void __launch_bounds__(256) k_fill_outflow(Pool<T> pool, int slot, int first, const Desc *__restrict__ desc,
                                                      int bc0, int bc1, int bc2, int bc3, int bc4, int bc5) {
  const int p = first + blockIdx.x;
  T *U = pool.patch(slot, p);
  __shared__ int s_nbr[27];
  if (threadIdx.x < 27) s_nbr[threadIdx.x] = desc[p].nbr[threadIdx.x];
  __syncthreads();
  const int bc[6] = {bc0, bc1, bc2, bc3, bc4, bc5};
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    bool any = false;
    for (int side = 0; side < 2; ++side) any |= (s_nbr[face_region(2 * d + side)] == -2 && bc[2 * d + side] == 1);
    if (!any) continue;                            // block-uniform
    __syncthreads();
    for (int side = 0; side < 2; ++side) {
      if (!(s_nbr[face_region(2 * d + side)] == -2 && bc[2 * d + side] == 1)) continue;
      const int src = side == 0 ? NG : NG + NI - 1;
      for (int t = threadIdx.x; t < NG * NP * NP; t += 256) {
        const int g = t / (NP * NP), a = (t / NP) % NP, b = t % NP;
        const int dst = side == 0 ? g : NG + NI + g;
        int cs, cd;
        if (d == 0) { cs = cell<T>(a, b, src); cd = cell<T>(a, b, dst); }
        else if (d == 1) { cs = cell<T>(a, src, b); cd = cell<T>(a, dst, b); }
        else { cs = cell<T>(src, a, b); cd = cell<T>(dst, a, b); }
#pragma unroll
        for (int v = 0; v < NV; ++v) U[size_t(v) * Layout<T>::VS + cd] = U[size_t(v) * Layout<T>::VS + cs];
      }
    }
  }
}

// ------------------------------------------------------------------ regrid steps (NEXT-3; S20, S21)
// S20: max over each 8^3 octant of |grad rho| / rho, centred differences over the ghost-filled box.
// One block per patch; thread (j, i) walks k; octant maxima by warp shuffles + shared memory.
// Always in double (it feeds a host-side threshold).  out[(patch_local)*8 + octant].
template <typename T>
__global__ void __launch_bounds__(256) k_refine_indicator(Pool<T> pool, int slot, int first, double inv2dx,
                                                          double *__restrict__ out) {
  const T *rho = pool.patch(slot, first + blockIdx.x);
  const int i = threadIdx.x & 15, j = threadIdx.x >> 4;
  constexpr int PX = Layout<T>::PX, PLANE = Layout<T>::PLANE;
  double best[2] = {0.0, 0.0};
  bool bad = false;
#pragma unroll 4
  for (int k = 0; k < NI; ++k) {
    const int c = cell<T>(k + NG, j + NG, i + NG);
    const double gx = (double(rho[c + 1]) - double(rho[c - 1])) * inv2dx;
    const double gy = (double(rho[c + PX]) - double(rho[c - PX])) * inv2dx;
    const double gz = (double(rho[c + PLANE]) - double(rho[c - PLANE])) * inv2dx;
    const double g = sqrt(gx * gx + gy * gy + gz * gz) / double(rho[c]);
    bad |= !(g - g == 0.0);
    best[k >> 3] = fmax(best[k >> 3], g);
  }
  // octant maxima on the bit pattern of a non-negative double (monotone as an unsigned integer; a NaN
  // pattern is larger than every finite one, so it survives the maximum)
  __shared__ unsigned long long smax[8];
  if (threadIdx.x < 8) smax[threadIdx.x] = 0ull;
  __syncthreads();
#pragma unroll
  for (int kz = 0; kz < 2; ++kz) {
    const double b = bad ? __longlong_as_double(0x7ff8000000000000LL) : best[kz];
    atomicMax(&smax[(i >> 3) | ((j >> 3) << 1) | (kz << 2)], (unsigned long long)__double_as_longlong(b));
  }
  __syncthreads();
  if (threadIdx.x < 8) out[size_t(blockIdx.x) * 8 + threadIdx.x] = __longlong_as_double((long long)smax[threadIdx.x]);
}

// S21: all interior cells of fine patch p from its parent's padded box (operator of S6, one slot).
template <typename T, int NV>
__global__ void __launch_bounds__(256) k_prolong_interior(Pool<T> pool, int slot, int pslot, int p,
                                                          const Desc *__restrict__ desc, const int *__restrict__ plist) {
  if (plist) p = plist[blockIdx.y];                              // batched: one grid row of 16 blocks per listed patch
  const Desc &D = desc[p];
  const int Q = D.parent;
  T *U = pool.patch(slot, p);
  const T *C = pool.patch(pslot, Q);
  const int ox = D.origin[0] - 2 * desc[Q].origin[0], oy = D.origin[1] - 2 * desc[Q].origin[1],
            oz = D.origin[2] - 2 * desc[Q].origin[2];           // 0 or 16: the octant
  const int k = blockIdx.x;                                      // one interior plane per block
  const int i = threadIdx.x & 15, j = threadIdx.x >> 4;
  const int g[3] = {ox + i, oy + j, oz + k};                     // fine index relative to the parent's corner
  int c0;
  T sg[3];
  {
    int pc[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      pc[d] = (g[d] >> 1) + NG;
      sg[d] = (g[d] & 1) ? T(0.25) : T(-0.25);
    }
    c0 = cell<T>(pc[2], pc[1], pc[0]);
  }
  const int st[3] = {1, Layout<T>::PX, Layout<T>::PLANE};
  const int me = cell<T>(k + NG, j + NG, i + NG);
#pragma unroll
  for (int v = 0; v < NV; ++v) {
    const T *c = C + size_t(v) * Layout<T>::VS;
    const T uc = c[c0];
    T val = uc;
#pragma unroll
    for (int d = 0; d < 3; ++d) val = val + sg[d] * minmod2(c[c0 + st[d]] - uc, uc - c[c0 - st[d]]);
    U[size_t(v) * Layout<T>::VS + me] = val;
  }
}

// Regrid (NEXT-3): surviving patches move to their index in the new table.  One block per new patch; map[q] = index
// in the old table or -1 (new patch: left for k_prolong_interior).  Whole padded boxes, 16-byte copies, from one
// slot to another (never in place).
template <typename T>
__global__ void __launch_bounds__(256) k_move_patches(Pool<T> pool, int src_slot, int dst_slot, const int *__restrict__ map) {
  const int q = blockIdx.x, o = map[q];
  if (o < 0) return;
  const uint4 *s = reinterpret_cast<const uint4 *>(pool.patch(src_slot, o));
  uint4 *d = reinterpret_cast<uint4 *>(pool.patch(dst_slot, q));
  const int n = int(size_t(pool.nv) * Layout<T>::VS * sizeof(T) / sizeof(uint4));
  for (int c = threadIdx.x; c < n; c += 256) d[c] = s[c];
}

// ------------------------------------------------------------------ a7: restriction (S8)
// One block per fine patch; each thread produces coarse cells (pairwise tree sum, so that a
// uniform state is restricted bitwise).
template <typename T, int NV>
__global__ void __launch_bounds__(256) k_restrict(Pool<T> pool, int fslot, int cslot, int first,
                                                  const Desc *__restrict__ desc, const int *__restrict__ octant) {
  const int p = first + blockIdx.x;
  const int Q = desc[p].parent, o = octant[p];
  const int ocx = o & 1, ocy = (o >> 1) & 1, ocz = (o >> 2) & 1;
  const T *Uf = pool.patch(fslot, p);
  T *Uc = pool.patch(cslot, Q);
  for (int t = threadIdx.x; t < 512 * NV; t += 256) {
    const int v = t / 512, c = t % 512;
    const int ci = c & 7, cj = (c >> 3) & 7, ck = c >> 6;
    const T *f = Uf + size_t(v) * Layout<T>::VS;
    auto F = [&](int dk, int dj, int di) { return f[cell<T>(NG + 2 * ck + dk, NG + 2 * cj + dj, NG + 2 * ci + di)]; };
    const T s = ((F(0, 0, 0) + F(0, 0, 1)) + (F(0, 1, 0) + F(0, 1, 1))) +
                ((F(1, 0, 0) + F(1, 0, 1)) + (F(1, 1, 0) + F(1, 1, 1)));
    Uc[size_t(v) * Layout<T>::VS + cell<T>(NG + 8 * ocz + ck, NG + 8 * ocy + cj, NG + 8 * ocx + ci)] = T(0.125) * s;
  }
}

// ------------------------------------------------------------------ flux registers (S10)
// rk_stage leaves the fluxes through the faces 0, 8 and 16 of every interior line in
// bflux[(patch_local*9 + d*3 + s)*NV + v][t2*16 + t1]  (s = face/8).  This kernel turns them
// into register increments in a fixed order: task < 6 = fine side of this patch's face;
// task >= 6 = coarse side under child (task-6)/6, face (task-6)%6.
template <typename T, int NV>
__global__ void __launch_bounds__(64) k_flux_registers(int first, int level, const Desc *__restrict__ desc,
                                                       const int *__restrict__ child, const T *__restrict__ bflux,
                                                       T *__restrict__ Rf, T *__restrict__ Rc, T wdt, double w, DtDev dtd,
                                                       const int *__restrict__ tasks) {
  if (dtd.p) wdt = T(w * (*dtd.p * dtd.pow2));
  // tasks (may be null): the (patch, face) and (patch, octant, face) pairs of the level that lie on a coarse-fine
  // boundary, packed as local patch * 64 + task, found once per hierarchy; null: every block tests its own pair
  const int pl = tasks ? tasks[blockIdx.x] >> 6 : blockIdx.x, p = first + pl, task = tasks ? tasks[blockIdx.x] & 63 : blockIdx.y;
  const int ca = threadIdx.x & 7, cb = threadIdx.x >> 3;
  if (task < 6) {
    const int f = task;
    if (level == 0 || desc[p].nbr[face_region(f)] != -1) return;
    const int d = f >> 1, s = (f & 1) ? 2 : 0;
    T *R = Rf + (size_t(p) * 6 + f) * NV * 64;
#pragma unroll
    for (int v = 0; v < NV; ++v) {
      const T *F = bflux + ((size_t(pl) * 9 + d * 3 + s) * NV + v) * 256;
      const T sum = (F[(2 * cb) * 16 + 2 * ca] + F[(2 * cb) * 16 + 2 * ca + 1]) +
                    (F[(2 * cb + 1) * 16 + 2 * ca] + F[(2 * cb + 1) * 16 + 2 * ca + 1]);
      R[v * 64 + cb * 8 + ca] += wdt * (T(0.25) * sum);
    }
  } else {
    const int o = (task - 6) / 6, f = (task - 6) % 6;
    const int ch = child[size_t(p) * 8 + o];
    if (ch < 0 || desc[ch].nbr[face_region(f)] != -1) return;
    const int oc[3] = {o & 1, (o >> 1) & 1, (o >> 2) & 1};
    const int d = f >> 1, s = oc[d] + (f & 1);
    const int d1 = (d == 0) ? 1 : 0, d2 = (d == 2) ? 1 : 2;
    T *R = Rc + (size_t(ch) * 6 + f) * NV * 64;
#pragma unroll
    for (int v = 0; v < NV; ++v) {
      const T *F = bflux + ((size_t(pl) * 9 + d * 3 + s) * NV + v) * 256;
      R[v * 64 + cb * 8 + ca] += wdt * F[(8 * oc[d2] + cb) * 16 + 8 * oc[d1] + ca];
    }
  }
}

// ------------------------------------------------------------------ a8: refluxing (S10)
// Launched once per axis with both faces of that axis (gridDim.y = 2), in the fixed order x, y, z: fine patches
// cover octants of 8 coarse cells, so an uncovered coarse cell cannot touch fine patches on both sides along
// one axis -- it is corrected by at most one face per launch (no races), and the launches keep the face order
// f = 0..5 of S10 for the cells that get corrections along several axes (deterministic rounding).
template <typename T, int NV>
__global__ void __launch_bounds__(64) k_reflux(Pool<T> pool, int slot, int first_fine, int f,
                                               const Desc *__restrict__ desc, const int *__restrict__ octant,
                                               T *__restrict__ Rf, T *__restrict__ Rc, T hc) {
  const int p = first_fine + blockIdx.x;
  f += blockIdx.y;                               // (launched per axis with gridDim.y = 2: the low and the high face)
  if (desc[p].nbr[face_region(f)] != -1) return;
  const int Q = desc[p].parent, o = octant[p];
  const int oc[3] = {o & 1, (o >> 1) & 1, (o >> 2) & 1};
  const int d = f >> 1, hi = f & 1;
  const int d1 = (d == 0) ? 1 : 0, d2 = (d == 2) ? 1 : 2;
  int cn = NG + 8 * oc[d] + (hi ? 8 : -1);
  int tgt = Q;
  if (cn < NG || cn >= NG + NI) {
    tgt = desc[Q].nbr[face_region(f)];
    if (tgt < 0) return;                        // improper nesting is rejected by set_hierarchy
    cn += hi ? -NI : NI;
  }
  T *U = pool.patch(slot, tgt);
  T *rf = Rf + (size_t(p) * 6 + f) * NV * 64, *rc = Rc + (size_t(p) * 6 + f) * NV * 64;
  const int ca = threadIdx.x & 7, cb = threadIdx.x >> 3;
  int pad[3];
  pad[d] = cn; pad[d1] = NG + 8 * oc[d1] + ca; pad[d2] = NG + 8 * oc[d2] + cb;
  const int c = cell<T>(pad[2], pad[1], pad[0]);
#pragma unroll
  for (int v = 0; v < NV; ++v) {
    const int r = v * 64 + cb * 8 + ca;
    const T corr = (rf[r] - rc[r]) / hc;
    T *u = U + size_t(v) * Layout<T>::VS + c;
    *u = hi ? (*u + corr) : (*u - corr);
    rf[r] = T(0); rc[r] = T(0);
  }
}

}  // namespace amr
