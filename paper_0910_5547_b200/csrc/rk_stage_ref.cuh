// rk_stage_ref.cuh -- reference stage kernel: one thread per interior cell, everything read
// straight from global memory, every face flux recomputed by both cells that share it.
// Slow (about 2x the flux work, 3x the slope work) but short enough to check by eye; the
// optimised kernel in rk_stage_tile.cuh is tested against the oracle AND against this one.
// Steps a3-a6 of the hot path: PAPER.md:79 Eq. 7, :94-98 Eq. 8, :104-118 Eq. 9-12.
#pragma once
#include "layout.cuh"
#include "physics.cuh"

namespace amr {

template <typename T, int NV, int D>
__device__ __forceinline__ void ref_direction(const T *__restrict__ Uin, int c, const Params<T> &P, int &hits,
                                              T (&Flo)[NV], T (&Fhi)[NV]) {
  constexpr int st = D == 0 ? 1 : (D == 1 ? Layout<T>::PX : Layout<T>::PLANE);
  T W[5][NV];
#pragma unroll
  for (int s = 0; s < 5; ++s) {
    T U[NV];
#pragma unroll
    for (int v = 0; v < NV; ++v) U[v] = Uin[size_t(v) * Layout<T>::VS + c + (s - 2) * st];
    cons_to_prim<T, NV>(U, W[s], P, hits);
  }
  T WLlo[NV], WRlo[NV], WLhi[NV], WRhi[NV];
#pragma unroll
  for (int v = 0; v < NV; ++v) {
    const T sm = limited_slope(W[0][v], W[1][v], W[2][v], P.theta);
    const T s0 = limited_slope(W[1][v], W[2][v], W[3][v], P.theta);
    const T sp = limited_slope(W[2][v], W[3][v], W[4][v], P.theta);
    WLlo[v] = W[1][v] + T(0.5) * sm;   // Eq. 9 at face i-1/2
    WRlo[v] = W[2][v] - T(0.5) * s0;   // Eq. 10 at face i-1/2
    WLhi[v] = W[2][v] + T(0.5) * s0;   // Eq. 9 at face i+1/2
    WRhi[v] = W[3][v] - T(0.5) * sp;   // Eq. 10 at face i+1/2
  }
  floor_state<T, NV>(WLlo, P, hits); floor_state<T, NV>(WRlo, P, hits);
  floor_state<T, NV>(WLhi, P, hits); floor_state<T, NV>(WRhi, P, hits);
  riemann_flux<T, NV, D>(WLlo, WRlo, P, Flo);
  riemann_flux<T, NV, D>(WLhi, WRhi, P, Fhi);
}

// grid: (npatches_of_level, 16 k-planes); block: 256 threads = one (j,i) plane.
// bflux (may be null): fluxes through faces 0, 8, 16 of every line, see k_flux_registers.
template <typename T, int NV>
__global__ void __launch_bounds__(256) k_rk_stage_ref(Pool<T> pool, int sin, int sbase, int sout, int first,
                                                      T a, T b, T dtdx, Params<T> P, T *__restrict__ bflux,
                                                      unsigned long long *__restrict__ floor_hits, DtDev dtd) {
  if (dtd.p) dtdx = T((*dtd.p * dtd.pow2) / dtd.hx);
  const int pl = blockIdx.x, p = first + pl;
  const int i = threadIdx.x & 15, j = threadIdx.x >> 4, k = blockIdx.y;
  const T *Uin = pool.patch(sin, p);
  const T *Ub = pool.patch(sbase, p);
  T *Uo = pool.patch(sout, p);
  const int c = cell<T>(k + NG, j + NG, i + NG);
  int hits = 0;
  T Fxl[NV], Fxh[NV], Fyl[NV], Fyh[NV], Fzl[NV], Fzh[NV];
  ref_direction<T, NV, 0>(Uin, c, P, hits, Fxl, Fxh);
  ref_direction<T, NV, 1>(Uin, c, P, hits, Fyl, Fyh);
  ref_direction<T, NV, 2>(Uin, c, P, hits, Fzl, Fzh);
#pragma unroll
  for (int v = 0; v < NV; ++v) {
    const T div = ((Fxh[v] - Fxl[v]) + (Fyh[v] - Fyl[v])) + (Fzh[v] - Fzl[v]);   // order x, y, z
    const size_t g = size_t(v) * Layout<T>::VS + c;
    Uo[g] = a * Ub[g] + b * (Uin[g] - dtdx * div);
  }
  if (bflux) {
    const int idx[3] = {i, j, k};
    const int t1[3] = {j, i, i}, t2[3] = {k, k, j};
    const T *lo[3] = {Fxl, Fyl, Fzl}, *hi[3] = {Fxh, Fyh, Fzh};
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      const int t = t2[d] * 16 + t1[d];
      T *B = bflux + (size_t(pl) * 9 + d * 3) * NV * 256;
      if (idx[d] == 0) for (int v = 0; v < NV; ++v) B[(0 * NV + v) * 256 + t] = lo[d][v];
      if (idx[d] == 8) for (int v = 0; v < NV; ++v) B[(1 * NV + v) * 256 + t] = lo[d][v];
      if (idx[d] == 15) for (int v = 0; v < NV; ++v) B[(2 * NV + v) * 256 + t] = hi[d][v];
    }
  }
  if (hits) atomicAdd(floor_hits, (unsigned long long)hits);
}

}  // namespace amr
