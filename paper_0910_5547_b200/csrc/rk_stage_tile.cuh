// rk_stage_tile.cuh -- the hot kernel: one method-of-lines stage of every 16^3 patch of a level
// (steps a3-a6: PAPER.md:79 Eq. 7, :94-98 Eq. 8, :104-112 Eq. 9-11, :114-118 Eq. 12).
//
// B200 design (not the paper's: its 1-D flattened sweeps with one global round trip per
// kernel, PAPER.md:139-153 / :226-248, are prior art):
//  * one CTA per patch, 10 warps: 8 "interior" warps own the 16x16 (i,j) columns and march
//    in z over the 20 padded planes; warp 8 owns the x-halo columns (i = -1 and 16), warp 9
//    the y-halo rows (j = -1 and 16).  Fluxes, L(U) and primitives never touch HBM.
//  * every cell is read from HBM exactly once per stage (coalesced 16-wide rows, prefetched
//    one plane ahead into registers), converted to primitives once (one reciprocal), and its
//    primitives are put in a double-buffered shared-memory plane for the x/y neighbours.
//  * z stencil lives in registers; x/y stencils exchange the cell-edge states q+ and the face
//    fluxes through shared memory (two barriers per plane), so each slope and each face flux
//    of a patch is computed exactly once.
//  * halo source is per face: own ghost zones (materialised by fill_ghosts) or, with
//    AMRHYDRO_OPT_HALO=1, the sibling's interior directly (no ghost round trip through HBM).
#pragma once
#include "layout.cuh"
#include "physics.cuh"

namespace amr {

template <typename T> struct TileCfg;
template <> struct TileCfg<double> { static constexpr int PW = 20, PQ = 18, PQ2 = 16; };
template <> struct TileCfg<float> { static constexpr int PW = 24, PQ = 24, PQ2 = 24; };   // rows j, j+2 hit disjoint banks

template <typename T, int NV> struct TileSmem {
  static constexpr int PW = TileCfg<T>::PW, PQ = TileCfg<T>::PQ, PQ2 = TileCfg<T>::PQ2;
  static constexpr int WP_ELEMS = 2 * NV * NP * PW;
  static constexpr int QX_ELEMS = NV * NI * PQ;
  static constexpr int QY_ELEMS = NV * (NI + 2) * PQ2;
  static constexpr int TOTAL = WP_ELEMS + 2 * QX_ELEMS + 2 * QY_ELEMS;
  static constexpr size_t BYTES = size_t(TOTAL) * sizeof(T);
};

constexpr int TILE_THREADS = 320;

template <typename T, int NV>
__global__ void __launch_bounds__(TILE_THREADS, (sizeof(T) == 4 ? 2 : 1))
k_rk_stage_tile(Pool<T> pool, int sin, int sbase, int sout, int first, T a, T b, T dtdx, Params<T> P,
                T *__restrict__ bflux, unsigned long long *__restrict__ floor_hits,
                const Desc *__restrict__ desc, int direct_halo) {
  using S = TileSmem<T, NV>;
  constexpr int PW = S::PW, PQ = S::PQ, PQ2 = S::PQ2;
  constexpr int PX = Layout<T>::PX, PLANE = Layout<T>::PLANE, VS = Layout<T>::VS;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  T *WP = reinterpret_cast<T *>(smem_raw);     // [2][NV][20][PW]   primitive planes
  T *QX = WP + S::WP_ELEMS;                    // [NV][16][PQ]      q+ of cell ci at ci+1
  T *FX = QX + S::QX_ELEMS;                    // [NV][16][PQ]      x flux at face fi
  T *QY = FX + S::QX_ELEMS;                    // [NV][18][PQ2]     q+ of cell cj at row cj+1
  T *FY = QY + S::QY_ELEMS;                    // [NV][18][PQ2]     y flux at face fj

  const int pl = blockIdx.x, p = first + pl;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const T *self = pool.patch(sin, p);
  // halo sources: own ghost zones, or the sibling's interior (shift = +-16 cells along the axis)
  const T *src[6];
  int shift[6];
#pragma unroll
  for (int f = 0; f < 6; ++f) {
    const int nb = direct_halo ? desc[p].nbr[face_region(f)] : -1;
    const int st = (f >> 1) == 0 ? 1 : ((f >> 1) == 1 ? PX : PLANE);
    src[f] = nb >= 0 ? pool.patch(sin, nb) : self;
    shift[f] = nb >= 0 ? ((f & 1) ? -NI * st : NI * st) : 0;
  }
  const T bdtdx = b * dtdx;
  int hits = 0;
  auto wp = [&](int buf, int v, int pj, int pi) -> T & { return WP[((buf * NV + v) * NP + pj) * PW + pi]; };

  if (warp < 8) {
    // ------------------------------------------------------------------ interior columns
    const int i = lane & 15, j = (warp & 1) + 2 * (lane >> 4) + 4 * (warp >> 1);
    const int pi = i + NG, pj = j + NG;
    const int off = Layout<T>::LEAD + pj * PX + pi;             // in-plane offset of this column
    const T *base = pool.patch(sbase, p) + off;
    T *out = pool.patch(sout, p) + off;
    const bool use_base = (a != T(0));
    auto plane_src = [&](int pk) -> const T * {
      return (pk < NG) ? src[4] + shift[4] + off + pk * PLANE
                       : (pk >= NG + NI ? src[5] + shift[5] + off + pk * PLANE : self + off + pk * PLANE);
    };
    T Wm[NV], Wc[NV], Wn[NV], Un[NV], Ubn[NV];
    T qpz[NV], Fzp[NV], accp[NV], pre0[NV], pre1[NV], pre2[NV];
    // prologue: planes 0 and 1 (z ghosts) -> Wm, Wc ; prefetch plane 2
    {
      const T *s0 = plane_src(0), *s1 = plane_src(1), *s2 = plane_src(2);
      T U0[NV], U1[NV];
#pragma unroll
      for (int v = 0; v < NV; ++v) { U0[v] = s0[size_t(v) * VS]; U1[v] = s1[size_t(v) * VS]; Un[v] = s2[size_t(v) * VS]; }
      if (use_base) {
#pragma unroll
        for (int v = 0; v < NV; ++v) Ubn[v] = base[size_t(v) * VS + 2 * PLANE];
      }
      cons_to_prim<T, NV>(U0, Wm, P, hits);
      cons_to_prim<T, NV>(U1, Wc, P, hits);
    }
#pragma unroll
    for (int v = 0; v < NV; ++v) { qpz[v] = Fzp[v] = accp[v] = pre0[v] = pre1[v] = pre2[v] = T(0); }

#pragma unroll 1
    for (int c = 1; c <= NG + NI; ++c) {          // current cell = padded plane c (cells k = -1..16)
      // 1. plane c+1: raw -> primitives (+ RK "pre" term), publish for the x/y neighbours
      cons_to_prim<T, NV>(Un, Wn, P, hits);
      const bool next_interior = (c + 1 >= NG) && (c + 1 < NG + NI);
#pragma unroll
      for (int v = 0; v < NV; ++v) {
        pre0[v] = pre1[v]; pre1[v] = pre2[v];
        pre2[v] = use_base ? (a * Ubn[v] + b * Un[v]) : (b * Un[v]);
      }
      if (next_interior) {
#pragma unroll
        for (int v = 0; v < NV; ++v) wp((c + 1) & 1, v, pj, pi) = Wn[v];
      }
      // 2. prefetch plane c+2
      if (c + 2 < NP) {
        const T *s = plane_src(c + 2);
#pragma unroll
        for (int v = 0; v < NV; ++v) Un[v] = s[size_t(v) * VS];
        if (use_base && c + 2 < NG + NI) {
#pragma unroll
          for (int v = 0; v < NV; ++v) Ubn[v] = base[size_t(v) * VS + (c + 2) * PLANE];
        }
      }
      // 3. z: slope of cell c, edge states, flux through the face between c-1 and c
      T qmz[NV], qpc[NV], Fz[NV];
#pragma unroll
      for (int v = 0; v < NV; ++v) {
        const T s = limited_slope(Wm[v], Wc[v], Wn[v], P.theta);
        qmz[v] = Wc[v] - T(0.5) * s;
        qpc[v] = Wc[v] + T(0.5) * s;
      }
      if (c >= NG) {
        T WL[NV], WR[NV];
#pragma unroll
        for (int v = 0; v < NV; ++v) { WL[v] = qpz[v]; WR[v] = qmz[v]; }
        floor_state<T, NV>(WL, P, hits); floor_state<T, NV>(WR, P, hits);
        riemann_flux<T, NV, 2>(WL, WR, P, Fz);
        if (bflux && ((c - NG) & 7) == 0) {
          T *B = bflux + ((size_t(pl) * 9 + 6 + ((c - NG) >> 3)) * NV) * 256 + j * 16 + i;
#pragma unroll
          for (int v = 0; v < NV; ++v) B[v * 256] = Fz[v];
        }
      }
      const bool cur_interior = (c >= NG) && (c < NG + NI);
      T acc[NV];
      if (cur_interior) {
        // 4. x/y phase 1: slopes of this cell along x and y, publish q+
        const int buf = c & 1;
        T qmx[NV], qmy[NV];
#pragma unroll
        for (int v = 0; v < NV; ++v) {
          const T sx = limited_slope(wp(buf, v, pj, pi - 1), Wc[v], wp(buf, v, pj, pi + 1), P.theta);
          const T sy = limited_slope(wp(buf, v, pj - 1, pi), Wc[v], wp(buf, v, pj + 1, pi), P.theta);
          qmx[v] = Wc[v] - T(0.5) * sx;
          qmy[v] = Wc[v] - T(0.5) * sy;
          QX[(v * NI + j) * PQ + i + 1] = Wc[v] + T(0.5) * sx;
          QY[(v * (NI + 2) + j + 1) * PQ2 + i] = Wc[v] + T(0.5) * sy;
        }
        __syncthreads();
        // 5. phase 2: fluxes through the low x and y faces of this cell
        T Fxl[NV], Fyl[NV];
        {
          T WL[NV];
#pragma unroll
          for (int v = 0; v < NV; ++v) WL[v] = QX[(v * NI + j) * PQ + i];
          floor_state<T, NV>(WL, P, hits); floor_state<T, NV>(qmx, P, hits);
          riemann_flux<T, NV, 0>(WL, qmx, P, Fxl);
#pragma unroll
          for (int v = 0; v < NV; ++v) { FX[(v * NI + j) * PQ + i] = Fxl[v]; WL[v] = QY[(v * (NI + 2) + j) * PQ2 + i]; }
          floor_state<T, NV>(WL, P, hits); floor_state<T, NV>(qmy, P, hits);
          riemann_flux<T, NV, 1>(WL, qmy, P, Fyl);
#pragma unroll
          for (int v = 0; v < NV; ++v) FY[(v * (NI + 2) + j) * PQ2 + i] = Fyl[v];
        }
        if (bflux) {
          if ((i & 7) == 0) {
            T *B = bflux + ((size_t(pl) * 9 + 0 + (i >> 3)) * NV) * 256 + (c - NG) * 16 + j;
#pragma unroll
            for (int v = 0; v < NV; ++v) B[v * 256] = Fxl[v];
          }
          if ((j & 7) == 0) {
            T *B = bflux + ((size_t(pl) * 9 + 3 + (j >> 3)) * NV) * 256 + (c - NG) * 16 + i;
#pragma unroll
            for (int v = 0; v < NV; ++v) B[v * 256] = Fyl[v];
          }
        }
        __syncthreads();
        // 6. phase 3: flux differences in x and y
#pragma unroll
        for (int v = 0; v < NV; ++v)
          acc[v] = (FX[(v * NI + j) * PQ + i + 1] - Fxl[v]) + (FY[(v * (NI + 2) + j + 1) * PQ2 + i] - Fyl[v]);
      }
      // 7. finish cell c-1: add the z difference, RK combination (Eq. 8), store
      if (c - 1 >= NG) {
        T *o = out + (c - 1) * PLANE;
#pragma unroll
        for (int v = 0; v < NV; ++v) o[size_t(v) * VS] = pre0[v] - bdtdx * (accp[v] + (Fz[v] - Fzp[v]));
      }
      // 8. rotate
#pragma unroll
      for (int v = 0; v < NV; ++v) {
        Wm[v] = Wc[v]; Wc[v] = Wn[v]; qpz[v] = qpc[v];
        if (c >= NG) Fzp[v] = Fz[v];
        if (cur_interior) accp[v] = acc[v];
      }
      if (c == 1) __syncthreads();   // plane 2's primitives were published without a phase barrier
    }
  } else if (warp == 8) {
    // ------------------------------------------------------------------ x-halo columns
    const int j = lane & 15, hi = lane >> 4;
    const int pj = j + NG, pi0 = hi ? NG + NI : 0;               // this lane owns cells pi0, pi0+1
    const int ci = hi ? NI : -1;                                 // the cell whose slope it computes
    const T *s = src[hi] + shift[hi] + Layout<T>::LEAD + pj * PX + pi0;
    T Ua[NV], Ub2[NV];
#pragma unroll
    for (int v = 0; v < NV; ++v) { Ua[v] = s[size_t(v) * VS + NG * PLANE]; Ub2[v] = s[size_t(v) * VS + NG * PLANE + 1]; }
#pragma unroll 1
    for (int c = 1; c <= NG + NI; ++c) {
      const bool next_interior = (c + 1 >= NG) && (c + 1 < NG + NI);
      if (next_interior) {
        T W0[NV], W1[NV];
        cons_to_prim<T, NV>(Ua, W0, P, hits);
        cons_to_prim<T, NV>(Ub2, W1, P, hits);
#pragma unroll
        for (int v = 0; v < NV; ++v) { wp((c + 1) & 1, v, pj, pi0) = W0[v]; wp((c + 1) & 1, v, pj, pi0 + 1) = W1[v]; }
        if (c + 2 < NG + NI) {
#pragma unroll
          for (int v = 0; v < NV; ++v) {
            Ua[v] = s[size_t(v) * VS + (c + 2) * PLANE];
            Ub2[v] = s[size_t(v) * VS + (c + 2) * PLANE + 1];
          }
        }
      }
      const bool cur_interior = (c >= NG) && (c < NG + NI);
      if (cur_interior) {
        const int buf = c & 1, pc = ci + NG;
        T qm[NV];
#pragma unroll
        for (int v = 0; v < NV; ++v) {
          const T w0 = wp(buf, v, pj, pc);
          const T sx = limited_slope(wp(buf, v, pj, pc - 1), w0, wp(buf, v, pj, pc + 1), P.theta);
          qm[v] = w0 - T(0.5) * sx;
          if (!hi) QX[(v * NI + j) * PQ + 0] = w0 + T(0.5) * sx;      // q+ of cell -1
        }
        __syncthreads();
        if (hi) {                                                     // face 16: q+ of cell 15 | q- of cell 16
          T WL[NV], F[NV];
#pragma unroll
          for (int v = 0; v < NV; ++v) WL[v] = QX[(v * NI + j) * PQ + NI];
          floor_state<T, NV>(WL, P, hits); floor_state<T, NV>(qm, P, hits);
          riemann_flux<T, NV, 0>(WL, qm, P, F);
#pragma unroll
          for (int v = 0; v < NV; ++v) FX[(v * NI + j) * PQ + NI] = F[v];
          if (bflux) {
            T *B = bflux + ((size_t(pl) * 9 + 2) * NV) * 256 + (c - NG) * 16 + j;
#pragma unroll
            for (int v = 0; v < NV; ++v) B[v * 256] = F[v];
          }
        }
        __syncthreads();
      }
      if (c == 1) __syncthreads();
    }
  } else {
    // ------------------------------------------------------------------ y-halo rows
    const int i = lane & 15, hi = lane >> 4;
    const int pi = i + NG, pj0 = hi ? NG + NI : 0;
    const int cj = hi ? NI : -1;
    const T *s = src[2 + hi] + shift[2 + hi] + Layout<T>::LEAD + pj0 * PX + pi;
    T Ua[NV], Ub2[NV];
#pragma unroll
    for (int v = 0; v < NV; ++v) { Ua[v] = s[size_t(v) * VS + NG * PLANE]; Ub2[v] = s[size_t(v) * VS + NG * PLANE + PX]; }
#pragma unroll 1
    for (int c = 1; c <= NG + NI; ++c) {
      const bool next_interior = (c + 1 >= NG) && (c + 1 < NG + NI);
      if (next_interior) {
        T W0[NV], W1[NV];
        cons_to_prim<T, NV>(Ua, W0, P, hits);
        cons_to_prim<T, NV>(Ub2, W1, P, hits);
#pragma unroll
        for (int v = 0; v < NV; ++v) { wp((c + 1) & 1, v, pj0, pi) = W0[v]; wp((c + 1) & 1, v, pj0 + 1, pi) = W1[v]; }
        if (c + 2 < NG + NI) {
#pragma unroll
          for (int v = 0; v < NV; ++v) {
            Ua[v] = s[size_t(v) * VS + (c + 2) * PLANE];
            Ub2[v] = s[size_t(v) * VS + (c + 2) * PLANE + PX];
          }
        }
      }
      const bool cur_interior = (c >= NG) && (c < NG + NI);
      if (cur_interior) {
        const int buf = c & 1, pc = cj + NG;
        T qm[NV];
#pragma unroll
        for (int v = 0; v < NV; ++v) {
          const T w0 = wp(buf, v, pc, pi);
          const T sy = limited_slope(wp(buf, v, pc - 1, pi), w0, wp(buf, v, pc + 1, pi), P.theta);
          qm[v] = w0 - T(0.5) * sy;
          if (!hi) QY[(v * (NI + 2) + 0) * PQ2 + i] = w0 + T(0.5) * sy;   // q+ of cell row -1
        }
        __syncthreads();
        if (hi) {
          T WL[NV], F[NV];
#pragma unroll
          for (int v = 0; v < NV; ++v) WL[v] = QY[(v * (NI + 2) + NI) * PQ2 + i];
          floor_state<T, NV>(WL, P, hits); floor_state<T, NV>(qm, P, hits);
          riemann_flux<T, NV, 1>(WL, qm, P, F);
#pragma unroll
          for (int v = 0; v < NV; ++v) FY[(v * (NI + 2) + NI) * PQ2 + i] = F[v];
          if (bflux) {
            T *B = bflux + ((size_t(pl) * 9 + 5) * NV) * 256 + (c - NG) * 16 + i;
#pragma unroll
            for (int v = 0; v < NV; ++v) B[v * 256] = F[v];
          }
        }
        __syncthreads();
      }
      if (c == 1) __syncthreads();
    }
  }
  if (hits) atomicAdd(floor_hits, (unsigned long long)hits);
}

// returns 0 or a cudaError_t
template <typename T, int NV>
int launch_rk_stage_tile(Pool<T> pool, int sin, int sbase, int sout, int first, int n, T a, T b, T dtdx,
                         Params<T> P, T *bflux, unsigned long long *floor_hits, const Desc *desc, int direct_halo,
                         cudaStream_t stream) {
  static bool configured = false;
  constexpr size_t bytes = TileSmem<T, NV>::BYTES;
  if (!configured) {
    cudaError_t e = cudaFuncSetAttribute(k_rk_stage_tile<T, NV>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(bytes));
    if (e != cudaSuccess) return int(e);
    configured = true;
  }
  k_rk_stage_tile<T, NV><<<n, TILE_THREADS, bytes, stream>>>(pool, sin, sbase, sout, first, a, b, dtdx, P, bflux,
                                                             floor_hits, desc, direct_halo);
  return 0;
}

}  // namespace amr
