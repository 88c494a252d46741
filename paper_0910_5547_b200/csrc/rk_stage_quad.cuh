// rk_stage_quad.cuh -- the stage kernel on quarter-patch tiles: one CTA of 3 warps advances an
// 8x8 column tile of a 16^3 patch through one method-of-lines stage (steps a3-a6: PAPER.md:79
// Eq. 7, :94-98 Eq. 8, :104-112 Eq. 9-11, :114-118 Eq. 12).
//
// Why: ncu on k_rk_stage_march (one 10-warp CTA per patch and SM; profiles/README.md r1b/r1c) shows
// the FP64 pipe, the issue slots and the shared-memory crossbar each ~40-45 % busy and adding up
// instead of overlapping: the two block barriers per plane keep all warps of the SM in the same
// phase (load-heavy slopes, then FP64-heavy fluxes).  The arithmetic and the z-marching scheme
// here are those of rk_stage_march.cuh; what changes is the granularity: 4-5 small independent
// CTAs per SM that drift out of phase, so that one tile's flux phase overlaps another tile's
// shared-memory phase.  Cost: the halo of a tile is relatively larger (one halo warp per two
// interior warps, and the faces between the four tiles of a patch are computed by both sides,
// bitwise identically).
//   warps 0-1 : interior columns, lane = (i, j) = (tid & 7, tid >> 3)
//   warp  2   : halo; lanes 0-15 the x ghost columns (8 rows x 2 sides), lanes 16-31 the y ghost
//               rows; lane 0 feeds the TMA ring (8x8xNV boxes)
// Shared memory (fp64, 5 variables): 44 kB per CTA; the flux arrays alias the q+ arrays (each slot
// has one reader, which reads the q+ before it overwrites the slot with its flux).
#pragma once
#include "rk_stage_march.cuh"

namespace amr {
namespace qk {

constexpr int TS = 8;                 // tile side
constexpr int TP = TS + 2 * NG;       // 12
constexpr int PW = 24, PQ = 24, PY = 8;   // pitches: rows of 8 cells land on disjoint banks (fp64 and fp32)
constexpr int NSLOT = 4;
constexpr int THREADS = 96;

template <typename T, int NV> struct Smem {
  static constexpr int RAWP = NV * TS * TS;        // one raw plane: [NV][8][8], dense TMA box
  static constexpr int WV = TP * PW;               // one variable of one primitive plane [12][PW]
  static constexpr int QXV = TS * PQ;              // [8][PQ]: slot s = q+ of cell s-1, then flux at face s
  static constexpr int QYV = (TS + 1) * PY;        // [9][PY]
  static constexpr int O_RAW = 0, O_W = O_RAW + NSLOT * RAWP, O_QX = O_W + 2 * NV * WV, O_QY = O_QX + NV * QXV,
                       O_END = O_QY + NV * QYV;
  static constexpr size_t BAR_OFF = ((size_t(O_END) * sizeof(T) + 15) / 16) * 16;
  static constexpr size_t BYTES = BAR_OFF + NSLOT * 8 + 128;   // + slack to align the ring to 128 B
};

// The halo warp.  Lane = (dirn, side, t): dirn 0 = the two ghost columns left/right of row t,
// dirn 1 = the two ghost rows below/above column t.  Converts its two cells of every interior
// plane, publishes them next to the interior cells, computes the slope of the ghost cell adjacent
// to the tile (q+ of cell -1 on the low side, q- of cell 8 on the high side) and, on the high
// side, the flux through face 8.  Sources: the tile's own patch, or across a patch face the
// neighbour's interior (direct halo) / the patch's own ghost zone.
template <typename T, int NV>
__device__ __forceinline__ void halo_warp(T *sm, const Pool<T> &pool, int sin, int p, const Desc &D, int direct_halo, int x0,
                                          int y0, int lane, const Params<T> &P, T th2, T *__restrict__ bflux, int pl, int &hits,
                                          const CUtensorMap *tmap, unsigned long long *bars) {
  using S = Smem<T, NV>;
  constexpr int WV = S::WV;
  constexpr int PX = Layout<T>::PX, PLANE = Layout<T>::PLANE, VS = Layout<T>::VS, LEAD = Layout<T>::LEAD;
  const int dirn = lane >> 4, hi = (lane >> 3) & 1, t = lane & 7;
  const T q4 = T(0.25);
  const int a = hi ? TS + NG : 0;                            // first of the two ghost cells, tile-padded coordinate along dirn
  // global source
  int px = dirn == 0 ? x0 + a : x0 + t + NG, py = dirn == 0 ? y0 + t + NG : y0 + a;
  int along = dirn == 0 ? px : py;
  int src = p;
  if (along < NG || along >= NG + NI) {
    const int nb = direct_halo ? D.nbr[face_region(2 * dirn + (along < NG ? 0 : 1))] : -1;
    if (nb >= 0) { src = nb; along += along < NG ? NI : -NI; }
  }
  if (dirn == 0) px = along; else py = along;
  const T *g = pool.patch(sin, src) + LEAD + py * PX + px;
  const int gst = dirn == 0 ? 1 : PX, rst = dirn == 0 ? 1 : PW;
  const int qv = dirn == 0 ? S::QXV : S::QYV;
  T *r = sm + S::O_W + (dirn == 0 ? (t + NG) * PW + a : a * PW + (t + NG));
  const T *st3 = r + (hi ? -rst : 0);                        // cells (7,8,9) or (-2,-1,0)
  T *Q = sm + (dirn == 0 ? S::O_QX + t * PQ : S::O_QY + t);
  T *qlo = Q;                                                // slot 0: q+ of cell -1
  T *qhi = Q + (dirn == 0 ? TS : TS * PY);                   // slot 8: q+ of cell 7, then the flux at face 8
  const bool rec = bflux && hi && (dirn == 0 ? x0 : y0) == TS;   // tile face 8 = patch face 16
  T Ua[NV], Ub[NV];
  auto load = [&](int pk) {
#pragma unroll
    for (int v = 0; v < NV; ++v) {
      const T *s = g + size_t(v) * VS + pk * PLANE;
      Ua[v] = s[0]; Ub[v] = s[gst];
    }
  };
  auto publish = [&](int pk) {
    T W0[NV], W1[NV];
    mk::prim<T, NV>(Ua, W0, P, hits);
    mk::prim<T, NV>(Ub, W1, P, hits);
    T *d = r + (pk & 1) * (NV * WV);
#pragma unroll
    for (int v = 0; v < NV; ++v) { d[v * WV] = W0[v]; d[v * WV + rst] = W1[v]; }
  };
  // TMA: interior box of padded plane pk (z ghost planes from the z neighbour when direct)
  const int nzl = direct_halo ? D.nbr[face_region(4)] : -1, nzh = direct_halo ? D.nbr[face_region(5)] : -1;
  const int qbase = sin * pool.max_patches;
  const int q_mid = (qbase + p) * NV, q_lo = (qbase + (nzl >= 0 ? nzl : p)) * NV, q_hi = (qbase + (nzh >= 0 ? nzh : p)) * NV;
  const int kz_lo = nzl >= 0 ? NI : 0, kz_hi = nzh >= 0 ? -NI : 0;
  const bool producer = lane == 0;
  auto issue = [&](int pk) {
    const int slot = pk % NSLOT;
    const int q = pk < NG ? q_lo : (pk >= NG + NI ? q_hi : q_mid);
    const int k = pk < NG ? pk + kz_lo : (pk >= NG + NI ? pk + kz_hi : pk);
    mk::mbar_expect_tx(&bars[slot], unsigned(S::RAWP * sizeof(T)));
    mk::tma_load_4d(sm + S::O_RAW + slot * S::RAWP, tmap, x0, NG + y0, k, q, &bars[slot]);
  };
  if (producer) {
#pragma unroll
    for (int s = 0; s < NSLOT; ++s) issue(s);
  }
  load(NG);
  publish(NG);
  load(NG + 1);
  __syncthreads();                                            // planes 0-2 converted by the interior warps
  if (producer) issue(NSLOT);                                 // slot of plane 0: converted, never needed again
#pragma unroll 1
  for (int c = NG; c < NG + NI; ++c) {
    if (c + 1 < NG + NI) {
      publish(c + 1);
      if (c + 2 < NG + NI) load(c + 2);
    }
    const T *s3 = st3 + (c & 1) * (NV * WV);
    T qm[NV];
#pragma unroll
    for (int v = 0; v < NV; ++v) {
      const T w0 = s3[v * WV], w1 = s3[v * WV + rst], w2 = s3[v * WV + 2 * rst];
      const T s = mk::slope4(w1 - w0, w2 - w1, w2 - w0, th2);
      qm[v] = fma(-q4, s, w1);                                // q- of cell 8 (high side)
      if (!hi) qlo[v * qv] = fma(q4, s, w1);                  // q+ of cell -1 (low side)
    }
    __syncthreads();
    if (producer && c + NSLOT - 1 < NP) issue(c + NSLOT - 1);   // slot of plane c-1 is free: cell c-1 is finished
    if (hi) {
      T WL[NV], G[NV];
#pragma unroll
      for (int v = 0; v < NV; ++v) WL[v] = qhi[v * qv];
      mk::floor_states<T, NV>(WL, qm, P, hits);
      if (dirn == 0) mk::face_flux<T, 0>(WL, qm, P, G);       // (both halves of the warp: same bits as the
      else           mk::face_flux<T, 1>(WL, qm, P, G);       //  interior warps' flux through the same face)
#pragma unroll
      for (int v = 0; v < NV; ++v) qhi[v * qv] = G[v];
      if (rec) {
        T *B = bflux + ((size_t(pl) * 9 + 3 * dirn + 2) * NV) * 256 + (c - NG) * 16 + (dirn == 0 ? y0 : x0) + t;
#pragma unroll
        for (int v = 0; v < NV; ++v) B[v * 256] = T(0.5) * G[v];
      }
    }
    __syncthreads();
  }
}

}  // namespace qk

#ifndef AMR_QUAD_MINB
#define AMR_QUAD_MINB 5
#endif

template <typename T, int NV, bool BASE>
__global__ void __launch_bounds__(qk::THREADS, (sizeof(T) == 8 && NV == 5) ? AMR_QUAD_MINB : (NV == 5 ? 8 : 3))
k_rk_stage_quad(const __grid_constant__ CUtensorMap tmap, Pool<T> pool, int sin, int sbase, int sout, int first, T a, T b,
                T dtdx, Params<T> P, T *__restrict__ bflux, unsigned long long *__restrict__ floor_hits,
                const Desc *__restrict__ desc, int direct_halo) {
  using S = qk::Smem<T, NV>;
  constexpr int TS = qk::TS, PW = qk::PW, PQ = qk::PQ, PY = qk::PY, NSLOT = qk::NSLOT;
  constexpr int WV = S::WV, QXV = S::QXV, QYV = S::QYV, RAWP = S::RAWP;
  constexpr int PX = Layout<T>::PX, PLANE = Layout<T>::PLANE, VS = Layout<T>::VS, LEAD = Layout<T>::LEAD;
  extern __shared__ unsigned char smem_raw[];
  // the TMA destination must be 128-byte aligned
  T *sm = reinterpret_cast<T *>(smem_raw + ((128u - (mk::smem_u32(smem_raw) & 127u)) & 127u));
  unsigned long long *bars = reinterpret_cast<unsigned long long *>(reinterpret_cast<unsigned char *>(sm) + S::BAR_OFF);

  const int pl = blockIdx.x >> 2, p = first + pl;
  const int x0 = (blockIdx.x & 1) * TS, y0 = ((blockIdx.x >> 1) & 1) * TS;       // tile origin inside the patch
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const T th2 = T(2) * P.theta, q4 = T(0.25);
  int hits = 0;

  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < NSLOT; ++s) mk::mbar_init(&bars[s], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  if (warp < 2) {
    // ------------------------------------------------------------------ interior columns
    const T kk = T(0.5) * b * dtdx;        // the 1/2 of Eq. 12 is applied here (G = 2F)
    const int i = tid & 7, j = tid >> 3;
    const int off = LEAD + (y0 + j + NG) * PX + (x0 + i + NG);  // in-plane offset of this column
    const T *base = pool.patch(sbase, p) + off;
    T *out = pool.patch(sout, p) + off;
    const T *raw = sm + S::O_RAW + j * TS + i;                   // this column in ring slot 0, v = 0
    T *wme = sm + S::O_W + (j + NG) * PW + (i + NG);             // this column in primitive plane 0, v = 0
    T *qx = sm + S::O_QX + j * PQ + i;                           // slot i: q+ of cell i-1, then flux at face i
    T *qy = sm + S::O_QY + j * PY + i;
    T Wc[NV], dzm[NV], qpz[NV], acc[NV];
    {
      T U0[NV], U1[NV], U2[NV], W0[NV], W1[NV];
      mk::mbar_wait(&bars[0], 0);
#pragma unroll
      for (int v = 0; v < NV; ++v) U0[v] = raw[v * (TS * TS)];
      mk::mbar_wait(&bars[1], 0);
#pragma unroll
      for (int v = 0; v < NV; ++v) U1[v] = raw[RAWP + v * (TS * TS)];
      mk::mbar_wait(&bars[2], 0);
#pragma unroll
      for (int v = 0; v < NV; ++v) U2[v] = raw[2 * RAWP + v * (TS * TS)];
      mk::prim<T, NV>(U0, W0, P, hits);
      mk::prim<T, NV>(U1, W1, P, hits);
      mk::prim<T, NV>(U2, Wc, P, hits);
#pragma unroll
      for (int v = 0; v < NV; ++v) {
        wme[v * WV] = Wc[v];                                        // plane 2 -> primitive buffer 0
        const T dm = W1[v] - W0[v];
        dzm[v] = Wc[v] - W1[v];
        const T s = mk::slope4(dm, dzm[v], Wc[v] - W0[v], th2);
        qpz[v] = fma(q4, s, W1[v]);                                 // q+ of the ghost cell below plane 2
        acc[v] = T(0);
      }
    }
    __syncthreads();

#pragma unroll 1
    for (int c = NG; c <= NG + NI; ++c) {            // current cell = padded plane c (2..17); c = 18: last z face only
      // 1. plane c+1: raw -> primitives, publish for the x/y neighbours
      T Wn[NV];
      {
        const int slot = (c + 1) % NSLOT;
        mk::mbar_wait(&bars[slot], unsigned((c + 1) / NSLOT) & 1u);
        T Un[NV];
#pragma unroll
        for (int v = 0; v < NV; ++v) Un[v] = raw[slot * RAWP + v * (TS * TS)];
        mk::prim<T, NV>(Un, Wn, P, hits);
      }
      if (c + 1 < NG + NI) {
        T *w = wme + ((c + 1) & 1) * (NV * WV);
#pragma unroll
        for (int v = 0; v < NV; ++v) w[v * WV] = Wn[v];
      }
      T ub[NV];
      if (BASE && c > NG) {
#pragma unroll
        for (int v = 0; v < NV; ++v) ub[v] = base[size_t(v) * VS + (c - 1) * PLANE];
      }
      // 2. z: slope of cell c, flux through the face between c-1 and c, finish cell c-1
      T Gz[NV];
      {
        T qm[NV], qp[NV];
#pragma unroll
        for (int v = 0; v < NV; ++v) {
          const T dp = Wn[v] - Wc[v];
          const T s = mk::slope4(dzm[v], dp, dzm[v] + dp, th2);
          qm[v] = fma(-q4, s, Wc[v]);
          qp[v] = fma(q4, s, Wc[v]);
          dzm[v] = dp;
        }
        mk::floor_states<T, NV>(qpz, qm, P, hits);
        mk::face_flux<T, 2>(qpz, qm, P, Gz);
#pragma unroll
        for (int v = 0; v < NV; ++v) qpz[v] = qp[v];
      }
      if (bflux && ((c - NG) & 7) == 0) {
        T *B = bflux + ((size_t(pl) * 9 + 6 + ((c - NG) >> 3)) * NV) * 256 + (y0 + j) * 16 + x0 + i;
#pragma unroll
        for (int v = 0; v < NV; ++v) B[v * 256] = T(0.5) * Gz[v];
      }
      if (c > NG) {
        const T *ui = raw + ((c - 1) % NSLOT) * RAWP;         // raw U of cell c-1 is still in the ring
        T *o = out + (c - 1) * PLANE;
#pragma unroll
        for (int v = 0; v < NV; ++v) {
          T pre = b * ui[v * (TS * TS)];
          if (BASE) pre = fma(a, ub[v], pre);
          o[size_t(v) * VS] = fma(-kk, acc[v] + Gz[v], pre);        // Eq. 7-8
        }
      }
      if (c < NG + NI) {
        // 3. x/y phase 1: slopes of this cell along x and y, publish q+
        const T *w = wme + (c & 1) * (NV * WV);
        T qmx[NV], qmy[NV];
#pragma unroll
        for (int v = 0; v < NV; ++v) {
          const T wl = w[v * WV - 1], wr = w[v * WV + 1], wd = w[v * WV - PW], wu = w[v * WV + PW];
          const T sx = mk::slope4(Wc[v] - wl, wr - Wc[v], wr - wl, th2);
          const T sy = mk::slope4(Wc[v] - wd, wu - Wc[v], wu - wd, th2);
          qmx[v] = fma(-q4, sx, Wc[v]);
          qmy[v] = fma(-q4, sy, Wc[v]);
          qx[v * QXV + 1] = fma(q4, sx, Wc[v]);
          qy[v * QYV + PY] = fma(q4, sy, Wc[v]);
        }
        __syncthreads();
        // 4. phase 2: fluxes through the low x and y faces of this cell (written over the q+ just read)
        T Gx[NV], Gy[NV];
        {
          T WL[NV], WD[NV];
#pragma unroll
          for (int v = 0; v < NV; ++v) { WL[v] = qx[v * QXV]; WD[v] = qy[v * QYV]; }
          mk::floor_states2<T, NV>(WL, qmx, WD, qmy, P, hits);
          mk::face_flux<T, 0>(WL, qmx, P, Gx);
          mk::face_flux<T, 1>(WD, qmy, P, Gy);
#pragma unroll
          for (int v = 0; v < NV; ++v) { qx[v * QXV] = Gx[v]; qy[v * QYV] = Gy[v]; }
        }
        if (bflux) {
          if (i == 0) {
            T *B = bflux + ((size_t(pl) * 9 + 0 + (x0 >> 3)) * NV) * 256 + (c - NG) * 16 + y0 + j;
#pragma unroll
            for (int v = 0; v < NV; ++v) B[v * 256] = T(0.5) * Gx[v];
          }
          if (j == 0) {
            T *B = bflux + ((size_t(pl) * 9 + 3 + (y0 >> 3)) * NV) * 256 + (c - NG) * 16 + x0 + i;
#pragma unroll
            for (int v = 0; v < NV; ++v) B[v * 256] = T(0.5) * Gy[v];
          }
        }
        __syncthreads();
        // 5. phase 3: flux differences in x and y; the low z face enters with its sign
#pragma unroll
        for (int v = 0; v < NV; ++v)
          acc[v] = ((qx[v * QXV + 1] - Gx[v]) + (qy[v * QYV + PY] - Gy[v])) - Gz[v];
      }
#pragma unroll
      for (int v = 0; v < NV; ++v) Wc[v] = Wn[v];
    }
  } else {
    qk::halo_warp<T, NV>(sm, pool, sin, p, desc[p], direct_halo, x0, y0, lane, P, th2, bflux, pl, hits, &tmap, bars);
  }
  if (hits) atomicAdd(floor_hits, (unsigned long long)hits);
}

// returns 0 or a cudaError_t; tmap8 = the pool's tensor map with 8x8 boxes
template <typename T, int NV>
int launch_rk_stage_quad(const CUtensorMap &tmap8, Pool<T> pool, int sin, int sbase, int sout, int first, int n, T a, T b,
                         T dtdx, Params<T> P, T *bflux, unsigned long long *floor_hits, const Desc *desc, int direct_halo,
                         cudaStream_t stream) {
  static bool configured = false;
  constexpr size_t bytes = qk::Smem<T, NV>::BYTES;
  if (!configured) {
    cudaError_t e = cudaFuncSetAttribute(k_rk_stage_quad<T, NV, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(bytes));
    if (e == cudaSuccess)
      e = cudaFuncSetAttribute(k_rk_stage_quad<T, NV, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(bytes));
    if (e != cudaSuccess) return int(e);
    configured = true;
  }
  if (a != T(0))
    k_rk_stage_quad<T, NV, true><<<4 * n, qk::THREADS, bytes, stream>>>(tmap8, pool, sin, sbase, sout, first, a, b, dtdx, P,
                                                                        bflux, floor_hits, desc, direct_halo);
  else
    k_rk_stage_quad<T, NV, false><<<4 * n, qk::THREADS, bytes, stream>>>(tmap8, pool, sin, sbase, sout, first, a, b, dtdx, P,
                                                                         bflux, floor_hits, desc, direct_halo);
  return 0;
}

}  // namespace amr
