// rk_stage_lite.cuh -- register-light variant of k_rk_stage_march for two CTAs per SM.
// (Steps a3-a6: PAPER.md:79 Eq. 7, :94-98 Eq. 8, :104-112 Eq. 9-11, :114-118 Eq. 12.)
//
// ncu on k_rk_stage_march (profiles/README.md, r1b): fp64 needs ~155 registers per thread, so one
// 10-warp CTA per SM, 2.5 warps per scheduler, issue slots 44 % busy, FP64 pipe 41 % busy: the
// stage is latency bound.  Forcing 96 registers spills to local memory, and with 2 x 108 kB of
// shared memory per SM the L1 is too small to hold the spills.  This variant keeps the same
// decomposition (one CTA per patch, z-marching, TMA ring, halo warps: see rk_stage_march.cuh)
// but moves the per-column state that lives across the x/y phases out of registers by hand:
//   * the running sum of flux differences and the z-face state q+ sit in per-thread slots of
//     shared memory (conflict-free: slot = thread index);
//   * the primitive state of the current cell is re-read from the published plane;
//   * the flux arrays alias the q+ arrays (every slot has one reader, which reads the q+ before
//     it overwrites the slot with its flux), and the ring has 3 slots: 105 kB per CTA (fp64).
#pragma once
#include "rk_stage_march.cuh"

namespace amr {

template <typename T, int NV, bool BASE>
__global__ void __launch_bounds__(mk::THREADS, 2)
k_rk_stage_lite(const __grid_constant__ CUtensorMap tmap, Pool<T> pool, int sin, int sbase, int sout, int first, T a, T b,
                T dtdx, Params<T> P, T *__restrict__ bflux, unsigned long long *__restrict__ floor_hits,
                const Desc *__restrict__ desc, int direct_halo) {
  using S = mk::Smem<T, NV, true>;
  constexpr int PW = S::PW, PQ = S::PQ, PY = S::PY, WV = S::WV, QXV = S::QXV, QYV = S::QYV, RAWP = S::RAWP, ACV = S::ACV;
  constexpr int PX = Layout<T>::PX, PLANE = Layout<T>::PLANE, VS = Layout<T>::VS, LEAD = Layout<T>::LEAD;
  extern __shared__ unsigned char smem_raw[];
  // the TMA destination must be 128-byte aligned
  T *sm = reinterpret_cast<T *>(smem_raw + ((128u - (mk::smem_u32(smem_raw) & 127u)) & 127u));
  unsigned long long *bars = reinterpret_cast<unsigned long long *>(reinterpret_cast<unsigned char *>(sm) + S::BAR_OFF);

  const int pl = blockIdx.x, p = first + pl;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const T th2 = T(2) * P.theta, q4 = T(0.25);
  int hits = 0;

  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < S::NSLOT; ++s) mk::mbar_init(&bars[s], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  if (warp < 8) {
    // ------------------------------------------------------------------ interior columns
    const T kk = T(0.5) * b * dtdx;        // the 1/2 of Eq. 12 is applied here (G = 2F)
    const int i = lane & 15, j = warp + 8 * (lane >> 4);
    const int off = LEAD + (j + NG) * PX + (i + NG);            // in-plane offset of this column
    const T *base = pool.patch(sbase, p) + off;
    T *out = pool.patch(sout, p) + off;
    const T *raw = sm + S::O_RAW + j * NI + i;                   // this column in ring slot 0, v = 0
    T *wme = sm + S::O_W + (j + NG) * PW + (i + NG);             // this column in primitive plane 0, v = 0
    T *qx = sm + S::O_QX + j * PQ + i;                           // slot i: q+ of cell i-1, then flux at face i
    T *qy = sm + S::O_QY + j * PY + i;
    T *accs = sm + S::O_ACC + tid, *qpzs = sm + S::O_QPZ + tid;  // per-thread slots
    T dzm[NV];
    {
      T U0[NV], U1[NV], U2[NV], W0[NV], W1[NV], W2[NV];
      mk::mbar_wait(&bars[0], 0);
#pragma unroll
      for (int v = 0; v < NV; ++v) U0[v] = raw[v * (NI * NI)];
      mk::mbar_wait(&bars[1], 0);
#pragma unroll
      for (int v = 0; v < NV; ++v) U1[v] = raw[RAWP + v * (NI * NI)];
      mk::mbar_wait(&bars[2], 0);
#pragma unroll
      for (int v = 0; v < NV; ++v) U2[v] = raw[2 * RAWP + v * (NI * NI)];
      mk::prim<T, NV>(U0, W0, P, hits);
      mk::prim<T, NV>(U1, W1, P, hits);
      mk::prim<T, NV>(U2, W2, P, hits);
#pragma unroll
      for (int v = 0; v < NV; ++v) {
        wme[v * WV] = W2[v];                                        // plane 2 -> primitive buffer 0
        const T dm = W1[v] - W0[v];
        dzm[v] = W2[v] - W1[v];
        const T s = mk::slope4(dm, dzm[v], W2[v] - W0[v], th2);
        qpzs[v * ACV] = fma(q4, s, W1[v]);                          // q+ of the ghost cell below plane 2
        accs[v * ACV] = T(0);
      }
    }
    __syncthreads();

#pragma unroll 1
    for (int c = NG; c <= NG + NI; ++c) {            // current cell = padded plane c (2..17); c = 18: last z face only
      const T *wc = wme + (c & 1) * (NV * WV);       // primitives of this cell (published one iteration ago)
      {
        // 1. plane c+1: raw -> primitives, publish for the x/y neighbours (plane 18 too: it is
        //    this column's own W(18) at c = 18)
        T Wn[NV];
        {
          const int slot = (c + 1) % S::NSLOT;
          mk::mbar_wait(&bars[slot], unsigned((c + 1) / S::NSLOT) & 1u);
          T Un[NV];
#pragma unroll
          for (int v = 0; v < NV; ++v) Un[v] = raw[slot * RAWP + v * (NI * NI)];
          mk::prim<T, NV>(Un, Wn, P, hits);
        }
        if (c + 1 <= NG + NI) {
          T *w = wme + ((c + 1) & 1) * (NV * WV);
#pragma unroll
          for (int v = 0; v < NV; ++v) w[v * WV] = Wn[v];
        }
        // 2. z: slope of cell c, flux through the face between c-1 and c, finish cell c-1
        T Gz[NV];
        {
          T qm[NV], ql[NV];
#pragma unroll
          for (int v = 0; v < NV; ++v) {
            const T w0 = wc[v * WV];
            const T dp = Wn[v] - w0;
            const T s = mk::slope4(dzm[v], dp, dzm[v] + dp, th2);
            qm[v] = fma(-q4, s, w0);
            ql[v] = qpzs[v * ACV];
            qpzs[v * ACV] = fma(q4, s, w0);
            dzm[v] = dp;
          }
          mk::floor_states<T, NV>(ql, qm, P, hits);
          mk::face_flux<T, 2>(ql, qm, P, Gz);
        }
        if (bflux && ((c - NG) & 7) == 0) {
          T *B = bflux + ((size_t(pl) * 9 + 6 + ((c - NG) >> 3)) * NV) * 256 + j * 16 + i;
#pragma unroll
          for (int v = 0; v < NV; ++v) B[v * 256] = T(0.5) * Gz[v];
        }
        if (c > NG) {
          const T *ui = raw + ((c - 1) % S::NSLOT) * RAWP;     // raw U of cell c-1 is still in the ring
          T *o = out + (c - 1) * PLANE;
#pragma unroll
          for (int v = 0; v < NV; ++v) {
            T pre = b * ui[v * (NI * NI)];
            if (BASE) pre = fma(a, base[size_t(v) * VS + (c - 1) * PLANE], pre);
            o[size_t(v) * VS] = fma(-kk, accs[v * ACV] + Gz[v], pre);   // Eq. 7-8
          }
        }
#pragma unroll
        for (int v = 0; v < NV; ++v) accs[v * ACV] = -Gz[v];     // the low z face enters cell c with its sign
      }
      if (c < NG + NI) {
        // 3. x/y phase 1: slopes of this cell along x and y, publish q+
        T qmx[NV], qmy[NV];
#pragma unroll
        for (int v = 0; v < NV; ++v) {
          const T w0 = wc[v * WV], wl = wc[v * WV - 1], wr = wc[v * WV + 1], wd = wc[v * WV - PW], wu = wc[v * WV + PW];
          const T sx = mk::slope4(w0 - wl, wr - w0, wr - wl, th2);
          const T sy = mk::slope4(w0 - wd, wu - w0, wu - wd, th2);
          qmx[v] = fma(-q4, sx, w0);
          qmy[v] = fma(-q4, sy, w0);
          qx[v * QXV + 1] = fma(q4, sx, w0);
          qy[v * QYV + PY] = fma(q4, sy, w0);
        }
        __syncthreads();
        // 4. phase 2: fluxes through the low x and y faces of this cell (written over the q+ just read)
        T Gx[NV], Gy[NV];
        {
          T WL[NV];
#pragma unroll
          for (int v = 0; v < NV; ++v) WL[v] = qx[v * QXV];
          mk::floor_states<T, NV>(WL, qmx, P, hits);
          mk::face_flux<T, 0>(WL, qmx, P, Gx);
#pragma unroll
          for (int v = 0; v < NV; ++v) qx[v * QXV] = Gx[v];
        }
        {
          T WD[NV];
#pragma unroll
          for (int v = 0; v < NV; ++v) WD[v] = qy[v * QYV];
          mk::floor_states<T, NV>(WD, qmy, P, hits);
          mk::face_flux<T, 1>(WD, qmy, P, Gy);
#pragma unroll
          for (int v = 0; v < NV; ++v) qy[v * QYV] = Gy[v];
        }
        if (bflux) {
          if ((i & 7) == 0) {
            T *B = bflux + ((size_t(pl) * 9 + 0 + (i >> 3)) * NV) * 256 + (c - NG) * 16 + j;
#pragma unroll
            for (int v = 0; v < NV; ++v) B[v * 256] = T(0.5) * Gx[v];
          }
          if ((j & 7) == 0) {
            T *B = bflux + ((size_t(pl) * 9 + 3 + (j >> 3)) * NV) * 256 + (c - NG) * 16 + i;
#pragma unroll
            for (int v = 0; v < NV; ++v) B[v * 256] = T(0.5) * Gy[v];
          }
        }
        __syncthreads();
        // 5. phase 3: flux differences in x and y join the low z face in the per-thread slot
#pragma unroll
        for (int v = 0; v < NV; ++v)
          accs[v * ACV] += (qx[v * QXV + 1] - Gx[v]) + (qy[v * QYV + PY] - Gy[v]);
      }
    }
  } else {
    // ------------------------------------------------------------------ halo warps (+ TMA producer)
    const Desc &D = desc[p];
    const T *self = pool.patch(sin, p);
    const int f0 = warp == 8 ? 0 : 2;
    const T *g[2];
#pragma unroll
    for (int s = 0; s < 2; ++s) {
      const int nb = direct_halo ? D.nbr[face_region(f0 + s)] : -1;
      const int st = warp == 8 ? 1 : PX;
      g[s] = nb >= 0 ? pool.patch(sin, nb) + (s ? -NI * st : NI * st) : self;
    }
    const int nzl = direct_halo ? D.nbr[face_region(4)] : -1, nzh = direct_halo ? D.nbr[face_region(5)] : -1;
    const int qbase = sin * pool.max_patches;
    const int q_mid = (qbase + p) * NV, q_lo = (qbase + (nzl >= 0 ? nzl : p)) * NV, q_hi = (qbase + (nzh >= 0 ? nzh : p)) * NV;
    const int kz_lo = nzl >= 0 ? NI : 0, kz_hi = nzh >= 0 ? -NI : 0;
    if (warp == 8)
      mk::halo_warp<T, NV, 0, S>(sm, g[0], g[1], lane, P, th2, bflux, pl, hits, lane == 0, &tmap, bars, q_mid, q_lo, q_hi, kz_lo, kz_hi);
    else
      mk::halo_warp<T, NV, 1, S>(sm, g[0], g[1], lane, P, th2, bflux, pl, hits, false, &tmap, bars, q_mid, q_lo, q_hi, kz_lo, kz_hi);
  }
  if (hits) atomicAdd(floor_hits, (unsigned long long)hits);
}

// returns 0 or a cudaError_t
template <typename T, int NV>
int launch_rk_stage_lite(const CUtensorMap &tmap, Pool<T> pool, int sin, int sbase, int sout, int first, int n, T a, T b,
                         T dtdx, Params<T> P, T *bflux, unsigned long long *floor_hits, const Desc *desc, int direct_halo,
                         cudaStream_t stream) {
  static bool configured = false;
  constexpr size_t bytes = mk::Smem<T, NV, true>::BYTES;
  if (!configured) {
    cudaError_t e = cudaFuncSetAttribute(k_rk_stage_lite<T, NV, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(bytes));
    if (e == cudaSuccess)
      e = cudaFuncSetAttribute(k_rk_stage_lite<T, NV, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(bytes));
    if (e != cudaSuccess) return int(e);
    configured = true;
  }
  if (a != T(0))
    k_rk_stage_lite<T, NV, true><<<n, mk::THREADS, bytes, stream>>>(tmap, pool, sin, sbase, sout, first, a, b, dtdx, P, bflux,
                                                                    floor_hits, desc, direct_halo);
  else
    k_rk_stage_lite<T, NV, false><<<n, mk::THREADS, bytes, stream>>>(tmap, pool, sin, sbase, sout, first, a, b, dtdx, P, bflux,
                                                                     floor_hits, desc, direct_halo);
  return 0;
}

}  // namespace amr
