// rk_stage_pair.cuh -- the hot kernel, second design: one method-of-lines stage of every 16^3 patch
// of a level (steps a3-a6: PAPER.md:79 Eq. 7, :94-98 Eq. 8, :104-112 Eq. 9-11, :114-118 Eq. 12).
//
// ncu on k_rk_stage_march (rk_stage_march.cuh) showed a latency-bound kernel: one 10-warp CTA per SM,
// 56 % of cycles with no eligible warp, 746 thread-instructions per cell of which 16 % in two halo
// warps and 11 % in shared-memory traffic (profiles/README.md, r1).  This kernel keeps what worked
// (z-march, TMA rings on mbarriers, every slope and face flux computed once, the arithmetic of
// mk::prim / mk::slope4 / mk::face_flux) and changes the decomposition:
//  * a thread owns TWO x-adjacent columns (2px, 2px+1) of row j: 128 threads (4 warps) per patch, two
//    CTAs per SM at up to 255 registers.  The two cells give every step two independent dependency
//    chains (ILP 2); the x face between them never leaves the registers; all own-cell and y-direction
//    shared-memory accesses are 16-byte (fp64) / 8-byte (fp32) vectors: about half the LDS/STS
//    instructions per cell; the update is stored with 16-byte stores.
//  * the x exchange (q+ of cell 2px+1 to the right neighbour, flux through face 2px to the left one) is a warp
//    shuffle inside the 8 lanes of a row; shared memory carries only the patch edge (q+ of the ghost cell -1,
//    q+ of cell 15 / flux through face 16) and the y exchange.
//  * no halo warps: each of the 128 threads also converts ONE of the 128 halo cells of a plane
//    (loaded one plane ahead straight from the sibling's interior or the own ghost zone); the ghost-cell
//    slopes (one warp pass per direction) and the fluxes through faces 16 (ONE warp pass for x and y, the
//    direction a run-time value of the lane) rotate over the four warps.
//  * CTA barriers are mbarrier arrive / wait halves with independent work between them (z slopes, z fluxes and
//    the update of the cell below after the first arrive; the conversion of plane c+2 after the second).
//  * the flux arrays alias the q+ arrays (a slot is read as q+ by its only reader before that same
//    thread overwrites it with its flux), U_base rides on a 2-slot TMA ring of its own: 87-107 kB of
//    shared memory per CTA (fp64 Euler), so that two CTAs fit an SM in both stages (fp32: three).
// Results are those of k_rk_stage_march up to the rounding of c = q_{i+1} - q_{i-1} (taken directly,
// as the oracle does, in x and y).  Measured alternatives (a warp-specialised split, other plane orders, one
// cell per thread with twice the warps) are in profiles/README.md; all were slower.
#pragma once
#include "rk_stage_march.cuh"

namespace amr {
namespace pk {

template <typename T> struct V2T;
template <> struct V2T<double> { using type = double2; };
template <> struct V2T<float> { using type = float2; };
template <typename T> __device__ __forceinline__ typename V2T<T>::type ld2(const T *p) {
  return *reinterpret_cast<const typename V2T<T>::type *>(p);
}
template <typename T> __device__ __forceinline__ void st2(T *p, T x, T y) {
  typename V2T<T>::type v;
  v.x = x; v.y = y;
  *reinterpret_cast<typename V2T<T>::type *>(p) = v;
}

constexpr int THREADS = 128;

// 64-bit shuffles inside the 8 lanes of one row (lane = (row & 3) * 8 + px)
__device__ __forceinline__ double shfl_up8(double x) { return __shfl_up_sync(0xffffffffu, x, 1, 8); }
__device__ __forceinline__ float shfl_up8(float x) { return __shfl_up_sync(0xffffffffu, x, 1, 8); }
__device__ __forceinline__ double shfl_down8(double x) { return __shfl_down_sync(0xffffffffu, x, 1, 8); }
__device__ __forceinline__ float shfl_down8(float x) { return __shfl_down_sync(0xffffffffu, x, 1, 8); }

template <typename T, int NV, bool WB> struct Smem {
  static constexpr int NSLOT = 4;                  // ring of raw conserved planes (TMA)
  static constexpr int BSLOT = 2;                  // ring of U_base planes (combination stage)
  static constexpr int RAWP = NV * NI * NI;        // one raw plane [NV][16][16], dense TMA box
  static constexpr int PW = NP;                    // primitive plane [20][20]: even pitch, pairs are 16-byte aligned
  static constexpr int WV = NP * PW;
  static constexpr int QXP = 1, QXV = 2 * NI;      // [2][16 rows]: column 0 = q+ of cell -1, column 1 = q+ of cell 15 / flux through face 16
  // fp32: a warp owns rows w, w+4, w+8, w+12 and the y array has pitch 20 (see the thread mapping in the kernel): measured
  // 5.55 -> 5.37 ms at 512^3; fp64 (16 bytes per lane, one row per wavefront anyway) keeps rows 4w..4w+3: 10.55 vs 10.84 ms
  static constexpr bool ROWS4 = sizeof(T) == 4;
  static constexpr int PY = ROWS4 ? NP : NI;       // pitch of the y exchange array
  static constexpr int QYV = (NI + 1) * PY;        // [17][PY]: slot j = q+ of row j-1 / flux through face j
  static constexpr int HQV = 16;                   // q- of the ghost cell 16 of every line (per direction)
  static constexpr int O_RAW = 0, O_W = O_RAW + NSLOT * RAWP, O_QX = O_W + 2 * NV * WV,
                       O_QY = ((O_QX + NV * QXV + 1) / 2) * 2, O_HQ = O_QY + NV * QYV,
                       O_BRAW = ((O_HQ + 2 * NV * HQV + 31) / 32) * 32;
  static constexpr int O_END = O_BRAW + (WB ? BSLOT * RAWP : 0);
  static constexpr size_t BAR_OFF = ((size_t(O_END) * sizeof(T) + 15) / 16) * 16;
  static constexpr size_t BYTES = BAR_OFF + (NSLOT + BSLOT + 2) * 8 + 128;   // + slack to align the ring to 128 B
};

// limited slope times 4 (fp64): mr = theta2 * m1 if |theta2 * m1| < |c| else c, m1 = the smaller of dm, dp in magnitude, and 0
// when dm and dp differ in sign: the value of mk::slope4 (the sign of m1 and of c is that of dm whenever the signs agree).
// The sign test is one LOP3 with a predicate result; q-+ = q0 -+ qs * mr with the constant qs = 1/4.
__device__ __forceinline__ double slope_mr(double dm, double dp, double c, double theta2, double &qs) {
  const double m1 = fabs(dm) < fabs(dp) ? dm : dp;
  const double t2 = theta2 * m1;
  double mr = fabs(t2) < fabs(c) ? t2 : c;
  int differ;
  asm("{\n .reg .pred p;\n .reg .b32 t;\n lop3.or.b32 t|p, %1, %2, 0x80000000, 0x28, 0;\n selp.b32 %0, 1, 0, p;\n}"
      : "=r"(differ) : "r"(__double2hiint(dm)), "r"(__double2hiint(dp)));
  if (differ) mr = 0.0;
  qs = 0.25;
  return mr;
}
__device__ __forceinline__ float slope_mr(float dm, float dp, float c, float theta2, float &qs) {
  qs = 0.25f;
  return mk::slope4(dm, dp, c, theta2);
}

// O1 for several cells with ONE rarely taken branch (S11): primitives without floors first, the floors of mk::prim only
// when a density or an internal energy is at or below its floor's high word.
template <typename T, int NV>
__device__ __forceinline__ void prim_nofloor(const T (&U)[NV], T (&W)[NV]) {
  const T rho = U[0];
  const T ir = mk::frcp(rho);
  const T vx = U[1] * ir, vy = U[2] * ir, vz = U[3] * ir;
  T et = U[4];
  if (NV >= 8) {
    et = fma(T(-0.5), fma(U[7 % NV], U[7 % NV], fma(U[6 % NV], U[6 % NV], U[5 % NV] * U[5 % NV])), et);
    W[5 % NV] = U[5 % NV]; W[6 % NV] = U[6 % NV]; W[7 % NV] = U[7 % NV];
  }
  if (NV == 9) W[8 % NV] = U[8 % NV];
  W[0] = rho; W[1] = fma(T(-0.5), fma(vz, vz, fma(vy, vy, vx * vx)), et * ir); W[2] = vx; W[3] = vy; W[4] = vz;
}
template <typename T, int NV>
__device__ __forceinline__ void prim3(const T (&Ua)[NV], const T (&Ub)[NV], const T (&Uc)[NV], bool with_c, T (&Wa)[NV],
                                      T (&Wb)[NV], T (&Wc)[NV], const Params<T> &P, int &hits) {
  using mk::hiw;
  prim_nofloor<T, NV>(Ua, Wa);
  prim_nofloor<T, NV>(Ub, Wb);
  int hr = min(hiw(Wa[0]), hiw(Wb[0])), he = min(hiw(Wa[1]), hiw(Wb[1]));
  if (with_c) {
    prim_nofloor<T, NV>(Uc, Wc);
    hr = min(hr, hiw(Wc[0])); he = min(he, hiw(Wc[1]));
  }
  if ((hr <= hiw(P.rho_floor)) | (he <= hiw(P.e_floor))) {
    mk::prim<T, NV>(Ua, Wa, P, hits);
    mk::prim<T, NV>(Ub, Wb, P, hits);
    if (with_c) mk::prim<T, NV>(Uc, Wc, P, hits);
  }
}

// S11 on reconstructed states: with the limiter of Eq. 9-11 and theta <= 2 a reconstructed density or internal energy
// lies between the values of the cell and of its neighbours (|slope/2| <= theta/2 min(|dm|, |dp|)), and those have
// been floored in the primitive recovery: the floors on l and r states cannot fire beyond one rounding of the floor
// itself, so this kernel does not test them (k_rk_stage_march and the oracle do, S11).

// ghost-cell slopes of one direction for one plane: lane = (line t, side).  Low side: q+ of cell -1 into
// slot 0 of the line; high side: q- of cell 16 into the stash (its flux follows after the barrier).
template <typename T, int NV, int D, typename S>
__device__ __forceinline__ void halo_slopes(T *sm, int buf, int lane, T th2) {
  constexpr int PW = S::PW, WV = S::WV;
  constexpr int rst = D == 0 ? 1 : PW;
  const int t = lane & 15, hi = lane >> 4;
  const T *s3 = sm + S::O_W + buf * (NV * WV) +
                (D == 0 ? (t + NG) * PW + (hi ? NG + NI - 1 : 0) : (hi ? NG + NI - 1 : 0) * PW + (t + NG));
  T *qlo = sm + (D == 0 ? S::O_QX + t * S::QXP : S::O_QY + t);      // (column 0 of the x edge array)
  T *hq = sm + S::O_HQ + D * (NV * S::HQV) + t;
  constexpr int qv = D == 0 ? S::QXV : S::QYV;
#pragma unroll
  for (int v = 0; v < NV; ++v) {
    const T w0 = s3[v * WV], w1 = s3[v * WV + rst], w2 = s3[v * WV + 2 * rst];
    T qs;
    const T mr = slope_mr(w1 - w0, w2 - w1, w2 - w0, th2, qs);
    if (hi) hq[v * S::HQV] = fma(-qs, mr, w1);
    else qlo[v * qv] = fma(qs, mr, w1);
  }
}
// both at once (Euler): lanes 0-15 the x faces, lanes 16-31 the y faces, with the direction a run-time value of the
// lane.  Same operations in the same order as mk::face_flux<T, 0> / <T, 1> (B * v is written fma(B, v, 0), which rounds
// identically), so a face shared by two patches still gets bitwise the same flux from both.
template <typename T>
__device__ __forceinline__ void face_flux_xy(const T (&L)[5], const T (&R)[5], const Params<T> &P, T (&G)[5], bool y) {
  const T rl = L[0], el = L[1], rr = R[0], er = R[1];
  const T vdl = y ? L[3] : L[2], vdr = y ? R[3] : R[2];
  const T pl = (P.gm1 * rl) * el, pr = (P.gm1 * rr) * er;
  const T q2l = fma(L[4], L[4], fma(L[3], L[3], L[2] * L[2]));
  const T q2r = fma(R[4], R[4], fma(R[3], R[3], R[2] * R[2]));
  const T hl = fma(T(0.5), q2l, el), hr = fma(T(0.5), q2r, er);
  const T sl = tabs(vdl) + mk::fsqrt(P.gg1 * el), sr = tabs(vdr) + mk::fsqrt(P.gg1 * er);
  const T lam = sl > sr ? sl : sr;
  const T A = rr * (vdr - lam), B = rl * (vdl + lam);
  const T pp = pl + pr;
  G[0] = A + B;
  G[1] = fma(A, R[2], fma(B, L[2], y ? T(0) : pp));
  G[2] = fma(A, R[3], fma(B, L[3], y ? pp : T(0)));
  G[3] = fma(A, R[4], B * L[4]);
  G[4] = fma(A, hr, fma(B, hl, fma(pr, vdr, pl * vdl)));
}
template <typename T, typename S>
__device__ __forceinline__ void halo_flux_xy(T *sm, int lane, const Params<T> &P, T *__restrict__ bflux, int pl, int zface,
                                             int bmask) {
  constexpr int NV = 5;
  const int t = lane & 15, d = lane >> 4;
  const int qv = d ? S::QYV : S::QXV;
  T *q16 = sm + (d ? S::O_QY + NI * S::PY + t : S::O_QX + (NI + t));
  const T *hq = sm + S::O_HQ + d * (NV * S::HQV) + t;
  T WL[NV], WR[NV], G[NV];
#pragma unroll
  for (int v = 0; v < NV; ++v) { WL[v] = q16[v * qv]; WR[v] = hq[v * S::HQV]; }
  face_flux_xy<T>(WL, WR, P, G, d != 0);
#pragma unroll
  for (int v = 0; v < NV; ++v) q16[v * qv] = G[v];
  if (bflux && ((bmask >> (3 * d + 2)) & 1)) {
    T *B = bflux + ((size_t(pl) * 9 + 3 * d + 2) * NV) * 256 + zface * 16 + t;
#pragma unroll
    for (int v = 0; v < NV; ++v) B[v * 256] = T(0.5) * G[v];
  }
}

}  // namespace pk

#ifndef AMR_PK_MINB
#define AMR_PK_MINB 2
#endif
#define AMR_PK_BOUNDS __launch_bounds__(pk::THREADS, (sizeof(T) == 4 ? AMR_PK_MINB + 1 : AMR_PK_MINB))   // fp32: three CTAs per SM (<= 168 registers)
template <typename T, int NV, bool BASE>
__global__ void AMR_PK_BOUNDS
k_rk_stage_pair(const __grid_constant__ CUtensorMap tmap, Pool<T> pool, int sin, int sbase, int sout, int first, T a, T b,
                T dtdx, Params<T> P, T *__restrict__ bflux, unsigned long long *__restrict__ floor_hits,
                const Desc *__restrict__ desc, int direct_halo, unsigned long long *__restrict__ smax_out, int zsplit, DtDev dtd,
                const int *__restrict__ bneed) {
  using S = pk::Smem<T, NV, BASE>;
  if (dtd.p) dtdx = T((*dtd.p * dtd.pow2) / dtd.hx);
  constexpr int PW = S::PW, WV = S::WV, QXV = S::QXV, QYV = S::QYV, RAWP = S::RAWP, NSLOT = S::NSLOT;
  constexpr int PX = Layout<T>::PX, PLANE = Layout<T>::PLANE, VS = Layout<T>::VS, LEAD = Layout<T>::LEAD;
  extern __shared__ unsigned char smem_raw[];
  T *sm = reinterpret_cast<T *>(smem_raw + ((128u - (mk::smem_u32(smem_raw) & 127u)) & 127u));   // TMA destination: 128-byte aligned
  unsigned long long *bars = reinterpret_cast<unsigned long long *>(reinterpret_cast<unsigned char *>(sm) + S::BAR_OFF);
  unsigned long long *bbars = bars + NSLOT;                   // U_base ring
  unsigned long long *xbar = bbars + S::BSLOT;                // [0]: q+ published (B1), [1]: fluxes published (B2)

  // zsplit = 1 (levels too small to fill the machine): two CTAs per patch, each marching over 8 of the 16 cells in z
  const int pl = blockIdx.x >> zsplit, p = first + pl;
  const int zlo = int(blockIdx.x & zsplit) * (NI / 2), nz = zsplit ? NI / 2 : NI;
  const int tid = threadIdx.x, lane = tid & 31;
  const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);     // (through a shuffle: the compiler then knows it is warp-uniform)
  // thread -> (row j, pair px).  8 lanes are one row.  fp32: the two rows of a half-warp are 4 apart, so that their 64-byte
  // segments of the primitive plane (pitch 20) and of the y array (pitch 20) fall into disjoint banks: 80 B x 4 = 320 B = 64 mod 128
  // (with adjacent rows every 8-byte vector access of a half-warp was a 2-way bank conflict)
  const int j = S::ROWS4 ? ((lane >> 3) << 2) + warp : tid >> 3, px = tid & 7, i0 = 2 * px;
  const T kk = T(0.5) * b * dtdx;        // the 1/2 of Eq. 12 is applied here (G = 2F)
  const T th2 = T(2) * P.theta;
  int hits = 0;
  // which of the nine boundary-flux planes of this patch a flux register will read (bit 3 d + s; all when no table)
  const int bmask = bflux ? (bneed ? bneed[p] : 0x1ff) : 0;

  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < NSLOT + S::BSLOT; ++s) mk::mbar_init(&bars[s], 1);
    mk::mbar_init(&xbar[0], pk::THREADS / 32);
    mk::mbar_init(&xbar[1], pk::THREADS / 32);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  const Desc &D = desc[p];
  // ---- this thread's halo cell: threads 0-63 the x-ghosts (row, cell -2,-1,16,17), 64-127 the y-ghosts (column, row ...)
  const T *hsrc;
  T *hdst;
  {
    int hrow, hcol, face;
    if (tid < 64) { const int q = tid & 3; hrow = (tid >> 2) + NG; hcol = q < 2 ? q : NI + q; face = q < 2 ? 0 : 1; }
    else { const int u = tid - 64, q = u >> 4; hcol = (u & 15) + NG; hrow = q < 2 ? q : NI + q; face = q < 2 ? 2 : 3; }
    hdst = sm + S::O_W + hrow * PW + hcol;
    const int nb = direct_halo ? D.nbr[face_region(face)] : -1;
    if (nb >= 0) {                        // the sibling's interior instead of the own ghost zone
      const int sh = (face & 1) ? -NI : NI;
      if (face < 2) hcol += sh; else hrow += sh;
    }
    hsrc = pool.patch(sin, nb >= 0 ? nb : p) + LEAD + hrow * PX + hcol;
  }
  // ---- TMA producer state (thread 0)
  int q_mid = 0, q_lo = 0, q_hi = 0, kz_lo = 0, kz_hi = 0, q_base = 0;
  if (tid == 0) {
    const int nzl = direct_halo ? D.nbr[face_region(4)] : -1, nzh = direct_halo ? D.nbr[face_region(5)] : -1;
    const int qb = sin * pool.max_patches;
    q_mid = (qb + p) * NV; q_lo = (qb + (nzl >= 0 ? nzl : p)) * NV; q_hi = (qb + (nzh >= 0 ? nzh : p)) * NV;
    kz_lo = nzl >= 0 ? NI : 0; kz_hi = nzh >= 0 ? -NI : 0;
    q_base = (sbase * pool.max_patches + p) * NV;
  }
  auto issue = [&](int pk_) {                                 // raw conserved interior box of padded plane pk_ of this march
    const int slot = pk_ % NSLOT, ap = pk_ + zlo;
    const int q = ap < NG ? q_lo : (ap >= NG + NI ? q_hi : q_mid);
    const int k = ap < NG ? ap + kz_lo : (ap >= NG + NI ? ap + kz_hi : ap);
    mk::mbar_expect_tx(&bars[slot], unsigned(RAWP * sizeof(T)));
    mk::tma_load_4d(sm + S::O_RAW + slot * RAWP, &tmap, 0, NG, k, q, &bars[slot]);
  };
  auto issue_base = [&](int c_) {                             // U_base of cell plane c_ (Eq. 8)
    const int slot = c_ & 1;
    mk::mbar_expect_tx(&bbars[slot], unsigned(RAWP * sizeof(T)));
    mk::tma_load_4d(sm + S::O_BRAW + slot * RAWP, &tmap, 0, NG, c_ + zlo, q_base, &bbars[slot]);
  };
  __syncthreads();
  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < NSLOT; ++s) issue(s);
    if (BASE) issue_base(NG);
  }

  const int off = LEAD + (j + NG) * PX + (i0 + NG);          // in-plane offset of this pair of columns (16-byte aligned)
  T *out = pool.patch(sout, p) + off;
  const T *raw = sm + S::O_RAW + j * NI + i0;                 // this pair in ring slot 0, v = 0
  T *wme = sm + S::O_W + (j + NG) * PW + (i0 + NG);           // this pair in primitive buffer 0, v = 0
  T *qx = sm + S::O_QX + j + (px == 7 ? NI : 0);              // px = 0: q+ of cell -1 of this row; px = 7: q+ of cell 15 / flux through face 16
  T *qy = sm + S::O_QY + j * S::PY + i0;                      // slot j: q+ of row j-1 / flux through face j

  T Uh[NV];                                                   // halo cell of the next plane to convert
  auto halo_load = [&](int pk_) {
#pragma unroll
    for (int v = 0; v < NV; ++v) Uh[v] = hsrc[size_t(v) * VS + (pk_ + zlo) * PLANE];
  };
  // raw plane pk_ -> primitives of this pair in primitive buffer pk_ & 1; with_halo: also this thread's halo cell (Uh)
  auto convert = [&](int pk_, bool with_halo, T (&W0)[NV], T (&W1)[NV]) {
    const int slot = pk_ % NSLOT;
    mk::mbar_wait(&bars[slot], unsigned(pk_ / NSLOT) & 1u);
    T U0[NV], U1[NV];
#pragma unroll
    for (int v = 0; v < NV; ++v) { const auto x = pk::ld2(raw + slot * RAWP + v * (NI * NI)); U0[v] = x.x; U1[v] = x.y; }
    T Wh[NV];
    pk::prim3<T, NV>(U0, U1, Uh, with_halo, W0, W1, Wh, P, hits);
    T *w = wme + (pk_ & 1) * (NV * WV);
#pragma unroll
    for (int v = 0; v < NV; ++v) pk::st2(w + v * WV, W0[v], W1[v]);
    if (with_halo) {
      T *d = hdst + (pk_ & 1) * (NV * WV);
#pragma unroll
      for (int v = 0; v < NV; ++v) d[v * WV] = Wh[v];
    }
  };
  // CTA barrier in two halves on an mbarrier: arrive (one lane per warp, after the warp's writes) ... wait
  auto arrive = [&](int which) {
    __syncwarp();
    if (lane == 0) asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(mk::smem_u32(&xbar[which])) : "memory");
  };

  T dzm[2][NV], qpz[2][NV], acc[2][NV];
  T best = T(0);                      // fused CFL reduction (a1) over the cells this thread finishes
  bool bad = false;
  halo_load(NG);
  {
    // planes 0, 1: only the z stencil of this pair needs them; planes 2 and 3 are published
    T W0[2][NV], W1[2][NV], W2[2][NV], W3[2][NV];
    {
      T U0[2][NV], U1[2][NV];
      mk::mbar_wait(&bars[0], 0);
#pragma unroll
      for (int v = 0; v < NV; ++v) { const auto x = pk::ld2(raw + v * (NI * NI)); U0[0][v] = x.x; U0[1][v] = x.y; }
      mk::mbar_wait(&bars[1], 0);
#pragma unroll
      for (int v = 0; v < NV; ++v) { const auto x = pk::ld2(raw + RAWP + v * (NI * NI)); U1[0][v] = x.x; U1[1][v] = x.y; }
#pragma unroll
      for (int s = 0; s < 2; ++s) { mk::prim<T, NV>(U0[s], W0[s], P, hits); mk::prim<T, NV>(U1[s], W1[s], P, hits); }
    }
    convert(NG, true, W2[0], W2[1]);
    if (nz > 1) halo_load(NG + 1);
    convert(NG + 1, nz > 1, W3[0], W3[1]);
    if (nz > 2) halo_load(NG + 2);
#pragma unroll
    for (int s = 0; s < 2; ++s)
#pragma unroll
      for (int v = 0; v < NV; ++v) {
        const T dm = W1[s][v] - W0[s][v];
        dzm[s][v] = W2[s][v] - W1[s][v];
        T qs;
        const T mr = pk::slope_mr(dm, dzm[s][v], dm + dzm[s][v], th2, qs);
        qpz[s][v] = fma(qs, mr, W1[s][v]);                       // q+ of the ghost cell below plane 2
        acc[s][v] = T(0);
      }
  }
  __syncthreads();
  if (tid == 0) issue(NSLOT);                                 // slot of plane 0: converted, never needed again

#pragma unroll 1
  for (int c = NG; c <= NG + nz; ++c) {            // current cell = plane c of this march (2..nz+1); c = nz+2: last z face only
    const bool live = c < NG + nz;                 // plane c is a cell of this march
    const unsigned par = unsigned(c - NG) & 1u;    // phase of the two exchange barriers
    const T *w = wme + (c & 1) * (NV * WV);
    T Wc[2][NV];
#pragma unroll
    for (int v = 0; v < NV; ++v) { const auto x = pk::ld2(w + v * WV); Wc[0][v] = x.x; Wc[1][v] = x.y; }
    T qmx0[NV], qpx0[NV], qmx1[NV], qmy0[NV], qmy1[NV];
    T WLs[NV];                                     // q+ of cell i0-1 from the left neighbour's registers (px > 0)
    if (live) {
      // 1. slopes of both cells along x and y; publish the q+ the neighbours need
#pragma unroll
      for (int v = 0; v < NV; ++v) {
        const T a0 = Wc[0][v], a1 = Wc[1][v];
        const T wl = w[v * WV - 1], wr = w[v * WV + 2];
        const auto wd = pk::ld2(w + v * WV - PW), wu = pk::ld2(w + v * WV + PW);
        const T d0 = a0 - wl, d1 = a1 - a0, d2 = wr - a1;
        T qs, mr;
        mr = pk::slope_mr(d0, d1, a1 - wl, th2, qs);
        qmx0[v] = fma(-qs, mr, a0); qpx0[v] = fma(qs, mr, a0);
        mr = pk::slope_mr(d1, d2, wr - a0, th2, qs);
        qmx1[v] = fma(-qs, mr, a1);
        const T qpx1 = fma(qs, mr, a1);
        WLs[v] = pk::shfl_up8(qpx1);
        if (px == 7) qx[v * QXV] = qpx1;           // for the flux through face 16 (halo_flux)
        mr = pk::slope_mr(a0 - wd.x, wu.x - a0, wu.x - wd.x, th2, qs);
        qmy0[v] = fma(-qs, mr, a0);
        const T qpy0 = fma(qs, mr, a0);
        mr = pk::slope_mr(a1 - wd.y, wu.y - a1, wu.y - wd.y, th2, qs);
        qmy1[v] = fma(-qs, mr, a1);
        pk::st2(qy + v * QYV + S::PY, qpy0, fma(qs, mr, a1));
      }
      if (warp == (c & 3)) pk::halo_slopes<T, NV, 0, S>(sm, c & 1, lane, th2);
      if (warp == ((c + 1) & 3)) pk::halo_slopes<T, NV, 1, S>(sm, c & 1, lane, th2);
      arrive(0);
    }
    // 2. z (between the two halves of the barrier): slope of cell c from this pair's own planes c-1 (dzm), c, c+1;
    //    flux through the face between c-1 and c; finish cell c-1
    {
      T Gz[2][NV], qm[2][NV];
      {
        const T *wn = wme + ((c + 1) & 1) * (NV * WV);
#pragma unroll
        for (int v = 0; v < NV; ++v) {
          const auto x = pk::ld2(wn + v * WV);
          const T dp0 = x.x - Wc[0][v], dp1 = x.y - Wc[1][v];
          T qs, mr;
          mr = pk::slope_mr(dzm[0][v], dp0, dzm[0][v] + dp0, th2, qs);
          qm[0][v] = fma(-qs, mr, Wc[0][v]);
          Gz[0][v] = fma(qs, mr, Wc[0][v]);                        // q+ of cell c, parked until qpz has been used
          mr = pk::slope_mr(dzm[1][v], dp1, dzm[1][v] + dp1, th2, qs);
          qm[1][v] = fma(-qs, mr, Wc[1][v]);
          Gz[1][v] = fma(qs, mr, Wc[1][v]);
          dzm[0][v] = dp0; dzm[1][v] = dp1;
        }
      }
      {
        T L0[NV], L1[NV];
#pragma unroll
        for (int v = 0; v < NV; ++v) { L0[v] = qpz[0][v]; L1[v] = qpz[1][v]; qpz[0][v] = Gz[0][v]; qpz[1][v] = Gz[1][v]; }
        mk::face_flux<T, 2>(L0, qm[0], P, Gz[0]);
        mk::face_flux<T, 2>(L1, qm[1], P, Gz[1]);
      }
      if (((c - NG + zlo) & 7) == 0 && ((bmask >> (6 + ((c - NG + zlo) >> 3))) & 1)) {
        T *B = bflux + ((size_t(pl) * 9 + 6 + ((c - NG + zlo) >> 3)) * NV) * 256 + j * 16 + i0;
#pragma unroll
        for (int v = 0; v < NV; ++v) pk::st2(B + v * 256, T(0.5) * Gz[0][v], T(0.5) * Gz[1][v]);
      }
      if (c > NG) {
        const T *ui = raw + ((c - 1) % NSLOT) * RAWP;        // raw U of cell c-1 is still in the ring
        const T *ub = raw + (S::O_BRAW - S::O_RAW) + ((c - 1) & 1) * RAWP;
        if (BASE) mk::mbar_wait(&bbars[(c - 1) & 1], unsigned((c - 1 - NG) >> 1) & 1u);
        T *o = out + (c - 1 + zlo) * PLANE;
        T un[2][NV];
#pragma unroll
        for (int v = 0; v < NV; ++v) {
          const auto x = pk::ld2(ui + v * (NI * NI));
          T pre0 = b * x.x, pre1 = b * x.y;
          if (BASE) {
            const auto y = pk::ld2(ub + v * (NI * NI));
            pre0 = fma(a, y.x, pre0); pre1 = fma(a, y.y, pre1);
          }
          un[0][v] = fma(-kk, acc[0][v] + Gz[0][v], pre0);          // Eq. 7-8
          un[1][v] = fma(-kk, acc[1][v] + Gz[1][v], pre1);
          pk::st2(o + size_t(v) * VS, un[0][v], un[1][v]);
        }
        if (BASE && smax_out) {
          // S4 on the state just produced: max_d |v_d| + c_d, with the NaN/inf test of k_cfl
#pragma unroll
          for (int s = 0; s < 2; ++s) {
            T Wq[NV];
            mk::prim<T, NV>(un[s], Wq, P, hits);
            const T sp = mk::max_speed_fast<T, NV>(Wq, P);
            const T chk = (((Wq[2] + Wq[3]) + Wq[4]) + sp) + (un[s][0] + un[s][4]);   // (the floors would hide a NaN density or energy)
            bad |= !(chk - chk == T(0));
            best = tmax(best, sp);
          }
        }
      }
#pragma unroll
      for (int v = 0; v < NV; ++v) { acc[0][v] = Gz[0][v]; acc[1][v] = Gz[1][v]; }     // the low z face (subtracted in step 5)
    }
    if (!live) break;
    mk::mbar_wait(&xbar[0], par);
    // 3. fluxes through the low x and y faces of both cells
    T Gx0[NV], Gx1[NV], Gy0[NV], Gy1[NV];
    {
      T WL[NV], WD0[NV], WD1[NV];
#pragma unroll
      for (int v = 0; v < NV; ++v) {
        WL[v] = WLs[v];
        if (px == 0) WL[v] = qx[v * QXV];          // q+ of the ghost cell -1 (halo_slopes)
        const auto y = pk::ld2(qy + v * QYV);
        WD0[v] = y.x; WD1[v] = y.y;
      }
      mk::face_flux<T, 0>(WL, qmx0, P, Gx0);
      mk::face_flux<T, 0>(qpx0, qmx1, P, Gx1);
      mk::face_flux<T, 1>(WD0, qmy0, P, Gy0);
      mk::face_flux<T, 1>(WD1, qmy1, P, Gy1);
#pragma unroll
      for (int v = 0; v < NV; ++v) {
        pk::st2(qy + v * QYV, Gy0[v], Gy1[v]);
      }
    }
    if (warp == ((c + 2) & 3)) pk::halo_flux_xy<T, S>(sm, lane, P, bflux, pl, c - NG + zlo, bmask);
    arrive(1);
    if (bmask) {
      if ((i0 & 7) == 0 && ((bmask >> (i0 >> 3)) & 1)) {
        T *B = bflux + ((size_t(pl) * 9 + 0 + (i0 >> 3)) * NV) * 256 + (c - NG + zlo) * 16 + j;
#pragma unroll
        for (int v = 0; v < NV; ++v) B[v * 256] = T(0.5) * Gx0[v];
      }
      if ((j & 7) == 0 && ((bmask >> (3 + (j >> 3))) & 1)) {
        T *B = bflux + ((size_t(pl) * 9 + 3 + (j >> 3)) * NV) * 256 + (c - NG + zlo) * 16 + i0;
#pragma unroll
        for (int v = 0; v < NV; ++v) pk::st2(B + v * 256, T(0.5) * Gy0[v], T(0.5) * Gy1[v]);
      }
    }
    // 4. (between the two halves of the second barrier) plane c+2: raw -> primitives, published for iteration c+2;
    //    every thread has passed the first barrier, so nobody reads plane c in that buffer any more
    if (c + 2 < nz + 2 * NG) {
      T Wa[NV], Wb[NV];
      const bool hl = c + 2 < NG + nz;
      convert(c + 2, hl, Wa, Wb);
      if (c + 3 < NG + nz) halo_load(c + 3);
    }
    mk::mbar_wait(&xbar[1], par);
    if (tid == 0) {                                // every thread is past step 2: these ring slots are free
      if (c + NSLOT - 1 < nz + 2 * NG) issue(c + NSLOT - 1);            // slot of plane c-1
      if (BASE && c + 1 < NG + nz) issue_base(c + 1);                   // slot of cell c-1
    }
    // 5. flux differences in x and y, minus the low z face parked in acc
#pragma unroll
    for (int v = 0; v < NV; ++v) {
      T fxh = pk::shfl_down8(Gx0[v]);               // flux through face i0+2 = the right neighbour's low face
      if (px == 7) fxh = qx[v * QXV];               // face 16 (halo_flux)
      const auto fyh = pk::ld2(qy + v * QYV + S::PY);
      acc[0][v] = ((Gx1[v] - Gx0[v]) + (fyh.x - Gy0[v])) - acc[0][v];
      acc[1][v] = ((fxh - Gx1[v]) + (fyh.y - Gy1[v])) - acc[1][v];
    }
  }
  if (BASE && smax_out) {
    // one atomicMax per warp on the bit pattern of a non-negative double (monotone as an unsigned integer)
    double bq = bad ? __longlong_as_double(0x7ff0000000000000LL) : double(best);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) bq = fmax(bq, __shfl_xor_sync(0xffffffffu, bq, o));
    if (lane == 0) atomicMax(smax_out, (unsigned long long)__double_as_longlong(bq));
  }
  if (hits) atomicAdd(floor_hits, (unsigned long long)hits);
}

// returns 0 or a cudaError_t
template <typename T, int NV>
int launch_rk_stage_pair(const CUtensorMap &tmap, Pool<T> pool, int sin, int sbase, int sout, int first, int n, T a, T b,
                         T dtdx, Params<T> P, T *bflux, unsigned long long *floor_hits, const Desc *desc, int direct_halo,
                         cudaStream_t stream, unsigned long long *smax_out = nullptr, int zmode = 0, int num_sms = 0, DtDev dtd = DtDev{nullptr, 0, 0},
                         const int *bneed = nullptr) {
  static bool configured = false;
  constexpr size_t bytes0 = pk::Smem<T, NV, false>::BYTES, bytes1 = pk::Smem<T, NV, true>::BYTES;
  if (!configured) {
    cudaError_t e = cudaFuncSetAttribute(k_rk_stage_pair<T, NV, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(bytes0));
    if (e == cudaSuccess)
      e = cudaFuncSetAttribute(k_rk_stage_pair<T, NV, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(bytes1));
    if (e != cudaSuccess) return int(e);
    configured = true;
  }
  // zmode 0: never split; 1: every patch; 2: every patch of a level of at most num_sms / 2 patches.  (The march kernel also
  // splits the thin last wave of a launch; here the block decode that takes costs the fp64 instantiation its last free
  // registers: 16-32 bytes of spills, 10.6 -> 12.8 ms at 512^3.)
  const int zsplit = (zmode == 1 || (zmode == 2 && 2 * n <= num_sms)) ? 1 : 0;
  if (a != T(0))
    k_rk_stage_pair<T, NV, true><<<n << zsplit, pk::THREADS, bytes1, stream>>>(tmap, pool, sin, sbase, sout, first, a, b, dtdx, P,
                                                                              bflux, floor_hits, desc, direct_halo, smax_out, zsplit, dtd, bneed);
  else
    k_rk_stage_pair<T, NV, false><<<n << zsplit, pk::THREADS, bytes0, stream>>>(tmap, pool, sin, sbase, sout, first, a, b, dtdx, P,
                                                                               bflux, floor_hits, desc, direct_halo, nullptr, zsplit, dtd, bneed);
  return 0;
}

}  // namespace amr
