// rk_stage_march.cuh -- the hot kernel: one method-of-lines stage of every 16^3 patch of a level
// (steps a3-a6: PAPER.md:79 Eq. 7, :94-98 Eq. 8, :104-112 Eq. 9-11, :114-118 Eq. 12).
//
// B200 design (the paper's 1-D flattened sweeps with one global round trip per kernel,
// PAPER.md:139-153 / :226-248, are prior art, not the blueprint).  ncu on the first versions of
// this kernel showed the stage is bound by instruction issue, the FP64 pipe and the shared-memory
// crossbar, not by HBM (profiles/README.md), so everything here is written for instruction count
// and for keeping global-memory latency off the critical path:
//  * one CTA per patch, 10 warps: 8 "interior" warps own the 16x16 (i,j) columns and march in z
//    over the 20 padded planes; warp 8 owns the x-halo columns, warp 9 the y-halo rows.
//    Fluxes, L(U) and primitives never touch HBM.
//  * the 16x16xNV interior box of every plane is brought in by TMA (cp.async.bulk.tensor, one
//    request per plane, 4-slot ring, mbarrier completion), issued three planes ahead by one
//    elected thread: no load instructions, address arithmetic or prefetch registers in the
//    interior warps, and the raw U of the cell being finished is still in the ring for the
//    Runge-Kutta combination.  z-ghost planes come through the same ring (from this patch's ghost
//    zones, or with AMRHYDRO_OPT_HALO=1 from the z-neighbour's interior).  In the combination
//    stage (a != 0) the planes of U_base ride on the same mbarriers into a second ring (fp64 and
//    fp32 Euler, fp64 8-variable MHD with the flux arrays aliased onto the q+ arrays): measured
//    -14 % on that stage against 5 global loads per cell in the warps.  Shared-memory layout and
//    launch bounds are per stage (fp32: 3 CTAs/SM at 64 registers without the ring, 2 at 96 with it).
//  * optional extras, all bitwise-neutral for the state: the CFL reduction of the next step fused
//    into the combination stage (smax_out); a z-split for levels too small to fill the machine
//    (two CTAs per patch, half a column each, about half the latency of a launch).
//  * each cell is converted to primitives once (one MUFU reciprocal + a third-order correction)
//    and published in a double-buffered shared-memory plane for the x/y neighbours; the z stencil
//    lives in registers; x/y exchange the cell-edge state q+ and the face fluxes through shared
//    memory (two barriers per plane): each slope and each face flux is computed once.
//  * the 1/2 of Eq. 12 and of the PLM half-slope are folded into constants (exact power-of-two
//    scalings): the kernel carries G = 2F and sm = 4*(half slope).  Limiter without explicit
//    |x| (the FP64 pipe would pay a DADD for each): compares and multiplies take |x| as an
//    operand modifier, the sign is restored on the integer pipe.  Floors are tested on the high
//    words (integer pipe) and applied in a rarely taken branch.
#pragma once
#include <cuda.h>

#include "layout.cuh"
#include "physics.cuh"

namespace amr {
namespace mk {

// ---- fast reciprocal / square root (MUFU seed + one third-order step: error ~ seed^3)
__device__ __forceinline__ double frcp(double x) {
  double y;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));   // >= 20 good bits
  double e = fma(-x, y, 1.0);
  e = fma(e, e, e);
  return fma(y, e, y);
}
__device__ __forceinline__ float frcp(float x) {
  float y;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
// sqrt of a strictly positive, finite x
__device__ __forceinline__ double fsqrt(double x) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  const double g = x * y;
  const double r = fma(-g, y, 1.0);              // 1 - x y^2
  return fma(g * r, fma(0.375, r, 0.5), g);      // g (1-r)^(-1/2) = g (1 + r/2 + 3/8 r^2 + O(r^3)): five FP64 operations
}
__device__ __forceinline__ float fsqrt(float x) {
  float y;
  asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
// x < fl for fl > 0 by integer order of the bit patterns (negative x and -0 compare below;
// a positive NaN does not -- NaNs are reported by cfl_dt, not repaired here)
__device__ __forceinline__ bool below(double x, double fl) { return __double_as_longlong(x) < __double_as_longlong(fl); }
__device__ __forceinline__ bool below(float x, float fl) { return __float_as_int(x) < __float_as_int(fl); }
__device__ __forceinline__ int hiw(double x) { return __double2hiint(x); }
__device__ __forceinline__ int hiw(float x) { return __float_as_int(x); }
// cheap necessary condition for "a or b is below fl": one integer min + one compare
template <typename T> __device__ __forceinline__ bool maybe_below(T a, T b, T fl) { return min(hiw(a), hiw(b)) <= hiw(fl); }

// sm = 4 * (1/2) minmod(theta dm, theta dp, c/2), c = qp - qm   (Eq. 9-11 with G1):
// q-(cell) = q0 - sm/4, q+(cell) = q0 + sm/4.  theta2 = 2 theta.  Exactly the oracle's value when
// c = qp - qm: min commutes with the monotone rounding of theta*x, all scalings are powers of two.
template <typename T> __device__ __forceinline__ T slope4(T dm, T dp, T c, T theta2) {
  const T m1 = tabs(dm) < tabs(dp) ? dm : dp;
  const T t2 = theta2 * tabs(m1);
  const T mr = t2 < tabs(c) ? t2 : c;
  return same_sign(dm, dp) ? with_sign_of(mr, dm) : T(0);
}

// O1: conserved -> primitive W = (rho, e, vx, vy, vz, [Bx, By, Bz]);  PAPER.md:59, :298; floors S11
template <typename T, int NV>
__device__ __forceinline__ void prim(const T (&U)[NV], T (&W)[NV], const Params<T> &P, int &hits) {
  T rho = U[0];
  if (hiw(rho) <= hiw(P.rho_floor)) {
    if (below(rho, P.rho_floor)) { rho = P.rho_floor; ++hits; }
  }
  const T ir = frcp(rho);
  const T vx = U[1] * ir, vy = U[2] * ir, vz = U[3] * ir;
  T et = U[4];
  if (NV >= 8) {
    et = fma(T(-0.5), fma(U[7 % NV], U[7 % NV], fma(U[6 % NV], U[6 % NV], U[5 % NV] * U[5 % NV])), et);
    W[5 % NV] = U[5 % NV]; W[6 % NV] = U[6 % NV]; W[7 % NV] = U[7 % NV];
  }
  if (NV == 9) W[8 % NV] = U[8 % NV];                               // psi (Eq. 14)
  T e = fma(T(-0.5), fma(vz, vz, fma(vy, vy, vx * vx)), et * ir);
  if (hiw(e) <= hiw(P.e_floor)) {
    if (below(e, P.e_floor)) { e = P.e_floor; ++hits; }
  }
  W[0] = rho; W[1] = e; W[2] = vx; W[3] = vy; W[4] = vz;
}

template <typename T, int NV>
__device__ __forceinline__ void floor_states2(T (&L)[NV], T (&R)[NV], T (&L2)[NV], T (&R2)[NV], const Params<T> &P, int &hits) {
  const int hr = min(min(hiw(L[0]), hiw(R[0])), min(hiw(L2[0]), hiw(R2[0])));
  const int he = min(min(hiw(L[1]), hiw(R[1])), min(hiw(L2[1]), hiw(R2[1])));
  if ((hr <= hiw(P.rho_floor)) | (he <= hiw(P.e_floor))) {
    if (below(L[0], P.rho_floor)) { L[0] = P.rho_floor; ++hits; }
    if (below(L[1], P.e_floor)) { L[1] = P.e_floor; ++hits; }
    if (below(R[0], P.rho_floor)) { R[0] = P.rho_floor; ++hits; }
    if (below(R[1], P.e_floor)) { R[1] = P.e_floor; ++hits; }
    if (below(L2[0], P.rho_floor)) { L2[0] = P.rho_floor; ++hits; }
    if (below(L2[1], P.e_floor)) { L2[1] = P.e_floor; ++hits; }
    if (below(R2[0], P.rho_floor)) { R2[0] = P.rho_floor; ++hits; }
    if (below(R2[1], P.e_floor)) { R2[1] = P.e_floor; ++hits; }
  }
}
template <typename T, int NV>
__device__ __forceinline__ void floor_states(T (&L)[NV], T (&R)[NV], const Params<T> &P, int &hits) {
  if (maybe_below(L[0], R[0], P.rho_floor) | maybe_below(L[1], R[1], P.e_floor)) {
    if (below(L[0], P.rho_floor)) { L[0] = P.rho_floor; ++hits; }
    if (below(L[1], P.e_floor)) { L[1] = P.e_floor; ++hits; }
    if (below(R[0], P.rho_floor)) { R[0] = P.rho_floor; ++hits; }
    if (below(R[1], P.e_floor)) { R[1] = P.e_floor; ++hits; }
  }
}

// O3, Eq. 12 doubled: G = F(L) + F(R) - lambda0 (U(R) - U(L)),
// lambda0 = max(|v_l| + c_l, |v_r| + c_r)  (= the max of Eq. 12 for single-valued c >= 0).
// Grouped by state instead of by term (45 instead of 57 FP64 instructions): with
//   A = rho_r (v_dr - lambda0),  B = rho_l (v_dl + lambda0),  h = v^2/2 + e
// Eq. 3-5 and Eq. 12 give  G_rho = A + B,  G_m = A v_r + B v_l (+ p_l + p_r along d),
// G_E = A h_r + B h_l + p_r v_dr + p_l v_dl.  No cancellation is introduced: |v_d -+ lambda0| >= c.
template <typename T, int D>
__device__ __forceinline__ void face_flux(const T (&L)[5], const T (&R)[5], const Params<T> &P, T (&G)[5]) {
  const T rl = L[0], el = L[1], rr = R[0], er = R[1];
  const T vdl = L[2 + D], vdr = R[2 + D];
  const T pl = (P.gm1 * rl) * el, pr = (P.gm1 * rr) * er;                         // Eq. 6
  const T q2l = fma(L[4], L[4], fma(L[3], L[3], L[2] * L[2]));
  const T q2r = fma(R[4], R[4], fma(R[3], R[3], R[2] * R[2]));
  const T hl = fma(T(0.5), q2l, el), hr = fma(T(0.5), q2r, er);
  const T sl = tabs(vdl) + fsqrt(P.gg1 * el), sr = tabs(vdr) + fsqrt(P.gg1 * er);   // S2
  const T lam = sl > sr ? sl : sr;
  const T A = rr * (vdr - lam), B = rl * (vdl + lam);
  G[0] = A + B;
#pragma unroll
  for (int t = 0; t < 3; ++t) {
    const T x = t == D ? fma(B, vdl, pl + pr) : B * L[2 + t];
    G[1 + t] = fma(A, R[2 + t], x);
  }
  G[4] = fma(A, hr, fma(B, hl, fma(pr, vdr, pl * vdl)));
}

// MHD, Eq. 15 with G3: NV = 8 ideal (psi == 0, S3'), NV = 9 GLM (F^d(B_d) = psi, F^d(psi) = c_h^2 B_d);
// fast magnetosonic speed along D (S3).  Per state: total pressure pt = p + B^2/2, total energy density
// E = rho (v^2/2 + e) + B^2/2, B.v and the signal speed; the doubled flux of Eq. 12 is then grouped by
// state as in the Euler version (A' = v_dr - lambda0, B' = v_dl + lambda0, A = rho_r A', B = rho_l B'):
//   G_rho = A + B;  G_m,i = A v_ir + B v_il - B_ir B_dr - B_il B_dl (+ pt_l + pt_r for i = d);
//   G_E = E_r A' + E_l B' + pt_r v_dr + pt_l v_dl - B_dr (B.v)_r - B_dl (B.v)_l;
//   G_B,i = A' B_ir + B' B_il - B_dr v_ir - B_dl v_il (i != d);  G_B,d = [psi_l + psi_r] - lambda0 (B_dr - B_dl);
//   G_psi = c_h^2 (B_dl + B_dr) - lambda0 (psi_r - psi_l)
template <typename T, int D, int NV>
__device__ __forceinline__ void mhd_scalars(const T (&W)[NV], const Params<T> &P, T &pt, T &E, T &Bv, T &speed) {
  static_assert(NV == 8 || NV == 9, "MHD variable sets");
  const T rho = W[0], e = W[1], vd = W[2 + D], Bd = W[5 + D];
  const T re = rho * e;
  const T q2 = fma(W[4], W[4], fma(W[3], W[3], W[2] * W[2]));
  const T B2 = fma(W[7], W[7], fma(W[6], W[6], W[5] * W[5]));
  Bv = fma(W[7], W[4], fma(W[6], W[3], W[5] * W[2]));
  const T hB2 = T(0.5) * B2;
  pt = fma(P.gm1, re, hB2);                                           // Eq. 6 + B^2/2
  E = fma(T(0.5) * rho, q2, re) + hB2;
  const T ir = frcp(rho);
  const T a2 = P.gg1 * e, s = fma(B2, ir, a2), bd2 = Bd * Bd * ir;
  const T disc = fma(s, s, T(-4) * a2 * bd2);
  // disc >= 0 analytically; rounding can leave it tiny or negative when a^2 = b^2 = b_d^2
  const T sq = disc > T(1e-30) * s * s ? fsqrt(disc) : T(0);
  speed = tabs(vd) + fsqrt(T(0.5) * (s + sq));
}
template <typename T, int D, int NV>
__device__ __forceinline__ void face_flux(const T (&L)[NV], const T (&R)[NV], const Params<T> &P, T (&G)[NV]) {
  T ptl, El, Bvl, sl, ptr, Er, Bvr, sr;
  mhd_scalars<T, D, NV>(L, P, ptl, El, Bvl, sl);
  mhd_scalars<T, D, NV>(R, P, ptr, Er, Bvr, sr);
  T lam = sl > sr ? sl : sr;
  if (NV == 9) lam = lam > P.ch ? lam : P.ch;                         // S17
  const T vdl = L[2 + D], vdr = R[2 + D], Bdl = L[5 + D], Bdr = R[5 + D];
  const T Ap = vdr - lam, Bp = vdl + lam;
  const T A = R[0] * Ap, B = L[0] * Bp;
  G[0] = A + B;
#pragma unroll
  for (int t = 0; t < 3; ++t) {
    T x = fma(-L[5 + t], Bdl, B * L[2 + t]);
    if (t == D) x += ptl + ptr;
    G[1 + t] = fma(A, R[2 + t], fma(-R[5 + t], Bdr, x));
    G[5 + t] = t == D ? -(lam * (Bdr - Bdl))
                      : fma(Ap, R[5 + t], fma(Bp, L[5 + t], fma(-Bdr, R[2 + t], -(Bdl * L[2 + t]))));
  }
  G[4] = fma(Er, Ap, fma(El, Bp, fma(ptr, vdr, fma(ptl, vdl, fma(-Bdr, Bvr, -(Bdl * Bvl))))));
  if (NV == 9) {
    G[5 + D] += L[8 % NV] + R[8 % NV];
    G[8 % NV] = fma(P.ch * P.ch, Bdl + Bdr, -(lam * (R[8 % NV] - L[8 % NV])));
  }
}

// fp32: the same value from the 3-input min/max of sm_100 (FMNMX3): with x = 2 theta dm, y = 2 theta dp,
// lo = min(x, y, c) <= hi = max(x, y, c), the minmod is the median of (0, lo, hi) = max(lo, min(0, hi))
// -- 6 instructions instead of 9, none of them a select.  (fp64 has no native min/max: it keeps
// the compare/select form above.)
__device__ __forceinline__ float slope4(float dm, float dp, float c, float theta2) {
  const float x = theta2 * dm, y = theta2 * dp;
  const float lo = fminf(fminf(x, y), c), hi = fmaxf(fmaxf(x, y), c);
  return fmaxf(lo, fminf(0.f, hi));
}

// S4 for the fused CFL reduction: max_d |v_d| + c_d.  Euler: the MUFU-seeded square root of this file
// (error ~1e-19 relative) instead of the IEEE one; MHD: the stand-alone formula of physics.cuh.
template <typename T, int NV> __device__ __forceinline__ T max_speed_fast(const T (&W)[NV], const Params<T> &P) {
  if (NV == 5) {
    const T ax = tabs(W[2]), ay = tabs(W[3]), az = tabs(W[4]);
    const T m1 = ax > ay ? ax : ay;
    return (m1 > az ? m1 : az) + fsqrt(P.gg1 * W[1]);
  } else {
    // S3 along the three directions with the MUFU-seeded reciprocal and square root of this file (the stand-alone
    // k_cfl keeps the IEEE forms of physics.cuh: six IEEE square roots and a division per cell are ~170 instructions)
    const T a2 = P.gg1 * W[1], ir = frcp(W[0]);
    const T B2 = fma(W[7 % NV], W[7 % NV], fma(W[6 % NV], W[6 % NV], W[5 % NV] * W[5 % NV]));
    const T s = fma(B2, ir, a2), s2 = s * s, a4 = T(4) * a2 * ir;
    T best = T(0);
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      const T Bd = W[(5 + d) % NV];
      const T disc = fma(-a4 * Bd, Bd, s2);
      const T sq = disc > T(1e-30) * s2 ? fsqrt(disc) : T(0);
      const T sp = tabs(W[2 + d]) + fsqrt(T(0.5) * (s + sq));
      best = sp > best ? sp : best;
    }
    if (NV == 9) best = best > P.ch ? best : P.ch;                // S17
    return best;
  }
}

// ---- TMA / mbarrier (PTX ISA: cp.async.bulk.tensor, mbarrier)
__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long *bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long *bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long *bar, unsigned parity) {
  unsigned ok;
  do {
    asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
                 : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
  } while (!ok);
}
__device__ __forceinline__ void tma_load_4d(void *dst, const CUtensorMap *tm, int x, int y, int z, int q,
                                            unsigned long long *bar) {
  asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];"
               ::"r"(smem_u32(dst)), "l"(tm), "r"(x), "r"(y), "r"(z), "r"(q), "r"(smem_u32(bar)) : "memory");
}

template <typename T> struct Cfg;
// shared-memory pitches: conflict-free for the row accesses of the interior warps (rows j, j+8
// per warp) and for the column accesses of the x-halo warp
#ifndef AMR_NSLOT64
#define AMR_NSLOT64 4
#endif
#ifndef AMR_NSLOT32
#define AMR_NSLOT32 4
#endif
// NSLOT: TMA ring depth (raw conserved planes), >= 3: planes c-1 (update), c, c+1 (conversion) are live
template <> struct Cfg<double> { static constexpr int PW = 21, PQ = 17, PY = 16, NSLOT = AMR_NSLOT64; };
template <> struct Cfg<float> { static constexpr int PW = 26, PQ = 18, PY = 18, NSLOT = AMR_NSLOT32; };

#ifndef AMR_BASE_TMA
#define AMR_BASE_TMA 1      // combination stage: U_base planes come through their own TMA ring (no global loads in the warps)
#endif
template <typename T, int NV, bool WB = true> struct Smem {   // WB: the kernel reads U_base (combination stage)
  static constexpr int PW = Cfg<T>::PW, PQ = Cfg<T>::PQ, PY = Cfg<T>::PY;
  // (the fp64 GLM-9 combination stage takes a ring of three, the minimum, so that its U_base ring fits beside it)
  // (and the MHD-8 one: 256^3 3.13 -> 3.05 ms per step with 33 kB less shared memory, i.e. more L1 for its 16-24 bytes of spills)
  static constexpr int NSLOT = (WB && AMR_BASE_TMA && sizeof(T) == 8 && NV >= 8) ? 3 : Cfg<T>::NSLOT;
  static constexpr int RAWP = NV * NI * NI;        // one raw plane: [NV][16][16], dense TMA box
  static constexpr int WV = NP * PW;               // one variable of one primitive plane [20][PW]
  static constexpr int QXV = NI * PQ;              // [16][PQ]: slot s = q+ of cell s-1 / flux at face s
  static constexpr int QYV = (NI + 1) * PY;        // [17][PY]
  // the flux arrays alias the q+ arrays (slot s is read as q+ by its only reader before that same thread overwrites it
  // with the flux) in the fp64 MHD combination stage, so that its U_base ring fits
  static constexpr bool ALIAS = WB && AMR_BASE_TMA && sizeof(T) == 8 && NV >= 8;
  static constexpr int O_RAW = 0, O_W = O_RAW + NSLOT * RAWP, O_QX = O_W + 2 * NV * WV,
                       O_FX = ALIAS ? O_QX : O_QX + NV * QXV, O_QY = O_FX + NV * QXV,
                       O_FY = ALIAS ? O_QY : O_QY + NV * QYV, O_ACC = O_FY + NV * QYV;
  // ring of U_base planes for the combination stage (128-byte aligned TMA destination).  fp32 Euler: the extra
  // 20 kB cost the third CTA per SM, so that instantiation also takes 96 registers instead of 64 (launch bounds)
  static constexpr int O_BRAW = ((O_ACC + 31) / 32) * 32;
  static constexpr bool BTMA = WB && AMR_BASE_TMA && (sizeof(T) == 8 || NV == 5) &&
                               size_t(O_BRAW + NSLOT * RAWP) * sizeof(T) + 256 <= 232448;   // 227 kB per CTA (Euler fits, fp64 GLM-9 does not)
  // fp64 GLM-9: q+ of the cell below (the z state carried from pass to pass) is parked here over the x/y phases, where the
  // nine variables do not fit into the 168 registers of a 10-warp CTA ([NV][256], one slot per interior thread)
#ifndef AMR_MK_PARK
#define AMR_MK_PARK 1
#endif
  static constexpr bool PARK = AMR_MK_PARK && sizeof(T) == 8 && NV == 9;   // (MHD-8, which does not spill in stage 1: 3.05 -> 3.37 ms with it)
  static constexpr int O_PARK = O_BRAW + (BTMA ? NSLOT * RAWP : 0);
  static constexpr int O_END = O_PARK + (PARK ? NV * NI * NI : 0);
  static constexpr size_t BAR_OFF = ((size_t(O_END) * sizeof(T) + 15) / 16) * 16;
  static constexpr size_t BYTES = BAR_OFF + NSLOT * 8 + 128;   // + slack to align the ring to 128 B
};

#ifndef AMR_MINB64
#define AMR_MINB64 1
#endif
#ifndef AMR_MINB32
#define AMR_MINB32 3
#endif
constexpr int THREADS = 320;

// One halo warp.  D = 0: lane = (row j, side): cells (-2,-1) or (16,17) of that row; D = 1: lane =
// (column i, side): rows (-2,-1) or (16,17).  Converts its two cells of every interior plane,
// publishes them next to the interior cells, computes the slope of the ghost cell adjacent to the
// patch (q+ of cell -1 on the low side, q- of cell 16 on the high side) and, on the high side,
// the flux through face 16.
template <typename T, int NV, int D, typename S = Smem<T, NV>>
__device__ __forceinline__ void halo_warp(T *sm, const T *glo, const T *ghi, int lane, const Params<T> &P, T th2,
                                          T *__restrict__ bflux, int pl, int &hits, bool producer,
                                          const CUtensorMap *tmap, unsigned long long *bars, int q_mid, int q_lo,
                                          int q_hi, int kz_lo, int kz_hi, int q_base = -1, int zlo = 0, int nz = NI) {
  // zlo, nz: the CTA marches over the nz cells starting at cell zlo of the column (z-split of small levels); plane
  // indices below are relative to that start, zlo converts them to planes of the patch
  constexpr int PW = S::PW, PQ = S::PQ, PY = S::PY, WV = S::WV;
  constexpr int PX = Layout<T>::PX, PLANE = Layout<T>::PLANE, VS = Layout<T>::VS, LEAD = Layout<T>::LEAD;
  constexpr int gst = D == 0 ? 1 : PX, rst = D == 0 ? 1 : PW;
  constexpr int qv = D == 0 ? S::QXV : S::QYV;
  const int t = lane & 15, hi = lane >> 4;
  const T q4 = T(0.25);
  // first of the two ghost cells (global, ring) and first of the three cells of the slope stencil
  const T *g = (hi ? ghi : glo) + LEAD + (D == 0 ? (t + NG) * PX + (hi ? NG + NI : 0) : (hi ? NG + NI : 0) * PX + (t + NG));
  T *W = sm + S::O_W;
  T *r = W + (D == 0 ? (t + NG) * PW + (hi ? NG + NI : 0) : (hi ? NG + NI : 0) * PW + (t + NG));
  const T *st3 = r + (hi ? -rst : 0);                       // cells (15,16,17) or (-2,-1,0)
  T *Q = sm + (D == 0 ? S::O_QX : S::O_QY), *F = sm + (D == 0 ? S::O_FX : S::O_FY);
  T *qlo = Q + (D == 0 ? t * PQ : t);                        // slot 0: q+ of cell -1
  const T *qhi = Q + (D == 0 ? t * PQ + NI : NI * PY + t);   // slot 16: q+ of cell 15
  T *fhi = F + (D == 0 ? t * PQ + NI : NI * PY + t);         // flux at face 16
  T Ua[NV], Ub[NV];
  auto load = [&](int pk) {
#pragma unroll
    for (int v = 0; v < NV; ++v) {
      const T *s = g + size_t(v) * VS + (pk + zlo) * PLANE;
      if (D == 0) {
        if (sizeof(T) == 8) { const double2 x = *reinterpret_cast<const double2 *>(s); Ua[v] = T(x.x); Ub[v] = T(x.y); }
        else                { const float2 x = *reinterpret_cast<const float2 *>(s);   Ua[v] = T(x.x); Ub[v] = T(x.y); }
      } else {
        Ua[v] = s[0]; Ub[v] = s[gst];
      }
    }
  };
  auto publish = [&](int pk) {
    T W0[NV], W1[NV];
    prim<T, NV>(Ua, W0, P, hits);
    prim<T, NV>(Ub, W1, P, hits);
    T *d = r + (pk & 1) * (NV * WV);
#pragma unroll
    for (int v = 0; v < NV; ++v) { d[v * WV] = W0[v]; d[v * WV + rst] = W1[v]; }
  };
  auto issue = [&](int pk) {                                  // TMA: interior box of padded plane pk
    const int slot = pk % S::NSLOT;
    const int ap = pk + zlo;
    const int q = ap < NG ? q_lo : (ap >= NG + NI ? q_hi : q_mid);
    const int k = ap < NG ? ap + kz_lo : (ap >= NG + NI ? ap + kz_hi : ap);
    // U_base of cell pk-2 rides on the same barrier: it is needed when plane pk has been converted (Eq. 8)
    const bool wb = q_base >= 0 && pk >= NG + 2;
    mbar_expect_tx(&bars[slot], unsigned(S::RAWP * sizeof(T)) * (wb ? 2u : 1u));
    tma_load_4d(sm + S::O_RAW + slot * S::RAWP, tmap, 0, NG, k, q, &bars[slot]);
    if (wb) tma_load_4d(sm + S::O_BRAW + slot * S::RAWP, tmap, 0, NG, ap - 2, q_base, &bars[slot]);
  };
  if (producer) {
#pragma unroll
    for (int s = 0; s < S::NSLOT; ++s) issue(s);
  }
  load(NG);
  publish(NG);
  load(NG + 1);
  __syncthreads();                                            // planes 0-2 converted by the interior warps
  if (producer) issue(S::NSLOT);                              // slot of plane 0: converted, never needed again
#pragma unroll 1
  for (int c = NG; c < NG + nz; ++c) {
    if (c + 1 < NG + nz) {
      publish(c + 1);
      if (c + 2 < NG + nz) load(c + 2);
    }
    const T *s3 = st3 + (c & 1) * (NV * WV);
    T qm[NV];
#pragma unroll
    for (int v = 0; v < NV; ++v) {
      const T w0 = s3[v * WV], w1 = s3[v * WV + rst], w2 = s3[v * WV + 2 * rst];
      const T s = slope4(w1 - w0, w2 - w1, w2 - w0, th2);
      qm[v] = fma(-q4, s, w1);                                // q- of cell 16 (high side)
      if (!hi) qlo[v * qv] = fma(q4, s, w1);                  // q+ of cell -1 (low side)
    }
    __syncthreads();
    if (producer && c + S::NSLOT - 1 < nz + 2 * NG) issue(c + S::NSLOT - 1);   // slot of plane c-1 is free: cell c-1 is finished
    if (hi) {
      T WL[NV], G[NV];
#pragma unroll
      for (int v = 0; v < NV; ++v) WL[v] = qhi[v * qv];
      floor_states<T, NV>(WL, qm, P, hits);
      face_flux<T, D>(WL, qm, P, G);
#pragma unroll
      for (int v = 0; v < NV; ++v) fhi[v * qv] = G[v];
      if (bflux) {
        T *B = bflux + ((size_t(pl) * 9 + 3 * D + 2) * NV) * 256 + (c - NG + zlo) * 16 + t;
#pragma unroll
        for (int v = 0; v < NV; ++v) B[v * 256] = T(0.5) * G[v];
      }
    }
    __syncthreads();
  }
}

}  // namespace mk

template <typename T, int NV, bool BASE>
__global__ void __launch_bounds__(mk::THREADS, (sizeof(T) == 8 ? (NV == 5 ? AMR_MINB64 : 1) : (NV == 5 ? (BASE && AMR_BASE_TMA ? 2 : AMR_MINB32) : 2)))
k_rk_stage_march(const __grid_constant__ CUtensorMap tmap, Pool<T> pool, int sin, int sbase, int sout, int first, T a, T b,
                 T dtdx, Params<T> P, T *__restrict__ bflux, unsigned long long *__restrict__ floor_hits,
                 const Desc *__restrict__ desc, int direct_halo, unsigned long long *__restrict__ smax_out, int nfull, DtDev dtd) {
  using S = mk::Smem<T, NV, BASE>;
  if (dtd.p) dtdx = T((*dtd.p * dtd.pow2) / dtd.hx);
  constexpr int PW = S::PW, PQ = S::PQ, PY = S::PY, WV = S::WV, QXV = S::QXV, QYV = S::QYV, RAWP = S::RAWP;
  constexpr int PX = Layout<T>::PX, PLANE = Layout<T>::PLANE, VS = Layout<T>::VS, LEAD = Layout<T>::LEAD;
  extern __shared__ unsigned char smem_raw[];
  // the TMA destination must be 128-byte aligned
  T *sm = reinterpret_cast<T *>(smem_raw + ((128u - (mk::smem_u32(smem_raw) & 127u)) & 127u));
  unsigned long long *bars = reinterpret_cast<unsigned long long *>(reinterpret_cast<unsigned char *>(sm) + S::BAR_OFF);

  // z-split: blocks 0 .. nfull-1 march over a whole patch; the blocks behind them come in pairs, two CTAs per patch, each
  // marching over 8 of the 16 cells in z (all patches of a level too small to fill the machine: nfull = 0; or the last,
  // less than half full wave of a launch, which then takes 0.6 instead of 1 wave time).  Bitwise the unsplit march.
  const bool zhalf = int(blockIdx.x) >= nfull;
  const int pl = zhalf ? nfull + ((int(blockIdx.x) - nfull) >> 1) : int(blockIdx.x), p = first + pl;
  const int zlo = zhalf ? ((int(blockIdx.x) - nfull) & 1) * (NI / 2) : 0, nz = zhalf ? NI / 2 : NI;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const T kk = T(0.5) * b * dtdx;        // the 1/2 of Eq. 12 is applied here (G = 2F)
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
    const int i = lane & 15, j = warp + 8 * (lane >> 4);
    const int off = LEAD + (j + NG) * PX + (i + NG);            // in-plane offset of this column
    const T *base = pool.patch(sbase, p) + off;
    T *out = pool.patch(sout, p) + off;
    const T *raw = sm + S::O_RAW + j * NI + i;                   // this column in ring slot 0, v = 0
    T *wme = sm + S::O_W + (j + NG) * PW + (i + NG);             // this column in primitive plane 0, v = 0
    T *qx = sm + S::O_QX + j * PQ + i, *fx = sm + S::O_FX + j * PQ + i;   // slot i: q+ of cell i-1 / flux at face i
    T *qy = sm + S::O_QY + j * PY + i, *fy = sm + S::O_FY + j * PY + i;
    T dzm[NV], qpz[NV], acc[NV];
    T *zpark = sm + S::O_PARK + tid;    // (S::PARK only)
    T best = T(0);                      // fused CFL reduction (a1) over the cells this thread finishes
    bool bad = false;
    // raw plane pk -> primitives of this column in primitive buffer pk & 1
    auto convert = [&](int pk) {
      const int slot = pk % S::NSLOT;
      mk::mbar_wait(&bars[slot], unsigned(pk / S::NSLOT) & 1u);
      T Un[NV], Wn[NV];
#pragma unroll
      for (int v = 0; v < NV; ++v) Un[v] = raw[slot * RAWP + v * (NI * NI)];
      mk::prim<T, NV>(Un, Wn, P, hits);
      T *w = wme + (pk & 1) * (NV * WV);
#pragma unroll
      for (int v = 0; v < NV; ++v) w[v * WV] = Wn[v];
    };
    {
      T U0[NV], U1[NV], U2[NV], W0[NV], W1[NV], Wc[NV];
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
      mk::prim<T, NV>(U2, Wc, P, hits);
#pragma unroll
      for (int v = 0; v < NV; ++v) {
        wme[v * WV] = Wc[v];                                        // plane 2 -> primitive buffer 0
        const T dm = W1[v] - W0[v];
        dzm[v] = Wc[v] - W1[v];
        const T s = mk::slope4(dm, dzm[v], dm + dzm[v], th2);            // (the sum, as in the loop: a z-split march must give the same bits)
        qpz[v] = fma(q4, s, W1[v]);                                 // q+ of the ghost cell below plane 2
        if (S::PARK) zpark[v * (NI * NI)] = qpz[v];
        acc[v] = T(0);
      }
    }
    __syncthreads();
    convert(NG + 1);

    // The primitives of this column live in the two primitive buffers, not in registers: plane c and c+1 are read where
    // the z slope needs them, and plane c+2 is converted at the END of pass c, when only dzm, qpz and acc are live (its
    // buffer, that of plane c, is free once every thread is past the x/y slopes: the second barrier of the pass)
#pragma unroll 1
    for (int c = NG; c <= NG + nz; ++c) {            // current cell = plane c of this march (2..nz+1); c = nz+2: last z face only
      const T *w = wme + (c & 1) * (NV * WV);
      T Wc[NV], Wn[NV];
      {
        const T *wn = wme + ((c + 1) & 1) * (NV * WV);
#pragma unroll
        for (int v = 0; v < NV; ++v) { Wc[v] = w[v * WV]; Wn[v] = wn[v * WV]; }
      }
      T ub[NV];
      if (BASE && !S::BTMA && c > NG) {             // (global loads: issued early; the TMA ring is read where it is used)
#pragma unroll
        for (int v = 0; v < NV; ++v) ub[v] = base[size_t(v) * VS + (c - 1 + zlo) * PLANE];
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
        if (S::PARK) {
#pragma unroll
          for (int v = 0; v < NV; ++v) qpz[v] = zpark[v * (NI * NI)];
        }
        mk::floor_states<T, NV>(qpz, qm, P, hits);
        mk::face_flux<T, 2>(qpz, qm, P, Gz);
        if (S::PARK) {
#pragma unroll
          for (int v = 0; v < NV; ++v) zpark[v * (NI * NI)] = qp[v];
        } else {
#pragma unroll
          for (int v = 0; v < NV; ++v) qpz[v] = qp[v];
        }
      }
      if (bflux && ((c - NG + zlo) & 7) == 0) {
        T *B = bflux + ((size_t(pl) * 9 + 6 + ((c - NG + zlo) >> 3)) * NV) * 256 + j * 16 + i;
#pragma unroll
        for (int v = 0; v < NV; ++v) B[v * 256] = T(0.5) * Gz[v];
      }
      if (c > NG) {
        const T *ui = raw + ((c - 1) % S::NSLOT) * RAWP;     // raw U of cell c-1 is still in the ring
        T *o = out + (c - 1 + zlo) * PLANE;
        T un[NV];
#pragma unroll
        for (int v = 0; v < NV; ++v) {
          T pre = b * ui[v * (NI * NI)];
          if (BASE) pre = fma(a, S::BTMA ? raw[S::O_BRAW - S::O_RAW + ((c + 1) % S::NSLOT) * RAWP + v * (NI * NI)]   // arrived with plane c+1
                                         : ub[v], pre);
          un[v] = fma(-kk, acc[v] + Gz[v], pre);                    // Eq. 7-8
          o[size_t(v) * VS] = un[v];
        }
        if (BASE && smax_out) {
          // S4 on the state just produced: max_d |v_d| + c_d, with the NaN/inf test of k_cfl
          T Wq[NV];
          mk::prim<T, NV>(un, Wq, P, hits);
          const T sp = mk::max_speed_fast<T, NV>(Wq, P);
          const T chk = (((Wq[2] + Wq[3]) + Wq[4]) + sp) + (un[0] + un[4]);   // (the floors would hide a NaN density or energy)
          bad |= !(chk - chk == T(0));
          best = tmax(best, sp);
        }
      }
      if (c < NG + nz) {
        // 3. x/y phase 1: slopes of this cell along x and y, publish q+
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
        // 4. phase 2: fluxes through the low x and y faces of this cell
        T Gx[NV], Gy[NV];
        {
          T WL[NV], WD[NV];
#pragma unroll
          for (int v = 0; v < NV; ++v) { WL[v] = qx[v * QXV]; WD[v] = qy[v * QYV]; }
          mk::floor_states2<T, NV>(WL, qmx, WD, qmy, P, hits);
          mk::face_flux<T, 0>(WL, qmx, P, Gx);
          mk::face_flux<T, 1>(WD, qmy, P, Gy);
#pragma unroll
          for (int v = 0; v < NV; ++v) { fx[v * QXV] = Gx[v]; fy[v * QYV] = Gy[v]; }
        }
        if (bflux) {
          if ((i & 7) == 0) {
            T *B = bflux + ((size_t(pl) * 9 + 0 + (i >> 3)) * NV) * 256 + (c - NG + zlo) * 16 + j;
#pragma unroll
            for (int v = 0; v < NV; ++v) B[v * 256] = T(0.5) * Gx[v];
          }
          if ((j & 7) == 0) {
            T *B = bflux + ((size_t(pl) * 9 + 3 + (j >> 3)) * NV) * 256 + (c - NG + zlo) * 16 + i;
#pragma unroll
            for (int v = 0; v < NV; ++v) B[v * 256] = T(0.5) * Gy[v];
          }
        }
        __syncthreads();
        // 5. phase 3: flux differences in x and y; the low z face enters with its sign
#pragma unroll
        for (int v = 0; v < NV; ++v)
          acc[v] = ((fx[v * QXV + 1] - Gx[v]) + (fy[v * QYV + PY] - Gy[v])) - Gz[v];
        // 6. plane c+2: raw -> primitives, for the z slope of the next pass and the x/y neighbours of the one after
        convert(c + 2);
      }
    }
    if (BASE && smax_out) {
      // one atomicMax per warp on the bit pattern of a non-negative double (monotone as an unsigned integer)
      double bq = bad ? __longlong_as_double(0x7ff0000000000000LL) : double(best);
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) bq = fmax(bq, __shfl_xor_sync(0xffffffffu, bq, o));
      if (lane == 0) atomicMax(smax_out, (unsigned long long)__double_as_longlong(bq));
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
      mk::halo_warp<T, NV, 0, S>(sm, g[0], g[1], lane, P, th2, bflux, pl, hits, lane == 0, &tmap, bars, q_mid, q_lo, q_hi, kz_lo, kz_hi,
                              (BASE && S::BTMA) ? (sbase * pool.max_patches + p) * NV : -1, zlo, nz);
    else
      mk::halo_warp<T, NV, 1, S>(sm, g[0], g[1], lane, P, th2, bflux, pl, hits, false, &tmap, bars, q_mid, q_lo, q_hi, kz_lo, kz_hi,
                                 -1, zlo, nz);
  }
  if (hits) atomicAdd(floor_hits, (unsigned long long)hits);
}

// 4-D tensor map over the pool: (i, pj, pk, q) with q = (slot*max_patches + patch)*nv + var; the
// origin is the first interior cell of a row, so that the global address is 32-byte aligned for
// both element types.  Box = one interior plane of all variables of one patch.
template <typename T, int NV>
int make_tensor_map(CUtensorMap *tm, void *pool_base, size_t max_patches, int nslots) {
  typedef CUresult (*encode_fn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
  static encode_fn enc = nullptr;
  if (!enc) {
    void *fp = nullptr;
    cudaDriverEntryPointQueryResult qr;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fp, cudaEnableDefault, &qr) != cudaSuccess || !fp) return -1;
    enc = (encode_fn)fp;
  }
  const cuuint64_t dims[4] = {cuuint64_t(NI), cuuint64_t(NP), cuuint64_t(NP), cuuint64_t(nslots) * max_patches * NV};
  const cuuint64_t strides[3] = {cuuint64_t(Layout<T>::PX) * sizeof(T), cuuint64_t(Layout<T>::PLANE) * sizeof(T),
                                 cuuint64_t(Layout<T>::VS) * sizeof(T)};
  const cuuint32_t box[4] = {cuuint32_t(NI), cuuint32_t(NI), 1, NV};
  const cuuint32_t estr[4] = {1, 1, 1, 1};
  void *origin = (char *)pool_base + size_t(Layout<T>::LEAD + NG) * sizeof(T);
  CUresult r = enc(tm, sizeof(T) == 8 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, origin, dims,
                   strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                   CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS ? 0 : -2;
}

// returns 0 or a cudaError_t
template <typename T, int NV>
int launch_rk_stage_march(const CUtensorMap &tmap, Pool<T> pool, int sin, int sbase, int sout, int first, int n, T a, T b,
                          T dtdx, Params<T> P, T *bflux, unsigned long long *floor_hits, const Desc *desc, int direct_halo,
                          cudaStream_t stream, unsigned long long *smax_out = nullptr, int zmode = 0, int num_sms = 0, DtDev dtd = DtDev{nullptr, 0, 0}) {
  static bool configured = false;
  static int cps[2] = {1, 1};               // resident CTAs per SM of the two instantiations
  constexpr size_t bytes0 = mk::Smem<T, NV, false>::BYTES, bytes1 = mk::Smem<T, NV, true>::BYTES;
  if (!configured) {
    cudaError_t e = cudaFuncSetAttribute(k_rk_stage_march<T, NV, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(bytes0));
    if (e == cudaSuccess)
      e = cudaFuncSetAttribute(k_rk_stage_march<T, NV, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(bytes1));
    if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&cps[0], k_rk_stage_march<T, NV, false>, mk::THREADS, bytes0);
    if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&cps[1], k_rk_stage_march<T, NV, true>, mk::THREADS, bytes1);
    if (e != cudaSuccess) return int(e);
    configured = true;
  }
  // zmode 0: never split; 1: every patch; 2: every patch of a level of at most num_sms / 2 patches, else the patches of
  // the last wave of the launch if that wave is less than half full (their half-CTAs then all fit into it)
  int nfull = n;
  if (zmode == 1 || (zmode == 2 && 2 * n <= num_sms)) nfull = 0;
  else if (zmode == 2) {
    const int slots = std::max(1, cps[a != T(0) ? 1 : 0]) * num_sms, tail = n % slots;
    if (n > slots && tail > 0 && 2 * tail <= slots) nfull = n - tail;
  }
  const int grid = nfull + 2 * (n - nfull);
  if (a != T(0))
    k_rk_stage_march<T, NV, true><<<grid, mk::THREADS, bytes1, stream>>>(tmap, pool, sin, sbase, sout, first, a, b, dtdx, P,
                                                                                bflux, floor_hits, desc, direct_halo, smax_out, nfull, dtd);
  else
    k_rk_stage_march<T, NV, false><<<grid, mk::THREADS, bytes0, stream>>>(tmap, pool, sin, sbase, sout, first, a, b, dtdx, P,
                                                                                 bflux, floor_hits, desc, direct_halo, nullptr, nfull, dtd);
  return 0;
}

}  // namespace amr
