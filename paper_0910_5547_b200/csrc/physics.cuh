// physics.cuh -- device-side variable sets, limiter and flux of the hot path (sm_100a).
//
// Euler: Eq. 1-6.  Ideal MHD (8 variables): Eq. 14-15 with
// reading G3 (B-slots of F^y/F^z permuted back) and psi == 0 (S3').  Reconstruction:
// PAPER.md:104-112 Eq. 9-11 with the factor 1/2 of reading G1.  Flux: Eq. 12
// (single-speed HLL = LLF, readings G2/G6), signal speeds S2/S3.  Floors: S11.
//
// Written for instruction count: one reciprocal per cell, one slope per cell and direction
// (shared by the two faces of the cell: Eq. 9 and Eq. 10 use the same minmod up to sign),
// sign logic of Eq. 11 on the integer pipe, lambda0 = max(|v_l|+c_l, |v_r|+c_r).
#pragma once
#include <cuda_runtime.h>

namespace amr {

template <typename T> struct Params {
  T gamma, gm1, gg1;   // gamma, gamma-1, gamma*(gamma-1)
  T theta;             // Eq. 9-10 (S1)
  T rho_floor, e_floor;
  T ch;                // c_h of Eq. 15 (9-variable GLM-MHD only; S17)
};

__device__ __forceinline__ float tsqrt(float x) { return sqrtf(x); }
__device__ __forceinline__ double tsqrt(double x) { return sqrt(x); }
__device__ __forceinline__ float tmax(float a, float b) { return fmaxf(a, b); }
__device__ __forceinline__ double tmax(double a, double b) { return fmax(a, b); }
__device__ __forceinline__ float tmin(float a, float b) { return fminf(a, b); }
__device__ __forceinline__ double tmin(double a, double b) { return fmin(a, b); }
__device__ __forceinline__ float tabs(float a) { return fabsf(a); }
__device__ __forceinline__ double tabs(double a) { return fabs(a); }
__device__ __forceinline__ float trcp(float a) { return 1.0f / a; }
__device__ __forceinline__ double trcp(double a) { return 1.0 / a; }

// same sign bit?  (integer pipe; +-0 is harmless because min(|a|,|b|,|c|) is then 0)
__device__ __forceinline__ bool same_sign(float a, float b) {
  return ((__float_as_int(a) ^ __float_as_int(b)) >= 0);
}
__device__ __forceinline__ bool same_sign(double a, double b) {
  return ((__double2hiint(a) ^ __double2hiint(b)) >= 0);
}
__device__ __forceinline__ float with_sign_of(float m, float s) { return copysignf(m, s); }
__device__ __forceinline__ double with_sign_of(double m, double s) { return copysign(m, s); }

// Limited slope of a cell from its left, own and right values:
//   sigma = minmod(theta (q0-qm), theta (qp-q0), (qp-qm)/2)            (Eq. 11)
// Eq. 9:  q_{i-1/2,l} = q_{i-1} + sigma_{i-1}/2 ;  Eq. 10: q_{i-1/2,r} = q_i - sigma_i/2
// (minmod is odd and symmetric in its first two arguments, so Eq. 10's minmod is -sigma_i).
// When a and b have the same strict sign, c has it too (q is then monotone over the 3 cells).
template <typename T> __device__ __forceinline__ T limited_slope(T qm, T q0, T qp, T theta) {
  T a = (q0 - qm) * theta;
  T b = (qp - q0) * theta;
  T c = (qp - qm) * T(0.5);
  T m = tmin(tabs(a), tmin(tabs(b), tabs(c)));
  return same_sign(a, b) ? with_sign_of(m, a) : T(0);
}

// O1: conserved -> primitive W = (rho, e, vx, vy, vz, [Bx, By, Bz]);  PAPER.md:59, :298.
template <typename T, int NV>
__device__ __forceinline__ void cons_to_prim(const T (&U)[NV], T (&W)[NV], const Params<T> &P, int &hits) {
  T rho = U[0];
  if (!(rho >= P.rho_floor)) { rho = P.rho_floor; ++hits; }
  T ir = trcp(rho);
  T vx = U[1] * ir, vy = U[2] * ir, vz = U[3] * ir;
  T et = U[4];
  if (NV >= 8) {
    et -= T(0.5) * (U[5 % NV] * U[5 % NV] + U[6 % NV] * U[6 % NV] + U[7 % NV] * U[7 % NV]);
    W[5 % NV] = U[5 % NV]; W[6 % NV] = U[6 % NV]; W[7 % NV] = U[7 % NV];
  }
  if (NV == 9) W[8 % NV] = U[8 % NV];                             // psi (Eq. 14)
  T e = et * ir - T(0.5) * (vx * vx + vy * vy + vz * vz);
  if (!(e >= P.e_floor)) { e = P.e_floor; ++hits; }
  W[0] = rho; W[1] = e; W[2] = vx; W[3] = vy; W[4] = vz;
}

template <typename T, int NV>
__device__ __forceinline__ void floor_state(T (&W)[NV], const Params<T> &P, int &hits) {
  if (!(W[0] >= P.rho_floor)) { W[0] = P.rho_floor; ++hits; }
  if (!(W[1] >= P.e_floor)) { W[1] = P.e_floor; ++hits; }
}

// conserved state, physical flux along D and signal speed of one primitive state
template <typename T, int NV, int D>
__device__ __forceinline__ void state_flux(const T (&W)[NV], const Params<T> &P, T (&U)[NV], T (&F)[NV], T &speed) {
  const T rho = W[0], e = W[1];
  const T vd = W[2 + D];
  const T p = P.gm1 * rho * e;                                   // Eq. 6
  const T ke = T(0.5) * (W[2] * W[2] + W[3] * W[3] + W[4] * W[4]);
  const T m = rho * vd;
  U[0] = rho; U[1] = rho * W[2]; U[2] = rho * W[3]; U[3] = rho * W[4];
  T E = rho * (ke + e);
  F[0] = m;
  if (NV == 5) {
    U[4] = E;
    F[1] = m * W[2]; F[2] = m * W[3]; F[3] = m * W[4];
    F[1 + D] += p;
    F[4] = (E + p) * vd;                                          // rho (v^2/2 + h) v_d, h = e + p/rho
    speed = tabs(vd) + tsqrt(P.gg1 * e);                          // S2: c_s^2 = gamma p / rho
  } else {
    const T Bx = W[5 % NV], By = W[6 % NV], Bz = W[7 % NV];
    const T Bd = W[(5 + D) % NV];
    const T B2 = Bx * Bx + By * By + Bz * Bz;
    const T Bv = Bx * W[2] + By * W[3] + Bz * W[4];
    const T pt = p + T(0.5) * B2;
    E += T(0.5) * B2;
    U[4] = E;
    U[5 % NV] = Bx; U[6 % NV] = By; U[7 % NV] = Bz;
    F[1] = m * W[2] - Bx * Bd; F[2] = m * W[3] - By * Bd; F[3] = m * W[4] - Bz * Bd;
    F[1 + D] += pt;
    F[4] = (E + pt) * vd - Bd * Bv;                               // Eq. 15 energy row
    F[5 % NV] = vd * Bx - Bd * W[2]; F[6 % NV] = vd * By - Bd * W[3]; F[7 % NV] = vd * Bz - Bd * W[4];
    F[(5 + D) % NV] = T(0);                                       // psi == 0 (S3')
    if (NV == 9) {                                                // Eq. 15: F^d(B_d) = psi, F^d(psi) = c_h^2 B_d
      U[8 % NV] = W[8 % NV];
      F[(5 + D) % NV] = W[8 % NV];
      F[8 % NV] = P.ch * P.ch * Bd;
    }
    const T ir = trcp(rho);                                       // S3: fast magnetosonic speed along D
    const T a2 = P.gg1 * e, b2 = B2 * ir, bd2 = Bd * Bd * ir;
    const T s = a2 + b2;
    const T disc = tmax(s * s - T(4) * a2 * bd2, T(0));
    speed = tabs(vd) + tsqrt(T(0.5) * (s + tsqrt(disc)));
  }
}

// O3, Eq. 12: F = 1/2 (F_l + F_r - lambda0 (U_r - U_l)),
// lambda0 = max(max(0, l_l^+, l_r^+), max(0, -l_l^-, -l_r^-)) = max(|v_l| + c_l, |v_r| + c_r).
template <typename T, int NV, int D>
__device__ __forceinline__ void riemann_flux(const T (&WL)[NV], const T (&WR)[NV], const Params<T> &P, T (&F)[NV]) {
  T UL[NV], UR[NV], FL[NV], FR[NV], sl, sr;
  state_flux<T, NV, D>(WL, P, UL, FL, sl);
  state_flux<T, NV, D>(WR, P, UR, FR, sr);
  T lam = tmax(sl, sr);
  if (NV == 9) lam = tmax(lam, P.ch);                             // S17
#pragma unroll
  for (int v = 0; v < NV; ++v) F[v] = T(0.5) * ((FL[v] + FR[v]) - lam * (UR[v] - UL[v]));
}

// max over directions of |v_d| + c_d for the CFL reduction (S4)
template <typename T, int NV>
__device__ __forceinline__ T max_signal_speed(const T (&W)[NV], const Params<T> &P) {
  const T a2 = P.gg1 * W[1];
  if (NV == 5) {
    return tmax(tabs(W[2]), tmax(tabs(W[3]), tabs(W[4]))) + tsqrt(a2);
  } else {
    const T ir = trcp(W[0]);
    const T B2 = W[5 % NV] * W[5 % NV] + W[6 % NV] * W[6 % NV] + W[7 % NV] * W[7 % NV];
    const T s = a2 + B2 * ir;
    T best = T(0);
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      const T bd2 = W[(5 + d) % NV] * W[(5 + d) % NV] * ir;
      const T disc = tmax(s * s - T(4) * a2 * bd2, T(0));
      best = tmax(best, tabs(W[2 + d]) + tsqrt(T(0.5) * (s + tsqrt(disc))));
    }
    if (NV == 9) best = tmax(best, P.ch);                         // S17: c_h bounds the time step too
    return best;
  }
}

}  // namespace amr
