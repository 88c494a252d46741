// amr_oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, obviously-correct CPU restatement of the per-patch finite-volume
// update of Wang, Abel & Kaehler, "Adaptive Mesh Fluid Simulations on GPU"
// (arXiv:0910.5547; text in /root/reference/PAPER.md, cited below as PAPER.md:<line>)
// plus the level-wide steps BASELINE.json's north_star names around it.
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
// legs may load this file.  It shares no code, header, table or constant with the
// CUDA path under paper_0910_5547_b200/csrc/.  Compiled with -ffp-contract=off so
// that what is written below is what is evaluated (no FMA contraction).
//
// Every function follows the paper's order and notation; the readings taken where
// PAPER.md is garbled (G1-G6) or silent (S1-S21) are those of SURVEY.md section 8(c)
// (S17-S21: DESIGN.md section 3) and are listed again in DESIGN.md.  Pins: tests/test_oracle_*.py
// (P1-P12 the hot path, P13-P17 the 9-variable GLM system, P18-P19 the regrid steps, P20 the floors of S11,
// P21 the global time step on several levels).
// Parity unpinned: none of the per-step functions (all have at least one pin);
// the long-time Brio-Wu / Sedov / KH *profiles* have no printed values in the paper.
//
// Storage (private to the oracle): pool[slot][patch][var][k][j][i] over the padded
// 20^3 box (2 ghost + 16 interior + 2 ghost per axis, i fastest).
//
// Variables (Eq. 2; Eq. 14; 8 variables = Eq. 14 without psi, reading S3';
// 9 variables = the GLM system the paper ran, readings S17-S19 of DESIGN.md):
//   U = (rho, rho vx, rho vy, rho vz, rho E [+ B^2/2], [Bx, By, Bz], [psi])
// Primitives handed to reconstruction ("Rho, Eint, Vx, Vy, Vz"):
//   W = (rho, e, vx, vy, vz, [Bx, By, Bz], [psi])

#include <algorithm>
#include <array>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <functional>
#include <thread>
#include <vector>

namespace {

constexpr int NI = 16;          // interior cells per side (BASELINE.json north_star)
constexpr int NG = 2;           // ghost zones per side (stencil i-2..i+1)
constexpr int NP = NI + 2 * NG; // padded side = 20
constexpr int NC = NP * NP * NP;
constexpr int MAXV = 9;

inline int cidx(int k, int j, int i) { return (k * NP + j) * NP + i; }

// ---------------------------------------------------------------- Eq. 11
// minmod(a,b,c) = 0.25 (sign a + sign b) |sign a + sign c| min(|a|,|b|,|c|)
template <class T> inline T sign_of(T x) { return (x > T(0)) ? T(1) : ((x < T(0)) ? T(-1) : T(0)); }

template <class T> inline T minmod3(T a, T b, T c) {
  T sa = sign_of(a), sb = sign_of(b), sc = sign_of(c);
  T m = std::min(std::fabs(a), std::min(std::fabs(b), std::fabs(c)));
  return T(0.25) * (sa + sb) * std::fabs(sa + sc) * m;
}

// two-argument minmod used by the prolongation operator (reading S6)
template <class T> inline T minmod2(T a, T b) {
  if (a > T(0) && b > T(0)) return std::min(a, b);
  if (a < T(0) && b < T(0)) return std::max(a, b);
  return T(0);
}

template <class T> struct Phys {
  int nv;        // 5 Euler, 8 ideal MHD, 9 GLM-MHD
  T gamma;       // PAPER.md:71 Eq. 6
  T theta;       // PAPER.md:110, reading S1
  T rho_floor;   // reading S11
  T e_floor;
  long *floor_hits;
  T ch = T(0);   // c_h of Eq. 15, reading S17: a constant given by the caller
  T cr = T(0);   // c_p^2 / c_h of Dedner et al. 2002 ("damping rate"), reading S18; 0 = no damping

  // O1: conserved -> primitive.  PAPER.md:59 (E = v^2/2 + e), PAPER.md:298 (energy slot rho E + B^2/2)
  inline void prim(const T *U, T *W) const {
    T rho = U[0];
    if (!(rho >= rho_floor)) { rho = rho_floor; if (floor_hits) ++*floor_hits; }
    T vx = U[1] / rho, vy = U[2] / rho, vz = U[3] / rho;
    T etot = U[4];
    if (nv >= 8) {
      T B2 = U[5] * U[5] + U[6] * U[6] + U[7] * U[7];
      etot = etot - T(0.5) * B2;
      W[5] = U[5]; W[6] = U[6]; W[7] = U[7];
    }
    if (nv == 9) W[8] = U[8];
    T e = etot / rho - T(0.5) * (vx * vx + vy * vy + vz * vz);
    if (!(e >= e_floor)) { e = e_floor; if (floor_hits) ++*floor_hits; }
    W[0] = rho; W[1] = e; W[2] = vx; W[3] = vy; W[4] = vz;
  }

  inline void floor_state(T *W) const {  // S11: same floors on reconstructed states
    if (!(W[0] >= rho_floor)) { W[0] = rho_floor; if (floor_hits) ++*floor_hits; }
    if (!(W[1] >= e_floor)) { W[1] = e_floor; if (floor_hits) ++*floor_hits; }
  }

  // conserved state of a primitive state (Eq. 2 / Eq. 14)
  inline void cons(const T *W, T *U) const {
    T rho = W[0], e = W[1], vx = W[2], vy = W[3], vz = W[4];
    T v2 = vx * vx + vy * vy + vz * vz;
    U[0] = rho; U[1] = rho * vx; U[2] = rho * vy; U[3] = rho * vz;
    U[4] = rho * (T(0.5) * v2 + e);
    if (nv >= 8) {
      T B2 = W[5] * W[5] + W[6] * W[6] + W[7] * W[7];
      U[4] = U[4] + T(0.5) * B2;
      U[5] = W[5]; U[6] = W[6]; U[7] = W[7];
    }
    if (nv == 9) U[8] = W[8];
  }

  // physical flux F^d(W).  Euler: Eq. 3-5 PAPER.md:63-67.  MHD: Eq. 15
  // with reading G3 (B-slots of F^y, F^z permuted back) and psi == 0 (S3').
  inline void flux(const T *W, int d, T *F) const {
    T rho = W[0], e = W[1];
    const T *v = W + 2;
    T vd = v[d];
    T p = (gamma - T(1)) * rho * e;             // Eq. 6
    T v2 = v[0] * v[0] + v[1] * v[1] + v[2] * v[2];
    T h = e + p / rho;
    F[0] = rho * vd;
    for (int i = 0; i < 3; ++i) F[1 + i] = rho * v[i] * vd;
    F[4] = rho * (T(0.5) * v2 + h) * vd;
    if (nv == 5) {
      F[1 + d] = F[1 + d] + p;
    } else {
      const T *B = W + 5;
      T B2 = B[0] * B[0] + B[1] * B[1] + B[2] * B[2];
      T Bd = B[d];
      T Bv = B[0] * v[0] + B[1] * v[1] + B[2] * v[2];
      for (int i = 0; i < 3; ++i) F[1 + i] = F[1 + i] - B[i] * Bd;
      F[1 + d] = F[1 + d] + p + T(0.5) * B2;
      F[4] = F[4] + B2 * vd - Bd * Bv;
      for (int i = 0; i < 3; ++i) F[5 + i] = vd * B[i] - Bd * v[i];
      F[5 + d] = T(0);                          // psi == 0 in the 8-variable system
      if (nv == 9) {                            // Eq. 15: F^d(B_d) = psi, F^d(psi) = c_h^2 B_d
        F[5 + d] = W[8];
        F[8] = ch * ch * Bd;
      }
    }
  }

  // signal speed along d: c_s (S2) or fast magnetosonic speed (S3)
  inline T speed(const T *W, int d) const {
    T rho = W[0], e = W[1];
    T p = (gamma - T(1)) * rho * e;
    T a2 = gamma * p / rho;
    if (nv == 5) return std::sqrt(a2);
    const T *B = W + 5;
    T b2 = (B[0] * B[0] + B[1] * B[1] + B[2] * B[2]) / rho;
    T bd2 = B[d] * B[d] / rho;
    T s = a2 + b2;
    T disc = s * s - T(4) * a2 * bd2;
    if (disc < T(0)) disc = T(0);
    return std::sqrt(T(0.5) * (s + std::sqrt(disc)));
  }

  // O2: PLM interface states at the face between cells i-1 and i from cells
  // i-2 (Wm2), i-1 (Wm1), i (W0), i+1 (Wp1).  Eq. 9-10 PAPER.md:106-108 with the
  // factor 1/2 of reading G1.
  inline void plm(const T *Wm2, const T *Wm1, const T *W0, const T *Wp1, T *WL, T *WR) const {
    for (int q = 0; q < nv; ++q) {
      WL[q] = Wm1[q] + T(0.5) * minmod3((Wm1[q] - Wm2[q]) * theta, (W0[q] - Wm1[q]) * theta,
                                         (W0[q] - Wm2[q]) / T(2));
      WR[q] = W0[q] + T(0.5) * minmod3((W0[q] - Wp1[q]) * theta, (Wm1[q] - W0[q]) * theta,
                                        (Wm1[q] - Wp1[q]) / T(2));
    }
    floor_state(WL);
    floor_state(WR);
  }

  // O3: Eq. 12 PAPER.md:116-118 (single-speed HLL = LLF, reading G6; conserved-state
  // difference, reading G2).
  inline T riemann(const T *WL, const T *WR, int d, T *F) const {
    T UL[MAXV], UR[MAXV], FL[MAXV], FR[MAXV];
    cons(WL, UL); cons(WR, UR);
    flux(WL, d, FL); flux(WR, d, FR);
    T cl = speed(WL, d), cr = speed(WR, d);
    T vl = WL[2 + d], vr = WR[2 + d];
    T lp = std::max(T(0), std::max(vl + cl, vr + cr));          // max(0, lambda_l^+, lambda_r^+)
    T lm = std::max(T(0), std::max(-(vl - cl), -(vr - cr)));    // max(0,-lambda_l^-,-lambda_r^-)
    T lam0 = std::max(lp, lm);
    if (nv == 9) lam0 = std::max(lam0, ch);    // the (B_d, psi) pair travels at +-c_h (reading S17)
    for (int q = 0; q < nv; ++q) F[q] = T(0.5) * (FL[q] + FR[q] - lam0 * (UR[q] - UL[q]));
    return lam0;
  }
};

// ------------------------------------------------------------------------------------
// Hierarchy state: flat patch-descriptor table (reading D4 of SURVEY.md: the Enzo grid
// tree of PAPER.md:43 flattened) + the padded pool + the coarse-fine flux registers.
// Neighbour table: nbr[p][r], r = (dz+1)*9 + (dy+1)*3 + (dx+1); entry >= 0 is a
// same-level patch, -1 a coarse-fine boundary, -2 a physical boundary.
// ------------------------------------------------------------------------------------
constexpr int FACE_REGION[6] = {12, 14, 10, 16, 4, 22};  // x-lo x-hi y-lo y-hi z-lo z-hi

template <class T> struct Hier {
  Phys<T> ph;
  int nv = 5, np = 0, nlev = 0, nslots = 0, nthreads = 1;
  double dx0 = 1.0;
  int bc[6] = {0, 0, 0, 0, 0, 0};  // 0 periodic (table wraps), 1 outflow
  std::vector<int> level, parent, origin, nbr, octant;
  std::vector<std::array<int, 8>> child;
  std::vector<std::vector<int>> lev_patches;
  std::vector<T> pool;
  std::vector<T> Rf, Rc;  // [patch][face][var][8*8]
  long floor_hits = 0;

  size_t patch_stride() const { return size_t(nv) * NC; }
  T *P(int slot, int p) { return pool.data() + (size_t(slot) * np + p) * patch_stride(); }
  T *reg(std::vector<T> &R, int p, int f) { return R.data() + (size_t(p) * 6 + f) * nv * 64; }
  double dx(int lev) const { return dx0 / double(1 << lev); }
  bool has_children(int lev) const { return lev + 1 < nlev && !lev_patches[lev + 1].empty(); }

  void parallel_for(int n, const std::function<void(int, Phys<T> &)> &fn) {
    int nt = std::max(1, std::min(nthreads, n));
    if (nt == 1) {
      Phys<T> q = ph; q.floor_hits = &floor_hits;
      for (int i = 0; i < n; ++i) fn(i, q);
      return;
    }
    std::vector<long> hits(nt, 0);
    std::vector<std::thread> th;
    for (int t = 0; t < nt; ++t)
      th.emplace_back([&, t]() {
        Phys<T> q = ph; q.floor_hits = &hits[t];
        for (int i = t; i < n; i += nt) fn(i, q);
      });
    for (auto &x : th) x.join();
    for (long h : hits) floor_hits += h;
  }

  // ---- S4: max over interior cells and directions of |v_d| + c_d
  double max_speed(int lev, int slot) {
    const auto &lp = lev_patches[lev];
    std::vector<double> smax(lp.size(), 0.0);
    parallel_for((int)lp.size(), [&](int n, Phys<T> &q) {
      const T *U = P(slot, lp[n]);
      double s = 0.0;
      T Uc[MAXV], W[MAXV];
      for (int k = NG; k < NG + NI; ++k)
        for (int j = NG; j < NG + NI; ++j)
          for (int i = NG; i < NG + NI; ++i) {
            for (int v = 0; v < nv; ++v) Uc[v] = U[size_t(v) * NC + cidx(k, j, i)];
            q.prim(Uc, W);
            for (int d = 0; d < 3; ++d) {
              double sd = double(std::fabs(W[2 + d]) + q.speed(W, d));
              if (nv == 9 && !(sd >= double(q.ch))) sd = double(q.ch);   // S17: c_h bounds the time step too
              if (!(sd <= s)) s = sd;  // NaN propagates
            }
          }
      smax[n] = s;
    });
    double s = 0.0;
    for (double x : smax) if (!(x <= s)) s = x;
    return s;
  }

  // ---- O6 / S5-S7: ghost fill of one level
  void fill_ghosts(int lev, int slot, int pold, int pnew, double alpha) {
    const auto &lp = lev_patches[lev];
    const T al = T(alpha);
    parallel_for((int)lp.size(), [&](int n, Phys<T> &) {
      int p = lp[n];
      T *U = P(slot, p);
      for (int r = 0; r < 27; ++r) {
        if (r == 13) continue;
        int off[3] = {r % 3 - 1, (r / 3) % 3 - 1, r / 9 - 1};
        int lo[3], hi[3];
        for (int d = 0; d < 3; ++d) {
          lo[d] = off[d] < 0 ? 0 : (off[d] == 0 ? NG : NG + NI);
          hi[d] = off[d] < 0 ? NG : (off[d] == 0 ? NG + NI : NP);
        }
        int nb = nbr[size_t(p) * 27 + r];
        if (nb >= 0) {                               // S5(1): same-level sibling copy
          const T *S = P(slot, nb);
          for (int v = 0; v < nv; ++v)
            for (int k = lo[2]; k < hi[2]; ++k)
              for (int j = lo[1]; j < hi[1]; ++j)
                for (int i = lo[0]; i < hi[0]; ++i)
                  U[size_t(v) * NC + cidx(k, j, i)] =
                      S[size_t(v) * NC + cidx(k - off[2] * NI, j - off[1] * NI, i - off[0] * NI)];
        } else if (nb == -1 && lev > 0) {            // S5(2): prolongation from the parent, S6-S7
          int Q = parent[p];
          const T *Co = P(pold, Q), *Cn = P(pnew, Q);
          for (int k = lo[2]; k < hi[2]; ++k)
            for (int j = lo[1]; j < hi[1]; ++j)
              for (int i = lo[0]; i < hi[0]; ++i) {
                int pad[3] = {i, j, k}, pc[3];
                T s[3];
                for (int d = 0; d < 3; ++d) {
                  int g = origin[size_t(p) * 3 + d] + pad[d] - NG;      // fine global index
                  int gc = (g >= 0) ? g / 2 : -((-g + 1) / 2);           // floor(g/2)
                  s[d] = (g - 2 * gc == 0) ? T(-0.25) : T(0.25);
                  pc[d] = gc - origin[size_t(Q) * 3 + d] + NG;           // parent padded index
                }
                int c0 = cidx(pc[2], pc[1], pc[0]);
                const int st[3] = {1, NP, NP * NP};
                for (int v = 0; v < nv; ++v) {
                  const T *o = Co + size_t(v) * NC, *nw = Cn + size_t(v) * NC;
                  auto UC = [&](int c) { return (T(1) - al) * o[c] + al * nw[c]; };   // S7
                  T uc = UC(c0), val = uc;
                  for (int d = 0; d < 3; ++d) {
                    T sig = minmod2(UC(c0 + st[d]) - uc, uc - UC(c0 - st[d]));
                    val = val + s[d] * sig;
                  }
                  U[size_t(v) * NC + cidx(k, j, i)] = val;
                }
              }
        }
      }
      // S5(3): outflow = zero-gradient, x then y then z over the full padded extent
      for (int d = 0; d < 3; ++d)
        for (int side = 0; side < 2; ++side) {
          int f = 2 * d + side;
          if (nbr[size_t(p) * 27 + FACE_REGION[f]] != -2 || bc[f] != 1) continue;
          int src = side == 0 ? NG : NG + NI - 1;
          for (int g = 0; g < NG; ++g) {
            int dst = side == 0 ? g : NG + NI + g;
            for (int v = 0; v < nv; ++v)
              for (int a = 0; a < NP; ++a)
                for (int b = 0; b < NP; ++b) {
                  int cs, cd;
                  if (d == 0) { cs = cidx(a, b, src); cd = cidx(a, b, dst); }
                  else if (d == 1) { cs = cidx(a, src, b); cd = cidx(a, dst, b); }
                  else { cs = cidx(src, a, b); cd = cidx(dst, a, b); }
                  U[size_t(v) * NC + cd] = U[size_t(v) * NC + cs];
                }
          }
        }
    });
  }

  // ---- regrid steps on either side of the hot path (readings S20-S21 of DESIGN.md)
  // S20: refinement indicator of BASELINE.json config 3, |grad rho| / rho with centred differences over the
  // ghost-filled padded box, reduced to its maximum over each 8^3 octant of every patch of the level (the
  // footprint of one would-be child patch).  out[n*8 + o], n = index in the level, o = octant (x bit 0).
  void refine_indicator(int lev, int slot, double *out) {
    const auto &lp = lev_patches[lev];
    const double dx = dx0 / double(1 << lev);
    for (size_t n = 0; n < lp.size(); ++n) {
      const T *rho = P(slot, lp[n]);
      for (int o = 0; o < 8; ++o) out[n * 8 + o] = 0.0;
      for (int k = NG; k < NG + NI; ++k)
        for (int j = NG; j < NG + NI; ++j)
          for (int i = NG; i < NG + NI; ++i) {
            double gx = (double(rho[cidx(k, j, i + 1)]) - double(rho[cidx(k, j, i - 1)])) / (2.0 * dx);
            double gy = (double(rho[cidx(k, j + 1, i)]) - double(rho[cidx(k, j - 1, i)])) / (2.0 * dx);
            double gz = (double(rho[cidx(k + 1, j, i)]) - double(rho[cidx(k - 1, j, i)])) / (2.0 * dx);
            double g = std::sqrt(gx * gx + gy * gy + gz * gz) / double(rho[cidx(k, j, i)]);
            int o = ((i - NG) >> 3) | (((j - NG) >> 3) << 1) | (((k - NG) >> 3) << 2);
            if (!(g <= out[n * 8 + o])) out[n * 8 + o] = g;   // NaN propagates
          }
    }
  }
  // S21: interior of a (new) fine patch from its parent's padded box with the operator of S6
  // (conservative limited-linear; the 8 children of a coarse cell average to it).
  void prolong_interior(int p, int slot, int pslot) {
    int Q = parent[p];
    T *U = P(slot, p);
    const T *C = P(pslot, Q);
    for (int k = NG; k < NG + NI; ++k)
      for (int j = NG; j < NG + NI; ++j)
        for (int i = NG; i < NG + NI; ++i) {
          int pad[3] = {i, j, k}, pc[3];
          T sg[3];
          for (int d = 0; d < 3; ++d) {
            int g = origin[size_t(p) * 3 + d] + pad[d] - NG;
            int gc = g / 2;                                              // g >= 0 on interior cells
            sg[d] = (g - 2 * gc == 0) ? T(-0.25) : T(0.25);
            pc[d] = gc - origin[size_t(Q) * 3 + d] + NG;
          }
          int c0 = cidx(pc[2], pc[1], pc[0]);
          const int st[3] = {1, NP, NP * NP};
          for (int v = 0; v < nv; ++v) {
            const T *c = C + size_t(v) * NC;
            T uc = c[c0], val = uc;
            for (int d = 0; d < 3; ++d) val = val + sg[d] * minmod2(c[c0 + st[d]] - uc, uc - c[c0 - st[d]]);
            U[size_t(v) * NC + cidx(k, j, i)] = val;
          }
        }
  }

  // ---- O1-O4: one RK stage on every patch of a level.
  // U_out = a U_base + b (U_in + dt L(U_in)) on interior cells; Eq. 7-8 PAPER.md:79-98.
  // w != 0 accumulates w*dt*F on coarse-fine faces (reading S10).
  void rk_stage(int lev, int sin, int sbase, int sout, double a_, double b_, double dt_, double w_) {
    const auto &lp = lev_patches[lev];
    const T a = T(a_), b = T(b_), dt = T(dt_), h = T(dx(lev));
    const T wdt = T(w_ * dt_);
    parallel_for((int)lp.size(), [&](int n, Phys<T> &q) {
      int p = lp[n];
      const T *Uin = P(sin, p), *Ub = P(sbase, p);
      T *Uo = P(sout, p);
      std::vector<T> Wc(size_t(NC) * MAXV, T(0));        // per-cell contiguous primitives
      // O1 on every cell the update reads: at most one index in the ghost range
      for (int k = 0; k < NP; ++k)
        for (int j = 0; j < NP; ++j)
          for (int i = 0; i < NP; ++i) {
            int ng = (i < NG || i >= NG + NI) + (j < NG || j >= NG + NI) + (k < NG || k >= NG + NI);
            if (ng > 1) continue;
            T Uc[MAXV];
            for (int v = 0; v < nv; ++v) Uc[v] = Uin[size_t(v) * NC + cidx(k, j, i)];
            q.prim(Uc, &Wc[size_t(cidx(k, j, i)) * MAXV]);
          }
      // O2+O3: fluxes on the 17 faces of every interior line, per direction
      const int NF = NI + 1;
      std::vector<T> F[3];
      for (int d = 0; d < 3; ++d) F[d].assign(size_t(nv) * NI * NI * NF, T(0));
      auto fidx = [&](int v, int t2, int t1, int f) { return ((size_t(v) * NI + t2) * NI + t1) * NF + f; };
      const int st[3] = {1, NP, NP * NP};
      for (int d = 0; d < 3; ++d)
        for (int t2 = 0; t2 < NI; ++t2)
          for (int t1 = 0; t1 < NI; ++t1)
            for (int f = 0; f < NF; ++f) {
              // face between cells (f-1) and f along d (interior numbering), transverse (t1,t2)
              int i, j, k;
              if (d == 0) { i = f + NG; j = t1 + NG; k = t2 + NG; }
              else if (d == 1) { j = f + NG; i = t1 + NG; k = t2 + NG; }
              else { k = f + NG; i = t1 + NG; j = t2 + NG; }
              int c = cidx(k, j, i);
              T WL[MAXV], WR[MAXV], Ff[MAXV];
              q.plm(&Wc[size_t(c - 2 * st[d]) * MAXV], &Wc[size_t(c - st[d]) * MAXV],
                    &Wc[size_t(c) * MAXV], &Wc[size_t(c + st[d]) * MAXV], WL, WR);
              q.riemann(WL, WR, d, Ff);
              for (int v = 0; v < nv; ++v) F[d][fidx(v, t2, t1, f)] = Ff[v];
            }
      // O4: flux divergence + RK combination, summation order x, y, z
      for (int v = 0; v < nv; ++v)
        for (int k = 0; k < NI; ++k)
          for (int j = 0; j < NI; ++j)
            for (int i = 0; i < NI; ++i) {
              T dFx = F[0][fidx(v, k, j, i + 1)] - F[0][fidx(v, k, j, i)];
              T dFy = F[1][fidx(v, k, i, j + 1)] - F[1][fidx(v, k, i, j)];
              T dFz = F[2][fidx(v, j, i, k + 1)] - F[2][fidx(v, j, i, k)];
              T L = -((dFx + dFy) + dFz) / h;
              size_t c = size_t(v) * NC + cidx(k + NG, j + NG, i + NG);
              Uo[c] = a * Ub[c] + b * (Uin[c] + dt * L);
            }
      if (w_ == 0.0) return;
      // S10 fine side: this patch's own coarse-fine faces, 4 fine faces -> 1 coarse face
      if (lev > 0)
        for (int f = 0; f < 6; ++f) {
          if (nbr[size_t(p) * 27 + FACE_REGION[f]] != -1) continue;
          int d = f / 2, ff = (f & 1) ? NI : 0;
          T *R = reg(Rf, p, f);
          for (int v = 0; v < nv; ++v)
            for (int cb = 0; cb < 8; ++cb)
              for (int ca = 0; ca < 8; ++ca) {
                T s = (F[d][fidx(v, 2 * cb, 2 * ca, ff)] + F[d][fidx(v, 2 * cb, 2 * ca + 1, ff)]) +
                      (F[d][fidx(v, 2 * cb + 1, 2 * ca, ff)] + F[d][fidx(v, 2 * cb + 1, 2 * ca + 1, ff)]);
                R[(size_t(v) * 8 + cb) * 8 + ca] += wdt * (T(0.25) * s);
              }
        }
      // S10 coarse side: the coarse faces under each child's coarse-fine faces
      for (int o = 0; o < 8; ++o) {
        int ch = child[p][o];
        if (ch < 0) continue;
        int oc[3] = {o & 1, (o >> 1) & 1, (o >> 2) & 1};
        for (int f = 0; f < 6; ++f) {
          if (nbr[size_t(ch) * 27 + FACE_REGION[f]] != -1) continue;
          int d = f / 2, ff = 8 * oc[d] + ((f & 1) ? 8 : 0);
          int d1 = (d == 0) ? 1 : 0, d2 = (d == 2) ? 1 : 2;     // transverse axes, t1 faster
          T *R = reg(Rc, ch, f);
          for (int v = 0; v < nv; ++v)
            for (int cb = 0; cb < 8; ++cb)
              for (int ca = 0; ca < 8; ++ca)
                R[(size_t(v) * 8 + cb) * 8 + ca] += wdt * F[d][fidx(v, 8 * oc[d2] + cb, 8 * oc[d1] + ca, ff)];
        }
      }
    });
  }

  // ---- O7 / S8: restriction, coarse cell = mean of its 8 fine cells
  void restrict_level(int fine_lev, int fslot, int cslot) {
    const auto &lp = lev_patches[fine_lev];
    parallel_for((int)lp.size(), [&](int n, Phys<T> &) {
      int p = lp[n], Q = parent[p], o = octant[p];
      int oc[3] = {o & 1, (o >> 1) & 1, (o >> 2) & 1};
      const T *Uf = P(fslot, p);
      T *Ucs = P(cslot, Q);
      for (int v = 0; v < nv; ++v)
        for (int ck = 0; ck < 8; ++ck)
          for (int cj = 0; cj < 8; ++cj)
            for (int ci = 0; ci < 8; ++ci) {
              // pairwise tree (x pairs, then y, then z): exact for 8 equal values, so a
              // uniform state is restricted bitwise (pin P5/P12)
              auto f = [&](int dk, int dj, int di) {
                return Uf[size_t(v) * NC + cidx(NG + 2 * ck + dk, NG + 2 * cj + dj, NG + 2 * ci + di)];
              };
              T s = ((f(0, 0, 0) + f(0, 0, 1)) + (f(0, 1, 0) + f(0, 1, 1))) +
                    ((f(1, 0, 0) + f(1, 0, 1)) + (f(1, 1, 0) + f(1, 1, 1)));
              Ucs[size_t(v) * NC + cidx(NG + 8 * oc[2] + ck, NG + 8 * oc[1] + cj, NG + 8 * oc[0] + ci)] = T(0.125) * s;
            }
    });
  }

  // ---- O8 / S10: refluxing of the uncovered coarse cells next to fine patches.
  // Faces are processed in the fixed order f = 0..5, patches in table order.
  int reflux(int clev, int slot) {
    if (clev + 1 >= nlev) return 0;
    const auto &lp = lev_patches[clev + 1];
    const T hc = T(dx(clev));
    for (int f = 0; f < 6; ++f)
      for (int p : lp) {
        if (nbr[size_t(p) * 27 + FACE_REGION[f]] != -1) continue;
        int Q = parent[p], o = octant[p];
        int oc[3] = {o & 1, (o >> 1) & 1, (o >> 2) & 1};
        int d = f / 2, hi = f & 1;
        int d1 = (d == 0) ? 1 : 0, d2 = (d == 2) ? 1 : 2;
        int cn = NG + 8 * oc[d] + (hi ? 8 : -1);      // uncovered cell, parent padded index along d
        int tgt = Q;
        if (cn < NG || cn >= NG + NI) {               // it lives in the parent's neighbour
          tgt = nbr[size_t(Q) * 27 + FACE_REGION[f]];
          if (tgt < 0) return -1;                     // improper nesting
          cn += hi ? -NI : NI;
        }
        T *U = P(slot, tgt);
        T *rf = reg(Rf, p, f), *rc = reg(Rc, p, f);
        for (int v = 0; v < nv; ++v)
          for (int cb = 0; cb < 8; ++cb)
            for (int ca = 0; ca < 8; ++ca) {
              int pad[3];
              pad[d] = cn; pad[d1] = NG + 8 * oc[d1] + ca; pad[d2] = NG + 8 * oc[d2] + cb;
              size_t c = size_t(v) * NC + cidx(pad[2], pad[1], pad[0]);
              size_t r = (size_t(v) * 8 + cb) * 8 + ca;
              T corr = (rf[r] - rc[r]) / hc;
              if (hi) U[c] = U[c] + corr; else U[c] = U[c] - corr;
              rf[r] = T(0); rc[r] = T(0);
            }
      }
    return 0;
  }

  // S18: the damping of psi in the mixed GLM form of Dedner et al. (2002), psi_t = ... - (c_h^2/c_p^2) psi,
  // integrated exactly over one step of the level, operator-split after the step: psi *= factor.
  void glm_damp(int lev, int slot, double factor) {
    if (nv != 9) return;
    for (int p : lev_patches[lev]) {
      T *psi = P(slot, p) + size_t(8) * NC;
      for (int k = NG; k < NG + NI; ++k)
        for (int j = NG; j < NG + NI; ++j)
          for (int i = NG; i < NG + NI; ++i) psi[cidx(k, j, i)] = psi[cidx(k, j, i)] * T(factor);
    }
  }

  void copy_slot(int lev, int src, int dst) {
    for (int p : lev_patches[lev]) std::memcpy(P(dst, p), P(src, p), patch_stride() * sizeof(T));
  }

  // ---- O5 + O9 / S9: recursive subcycled advance.  Slots: 0 = A (U^n -> U^{n+1}),
  // 1 = B (U^(1)), 2 = C (U^n of a level with children, ghosts included).
  // a1, a2: time-interpolation weights of the parent data for the two ghost fills (S7).
  int advance(int lev, double dt, double a1, double a2) {
    bool kids = has_children(lev);
    double w = (nlev > 1) ? 0.5 : 0.0;
    fill_ghosts(lev, 0, 2, 0, a1);
    if (kids) copy_slot(lev, 0, 2);
    rk_stage(lev, 0, 0, 1, 0.0, 1.0, dt, w);             // U1 = Un + dt L(Un)
    fill_ghosts(lev, 1, 2, 0, a2);
    rk_stage(lev, 1, 0, 0, 0.5, 0.5, dt, w);             // Un+1 = 1/2 Un + 1/2 (U1 + dt L(U1))
    if (nv == 9 && ph.cr > T(0)) glm_damp(lev, 0, std::exp(-dt * double(ph.ch) / double(ph.cr)));
    if (kids) {
      fill_ghosts(lev, 0, 2, 0, a2);                     // new-time ghosts for the children's prolongation
      if (advance(lev + 1, 0.5 * dt, 0.0, 0.5)) return -1;
      if (advance(lev + 1, 0.5 * dt, 0.5, 1.0)) return -1;
      restrict_level(lev + 1, 0, 0);
      if (reflux(lev, 0)) return -1;
    }
    return 0;
  }

  double global_dt(double cfl) {                         // S4: dt0 = CFL dx0 / max_l S_max,l
    double s = 0.0;
    for (int l = 0; l < nlev; ++l) {
      if (lev_patches[l].empty()) continue;
      double sl = max_speed(l, 0);
      if (!(sl <= s)) s = sl;
    }
    return cfl * dx0 / s;
  }
};

struct Handle {
  int bits;
  Hier<double> *d = nullptr;
  Hier<float> *f = nullptr;
};

template <class T>
int set_hierarchy(Hier<T> &H, int np, int nlev, const int *level, const int *origin, const int *parent,
                  const int *nbr, double dx0, const int *bc, int nslots) {
  H.np = np; H.nlev = nlev; H.nslots = nslots; H.dx0 = dx0;
  for (int i = 0; i < 6; ++i) H.bc[i] = bc[i];
  H.level.assign(level, level + np);
  H.parent.assign(parent, parent + np);
  H.origin.assign(origin, origin + 3 * size_t(np));
  H.nbr.assign(nbr, nbr + 27 * size_t(np));
  H.octant.assign(np, 0);
  H.child.assign(np, std::array<int, 8>{-1, -1, -1, -1, -1, -1, -1, -1});
  H.lev_patches.assign(nlev, {});
  for (int p = 0; p < np; ++p) {
    if (level[p] < 0 || level[p] >= nlev) return -1;
    H.lev_patches[level[p]].push_back(p);
    if (level[p] > 0) {
      int Q = parent[p];
      if (Q < 0 || Q >= np || level[Q] != level[p] - 1) return -2;
      int o = 0;
      for (int d = 0; d < 3; ++d) {
        int rel = origin[3 * p + d] - 2 * origin[3 * Q + d];
        if (rel != 0 && rel != NI) return -3;
        if (rel == NI) o |= (1 << d);
      }
      H.octant[p] = o;
      H.child[Q][o] = p;
    }
  }
  H.pool.assign(size_t(nslots) * np * H.patch_stride(), T(0));
  H.Rf.assign(size_t(np) * 6 * H.nv * 64, T(0));
  H.Rc.assign(size_t(np) * 6 * H.nv * 64, T(0));
  return 0;
}

}  // namespace

#define DISPATCH(h, expr)                         \
  do {                                            \
    Handle *H_ = (Handle *)(h);                   \
    if (H_->bits == 64) { auto &H = *H_->d; expr; } \
    else { auto &H = *H_->f; expr; }              \
  } while (0)

extern "C" {

void *orc_create(int bits, double gamma, int nvars, double theta, double rho_floor, double e_floor) {
  if ((bits != 32 && bits != 64) || (nvars != 5 && nvars != 8 && nvars != 9)) return nullptr;
  Handle *h = new Handle;
  h->bits = bits;
  if (bits == 64) {
    h->d = new Hier<double>;
    h->d->nv = nvars;
    h->d->ph = Phys<double>{nvars, gamma, theta, rho_floor, e_floor, nullptr};
  } else {
    h->f = new Hier<float>;
    h->f->nv = nvars;
    h->f->ph = Phys<float>{nvars, float(gamma), float(theta), float(rho_floor), float(e_floor), nullptr};
  }
  return h;
}
void orc_destroy(void *h) { Handle *H = (Handle *)h; delete H->d; delete H->f; delete H; }
void orc_set_threads(void *h, int n) { DISPATCH(h, H.nthreads = n); }
void orc_set_theta(void *h, double th) { DISPATCH(h, H.ph.theta = decltype(H.ph.theta)(th)); }
void orc_set_glm(void *h, double ch, double cr) {
  DISPATCH(h, { H.ph.ch = decltype(H.ph.ch)(ch); H.ph.cr = decltype(H.ph.cr)(cr); });
}
int orc_glm_damp(void *h, int lev, int slot, double factor) { DISPATCH(h, H.glm_damp(lev, slot, factor)); return 0; }
long orc_floor_hits(void *h) { long r = 0; DISPATCH(h, r = H.floor_hits); return r; }

int orc_set_hierarchy(void *h, int np, int nlev, const int *level, const int *origin, const int *parent,
                      const int *nbr, double dx0, const int *bc, int nslots) {
  int r = 0;
  DISPATCH(h, r = set_hierarchy(H, np, nlev, level, origin, parent, nbr, dx0, bc, nslots));
  return r;
}
// interior [var][16][16][16] doubles in/out (converted to the oracle's T)
int orc_upload(void *h, int slot, int p, const double *in) {
  DISPATCH(h, {
    auto *U = H.P(slot, p);
    for (int v = 0; v < H.nv; ++v)
      for (int k = 0; k < NI; ++k) for (int j = 0; j < NI; ++j) for (int i = 0; i < NI; ++i)
        U[size_t(v) * NC + cidx(k + NG, j + NG, i + NG)] =
            (std::remove_reference_t<decltype(*U)>)in[((size_t(v) * NI + k) * NI + j) * NI + i];
  });
  return 0;
}
int orc_download(void *h, int slot, int p, double *out) {
  DISPATCH(h, {
    auto *U = H.P(slot, p);
    for (int v = 0; v < H.nv; ++v)
      for (int k = 0; k < NI; ++k) for (int j = 0; j < NI; ++j) for (int i = 0; i < NI; ++i)
        out[((size_t(v) * NI + k) * NI + j) * NI + i] = double(U[size_t(v) * NC + cidx(k + NG, j + NG, i + NG)]);
  });
  return 0;
}
// padded [var][20][20][20] doubles in/out (tests of the ghost fill)
int orc_upload_padded(void *h, int slot, int p, const double *in) {
  DISPATCH(h, { auto *U = H.P(slot, p); for (size_t c = 0; c < H.patch_stride(); ++c) U[c] = (std::remove_reference_t<decltype(*U)>)in[c]; });
  return 0;
}
int orc_download_padded(void *h, int slot, int p, double *out) {
  DISPATCH(h, { auto *U = H.P(slot, p); for (size_t c = 0; c < H.patch_stride(); ++c) out[c] = double(U[c]); });
  return 0;
}
int orc_download_registers(void *h, int p, double *rf, double *rc) {   // [6][var][8][8] each
  DISPATCH(h, {
    size_t n = size_t(6) * H.nv * 64;
    for (size_t c = 0; c < n; ++c) { rf[c] = double(H.Rf[size_t(p) * n + c]); rc[c] = double(H.Rc[size_t(p) * n + c]); }
  });
  return 0;
}
double orc_max_speed(void *h, int lev, int slot) { double r = 0; DISPATCH(h, r = H.max_speed(lev, slot)); return r; }
int orc_cfl_dt(void *h, int lev, int slot, double cfl, double *dt) {
  double s = orc_max_speed(h, lev, slot);
  if (!(s > 0.0) || !std::isfinite(s)) return -5;
  DISPATCH(h, *dt = cfl * H.dx(lev) / s);
  return 0;
}
int orc_fill_ghosts(void *h, int lev, int slot, int pold, int pnew, double alpha) {
  DISPATCH(h, H.fill_ghosts(lev, slot, pold, pnew, alpha));
  return 0;
}
int orc_rk_stage(void *h, int lev, int sin, int sbase, int sout, double a, double b, double dt, double w) {
  if (sin == sout) return -1;
  DISPATCH(h, H.rk_stage(lev, sin, sbase, sout, a, b, dt, w));
  return 0;
}
int orc_restrict(void *h, int flev, int fslot, int cslot) { DISPATCH(h, H.restrict_level(flev, fslot, cslot)); return 0; }
int orc_reflux(void *h, int clev, int slot) { int r = 0; DISPATCH(h, r = H.reflux(clev, slot)); return r; }
int orc_refine_indicator(void *h, int lev, int slot, double *out) { DISPATCH(h, H.refine_indicator(lev, slot, out)); return 0; }
int orc_prolong_interior(void *h, int p, int slot, int pslot) {
  int r = 0;
  DISPATCH(h, { if (p < 0 || p >= H.np || H.level[p] == 0) r = -1; else H.prolong_interior(p, slot, pslot); });
  return r;
}
int orc_copy_slot(void *h, int lev, int src, int dst) { DISPATCH(h, H.copy_slot(lev, src, dst)); return 0; }
// one coarse step of the whole hierarchy (O5 when nlev == 1); returns dt0 used
int orc_advance(void *h, double cfl, double dt_fixed, double *dt_out) {
  int r = 0;
  DISPATCH(h, {
    double dt = dt_fixed > 0.0 ? dt_fixed : H.global_dt(cfl);
    if (!(dt > 0.0) || !std::isfinite(dt)) return -5;
    *dt_out = dt;
    r = H.advance(0, dt, 0.0, 0.0);
  });
  return r;
}

// ---- single-face helpers for the pins (P1, P2, P8): double precision only
double orc_minmod(double a, double b, double c) { return minmod3(a, b, c); }
double orc_face(int nvars, double gamma, double theta, int dir, const double *Wm2, const double *Wm1,
                const double *W0, const double *Wp1, double *WL, double *WR, double *F) {
  Phys<double> q{nvars, gamma, theta, 1e-300, 1e-300, nullptr};
  q.plm(Wm2, Wm1, W0, Wp1, WL, WR);
  return q.riemann(WL, WR, dir, F);
}
// the same two helpers with the floors of S11 given by the caller and their activations counted (pin P20:
// tests/test_oracle_pins.py drives states below the floors through them); no arithmetic of their own
double orc_face_floors(int nvars, double gamma, double theta, int dir, double rho_floor, double e_floor, const double *Wm2,
                       const double *Wm1, const double *W0, const double *Wp1, double *WL, double *WR, double *F,
                       long *hits) {
  Phys<double> q{nvars, gamma, theta, rho_floor, e_floor, hits};
  q.plm(Wm2, Wm1, W0, Wp1, WL, WR);
  return q.riemann(WL, WR, dir, F);
}
void orc_prim_floors(int nvars, double gamma, double rho_floor, double e_floor, const double *U, double *W, long *hits) {
  Phys<double> q{nvars, gamma, 1.5, rho_floor, e_floor, hits};
  q.prim(U, W);
}
void orc_prim(int nvars, double gamma, const double *U, double *W) {
  Phys<double> q{nvars, gamma, 1.5, 1e-300, 1e-300, nullptr};
  q.prim(U, W);
}
void orc_flux(int nvars, double gamma, int dir, const double *W, double *U, double *F, double *c) {
  Phys<double> q{nvars, gamma, 1.5, 1e-300, 1e-300, nullptr};
  q.cons(W, U); q.flux(W, dir, F); *c = q.speed(W, dir);
}
// the same for the 9-variable system with its c_h; face flux of Eq. 12 from two given states
void orc_flux_glm(double gamma, double ch, int dir, const double *W, double *U, double *F) {
  Phys<double> q{9, gamma, 1.5, 1e-300, 1e-300, nullptr};
  q.ch = ch;
  q.cons(W, U); q.flux(W, dir, F);
}
double orc_riemann_glm(double gamma, double ch, int dir, const double *WL, const double *WR, double *F) {
  Phys<double> q{9, gamma, 1.5, 1e-300, 1e-300, nullptr};
  q.ch = ch;
  return q.riemann(WL, WR, dir, F);
}
}  // extern "C"
