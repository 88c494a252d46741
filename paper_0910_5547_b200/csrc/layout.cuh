// layout.cuh -- private HBM layout of the patch pool (sm_100a build).
//
// pool[slot][patch][var][VS] ; inside a var block the padded 20x20x20 box (2 ghost + 16
// interior + 2 ghost per axis, PAPER.md:104 / BASELINE.json north_star) is stored x-fastest
// with an x pitch PX and a lead pad LEAD chosen so that every interior row of 16 cells starts
// on a 32-byte DRAM sector boundary:
//   fp64: PX = 20 (160 B rows), LEAD = 2  -> interior row = bytes [32,160) of its row group
//   fp32: PX = 24 ( 96 B rows), LEAD = 6  -> interior row = bytes [32, 96)
// so interior loads/stores touch only whole sectors and the ghost cells of consecutive rows
// share "ghost-only" sectors.  VS is rounded up to a multiple of 128 bytes.
#pragma once
#include <cstddef>
#include <cstdint>

namespace amr {

constexpr int NI = 16;            // interior cells per side
constexpr int NG = 2;             // ghost zones per side
constexpr int NP = NI + 2 * NG;   // 20
// index of the face-neighbour block in the 27-entry table: x-lo x-hi y-lo y-hi z-lo z-hi
__host__ __device__ __forceinline__ int face_region(int f) {
  const int d = f >> 1, st = d == 0 ? 1 : (d == 1 ? 3 : 9);
  return 13 + ((f & 1) ? st : -st);
}

template <typename T> struct Layout;
template <> struct Layout<double> {
  static constexpr int PX = 20, LEAD = 2;
  static constexpr int PLANE = PX * NP;
  static constexpr int VS = ((LEAD + PLANE * NP + 15) / 16) * 16;   // 8016 elements
};
template <> struct Layout<float> {
  static constexpr int PX = 24, LEAD = 6;
  static constexpr int PLANE = PX * NP;
  static constexpr int VS = ((LEAD + PLANE * NP + 31) / 32) * 32;   // 9632 elements
};

template <typename T> __host__ __device__ __forceinline__ int cell(int k, int j, int i) {
  return Layout<T>::LEAD + (k * NP + j) * Layout<T>::PX + i;
}

// 128-byte descriptor row as declared in include/amrhydro.h (kept in sync by a static_assert
// in amrhydro.cu); plus the derived child table.
struct Desc {
  int level;
  int origin[3];
  int parent;
  int nbr[27];
};

// Time step of a launch when it lives in device memory (CUDA-graph replay of the subcycled step: the graph's kernel
// arguments are frozen, the step size is not): dt = dt0[0] * pow2 with pow2 = 2^-level exactly, i.e. bitwise the value the
// host recursion dt/2 hands down.  p == nullptr: the launch carries dt as a plain argument.
struct DtDev {
  const double *p;
  double pow2;
  double hx;       // cell width of the level (rk_stage: dt/dx is formed as on the host, (dt0 * pow2) / hx)
};

template <typename T> struct Pool {
  T *base;
  int max_patches;
  int nv;
  __host__ __device__ __forceinline__ T *patch(int slot, int p) const {
    return base + (size_t(slot) * max_patches + p) * size_t(nv) * Layout<T>::VS;
  }
};

}  // namespace amr
