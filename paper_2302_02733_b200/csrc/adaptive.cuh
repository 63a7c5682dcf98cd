// Adaptive ray tracing ("adaptive ray tracing which reduces the number of light rays to follow"; SURVEY.md
// 8(f)-3; reading R-11 in DESIGN.md).  The per-ray kernels are reused unchanged: these kernels only choose which pixels
// are traced at each lattice level, interpolate the others and decide where to refine.
//
//   lattice of level l (stride s_l = 2^(L-l)): pixel indices {0, s_l, 2 s_l, ...} and n-1, in x and y; a cell is the
//   rectangle between consecutive lines.  Level 0: all lattice points traced, all cells flagged.  Level l >= 1: a new
//   lattice point is traced if a level-(l-1) cell containing it is flagged, else it takes the bilinear interpolation
//   of that cell's corners; a flagged level-(l-1) cell P needs refinement if |S_k(p) - B_P,k(p)| > rel_tol |I(p)| +
//   abs_tol for some new point p in it and some Stokes parameter k, or if it has no new point at this level (narrower
//   than the stride both ways: the flag is carried down); its level-l cells are flagged iff it does.
//
// Arrays are indexed by flat pixel j*nx+i; a cell's flag lives at its lower-left corner pixel.
#pragma once
#include <stdint.h>

namespace ipole {

struct AdaArgs {
  int nx, ny;
  int s;                      // stride of this level; the parent level has stride 2 s
  double rel_tol, abs_tol;
  double* img[4];             // I, Q, U, V planes [ny][nx]
  uint8_t* state;             // 0 unknown, 1 traced, 2 interpolated
  const uint8_t* flag_prev;   // flags of the level-(l-1) cells
  uint8_t* flag_cur;          // flags of the level-l cells (cleared by the host before k_ada_flag)
  int64_t* list; int* count;  // pixels to trace at this level
  const double* val[4];       // traced values of the list entries (k_ada_scatter)
};

__device__ __forceinline__ bool ada_on_line(int i, int n, int s) { return (i % s) == 0 || i == n - 1; }
__device__ __forceinline__ int ada_floor_line(int i, int n, int s) { return (i == n - 1) ? n - 1 : (i / s) * s; }
__device__ __forceinline__ int ada_next_line(int a, int n, int s) { return min(a + s, n - 1); }
__device__ __forceinline__ int ada_prev_line(int i, int n, int s) { return (i == n - 1) ? ((n - 2) / s) * s : i - s; }

// bilinear interpolant of the corners (i0|i1, j0|j1) at (i, j); products and sums rounded one by one, in the oracle's
// order, so that equal corner values give equal bits
__device__ __forceinline__ double ada_bilinear(const double* p, int nx, int i0, int i1, int j0, int j1, int i, int j) {
  const double t = (i1 > i0) ? (double)(i - i0) / (double)(i1 - i0) : 0.0;
  const double u = (j1 > j0) ? (double)(j - j0) / (double)(j1 - j0) : 0.0;
  const double w00 = __dmul_rn(1.0 - t, 1.0 - u), w10 = __dmul_rn(t, 1.0 - u), w01 = __dmul_rn(1.0 - t, u), w11 = __dmul_rn(t, u);
  const double a = p[(size_t)j0 * nx + i0], b = p[(size_t)j0 * nx + i1], c = p[(size_t)j1 * nx + i0], d = p[(size_t)j1 * nx + i1];
  return __dadd_rn(__dadd_rn(__dadd_rn(__dmul_rn(w00, a), __dmul_rn(w10, b)), __dmul_rn(w01, c)), __dmul_rn(w11, d));
}

// levels 0 and 1 in one go (both are traced everywhere, so one launch of the per-ray kernels serves them): list every
// level-1 lattice point (stride A.s), flag every level-0 cell (stride s0 = 2 A.s)
__global__ void k_ada_level01(AdaArgs A, uint8_t* flag0, int s0) {
  const int64_t n = (int64_t)A.nx * A.ny;
  for (int64_t p = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; p < n; p += (int64_t)gridDim.x * blockDim.x) {
    const int i = (int)(p % A.nx), j = (int)(p / A.nx);
    A.state[p] = 0;
    flag0[p] = ((i % s0) == 0 && (j % s0) == 0 && i < A.nx - 1 && j < A.ny - 1) ? 1 : 0;
    if (ada_on_line(i, A.nx, A.s) && ada_on_line(j, A.ny, A.s)) A.list[atomicAdd(A.count, 1)] = p;
  }
}

// level l: new lattice points are listed for tracing or interpolated from the parent cell
__global__ void k_ada_select(AdaArgs A) {
  const int64_t n = (int64_t)A.nx * A.ny;
  const int s = A.s, ps = 2 * A.s;
  for (int64_t p = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; p < n; p += (int64_t)gridDim.x * blockDim.x) {
    const int i = (int)(p % A.nx), j = (int)(p / A.nx);
    if (!(ada_on_line(i, A.nx, s) && ada_on_line(j, A.ny, s))) continue;
    const bool xl = ada_on_line(i, A.nx, ps), yl = ada_on_line(j, A.ny, ps);
    if (xl && yl) continue;   // a point of the parent lattice: known already
    // lower-left corners of the parent cells whose closed rectangle contains (i, j)
    int xa[2], ya[2], nxa = 0, nya = 0;
    if (xl) { if (i > 0) xa[nxa++] = ada_prev_line(i, A.nx, ps); if (i < A.nx - 1) xa[nxa++] = i; }
    else xa[nxa++] = ada_floor_line(i, A.nx, ps);
    if (yl) { if (j > 0) ya[nya++] = ada_prev_line(j, A.ny, ps); if (j < A.ny - 1) ya[nya++] = j; }
    else ya[nya++] = ada_floor_line(j, A.ny, ps);
    bool flagged = false;
    for (int a = 0; a < nxa; ++a) for (int b = 0; b < nya; ++b) flagged |= A.flag_prev[(size_t)ya[b] * A.nx + xa[a]] != 0;
    if (flagged) { A.list[atomicAdd(A.count, 1)] = p; continue; }
    // the cell to the right / above when there are two
    const int i0 = xa[nxa - 1], j0 = ya[nya - 1];
    const int i1 = ada_next_line(i0, A.nx, ps), j1 = ada_next_line(j0, A.ny, ps);
#pragma unroll
    for (int k = 0; k < 4; ++k) A.img[k][p] = ada_bilinear(A.img[k], A.nx, i0, i1, j0, j1, i, j);
    A.state[p] = 2;
  }
}

__global__ void k_ada_scatter(AdaArgs A, int n_list) {
  for (int q = blockIdx.x * blockDim.x + threadIdx.x; q < n_list; q += gridDim.x * blockDim.x) {
    const int64_t p = A.list[q];
#pragma unroll
    for (int k = 0; k < 4; ++k) A.img[k][p] = A.val[k][q];
    A.state[p] = 1;
  }
}

// level l: every flagged parent cell compares its new points with its own bilinear interpolant
__global__ void k_ada_flag(AdaArgs A) {
  const int64_t n = (int64_t)A.nx * A.ny;
  const int s = A.s, ps = 2 * A.s;
  for (int64_t p = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; p < n; p += (int64_t)gridDim.x * blockDim.x) {
    const int i0 = (int)(p % A.nx), j0 = (int)(p / A.nx);
    if (i0 >= A.nx - 1 || j0 >= A.ny - 1 || (i0 % ps) != 0 || (j0 % ps) != 0) continue;   // not a parent cell's corner
    if (!A.flag_prev[p]) continue;
    const int i1 = ada_next_line(i0, A.nx, ps), j1 = ada_next_line(j0, A.ny, ps);
    int xs[3], ys[3], nxs = 0, nys = 0;
    xs[nxs++] = i0; if (i0 + s < i1) xs[nxs++] = i0 + s; xs[nxs++] = i1;
    ys[nys++] = j0; if (j0 + s < j1) ys[nys++] = j0 + s; ys[nys++] = j1;
    bool refine = (nxs == 2 && nys == 2);   // no new point in this cell: its flag is carried down
    for (int b = 0; b < nys; ++b)
      for (int a = 0; a < nxs; ++a) {
        const int i = xs[a], j = ys[b];
        if ((i == i0 || i == i1) && (j == j0 || j == j1)) continue;   // a corner of the cell
        const size_t q = (size_t)j * A.nx + i;
        const double lim = __dadd_rn(__dmul_rn(A.rel_tol, fabs(A.img[0][q])), A.abs_tol);
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          const double bl = ada_bilinear(A.img[k], A.nx, i0, i1, j0, j1, i, j);
          refine |= fabs(__dadd_rn(A.img[k][q], -bl)) > lim;
        }
      }
    if (refine)
      for (int b = 0; b + 1 < nys; ++b) for (int a = 0; a + 1 < nxs; ++a) A.flag_cur[(size_t)ys[b] * A.nx + xs[a]] = 1;
  }
}

}  // namespace ipole
