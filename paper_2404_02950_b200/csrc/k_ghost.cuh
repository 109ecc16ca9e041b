// k_ghost.cuh -- K2: ghost fill of one stage buffer of one level.
//
// One thread per ghost cell.  For the ghost cell at unwrapped level index f:
//   * wrap f periodically (L23); if a box of the same level owns the wrapped cell, copy its VALID value
//     (same-level copy wins over interpolation, R9);
//   * else (level > 0) trilinear interpolation of the coarse state, itself linearly interpolated in time
//     between the coarse level's old and new states: c = (1-alpha) c_old + alpha c_new (L70-72).
//     f = 2c + r sits -1/4 (r = 0) or +1/4 (r = 1) of a coarse cell from the centre of c: per-axis weights
//     3/4 on c and 1/4 on c-1 (r = 0) or c+1 (r = 1).  Only VALID coarse cells are read, found through the
//     coarse owner table (their existence is what proper nesting guarantees, L70).
// Only valid cells are read and only ghost cells are written, so one launch per level has no hazards.
//
// Work distribution: the ghost shell of a box is cut into three slab pairs (z-low/high: full ghosted
// xy-planes; y-low/high: full ghosted x-rows; x-low/high), enumerated x-fastest so that the wide slabs are
// written with coalesced rows.  A prefix table over boxes (in CTAs) maps blockIdx.x -> box by bisection.
#pragma once
#include "layout.h"

namespace sledge {

constexpr int GHOST_THREADS = 256;

template <typename T>
struct GhostArgs {
  using P = typename PairOf<T>::type;
  const BoxDev* boxes;
  const int* blk_prefix;  // nbox + 1 entries, CTAs before box b
  int nbox;
  P* psi;
  P* pi;             // used only when FILL_PI
  const int* owner;  // this level's owner grid (box index or -1), granularity = blocking factor
  LevelGeom geom;
  // next coarser level (level > 0 only)
  const BoxDev* cboxes;
  const int* cowner;
  LevelGeom cgeom;
  const P* c_old_psi;
  const P* c_new_psi;
  const P* c_old_pi;
  const P* c_new_pi;
  T alpha;
  int has_coarse;
  int* err_flag;  // set to 1 if a ghost cell has neither a same-level owner nor coarse data
};

__device__ __forceinline__ long long cell_offset(const BoxDev& b, int g, int ox, int i, int j, int k) {
  return b.base + ((long long)(k + g) * b.sy + (j + g)) * b.sx + (i + ox);
}

__device__ __forceinline__ int owner_lookup(const int* owner, const LevelGeom& gm, int wi, int wj, int wk) {
  return owner[((long long)(wk >> gm.bf_shift) * gm.no[1] + (wj >> gm.bf_shift)) * gm.no[0] + (wi >> gm.bf_shift)];
}

template <typename T>
__device__ __forceinline__ typename PairOf<T>::type interp_coarse(
    const typename PairOf<T>::type* c_old, const typename PairOf<T>::type* c_new, const BoxDev* cboxes,
    const int* cowner, const LevelGeom& cg, T alpha, const int c0[3], const int c1[3], bool& ok) {
  using P = typename PairOf<T>::type;
  const T w[2] = {T(0.75), T(0.25)};
  const T oma = T(1) - alpha;
  T s0 = T(0), s1 = T(0);
#pragma unroll
  for (int dz = 0; dz < 2; ++dz)
#pragma unroll
    for (int dy = 0; dy < 2; ++dy)
#pragma unroll
      for (int dx = 0; dx < 2; ++dx) {
        const int ci = wrap_idx(dx ? c1[0] : c0[0], cg.n[0]);
        const int cj = wrap_idx(dy ? c1[1] : c0[1], cg.n[1]);
        const int ck = wrap_idx(dz ? c1[2] : c0[2], cg.n[2]);
        const int ow = owner_lookup(cowner, cg, ci, cj, ck);
        if (ow < 0) {
          ok = false;
          continue;
        }
        const BoxDev cb = cboxes[ow];
        const long long o = cell_offset(cb, cg.g, cg.ox, ci - cb.lo[0], cj - cb.lo[1], ck - cb.lo[2]);
        const P vo = c_old[o];
        const P vn = c_new[o];
        const T cv0 = oma * vo.x + alpha * vn.x;
        const T cv1 = oma * vo.y + alpha * vn.y;
        const T wt = (w[dz] * w[dy]) * w[dx];
        s0 += wt * cv0;
        s1 += wt * cv1;
      }
  return mkpair(s0, s1);
}

template <typename T, bool FILL_PI>
__global__ void __launch_bounds__(GHOST_THREADS) k_fill_ghosts(const GhostArgs<T> a) {
  using P = typename PairOf<T>::type;
  // blockIdx.x -> box
  int lo_b = 0, hi_b = a.nbox;
  const int blk = blockIdx.x;
  while (hi_b - lo_b > 1) {
    const int mid = (lo_b + hi_b) >> 1;
    if (a.blk_prefix[mid] <= blk) lo_b = mid; else hi_b = mid;
  }
  const BoxDev b = a.boxes[lo_b];
  const int g = a.geom.g;
  const int nx = b.n[0], ny = b.n[1], nz = b.n[2];
  const int Gx = nx + 2 * g, Gy = ny + 2 * g;
  const long long nA = (long long)Gx * Gy * (2 * g);  // z slabs
  const long long nB = (long long)Gx * (2 * g) * nz;  // y slabs
  const long long nC = (long long)(2 * g) * ny * nz;  // x slabs
  const long long q = (long long)(blk - a.blk_prefix[lo_b]) * GHOST_THREADS + threadIdx.x;
  if (q >= nA + nB + nC) return;
  int i, j, k;
  if (q < nA) {
    const int zz = (int)(q / ((long long)Gx * Gy));
    const int r = (int)(q - (long long)zz * Gx * Gy);
    j = r / Gx - g;
    i = r % Gx - g;
    k = zz < g ? zz - g : nz + (zz - g);
  } else if (q < nA + nB) {
    const long long p = q - nA;
    const int rowlen = Gx * 2 * g;
    k = (int)(p / rowlen);
    const int r = (int)(p - (long long)k * rowlen);
    const int yy = r / Gx;
    i = r % Gx - g;
    j = yy < g ? yy - g : ny + (yy - g);
  } else {
    const long long p = q - nA - nB;
    const int rowlen = 2 * g * ny;
    k = (int)(p / rowlen);
    const int r = (int)(p - (long long)k * rowlen);
    j = r / (2 * g);
    const int xx = r % (2 * g);
    i = xx < g ? xx - g : nx + (xx - g);
  }
  const int f0 = b.lo[0] + i, f1 = b.lo[1] + j, f2 = b.lo[2] + k;  // unwrapped level index
  const int wi = wrap_idx(f0, a.geom.n[0]), wj = wrap_idx(f1, a.geom.n[1]), wk = wrap_idx(f2, a.geom.n[2]);
  const long long dst = cell_offset(b, g, a.geom.ox, i, j, k);
  const int ow = owner_lookup(a.owner, a.geom, wi, wj, wk);
  if (ow >= 0) {
    const BoxDev sb = a.boxes[ow];
    const long long src = cell_offset(sb, g, a.geom.ox, wi - sb.lo[0], wj - sb.lo[1], wk - sb.lo[2]);
    a.psi[dst] = a.psi[src];
    if (FILL_PI) a.pi[dst] = a.pi[src];
    return;
  }
  if (!a.has_coarse) {
    *a.err_flag = 1;
    return;
  }
  int c0[3], c1[3];
  const int f[3] = {f0, f1, f2};
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    c0[d] = floordiv2(f[d]);
    const int r = f[d] - 2 * c0[d];
    c1[d] = r == 0 ? c0[d] - 1 : c0[d] + 1;
  }
  bool ok = true;
  a.psi[dst] = interp_coarse<T>(a.c_old_psi, a.c_new_psi, a.cboxes, a.cowner, a.cgeom, a.alpha, c0, c1, ok);
  if (FILL_PI)
    a.pi[dst] = interp_coarse<T>(a.c_old_pi, a.c_new_pi, a.cboxes, a.cowner, a.cgeom, a.alpha, c0, c1, ok);
  if (!ok) *a.err_flag = 1;
}

}  // namespace sledge
