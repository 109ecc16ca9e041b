// k_tag.cuh -- K3: string tagging + per-32^3-block flag reduction.
//
// The paper only gives the bool-per-cell hook TagCellForRefinement; the winding rule
// is DESIGN.md reading R8: for cell P and (d1,d2) in {(x,y),(y,z),(z,x)} take the plaquette
// A=P, B=P+e_d1, C=P+e_d1+e_d2, D=P+e_d2 and count signed crossings of the positive psi1 axis along
// A->B->C->D->A.  Edge a->b: up = a2<0 && b2>=0, dn = a2>=0 && b2<0, cr = a1*b2 - a2*b1 with both products
// and the difference individually rounded (no FMA); +1 if up && cr>0, -1 if dn && cr<0.
// tag bit0/1/2 = winding(xy / yz / zx) != 0.  Per aligned 32^3 block of the level index space: number of
// cells with tag != 0 (tagging statistics, L776).
//
// Mapping: a warp owns 32 consecutive x cells of one row and marches along z; a CTA is TAG_TY such rows.
// Every thread loads its own cell (x,y) and (x,y+1) of each new plane; the +x neighbours come from the
// next lane by shuffle (lane 31 loads them).  The previous plane stays in registers, so each psi value is
// fetched from L1/L2 at most twice and from HBM once.  Counts: ballot + popc per plane, accumulated per
// warp across the march and flushed with one atomicAdd whenever the warp leaves a 32-block in z.
#pragma once
#include "layout.h"

namespace sledge {

constexpr int TAG_TX = 32;
constexpr int TAG_TY = 8;

template <typename T>
struct TagArgs {
  using P = typename PairOf<T>::type;
  const BoxDev* boxes;
  const TileDev* tiles;
  const P* psi;
  uint8_t* tags;     // may be null
  uint32_t* counts;  // may be null
  int g, ox;
  int nb0, nb1;  // count blocks per axis (x, y)
};

template <typename T>
__device__ __forceinline__ int edge_cross(T a1, T a2, T b1, T b2);
template <>
__device__ __forceinline__ int edge_cross<double>(double a1, double a2, double b1, double b2) {
  const bool up = (a2 < 0.0) && (b2 >= 0.0);
  const bool dn = (a2 >= 0.0) && (b2 < 0.0);
  const double cr = __dsub_rn(__dmul_rn(a1, b2), __dmul_rn(a2, b1));
  return (up && cr > 0.0) ? 1 : ((dn && cr < 0.0) ? -1 : 0);
}
template <>
__device__ __forceinline__ int edge_cross<float>(float a1, float a2, float b1, float b2) {
  const bool up = (a2 < 0.f) && (b2 >= 0.f);
  const bool dn = (a2 >= 0.f) && (b2 < 0.f);
  const float cr = __fsub_rn(__fmul_rn(a1, b2), __fmul_rn(a2, b1));
  return (up && cr > 0.f) ? 1 : ((dn && cr < 0.f) ? -1 : 0);
}

template <typename T, typename P>
__device__ __forceinline__ int winding(const P& A, const P& B, const P& C, const P& D) {
  return edge_cross<T>(A.x, A.y, B.x, B.y) + edge_cross<T>(B.x, B.y, C.x, C.y) + edge_cross<T>(C.x, C.y, D.x, D.y) +
         edge_cross<T>(D.x, D.y, A.x, A.y);
}

template <typename P>
__device__ __forceinline__ P shfl_down_pair(const P& v, int delta);
template <>
__device__ __forceinline__ double2 shfl_down_pair<double2>(const double2& v, int delta) {
  return make_double2(__shfl_down_sync(0xffffffffu, v.x, delta), __shfl_down_sync(0xffffffffu, v.y, delta));
}
template <>
__device__ __forceinline__ float2 shfl_down_pair<float2>(const float2& v, int delta) {
  return make_float2(__shfl_down_sync(0xffffffffu, v.x, delta), __shfl_down_sync(0xffffffffu, v.y, delta));
}

template <typename T>
__global__ void __launch_bounds__(TAG_TX* TAG_TY) k_tag_strings(const TagArgs<T> a) {
  using P = typename PairOf<T>::type;
  const TileDev t = a.tiles[blockIdx.x];
  const BoxDev b = a.boxes[t.box];
  const int lane = threadIdx.x % TAG_TX, ty = threadIdx.x / TAG_TX;
  const int x = t.x0 + lane, y = t.y0 + ty;
  if (y >= b.n[1]) return;  // whole warp leaves together (a warp is one row)
  // lanes past the box edge clamp to the last valid cell: they load valid memory and write nothing
  const bool act = x < b.n[0];
  const int xc = act ? x : b.n[0] - 1;
  const bool edge = (lane == TAG_TX - 1) || (x == b.n[0] - 1);  // must load its own +x neighbour
  const long long plane = (long long)b.sx * b.sy;
  long long off = b.base + ((long long)(t.z0 + a.g) * b.sy + (y + a.g)) * b.sx + (xc + a.ox);

  auto load_plane = [&](long long o, P& c00, P& c10, P& c01, P& c11) {
    c00 = __ldg(a.psi + o);
    c01 = __ldg(a.psi + o + b.sx);
    P e0 = c00, e1 = c01;
    if (edge) {
      e0 = __ldg(a.psi + o + 1);
      e1 = __ldg(a.psi + o + b.sx + 1);
    }
    c10 = shfl_down_pair<P>(c00, 1);
    c11 = shfl_down_pair<P>(c01, 1);
    if (edge) {
      c10 = e0;
      c11 = e1;
    }
  };

  P c00, c10, c01, c11;  // plane k:   (x,y) (x+1,y) (x,y+1) (x+1,y+1)
  load_plane(off, c00, c10, c01, c11);

  const int gx = b.lo[0] + xc, gy = b.lo[1] + y;
  const int bi = gx >> 5, bj = gy >> 5;
  const int bi0 = __shfl_sync(0xffffffffu, bi, 0);
  int cnt0 = 0, cnt1 = 0;  // tagged cells in x-block bi0 / bi0+1 (a warp can straddle two when lo % 32 != 0)
  int cur_bk = (b.lo[2] + t.z0) >> 5;
  auto flush = [&](int bk) {
    if (a.counts && lane == 0) {
      if (cnt0) atomicAdd(a.counts + ((long long)bk * a.nb1 + bj) * a.nb0 + bi0, (uint32_t)cnt0);
      if (cnt1) atomicAdd(a.counts + ((long long)bk * a.nb1 + bj) * a.nb0 + bi0 + 1, (uint32_t)cnt1);
    }
    cnt0 = cnt1 = 0;
  };

  for (int zz = 0; zz < t.nz; ++zz) {
    const int z = t.z0 + zz;
    P n00, n10, n01, n11;  // plane k+1
    load_plane(off + plane, n00, n10, n01, n11);
    const int wxy = winding<T, P>(c00, c10, c11, c01);  // A=P, B=P+x, C=P+x+y, D=P+y
    const int wyz = winding<T, P>(c00, c01, n01, n00);  // A=P, B=P+y, C=P+y+z, D=P+z
    const int wzx = winding<T, P>(c00, n00, n10, c10);  // A=P, B=P+z, C=P+z+x, D=P+x
    const uint8_t tag = (uint8_t)((wxy != 0 ? 1 : 0) | (wyz != 0 ? 2 : 0) | (wzx != 0 ? 4 : 0));
    if (a.tags && act) a.tags[b.tag_base + ((long long)z * b.n[1] + y) * b.n[0] + x] = tag;
    const int bk = (b.lo[2] + z) >> 5;
    if (bk != cur_bk) {
      flush(cur_bk);
      cur_bk = bk;
    }
    const bool hit = act && tag != 0;
    cnt0 += __popc(__ballot_sync(0xffffffffu, hit && bi == bi0));
    cnt1 += __popc(__ballot_sync(0xffffffffu, hit && bi != bi0));
    c00 = n00;
    c10 = n10;
    c01 = n01;
    c11 = n11;
    off += plane;
  }
  flush(cur_bk);
}

}  // namespace sledge
