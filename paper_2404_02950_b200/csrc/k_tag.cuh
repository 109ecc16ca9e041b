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
// Mapping (edge form).  The contribution E(a->b) of an edge is antisymmetric bit for bit: the reversed edge
// swaps up/dn and negates cr exactly (same two rounded products, x - y = -(y - x) in IEEE), so
//   W_xy(P) = Ex(P) + Ey(P+x) - Ex(P+y) - Ey(P)      Ex/Ey/Ez(P) = E(P -> P+e_x / e_y / e_z)
//   W_yz(P) = Ey(P) + Ez(P+y) - Ey(P+z) - Ez(P)
//   W_zx(P) = Ez(P) + Ex(P+z) - Ez(P+x) - Ex(P)
// and only the edges that START at a cell are ever evaluated (3 cross products per cell instead of 12).
// A warp owns a 31 x TAG_RY patch of cells and marches along z without any block-level synchronisation: lane l
// holds the column x0+l of TAG_RY+1 rows (the last row and lane 31 are halo: they only supply edges), the
// plane below stays in registers, loads run TAG_PF planes ahead, psi(P+x) and the packed edges of P+x come from
// lane l+1 by shuffle.  Per plane and thread: Ex, Ez on TAG_RY+1 rows and Ey on TAG_RY rows (3.5 edges per cell
// for TAG_RY = 4).  Warps step by 31 cells in x so that every lane's +x partner is in the warp.
// Counts: per-thread counters, reduced over the warp (redux) and flushed with one atomicAdd per 32-block
// whenever the warp leaves a 32-block in z.
#pragma once
#include "layout.h"
#include "k_rk_pipe.cuh"  // cp.async helpers

namespace sledge {

constexpr int TAG_TX = 31;                 // cells per warp row that produce tags (lane 31 is the +x halo)
#ifndef SLEDGE_TAG_RY
#define SLEDGE_TAG_RY 4
#endif
constexpr int TAG_RY = SLEDGE_TAG_RY;                  // rows per warp
#ifndef SLEDGE_TAG_WARPS
#define SLEDGE_TAG_WARPS 4
#endif
constexpr int TAG_WARPS = SLEDGE_TAG_WARPS;               // warps per CTA, stacked in y
constexpr int TAG_TY = TAG_RY * TAG_WARPS; // rows per CTA tile
constexpr int TAG_THREADS = TAG_WARPS * 32;
template <typename T> constexpr size_t tag_smem_bytes();
#ifndef SLEDGE_TAG_PF
#define SLEDGE_TAG_PF 4
#endif
constexpr int TAG_PF = SLEDGE_TAG_PF;       // planes in flight per thread (cp.async ring depth)
static_assert(TAG_RY <= 32, "a warp's rows may straddle at most two 32-blocks");

template <typename T>
struct TagArgs {
  using P = typename PairOf<T>::type;
  const BoxDev* boxes;
  const TileDev* tiles;
  const P* psi;
  uint8_t* tags;     // may be null
  uint32_t* counts;  // may be null
  int g, ox;
  int wrap;      // the level is ONE box covering the periodic domain: +1 neighbours past the box edge are read at
                 // their wrapped position instead of from the ghost layer (L23), no ghost fill needed
  int nb0, nb1;  // count blocks per axis (x, y)
};

// individually rounded a1*b2 - a2*b1 (R8: no FMA)
__device__ __forceinline__ double cross_rn(double a1, double a2, double b1, double b2) {
  return __dsub_rn(__dmul_rn(a1, b2), __dmul_rn(a2, b1));
}
__device__ __forceinline__ float cross_rn(float a1, float a2, float b1, float b2) {
  return __fsub_rn(__fmul_rn(a1, b2), __fmul_rn(a2, b1));
}

__device__ __forceinline__ double mul_rn(double a, double b) { return __dmul_rn(a, b); }
__device__ __forceinline__ float mul_rn(float a, float b) { return __fmul_rn(a, b); }

// E(a -> b): +1 if up && cr > 0, -1 if dn && cr < 0, else 0, with up = a2<0 && b2>=0, dn = a2>=0 && b2<0.
// sa = (a2 < 0) and sb = (b2 < 0) are evaluated once per loaded value.  Writing b2 >= 0 as !(b2 < 0) differs from
// the definition only when a2 or b2 is NaN, and then cr is NaN and the edge is 0 either way; -0 is not < 0 in
// both forms.
// cr = RN(p - q) with p = RN(a1 b2), q = RN(a2 b1): the rounded difference of two floating-point numbers has the sign
// of the exact difference (gradual underflow keeps a non-zero difference non-zero; inf - inf and NaN give NaN, for
// which both orderings are false as well), so cr > 0 <=> p > q and cr < 0 <=> p < q: the subtraction is not needed.
template <typename T, typename P>
__device__ __forceinline__ int edge_of(const P& a, bool sa, const P& b, bool sb) {
  const T p = mul_rn(a.x, b.y), q = mul_rn(a.y, b.x);
  const bool up = sa && !sb, dn = !sa && sb;
  return (int)(up && p > q) - (int)(dn && p < q);
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



template <typename T> constexpr size_t tag_smem_bytes() {
  return ((size_t)TAG_WARPS * TAG_PF * (TAG_RY + 1) * 32 + 1) * sizeof(typename PairOf<T>::type);
}

// edges of P+x packed for the shuffle: (Ey+1) | (Ez+1)<<2
template <typename T>
__global__ void __launch_bounds__(TAG_THREADS) k_tag_strings(const TagArgs<T> a) {
  using P = typename PairOf<T>::type;
  constexpr int RY = TAG_RY;
  const TileDev t = a.tiles[blockIdx.x];
  const BoxDev b = a.boxes[t.box];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int x = t.x0 + lane, y0 = t.y0 + warp * RY;
  if (y0 >= b.n[1]) return;  // whole warp leaves together; there is no block-level synchronisation
  // cells past the box edge clamp to the first ghost layer (g >= 1): valid memory, results unused
  const bool wr = a.wrap != 0;
  const int xc = (wr && x >= b.n[0]) ? 0 : min(x, b.n[0]);
  const bool actx = lane < TAG_TX && x < b.n[0];
  const long long plane = (long long)b.sx * b.sy;
  const long long org = b.base + (long long)(t.z0 + a.g) * plane + (xc + a.ox);
  long long orow[RY + 1];
#pragma unroll
  for (int r = 0; r <= RY; ++r) orow[r] = org + (long long)(((wr && y0 + r >= b.n[1]) ? 0 : min(y0 + r, b.n[1])) + a.g) * b.sx;

  // plane index n is relative to t.z0; n = nz is the first plane above the tile (a ghost plane or the next tile)
  // Every lane streams its own column through a per-warp shared-memory ring with cp.async, TAG_PF planes ahead:
  // the bytes in flight cost no registers.  ring[slot][row][lane]; lane l reads its +x partner at [lane + 1].
  extern __shared__ __align__(16) unsigned char tag_smem[];
  P* const ring = reinterpret_cast<P*>(tag_smem) + (size_t)warp * (TAG_PF * (RY + 1) * 32) + lane;
  auto issue = [&](int n) {
    P* const dst = ring + (n % TAG_PF) * ((RY + 1) * 32);
    const int pn = min(n, t.nz);
    const long long po = (long long)((wr && t.z0 + pn >= b.n[2]) ? -t.z0 : pn) * plane;
#pragma unroll
    for (int r = 0; r <= RY; ++r) cp_async_pair(dst + r * 32, a.psi + orow[r] + po);
  };
#pragma unroll
  for (int d = 0; d < TAG_PF; ++d) {
    issue(d);
    cp_async_commit();
  }
  P cur[RY + 1];
  cp_async_wait<TAG_PF - 1>();
#pragma unroll
  for (int r = 0; r <= RY; ++r) cur[r] = ring[r * 32];  // plane 0 (slot 0), own entries only
  int exc[RY], eyc[RY], wxyc[RY];  // in-plane edges and W_xy of the plane below
#pragma unroll
  for (int r = 0; r < RY; ++r) exc[r] = eyc[r] = wxyc[r] = 0;
  bool sc[RY + 1];  // (psi2 < 0) of cur
#pragma unroll
  for (int r = 0; r <= RY; ++r) sc[r] = cur[r].y < T(0);

  // count blocks: lanes split over at most two x-blocks, rows over at most two y-blocks
  const int bi = (b.lo[0] + min(x, b.n[0] - 1)) >> 5;
  const int bi0 = __shfl_sync(0xffffffffu, bi, 0);
  const int bj0 = (b.lo[1] + y0) >> 5;
  int cntA = 0, cntB = 0;  // this thread's tagged cells in y-block bj0 / bj0 + 1
  int cur_bk = (b.lo[2] + t.z0) >> 5;
  auto flush = [&](int bk) {
    if (a.counts) {
      const unsigned m = 0xffffffffu;
      const int v00 = __reduce_add_sync(m, bi == bi0 ? cntA : 0), v10 = __reduce_add_sync(m, bi == bi0 ? 0 : cntA);
      const int v01 = __reduce_add_sync(m, bi == bi0 ? cntB : 0), v11 = __reduce_add_sync(m, bi == bi0 ? 0 : cntB);
      if (lane == 0) {
        uint32_t* const c0 = a.counts + ((long long)bk * a.nb1 + bj0) * a.nb0 + bi0;
        if (v00) atomicAdd(c0, (uint32_t)v00);
        if (v10) atomicAdd(c0 + 1, (uint32_t)v10);
        if (v01) atomicAdd(c0 + a.nb0, (uint32_t)v01);
        if (v11) atomicAdd(c0 + a.nb0 + 1, (uint32_t)v11);
      }
    }
    cntA = cntB = 0;
  };

#pragma unroll 2
  for (int n = 0; n <= t.nz; ++n) {
    P nO[RY + 1], nX[RY + 1];
    bool so[RY + 1], sx[RY + 1];
    unsigned sbits = 0;
#pragma unroll
    cp_async_wait<TAG_PF - 1>();  // this lane's copies of plane n have landed ...
    __syncwarp();                 // ... and its neighbour's
    const P* const src = ring + (n % TAG_PF) * ((RY + 1) * 32);
#pragma unroll
    for (int r = 0; r <= RY; ++r) {
      nO[r] = src[r * 32];
      nX[r] = src[r * 32 + 1];  // lane 31 reads a foreign entry: its Ex is never used
      so[r] = nO[r].y < T(0);
      sbits |= (so[r] ? 1u : 0u) << r;
    }
    __syncwarp();  // everybody has read slot n % TAG_PF before it is refilled
    issue(n + TAG_PF);
    cp_async_commit();
    sbits = __shfl_down_sync(0xffffffffu, sbits, 1);
#pragma unroll
    for (int r = 0; r <= RY; ++r) sx[r] = (sbits >> r) & 1u;
    int ex[RY + 1], ez[RY + 1], ey[RY];
#pragma unroll
    for (int r = 0; r <= RY; ++r) {
      ex[r] = edge_of<T, P>(nO[r], so[r], nX[r], sx[r]);   // plane n
      ez[r] = edge_of<T, P>(cur[r], sc[r], nO[r], so[r]);  // plane n-1 -> n (0 at n = 0: cur == nO)
    }
#pragma unroll
    for (int r = 0; r < RY; ++r) ey[r] = edge_of<T, P>(nO[r], so[r], nO[r + 1], so[r + 1]);
    int pk = 0;  // (Ey+1) | (Ez+1)<<2 of every row, 4 bits per row, for the lane on the left
#pragma unroll
    for (int r = 0; r < RY; ++r) pk |= ((ey[r] + 1) | ((ez[r] + 1) << 2)) << (4 * r);
    const int nb = __shfl_down_sync(0xffffffffu, pk, 1);
    const int z = t.z0 + n - 1;
    const int bk = (b.lo[2] + z) >> 5;
    if (n > 0 && bk != cur_bk) {
      flush(cur_bk);
      cur_bk = bk;
    }
#pragma unroll
    for (int r = 0; r < RY; ++r) {
      const int eyx = ((nb >> (4 * r)) & 3) - 1, ezx = ((nb >> (4 * r + 2)) & 3) - 1;  // Ey(P+x), Ez(P+x)
      const int wxyn = ex[r] + eyx - ex[r + 1] - ey[r];
      if (n > 0) {
        const int wyz = eyc[r] + ez[r + 1] - ey[r] - ez[r];
        const int wzx = ez[r] + ex[r] - ezx - exc[r];
        const uint8_t tag = (uint8_t)((wxyc[r] != 0 ? 1 : 0) | (wyz != 0 ? 2 : 0) | (wzx != 0 ? 4 : 0));
        const int y = y0 + r;
        const bool act = actx && y < b.n[1];
        if (a.tags && act) a.tags[b.tag_base + ((long long)z * b.n[1] + y) * b.n[0] + x] = tag;
        const int hit = (act && tag != 0) ? 1 : 0;
        if (((b.lo[1] + y) >> 5) == bj0) cntA += hit; else cntB += hit;
      }
      wxyc[r] = wxyn;
      exc[r] = ex[r];
      eyc[r] = ey[r];
    }
#pragma unroll
    for (int r = 0; r <= RY; ++r) {
      cur[r] = nO[r];
      sc[r] = so[r];
    }
  }
  flush(cur_bk);
}

}  // namespace sledge
