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
//
// One comparison per edge.  With s(v) = (v2 < 0), an edge contributes only if s(a) != s(b), and then
//   up (s(a), !s(b)):  p > q  with p = RN(a1 b2) = RN(a1 |b2|) =: P,  q = RN(a2 b1) = -RN(|a2| b1) =: -Q
//   dn (!s(a), s(b)):  p < q  with p = -P, q = Q
// (rounding to nearest is symmetric in sign, so the identities hold bit for bit, zeros, infinities and NaNs
// included: a comparison with NaN is false on both sides, +0 and -0 compare equal on both sides), i.e. in both
// cases the edge counts iff P > -Q, and its sign is +1 if s(a), else -1.  The comparison "cr > 0" of the
// definition equals "p > q" because the rounded difference of two floating-point numbers has the sign of the
// exact difference (gradual underflow).
//
// Bit-sliced windings.  A warp owns a 31 x TAG_RY patch of cells (lane 31 and a (TAG_RY+1)-th row are halo: they
// only supply edges) and marches along z with no block-level synchronisation.  A lane keeps, per plane, ONE word
// per quantity with a 3-bit field per row (bit 3r = row r): S = s(psi), G = the comparison results of its x / y / z
// edges.  Edges that count: N = G & (S ^ S_partner), split by sign into N & S_a and N & ~S_a; the four signed
// terms of a winding are added as 3-bit integers for all rows at once (two 3-input adds), positive and negative
// terms separately, and W != 0 <=> the two sums differ.  The three winding masks interleave into the tag bits:
// (m_xy | m_yz << 1 | m_zx << 2) >> 3r & 7 is the tag byte of row r.  The masks of P+x come from lane + 1 by
// shuffle.  ~40 instructions per cell instead of ~130 with per-cell integer arithmetic.
// Loads: every lane streams its column through a per-warp cp.async ring, TAG_PF planes ahead (bytes in flight cost
// no registers); psi(P+x) is read from the neighbouring lane's ring entry.
// Counts: per-thread counters, reduced over the warp (redux) and flushed with one atomicAdd per 32-block
// whenever the warp leaves a 32-block in z.
#pragma once
#include "layout.h"
#include "k_rk_pipe.cuh"  // cp.async helpers

namespace sledge {

constexpr int TAG_TX = 31;                 // cells per warp row that produce tags (lane 31 is the +x halo)
#ifndef SLEDGE_TAG_RY
#define SLEDGE_TAG_RY 8
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
#define SLEDGE_TAG_PF 3
#endif
constexpr int TAG_PF = SLEDGE_TAG_PF;       // planes in flight per thread (cp.async ring depth)
static_assert(TAG_RY <= 9, "3-bit fields of TAG_RY + 1 rows must fit a 32-bit word with the << 2 of the tag interleave");

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
  // Tiles over STORAGE boxes (several caller's boxes coalesced, sledge.cu "storage boxes"): the tag bytes keep the
  // caller's layout, found per blocking-factor cell (the granularity of box ownership, >= TAG_RY here) in this table:
  // {x, y} = offset of the cell's first tag byte (low, high word), z = n0 and w = n1 of the caller's box it lies in.
  // Null: `boxes` are the caller's boxes themselves.
  const int4* tag_cells;
  int bfs, no0, no1;  // log2(blocking factor), owner grid extent (x, y)
};

__device__ __forceinline__ double mul_rn(double a, double b) { return __dmul_rn(a, b); }
__device__ __forceinline__ float mul_rn(float a, float b) { return __fmul_rn(a, b); }

// the comparison of edge a -> b (see the header): P > -Q with P = RN(a1 |b2|), Q = RN(|a2| b1)
template <typename T, typename P>
__device__ __forceinline__ bool edge_cmp(const P& a, const P& b) {
  return mul_rn(a.x, fabs(b.y)) > -mul_rn(fabs(a.y), b.x);
}

template <typename T> constexpr size_t tag_smem_bytes() {
  return ((size_t)TAG_WARPS * TAG_PF * (TAG_RY + 1) * 32 + 1) * sizeof(typename PairOf<T>::type);
}

// one 3-bit field per row: bit 3r
__host__ __device__ constexpr unsigned tag_rowbits(int rows) {
  unsigned m = 0;
  for (int r = 0; r < rows; ++r) m |= 1u << (3 * r);
  return m;
}
// field-wise "a != b" of two words of 3-bit integers -> bit 3r
__device__ __forceinline__ unsigned tag_differs(unsigned a, unsigned b) {
  const unsigned v = a ^ b;
  constexpr unsigned ROWS = tag_rowbits(TAG_RY);
  return (v | (v >> 1) | (v >> 2)) & ROWS;
}

#ifndef SLEDGE_TAG_MINB
#define SLEDGE_TAG_MINB 3  // <= 168 registers: three CTAs of four warps per SM (fp64 needs 182 without the cap; no spills with it)
#endif
#ifndef SLEDGE_TAG_MINB_LOOKUP
#define SLEDGE_TAG_MINB_LOOKUP SLEDGE_TAG_MINB
#endif
// LOOKUP: tiles over storage boxes, tag addresses through a.tag_cells (its own instantiation: the extra registers must
// not cost the plain pass its third CTA per SM)
template <typename T, bool LOOKUP = false>
__global__ void __launch_bounds__(TAG_THREADS, LOOKUP ? SLEDGE_TAG_MINB_LOOKUP : SLEDGE_TAG_MINB) k_tag_strings(const TagArgs<T> a) {
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
  const char* prow[RY + 1];  // this lane's cell of row r in plane t.z0
#pragma unroll
  for (int r = 0; r <= RY; ++r)
    prow[r] = reinterpret_cast<const char*>(
        a.psi + org + (long long)(((wr && y0 + r >= b.n[1]) ? 0 : min(y0 + r, b.n[1])) + a.g) * b.sx);

  // plane index n is relative to t.z0; n = nz is the first plane above the tile (a ghost plane, the next tile, or
  // plane 0 of the periodic box); planes past it are never used and re-read plane nz.
  // ring[slot][row][lane]; lane l reads its +x partner at [lane + 1].
  extern __shared__ __align__(16) unsigned char tag_smem[];
  constexpr int SLOT = (RY + 1) * 32;  // pairs per ring slot
  P* const ring = reinterpret_cast<P*>(tag_smem) + (size_t)warp * (TAG_PF * SLOT) + lane;
  const long long plane_bytes = plane * (long long)sizeof(P);
  const long long top_bytes = (wr && t.z0 + t.nz >= b.n[2]) ? -(long long)t.z0 * plane_bytes : (long long)t.nz * plane_bytes;
  long long po = 0;  // byte offset of the next plane to issue
  int pn = 0;        // its index
  auto issue = [&](P* dst) {
#pragma unroll
    for (int r = 0; r <= RY; ++r) cp_async_pair(dst + r * 32, reinterpret_cast<const P*>(prow[r] + po));
    ++pn;
    po = pn < t.nz ? po + plane_bytes : top_bytes;
  };
#pragma unroll
  for (int d = 0; d < TAG_PF; ++d) {
    issue(ring + d * SLOT);
    cp_async_commit();
  }

  // rows of this warp that exist and produce tags, as 3-bit fields; rows in the first of the (at most two) y count blocks
  const int nrows = min(RY, b.n[1] - y0);
  const int bj0 = (b.lo[1] + y0) >> 5;
  unsigned act = 0, rowsA = 0;
#pragma unroll
  for (int r = 0; r < RY; ++r) {
    if (actx && r < nrows) act |= 1u << (3 * r);
    if (((b.lo[1] + y0 + r) >> 5) == bj0) rowsA |= 1u << (3 * r);
  }
  // count blocks: lanes split over at most two x-blocks
  const int bi = (b.lo[0] + min(x, b.n[0] - 1)) >> 5;
  const int bi0 = __shfl_sync(0xffffffffu, bi, 0);
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
  uint8_t* tagp = a.tags ? a.tags + b.tag_base + ((long long)(t.z0 - 1) * b.n[1] + y0) * b.n[0] + x : nullptr;
  long long tag_plane = (long long)b.n[1] * b.n[0];
  int tag_row = b.n[0];
  // lookup mode: this lane's column of blocking-factor cells (x and y cell fixed, z varies), next entry prefetched
  const bool lookup = LOOKUP && a.tags != nullptr;
  const int bfm = (1 << a.bfs) - 1;
  const int gx = b.lo[0] + min(x, b.n[0] - 1), gy = b.lo[1] + y0;
  const int4* cellp = nullptr;
  int4 nextc = make_int4(0, 0, 0, 0);
  if (lookup) {
    cellp = a.tag_cells + ((long long)((b.lo[2] + t.z0) >> a.bfs) * a.no1 + (gy >> a.bfs)) * a.no0 + (gx >> a.bfs);
    nextc = __ldg(cellp);
  }

  // state carried from plane n-1: its values, sign word, signed in-plane edges (x, y) and W_xy mask
  P cur[RY + 1];
#pragma unroll
  for (int r = 0; r <= RY; ++r) cur[r] = mkpair(T(0), T(0));
  unsigned Sp = 0, Spx = 0, XPp = 0, XNp = 0, YPp = 0, YNp = 0, mxy_p = 0;
  int slot = 0;

#pragma unroll 2
  for (int n = 0; n <= t.nz; ++n) {
    P nO[RY + 1], nX[RY + 1];
    cp_async_wait<TAG_PF - 1>();  // this lane's copies of plane n have landed ...
    __syncwarp();                 // ... and its neighbour's
    P* const src = ring + slot * SLOT;
#pragma unroll
    for (int r = 0; r <= RY; ++r) {
      nO[r] = src[r * 32];
      nX[r] = src[r * 32 + 1];  // lane 31 reads a foreign entry: its results are never used
    }
    __syncwarp();  // everybody has read slot n % TAG_PF before it is refilled
    issue(src);  // plane n + TAG_PF goes into the slot just drained
    cp_async_commit();
    slot = slot + 1 == TAG_PF ? 0 : slot + 1;

    unsigned S = 0, Gx = 0, Gy = 0, Gz = 0;
#pragma unroll
    for (int r = 0; r <= RY; ++r) {
      if (nO[r].y < T(0)) S |= 1u << (3 * r);
      if (edge_cmp<T, P>(nO[r], nX[r])) Gx |= 1u << (3 * r);   // plane n
      if (edge_cmp<T, P>(cur[r], nO[r])) Gz |= 1u << (3 * r);  // plane n-1 -> n
    }
#pragma unroll
    for (int r = 0; r < RY; ++r)
      if (edge_cmp<T, P>(nO[r], nO[r + 1])) Gy |= 1u << (3 * r);
    const unsigned Sx = __shfl_down_sync(0xffffffffu, S, 1);
    const unsigned X = Gx & (S ^ Sx), Y = Gy & (S ^ (S >> 3)), Z = Gz & (Sp ^ S);  // edges that count
    const unsigned XP = X & S, XN = X & ~S, YP = Y & S, YN = Y & ~S, ZP = Z & Sp, ZN = Z & ~Sp;
    // Y and Z of the lane on the right (P + x): one shuffle, signs from Sx (plane n) and Spx (plane n - 1)
    const unsigned YZx = __shfl_down_sync(0xffffffffu, Y | (Z << 1), 1);
    constexpr unsigned ROWS = tag_rowbits(RY);
    const unsigned Yx = YZx & ROWS, Zx = (YZx >> 1) & ROWS;
    const unsigned YPx = Yx & Sx, YNx = Yx & ~Sx, ZPx = Zx & Spx, ZNx = Zx & ~Spx;
    // W_xy of plane n (tagged one iteration later, with the plane's other two windings)
    const unsigned mxy = tag_differs(XP + YPx + ((XN >> 3) + YN), XN + YNx + ((XP >> 3) + YP));
    const int z = t.z0 + n - 1;
    const int bk = (b.lo[2] + z) >> 5;
    if (n > 0) {
      if (bk != cur_bk) {
        flush(cur_bk);
        cur_bk = bk;
      }
      const unsigned myz = tag_differs(YPp + (ZP >> 3) + (YN + ZN), YNp + (ZN >> 3) + (YP + ZP));
      const unsigned mzx = tag_differs(ZP + XP + (ZNx + XNp), ZN + XN + (ZPx + XPp));
      const unsigned c3 = mxy_p | (myz << 1) | (mzx << 2);  // field r = tag byte of row r
      if (lookup && (n == 1 || ((b.lo[2] + z) & bfm) == 0)) {  // entering a blocking-factor cell: its caller's box
        const int4 c = nextc;
        tag_row = c.z;
        tag_plane = (long long)c.z * c.w;
        tagp = a.tags + (((long long)(unsigned)c.y << 32) | (unsigned)c.x) +
               ((long long)((b.lo[2] + z) & bfm) * c.w + (gy & bfm)) * c.z + (gx & bfm);
        cellp += (long long)a.no1 * a.no0;
        if (z + (bfm - ((b.lo[2] + z) & bfm)) + 1 < t.z0 + t.nz) nextc = __ldg(cellp);  // next cell of this tile, used planes later
      }
      if (a.tags) {
#pragma unroll
        for (int r = 0; r < RY; ++r)
          if ((act >> (3 * r)) & 1u) tagp[(long long)r * tag_row] = (uint8_t)((c3 >> (3 * r)) & 7u);
      }
      const unsigned any = (mxy_p | myz | mzx) & act;
      cntA += __popc(any & rowsA);
      cntB += __popc(any & ~rowsA);
    }
    tagp += tag_plane;
    mxy_p = mxy;
    Sp = S;
    Spx = Sx;
    XPp = XP;
    XNp = XN;
    YPp = YP;
    YNp = YN;
#pragma unroll
    for (int r = 0; r <= RY; ++r) cur[r] = nO[r];
  }
  flush(cur_bk);
}

}  // namespace sledge
