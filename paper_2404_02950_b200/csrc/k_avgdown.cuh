// k_avgdown.cuh -- K4: level synchronisation, coarse <- mean of the 8 fine children,
// all four components, and the dense <-> padded state copies behind sledge_set_state / sledge_get_state.
//
// K4 mapping: one thread per coarse cell under a fine box (n/2 per axis), x fastest, so a warp reads
// 32 x 2 consecutive fine pairs per row (coalesced) and writes 32 consecutive coarse pairs.  The coarse
// destination is found through the coarse owner table (a fine box may lie over several coarse boxes).
// Children are summed in the fixed order z, y, x (x fastest) starting from 0, then scaled by 1/8.
//
// TEE variant (Eq.5-6, L373-380 Eq.12; self-shadow method, f = identity): the same thread reads the
// coarse value BEFORE overwriting it, Delta_c = |coarse_c - mean_c| for c = psi1, psi2, tag = (Delta_psi1 > eps1) |
// (Delta_psi2 > eps2) << 1 in the kernel's precision, writes the byte to the 8 children (four 2-byte stores) and adds
// 8 to the fine level's 32^3 block count when the tag is set.  No extra pass over the data: the truncation-error
// estimate rides on the synchronisation.
#pragma once
#include "k_ghost.cuh"

namespace sledge {

constexpr int AVG_THREADS = 256;

template <typename T>
struct AvgArgs {
  using P = typename PairOf<T>::type;
  const BoxDev* fboxes;
  const int* blk_prefix;  // CTAs before fine box b
  int nfbox;
  const P* f_psi;
  const P* f_pi;
  LevelGeom fgeom;
  const BoxDev* cboxes;
  const int* cowner;
  LevelGeom cgeom;
  P* c_psi;
  P* c_pi;
  int* err_flag;
  // TEE variant only
  T tee_eps[4];          // threshold per component psi1, psi2, Pi1, Pi2 (L781-782); +inf = never tags
  uint8_t* tee_tags;     // dense tags of the FINE level (boxes back to back, x fastest); may be null
  uint32_t* tee_counts;  // tagged fine cells per aligned 32^3 block of the fine level; may be null
  int nb0, nb1;          // count blocks per axis (x, y) of the fine level
};

template <typename T>
__device__ __forceinline__ typename PairOf<T>::type mean8(const typename PairOf<T>::type* f, long long o, int sx,
                                                          long long plane) {
  T s0 = T(0), s1 = T(0);
#pragma unroll
  for (int rz = 0; rz < 2; ++rz)
#pragma unroll
    for (int ry = 0; ry < 2; ++ry)
#pragma unroll
      for (int rx = 0; rx < 2; ++rx) {
        const typename PairOf<T>::type v = f[o + rz * plane + (long long)ry * sx + rx];
        s0 += v.x;
        s1 += v.y;
      }
  return mkpair(T(0.125) * s0, T(0.125) * s1);
}

template <typename T, bool TEE>
__global__ void __launch_bounds__(AVG_THREADS) k_average_down(const AvgArgs<T> a) {
  int lo_b = 0, hi_b = a.nfbox;
  const int blk = blockIdx.x;
  while (hi_b - lo_b > 1) {
    const int mid = (lo_b + hi_b) >> 1;
    if (a.blk_prefix[mid] <= blk) lo_b = mid; else hi_b = mid;
  }
  const BoxDev fb = a.fboxes[lo_b];
  const int cx = fb.n[0] >> 1, cy = fb.n[1] >> 1, cz = fb.n[2] >> 1;
  const long long q = (long long)(blk - a.blk_prefix[lo_b]) * AVG_THREADS + threadIdx.x;
  if (q >= (long long)cx * cy * cz) return;
  const int I = (int)(q % cx);
  const int J = (int)((q / cx) % cy);
  const int K = (int)(q / ((long long)cx * cy));
  const int ci = (fb.lo[0] >> 1) + I, cj = (fb.lo[1] >> 1) + J, ck = (fb.lo[2] >> 1) + K;
  const int ow = owner_lookup(a.cowner, a.cgeom, ci, cj, ck);
  if (ow < 0) {
    *a.err_flag = 1;
    return;
  }
  const BoxDev cb = a.cboxes[ow];
  const long long fo = cell_offset(fb, a.fgeom.g, a.fgeom.ox, 2 * I, 2 * J, 2 * K);
  const long long co = cell_offset(cb, a.cgeom.g, a.cgeom.ox, ci - cb.lo[0], cj - cb.lo[1], ck - cb.lo[2]);
  const long long fplane = (long long)fb.sx * fb.sy;
  const typename PairOf<T>::type m = mean8<T>(a.f_psi, fo, fb.sx, fplane);
  const typename PairOf<T>::type mp = mean8<T>(a.f_pi, fo, fb.sx, fplane);
  if (TEE) {
    const typename PairOf<T>::type c = a.c_psi[co];  // the coarse level's own result, before the overwrite
    const typename PairOf<T>::type cp = a.c_pi[co];
    const T d1 = fabs(c.x - m.x), d2 = fabs(c.y - m.y), d3 = fabs(cp.x - mp.x), d4 = fabs(cp.y - mp.y);
    const unsigned tag = (d1 > a.tee_eps[0] ? 1u : 0u) | (d2 > a.tee_eps[1] ? 2u : 0u) |
                         (d3 > a.tee_eps[2] ? 4u : 0u) | (d4 > a.tee_eps[3] ? 8u : 0u);
    if (a.tee_tags) {
      const unsigned short two = (unsigned short)(tag | (tag << 8));
#pragma unroll
      for (int rz = 0; rz < 2; ++rz)
#pragma unroll
        for (int ry = 0; ry < 2; ++ry) {
          const long long o = fb.tag_base + ((long long)(2 * K + rz) * fb.n[1] + (2 * J + ry)) * fb.n[0] + 2 * I;
          *reinterpret_cast<unsigned short*>(a.tee_tags + o) = two;  // o is even: n0 and tag_base are
        }
    }
    if (tag && a.tee_counts) {
      const int bi = (fb.lo[0] + 2 * I) >> 5, bj = (fb.lo[1] + 2 * J) >> 5, bk = (fb.lo[2] + 2 * K) >> 5;
      atomicAdd(a.tee_counts + ((long long)bk * a.nb1 + bj) * a.nb0 + bi, 8u);
    }
  }
  a.c_psi[co] = m;
  a.c_pi[co] = mp;
}

// ---- dense <-> padded copies (one component of one box) -------------------------------------------

// dense: (n0 + 2e) x (n1 + 2e) x (n2 + 2e) reals, x fastest, e = 0 (valid region) or g (with ghosts)
template <typename T, bool TO_STATE>
__global__ void k_copy_comp(const BoxDev b, int g, int ox, int e, int comp, typename PairOf<T>::type* plane_ptr,
                            T* dense) {
  const int ex = b.n[0] + 2 * e, ey = b.n[1] + 2 * e, ez = b.n[2] + 2 * e;
  const long long total = (long long)ex * ey * ez;
  for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < total;
       q += (long long)gridDim.x * blockDim.x) {
    const int i = (int)(q % ex) - e;
    const int j = (int)((q / ex) % ey) - e;
    const int k = (int)(q / ((long long)ex * ey)) - e;
    T* cell = reinterpret_cast<T*>(plane_ptr + cell_offset(b, g, ox, i, j, k)) + (comp & 1);
    if (TO_STATE) *cell = dense[q]; else dense[q] = *cell;
  }
}

}  // namespace sledge
