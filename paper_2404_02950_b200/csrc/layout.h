// layout.h -- device-side descriptors and vector helpers shared by the sledge kernels.
//
// Data layout in HBM: a level's field plane is an array of PAIRS (psi1,psi2) or (Pi1,Pi2).
// Box b of the level occupies cells [base, base + sx*sy*sz); cell (i,j,k) relative to the box's valid
// low corner (ghosts: negative / >= n) sits at base + ((k+g)*sy + (j+g))*sx + (i+ox).  ox >= g is the
// x offset of the first valid cell, chosen so that it is 128-byte aligned; sx is a multiple of the
// 128-byte cell count, so every row start is 128-byte aligned as well.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace sledge {

struct BoxDev {
  long long base;  // first cell of the box (in pairs) inside the level plane
  int n[3];        // valid cells
  int lo[3];       // low corner in the level's index space
  int sx, sy;      // row pitch and rows per z-plane (in cells)
  long long tag_base;  // offset of this box's first cell in the level's dense tag array
};

struct TileDev {
  int box;         // index into the level's BoxDev table
  int x0, y0, z0;  // box-relative origin of the tile
  int nz;          // z planes this tile marches through
};

struct LevelGeom {
  int n[3];   // index-space extent of the level
  int no[3];  // owner grid extent = n / blocking_factor
  int bf_shift;
  int g, ox;
};

template <typename T> struct PairOf;
template <> struct PairOf<double> { using type = double2; };
template <> struct PairOf<float> { using type = float2; };

__device__ __forceinline__ double2 mkpair(double a, double b) { return make_double2(a, b); }
__device__ __forceinline__ float2 mkpair(float a, float b) { return make_float2(a, b); }

// 16-byte vector = CPT pairs (1 for fp64, 2 for fp32); all streaming accesses use it.
template <typename T> struct Vec16;
template <> struct Vec16<double> {
  static constexpr int CPT = 1;
  double2 p[1];
};
template <> struct Vec16<float> {
  static constexpr int CPT = 2;
  float2 p[2];
};

template <typename T>
__device__ __forceinline__ Vec16<T> ldg16(const typename PairOf<T>::type* ptr) {
  Vec16<T> r;
  const int4 raw = __ldg(reinterpret_cast<const int4*>(ptr));
  *reinterpret_cast<int4*>(&r) = raw;
  return r;
}
// L2 eviction-priority policies (createpolicy): stencil data that a neighbouring CTA re-reads as halo is
// loaded evict_last, pure streams (pointwise inputs, all outputs) evict_first.
__device__ __forceinline__ uint64_t l2_policy_evict_first() {
  uint64_t p;
  asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
  return p;
}
__device__ __forceinline__ uint64_t l2_policy_evict_last() {
  uint64_t p;
  asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
  return p;
}
#ifndef SLEDGE_POL
#define SLEDGE_POL 0
#endif
// streaming variant: the data is touched once per launch, keep it out of L1
template <typename T>
__device__ __forceinline__ Vec16<T> ldg16_stream(const typename PairOf<T>::type* ptr) {
  Vec16<T> r;
  int4 raw;
#if SLEDGE_POL == 2
  asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.v4.s32 {%0,%1,%2,%3}, [%4], %5;"
               : "=r"(raw.x), "=r"(raw.y), "=r"(raw.z), "=r"(raw.w)
               : "l"(ptr), "l"(l2_policy_evict_first()));
#else
  asm volatile("ld.global.nc.L1::no_allocate.v4.s32 {%0,%1,%2,%3}, [%4];"
               : "=r"(raw.x), "=r"(raw.y), "=r"(raw.z), "=r"(raw.w)
               : "l"(ptr));
#endif
  *reinterpret_cast<int4*>(&r) = raw;
  return r;
}
// stencil variant: a neighbouring CTA reads the same line as halo shortly before / after
template <typename T>
__device__ __forceinline__ Vec16<T> ldg16_keep(const typename PairOf<T>::type* ptr) {
  Vec16<T> r;
  int4 raw;
#if SLEDGE_POL == 2
  asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.v4.s32 {%0,%1,%2,%3}, [%4], %5;"
               : "=r"(raw.x), "=r"(raw.y), "=r"(raw.z), "=r"(raw.w)
               : "l"(ptr), "l"(l2_policy_evict_last()));
#elif SLEDGE_POL == 1
  asm volatile("ld.global.v4.s32 {%0,%1,%2,%3}, [%4];"
               : "=r"(raw.x), "=r"(raw.y), "=r"(raw.z), "=r"(raw.w)
               : "l"(ptr));
#else
  asm volatile("ld.global.nc.L1::no_allocate.v4.s32 {%0,%1,%2,%3}, [%4];"
               : "=r"(raw.x), "=r"(raw.y), "=r"(raw.z), "=r"(raw.w)
               : "l"(ptr));
#endif
  *reinterpret_cast<int4*>(&r) = raw;
  return r;
}
template <typename T>
__device__ __forceinline__ void stg16(typename PairOf<T>::type* ptr, const Vec16<T>& v) {
  const int4 raw = *reinterpret_cast<const int4*>(&v);
#if SLEDGE_POL == 2
  asm volatile("st.global.L1::no_allocate.L2::cache_hint.v4.s32 [%0], {%1,%2,%3,%4}, %5;" ::"l"(ptr), "r"(raw.x),
               "r"(raw.y), "r"(raw.z), "r"(raw.w), "l"(l2_policy_evict_first())
               : "memory");
#else
  asm volatile("st.global.L1::no_allocate.v4.s32 [%0], {%1,%2,%3,%4};" ::"l"(ptr), "r"(raw.x), "r"(raw.y),
               "r"(raw.z), "r"(raw.w)
               : "memory");
#endif
}

__host__ __device__ __forceinline__ int wrap_idx(int i, int n) {
  int r = i % n;
  return r < 0 ? r + n : r;
}
__host__ __device__ __forceinline__ int floordiv2(int i) { return i >> 1; }  // arithmetic shift = floor

}  // namespace sledge
