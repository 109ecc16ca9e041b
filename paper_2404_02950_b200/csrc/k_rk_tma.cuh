// k_rk_tma.cuh -- K1, TMA-staged variant of the plane-ring sweeps of k_rk_plane.cuh: same modes, same per-cell
// arithmetic (rk_cell / lap_from, Eq.10-11), same ring of ghosted tile planes and
// register z-windows; what changes is who moves the planes.
//
// k_rk_plane copies a ghosted tile plane with 16-byte cp.async issued by every thread: RY own vectors plus HPT
// halo pairs per field, each with its own 64-bit address, ~8 LSU cycles per warp instruction (4 issue + 4 shared-
// memory write): in the FUSED sweeps these copies take a third of the LSU / shared-memory pipe that the stencil
// reads also need, which is what bounds those sweeps (profiles/r01_c3_ncu_full_final.md: l1tex 69-72 %, DRAM 80 %).
// Here ONE thread issues one cp.async.bulk.tensor.3d (TMA) per differenced field and plane: the box
// (SW x SH pairs, halo included) lands in shared memory in exactly the layout the stencil reads, completion is
// signalled on an mbarrier, and no thread spends an instruction, an address register or an LSU slot on it.
// A tensor map per (box, state buffer, plane) is built at create time (sledge.cu: make_tensor_maps) and lives in
// the arena; the boxes' ghost layers (>= R) and the 128-byte row padding make every tile box start inside the
// stored array, and what sticks out at the high end of a partial tile is zero-filled by the TMA unit and never read.
//
// TMA has no periodic wrap, so on a level that is ONE box over the periodic domain (a.wrap) the sweep keeps the
// star ghost cells of its OUTPUT valid instead: a thread whose cell lies within R of a box face also stores its
// result at the periodic image just outside the opposite face (L23).  The host fills the ghosts of a state that
// no such sweep has written (after sledge_set_state, an average-down) with K2 once.
//
// Pipeline per CTA (z-march, ring of S = R + 1 + PD planes per field, as in k_rk_plane): iteration zz waits for
// the mbarrier of plane zz + R, passes ONE __syncthreads (which retires plane zz - 1), thread 0 re-arms that
// slot's mbarrier and issues the TMA of plane zz + R + PD into it.  Pointwise inputs keep their per-thread
// cp.async ring.  (A variant without the block-wide barrier -- an "empty" mbarrier per slot on which every warp
// arrives after its shared-memory reads, so that the warps of a CTA drift apart -- was measured 2.5 % SLOWER on
// C3 and is not kept: profiles/r02_k1_variants.md.)
#pragma once
#include <cuda.h>  // CUtensorMap (type only)

#include <utility>

#include "k_rk_plane.cuh"

namespace sledge {

// f(integral_constant<int, 0>) ... f(integral_constant<int, N-1>): a loop whose index is a compile-time constant in
// the body (the register z-windows rotate through their slots instead of being shifted)
template <class F, int... I>
__device__ __forceinline__ void static_for_impl(F&& f, std::integer_sequence<int, I...>) {
  (f(std::integral_constant<int, I>{}), ...);
}
template <int N, class F>
__device__ __forceinline__ void static_for(F&& f) {
  static_for_impl(f, std::make_integer_sequence<int, N>{});
}

__device__ __forceinline__ void mbar_init(uint64_t* bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(bytes)
               : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t* bar, unsigned parity) {
  unsigned ok;
  asm volatile(
      "{\n\t"
      ".reg .pred p;\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
      "selp.u32 %0, 1, 0, p;\n\t"
      "}"
      : "=r"(ok)
      : "r"((unsigned)__cvta_generic_to_shared(bar)), "r"(parity)
      : "memory");
  return ok != 0;
}
// try_wait suspends the thread for a hardware time slice per attempt; a load that never completes (a bad tensor
// map) becomes a trap -- reported as SLEDGE_ECUDA by the next call -- instead of a hung GPU
__device__ __forceinline__ void mbar_wait(uint64_t* bar, unsigned parity) {
  unsigned spins = 0;
  while (!mbar_try_wait(bar, parity))
    if (++spins > (1u << 22)) __trap();
}
// one tile box: coordinates (c0 = first real, c1 = row, c2 = plane) in the box's stored array
__device__ __forceinline__ void tma_load_3d(void* smem_dst, const CUtensorMap* map, uint64_t* bar, int c0, int c1, int c2) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cta.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];" ::"r"(
          (unsigned)__cvta_generic_to_shared(smem_dst)),
      "l"(map), "r"((unsigned)__cvta_generic_to_shared(bar)), "r"(c0), "r"(c1), "r"(c2)
      : "memory");
}

template <typename T, int ORDER, int MODE, int TX, int TY, int PD, int RY = 1>
struct TmaCfg {
  using PC = PlaneCfg<T, ORDER, MODE, TX, TY, PD, RY>;
  static constexpr int R = PC::R, CPT = PC::CPT, TXC = PC::TXC, XO = PC::XO, SW = PC::SW, SH = PC::SH, NT = PC::NT;
  static constexpr int NF = PC::NF, NP = PC::NP, NOUT = PC::NOUT, S = PC::S;
  static constexpr size_t PAIR = PC::PAIR;
  static constexpr int BOX_BYTES = SH * SW * (int)PAIR;             // what one TMA load writes
  static constexpr int PSZ = ((BOX_BYTES + 127) / 128 * 128) / (int)PAIR;  // pairs per field plane, 128-byte multiple
  static constexpr size_t PLANE_BYTES = (size_t)S * NF * PSZ * PAIR;
  static constexpr size_t PNT_BYTES = (size_t)PD * NP * RY * NT * 16;
  static constexpr size_t BAR_OFF = PLANE_BYTES + PNT_BYTES;
  static constexpr size_t SMEM_BYTES = BAR_OFF + (size_t)S * 8;
};

template <typename T, int ORDER, int MODE, int TX, int TY, int RY = 1>
constexpr int tma_depth(size_t budget, int pdmax) {
  int d = 1;
  if (pdmax >= 2 && TmaCfg<T, ORDER, MODE, TX, TY, 2, RY>::SMEM_BYTES <= budget) d = 2;
  if (pdmax >= 3 && TmaCfg<T, ORDER, MODE, TX, TY, 3, RY>::SMEM_BYTES <= budget) d = 3;
  if (pdmax >= 4 && TmaCfg<T, ORDER, MODE, TX, TY, 4, RY>::SMEM_BYTES <= budget) d = 4;
  return d;
}

template <typename T, int ORDER, int MODE, int TX, int TY, int PD, int RY, int MINB>
__global__ void __launch_bounds__(TX* TY / RY, MINB) k_rk_tma(const PipeArgs<T> a) {
  using P = typename PairOf<T>::type;
  using V = Vec16<T>;
  using C = TmaCfg<T, ORDER, MODE, TX, TY, PD, RY>;
  constexpr int R = C::R, CPT = C::CPT, XO = C::XO, SW = C::SW, NT = C::NT;
  constexpr int NF = C::NF, NP = C::NP, NOUT = C::NOUT, S = C::S, PSZ = C::PSZ;
  constexpr int NPA = NP > 0 ? NP : 1;

  extern __shared__ __align__(128) unsigned char smem_raw[];
  P* const planes = reinterpret_cast<P*>(smem_raw);                  // [S][NF][PSZ]
  V* const pring = reinterpret_cast<V*>(smem_raw + C::PLANE_BYTES);  // [PD][NP][RY][NT]
  uint64_t* const full = reinterpret_cast<uint64_t*>(smem_raw + C::BAR_OFF);  // [S]

  const TileDev t = a.tiles[blockIdx.x];
  const BoxDev b = a.boxes[t.box];
  const int tid = threadIdx.x;
  const int tx = tid % TX, ty = (tid / TX) * RY;  // ty = first of this thread's rows
  const int x = t.x0 + tx * CPT, y = t.y0 + ty;
  bool active[RY];
#pragma unroll
  for (int j = 0; j < RY; ++j) active[j] = (x < b.n[0]) && (y + j < b.n[1]);
  const long long plane = (long long)b.sx * b.sy;
  const long long off = b.base + (long long)(t.z0 + a.g) * plane + (long long)(y + a.g) * b.sx + (x + a.ox);
  const int s_own = (ty + R) * SW + (tx * CPT + XO);  // row j of this thread: s_own + j * SW

  // tile box origin in the box's stored array: reals along x (two per pair), rows, planes
  const int c0 = 2 * (t.x0 + a.ox - XO), c1 = t.y0 + a.g - R, c2 = t.z0 + a.g;
  const CUtensorMap* tmap[NF];
#pragma unroll
  for (int f = 0; f < NF; ++f) tmap[f] = reinterpret_cast<const CUtensorMap*>(a.tmap[f]) + t.box;
  auto issue_plane = [&](int p, int slot) {  // thread 0 only
    mbar_expect_tx(full + slot, (unsigned)(NF * C::BOX_BYTES));
#pragma unroll
    for (int f = 0; f < NF; ++f) tma_load_3d(planes + ((size_t)slot * NF + f) * PSZ, tmap[f], full + slot, c0, c1, c2 + p);
  };
  auto issue_pnt = [&](int st) {
    if (NP > 0) {
      V* const o = pring + (size_t)(st % PD) * NP * RY * NT + tid;
#pragma unroll
      for (int j = 0; j < RY; ++j)
        if (active[j]) {
#pragma unroll
          for (int q = 0; q < NP; ++q)
            cp_async_16(o + (q * RY + j) * NT, a.pnt[q] + off + (long long)st * plane + (long long)j * b.sx);
        }
    }
  };

  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < S; ++s) mbar_init(full + s, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  // prologue: centre planes 0..R-1, then stages 0..PD-1 (stage st = plane st+R and pointwise inputs of plane st)
  const int np = t.nz + R;  // planes 0 .. np-1 are copied
  if (tid == 0) {
#pragma unroll
    for (int p = 0; p < R + PD; ++p)
      if (p < np) issue_plane(p, p % S);
  }
#pragma unroll
  for (int st = 0; st < PD; ++st) {
    if (st < t.nz) issue_pnt(st);
    cp_async_commit();
  }
  // lower 2R planes of the z-windows straight into registers
  // The window ROTATES: in the iteration with zz % W == u the value of plane z + m - R sits in w[f][j][(m + u) % W]
  // (W = 2R + 1), so that nothing is moved from one iteration to the next; the z loop is unrolled W times for it.
  constexpr int W = 2 * R + 1;
  V w[NF][RY][W];
#pragma unroll
  for (int f = 0; f < NF; ++f)
#pragma unroll
    for (int j = 0; j < RY; ++j)
#pragma unroll
      for (int m = 0; m < 2 * R; ++m)
        if (active[j]) w[f][j][m] = ldg16_keep<T>(a.sten[f] + off + (long long)j * b.sx + (long long)(m - R) * plane);
#pragma unroll
  for (int p = 0; p < R; ++p) mbar_wait(full + p, 0);

  // periodic one-box level: which periodic images of this thread's results are star ghost cells (L23)
  const bool wr = a.wrap != 0;
  int gx_lo = 0, gx_hi = 0;  // bit p: pair p of the vector also goes to x + n / x - n
  bool gy_lo[RY], gy_hi[RY];
#pragma unroll
  for (int p = 0; p < CPT; ++p) {
    if (wr && x + p < R) gx_lo |= 1 << p;
    if (wr && x + p >= b.n[0] - R && x + p < b.n[0]) gx_hi |= 1 << p;
  }
#pragma unroll
  for (int j = 0; j < RY; ++j) {
    gy_lo[j] = wr && (y + j < R);
    gy_hi[j] = wr && (y + j >= b.n[1] - R) && (y + j < b.n[1]);
  }

  int slot_c = 0;             // slot of the centre plane zz
  int slot_t = R % S;         // slot of plane zz + R
  int slot_n = (R + PD) % S;  // slot of plane zz + R + PD
  unsigned par_t = 0;         // parity of the phase that completes plane zz + R in slot_t
  auto step = [&](const int zz, auto uc) {
    constexpr int u = decltype(uc)::value;  // zz % W
    mbar_wait(full + slot_t, par_t);  // plane zz + R has landed
    cp_async_wait<PD - 1>();          // this thread's pointwise inputs of plane zz
    __syncthreads();                  // plane zz-1 is retired
    const P* const cb = planes + (size_t)slot_c * NF * PSZ;
    const P* const tb = planes + (size_t)slot_t * NF * PSZ;
    V pv[RY][NPA];
#pragma unroll
    for (int f = 0; f < NF; ++f)
#pragma unroll
      for (int j = 0; j < RY; ++j) {
        w[f][j][(2 * R + u) % W] = *reinterpret_cast<const V*>(tb + f * PSZ + s_own + j * SW);
      }
    if (NP > 0) {
      const V* const o = pring + (size_t)(zz % PD) * NP * RY * NT + tid;
#pragma unroll
      for (int j = 0; j < RY; ++j)
        if (active[j]) {
#pragma unroll
          for (int q = 0; q < NP; ++q) pv[j][q] = o[(q * RY + j) * NT];
        }
    }
    // stage zz + PD reuses the slot of plane zz-1 and the pointwise entries just drained
    if (tid == 0 && zz + PD + R < np) issue_plane(zz + PD + R, slot_n);
    if (zz + PD < t.nz) issue_pnt(zz + PD);
    cp_async_commit();

    if (active[0]) {
      V o_psi[RY][NOUT], o_pi[RY][NOUT];
#pragma unroll
      for (int p = 0; p < CPT; ++p) {
        T lap[RY][NF][2];
#pragma unroll
        for (int f = 0; f < NF; ++f) {
          const P* const s = cb + f * PSZ + s_own + p;
          // this thread's column of the centre plane, rows -R .. RY-1+R: own rows from registers
          P col[RY + 2 * R];
#pragma unroll
          for (int i = 0; i < RY + 2 * R; ++i) {
            if (i >= R && i < R + RY) col[i] = w[f][i - R][(R + u) % W].p[p];
            else col[i] = s[(i - R) * SW];
          }
#pragma unroll
          for (int j = 0; j < RY; ++j) {
            P xn[2 * R];  // x-r, x+r
#pragma unroll
            for (int r = 1; r <= R; ++r) {
              xn[2 * (r - 1) + 0] = s[j * SW - r];
              xn[2 * (r - 1) + 1] = s[j * SW + r];
            }
#pragma unroll
            for (int c = 0; c < 2; ++c) {
              auto comp = [c](const P& v) -> T { return c == 0 ? v.x : v.y; };
              T xm[3], xp[3], ym[3], yp[3], zm[3], zp[3];
#pragma unroll
              for (int r = 1; r <= R; ++r) {
                xm[r - 1] = comp(xn[2 * (r - 1) + 0]);
                xp[r - 1] = comp(xn[2 * (r - 1) + 1]);
                ym[r - 1] = comp(col[j + R - r]);
                yp[r - 1] = comp(col[j + R + r]);
                zm[r - 1] = comp(w[f][j][(R - r + u) % W].p[p]);
                zp[r - 1] = comp(w[f][j][(R + r + u) % W].p[p]);
              }
              lap[j][f][c] = lap_from<T, ORDER>(comp(w[f][j][(R + u) % W].p[p]), xm, xp, ym, yp, zm, zp, a.inv_h2);
            }
          }
        }
#pragma unroll
        for (int j = 0; j < RY; ++j) {
          P wc[NF], pc[NPA], opsi[NOUT], opi[NOUT];
#pragma unroll
          for (int f = 0; f < NF; ++f) wc[f] = w[f][j][(R + u) % W].p[p];
#pragma unroll
          for (int q = 0; q < NPA; ++q) pc[q] = pv[j][q].p[p];
          rk_cell<T, MODE>(a, lap[j], wc, pc, opsi, opi);
#pragma unroll
          for (int q = 0; q < NOUT; ++q) {
            o_psi[j][q].p[p] = opsi[q];
            o_pi[j][q].p[p] = opi[q];
          }
        }
      }
      const int z = t.z0 + zz;
      const long long gz = !wr ? 0 : (z < R ? (long long)b.n[2] * plane : (z >= b.n[2] - R ? -(long long)b.n[2] * plane : 0));
#pragma unroll
      for (int j = 0; j < RY; ++j)
        if (active[j]) {
          const long long oo = off + (long long)zz * plane + (long long)j * b.sx;
#pragma unroll
          for (int q = 0; q < NOUT; ++q) {
            stg16<T>(a.out_psi[q] + oo, o_psi[j][q]);
            stg16<T>(a.out_pi[q] + oo, o_pi[j][q]);
          }
          if (wr) {  // periodic images that are star ghost cells of this box
            if (gz != 0) {
#pragma unroll
              for (int q = 0; q < NOUT; ++q) {
                stg16<T>(a.out_psi[q] + oo + gz, o_psi[j][q]);
                stg16<T>(a.out_pi[q] + oo + gz, o_pi[j][q]);
              }
            }
            if (gy_lo[j] || gy_hi[j]) {
              const long long gy = (gy_lo[j] ? (long long)b.n[1] : -(long long)b.n[1]) * b.sx;
#pragma unroll
              for (int q = 0; q < NOUT; ++q) {
                stg16<T>(a.out_psi[q] + oo + gy, o_psi[j][q]);
                stg16<T>(a.out_pi[q] + oo + gy, o_pi[j][q]);
              }
            }
            if (gx_lo | gx_hi) {
#pragma unroll
              for (int p = 0; p < CPT; ++p)
                if (((gx_lo | gx_hi) >> p) & 1) {
                  const long long gx = oo + p + (((gx_lo >> p) & 1) ? b.n[0] : -b.n[0]);
#pragma unroll
                  for (int q = 0; q < NOUT; ++q) {
                    a.out_psi[q][gx] = o_psi[j][q].p[p];
                    a.out_pi[q][gx] = o_pi[j][q].p[p];
                  }
                }
            }
          }
        }
    }
    slot_c = slot_c + 1 == S ? 0 : slot_c + 1;
    if (slot_t + 1 == S) {
      slot_t = 0;
      par_t ^= 1u;
    } else {
      ++slot_t;
    }
    slot_n = slot_n + 1 == S ? 0 : slot_n + 1;
  };
  for (int zz0 = 0; zz0 < t.nz; zz0 += W)
    static_for<W>([&](auto uc) {
      if (zz0 + decltype(uc)::value < t.nz) step(zz0 + decltype(uc)::value, uc);  // uniform over the CTA
    });
}

}  // namespace sledge
