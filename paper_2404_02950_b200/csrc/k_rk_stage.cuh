// k_rk_stage.cuh -- K1: fused Laplacian + Mexican-hat potential + RK4 stage update.
//
// What it computes (Eq.10-11; Laplacian<order> L649; RK4 = integrator.type 4, L808):
//   k_psi_c = Pi_c(U)
//   k_Pi_c  = Lap_h psi_c(U) - psi_c (lambda eta_s^2 (psi1^2 + psi2^2 - 1) + a) - (kappa/eta_s) Pi_c(U)
// and one of the stage updates below, for every valid cell of every box of a level in ONE launch.
//
// Data flow per cell-stage (words = reals, R + W):
//   LEAN    (52 words / cell-step)   S1: U2 = Y + dt/2 k            4R + 4W
//                                    S2: U3 = Y + dt/2 k            8R + 4W
//                                    S3: U4 = Y + dt k              8R + 4W
//                                    S4: Ynew = (U2 + 2U3 + U4 - Y)/3 + dt/6 k   16R + 4W
//   CLASSIC (64 words / cell-step)   S1: U2 = Y + dt/2 k ; ACC = Y + dt/6 k      4R + 8W
//                                    S2/S3: U = Y + a dt k ; ACC += dt/3 k       12R + 8W
//                                    S4: Ynew = ACC + dt/6 k                     8R + 4W
// (LEAN S4 is the classic combination rewritten with dt k1 = 2(U2-Y), dt k2 = 2(U3-Y), dt k3 = U4-Y.)
//
// Mapping: a CTA owns a TXC x TY column tile of one box and marches along z.  Each thread keeps the
// 2R+1 z-window of its own psi column in registers; only the centre plane goes through shared memory
// (double buffered, one __syncthreads per plane) so that x/y neighbours come from on-chip memory.
// Everything that is not differenced (Pi, Y, U2, U3, ACC) streams HBM -> registers -> HBM with 16-byte
// accesses, prefetched one plane ahead so that >= 9 independent 16-byte loads per thread are in flight.
#pragma once
#include "layout.h"

namespace sledge {

enum StageMode {
  LEAN_S1 = 0,
  LEAN_S23 = 1,
  LEAN_S4 = 2,
  CLASSIC_S1 = 3,
  CLASSIC_S23 = 4,
  CLASSIC_S4 = 5
};

template <int MODE> struct ModeInfo;
// NIN: pointwise input buffers besides the stage state U;  NOUT: output buffers
template <> struct ModeInfo<LEAN_S1> { static constexpr int NIN = 0, NOUT = 1; };
template <> struct ModeInfo<LEAN_S23> { static constexpr int NIN = 1, NOUT = 1; };
template <> struct ModeInfo<LEAN_S4> { static constexpr int NIN = 3, NOUT = 1; };
template <> struct ModeInfo<CLASSIC_S1> { static constexpr int NIN = 0, NOUT = 2; };
template <> struct ModeInfo<CLASSIC_S23> { static constexpr int NIN = 2, NOUT = 2; };
template <> struct ModeInfo<CLASSIC_S4> { static constexpr int NIN = 1, NOUT = 1; };

template <typename T>
struct StageArgs {
  using P = typename PairOf<T>::type;
  const BoxDev* boxes;
  const TileDev* tiles;
  const P* u_psi;      // stage state U: differenced
  const P* u_pi;
  const P* in_psi[3];  // pointwise inputs (meaning depends on MODE)
  const P* in_pi[3];
  P* out_psi[2];
  P* out_pi[2];
  int g, ox;
  T inv_h2;      // 1/h^2 (order 1) or 1/(12 h^2) (order 2)
  T lam_eta2;    // lambda * eta_s^2
  T a_mass;
  T fric;        // kappa / eta_s
  T adt;         // a_s * dt (S1-S3) or dt/6 (S4)
  T bdt;         // classic: b_s * dt for the accumulator
};

template <typename T, int ORDER>
__device__ __forceinline__ T lap_from(T u, const T* xm, const T* xp, const T* ym, const T* yp, const T* zm,
                                      const T* zp, T inv_h2) {
  // same association as the definition: sum_d [(u+ - u) + (u- - u)], x then y then z
  T n1x = (xp[0] - u) + (xm[0] - u);
  T n1y = (yp[0] - u) + (ym[0] - u);
  T n1z = (zp[0] - u) + (zm[0] - u);
  T s1 = (n1x + n1y) + n1z;
  if (ORDER == 1) return s1 * inv_h2;
  T n2x = (xp[1] - u) + (xm[1] - u);
  T n2y = (yp[1] - u) + (ym[1] - u);
  T n2z = (zp[1] - u) + (zm[1] - u);
  T s2 = (n2x + n2y) + n2z;
  return (T(16) * s1 - s2) * inv_h2;
}

template <typename T, int ORDER, int MODE, int TX, int TY>
__global__ void __launch_bounds__(TX* TY) k_rk_stage(const StageArgs<T> a) {
  using P = typename PairOf<T>::type;
  using V = Vec16<T>;
  constexpr int R = ORDER;
  constexpr int CPT = V::CPT;
  constexpr int TXC = TX * CPT;
  constexpr int SW = TXC + 2 * R;
  constexpr int SH = TY + 2 * R;
  constexpr int NT = TX * TY;
  constexpr int NH = 2 * R * (TXC + TY);  // halo pairs per plane (star stencil: no corners)
  constexpr int HPT = (NH + NT - 1) / NT;
  constexpr int NIN = ModeInfo<MODE>::NIN;
  constexpr int NOUT = ModeInfo<MODE>::NOUT;

  __shared__ P sm[2][SH * SW];

  const TileDev t = a.tiles[blockIdx.x];
  const BoxDev b = a.boxes[t.box];
  const int tid = threadIdx.x;
  const int tx = tid % TX, ty = tid / TX;
  const int x = t.x0 + tx * CPT, y = t.y0 + ty;
  const bool active = (x < b.n[0]) && (y < b.n[1]);
  // in a partial tile the columns/rows just past the box edge are ghost cells that the edge cells need as
  // +x / +y neighbours: threads sitting there still stream their psi column through shared memory
  const bool loader = (x < b.n[0] + R) && (y < b.n[1] + R);
  const long long plane = (long long)b.sx * b.sy;
  const long long tile_org = b.base + (long long)(t.z0 + a.g) * plane + (long long)(t.y0 + a.g) * b.sx + (t.x0 + a.ox);
  long long off = tile_org + (long long)ty * b.sx + tx * CPT;  // this thread's cell in plane z0

  // halo assignment: pair index -> (hx, hy) relative to the tile origin
  int h_goff[HPT];   // global offset relative to tile_org (within a plane)
  int h_soff[HPT];   // shared offset, -1 = none
#pragma unroll
  for (int q = 0; q < HPT; ++q) {
    int idx = tid + q * NT;
    int hx = 0, hy = 0;
    bool ok = idx < NH;
    if (idx < 2 * R * TXC) {  // bottom / top strips, x fastest
      int row = idx / TXC;    // 0..2R-1
      hx = idx % TXC;
      hy = (row < R) ? (row - R) : (TY + row - R);
    } else {
      int j = idx - 2 * R * TXC;  // left / right strips
      int col = j % (2 * R);
      hy = j / (2 * R);
      hx = (col < R) ? (col - R) : (TXC + col - R);
    }
    // stay inside the box's ghosted extent (partial tiles at the high end of a box)
    ok = ok && (t.x0 + hx < b.n[0] + R) && (t.y0 + hy < b.n[1] + R);
    h_goff[q] = hy * b.sx + hx;
    h_soff[q] = ok ? ((hy + R) * SW + (hx + R)) : -1;
  }

  const int s_own = (ty + R) * SW + (tx * CPT + R);

  // z-window of the own column: w[m] = psi(z + m - R)
  V w[2 * R + 1];
#pragma unroll
  for (int m = 0; m < 2 * R; ++m) {
    if (loader) w[m + 1] = ldg16_stream<T>(a.u_psi + off + (long long)(m - R) * plane);
  }
  // prefetch registers for the first plane
  V n_psi, n_upi, n_in_psi[NIN > 0 ? NIN : 1], n_in_pi[NIN > 0 ? NIN : 1];
  P n_halo[HPT];
  if (loader) n_psi = ldg16_stream<T>(a.u_psi + off + (long long)R * plane);
  if (active) {
    n_upi = ldg16_stream<T>(a.u_pi + off);
#pragma unroll
    for (int q = 0; q < NIN; ++q) {
      n_in_psi[q] = ldg16_stream<T>(a.in_psi[q] + off);
      n_in_pi[q] = ldg16_stream<T>(a.in_pi[q] + off);
    }
  }
#pragma unroll
  for (int q = 0; q < HPT; ++q)
    if (h_soff[q] >= 0) n_halo[q] = a.u_psi[tile_org + h_goff[q]];

  for (int zz = 0; zz < t.nz; ++zz) {
    P* s = sm[zz & 1];
    // shift the window, take delivery of the prefetched plane
#pragma unroll
    for (int m = 0; m < 2 * R; ++m) w[m] = w[m + 1];
    w[2 * R] = n_psi;
    const V upi = n_upi;
    V in_psi[NIN > 0 ? NIN : 1], in_pi[NIN > 0 ? NIN : 1];
#pragma unroll
    for (int q = 0; q < NIN; ++q) {
      in_psi[q] = n_in_psi[q];
      in_pi[q] = n_in_pi[q];
    }
    // centre plane -> shared
    if (loader) {
#pragma unroll
      for (int p = 0; p < CPT; ++p) s[s_own + p] = w[R].p[p];
    }
#pragma unroll
    for (int q = 0; q < HPT; ++q)
      if (h_soff[q] >= 0) s[h_soff[q]] = n_halo[q];
    __syncthreads();

    // issue next plane's loads before computing this one
    if (zz + 1 < t.nz) {
      const long long o1 = off + plane;
      if (loader) n_psi = ldg16_stream<T>(a.u_psi + o1 + (long long)R * plane);
      if (active) {
        n_upi = ldg16_stream<T>(a.u_pi + o1);
#pragma unroll
        for (int q = 0; q < NIN; ++q) {
          n_in_psi[q] = ldg16_stream<T>(a.in_psi[q] + o1);
          n_in_pi[q] = ldg16_stream<T>(a.in_pi[q] + o1);
        }
      }
      const long long h1 = tile_org + (long long)(zz + 1) * plane;
#pragma unroll
      for (int q = 0; q < HPT; ++q)
        if (h_soff[q] >= 0) n_halo[q] = a.u_psi[h1 + h_goff[q]];
    }

    if (active) {
      V o_psi[NOUT], o_pi[NOUT];
#pragma unroll
      for (int p = 0; p < CPT; ++p) {
        const int sc = s_own + p;
        T lap[2];
#pragma unroll
        for (int c = 0; c < 2; ++c) {
          auto comp = [c](const P& v) -> T { return c == 0 ? v.x : v.y; };
          T xm[2], xp[2], ym[2], yp[2], zm[2], zp[2];
#pragma unroll
          for (int r = 1; r <= R; ++r) {
            xm[r - 1] = comp(s[sc - r]);
            xp[r - 1] = comp(s[sc + r]);
            ym[r - 1] = comp(s[sc - r * SW]);
            yp[r - 1] = comp(s[sc + r * SW]);
            zm[r - 1] = comp(w[R - r].p[p]);
            zp[r - 1] = comp(w[R + r].p[p]);
          }
          lap[c] = lap_from<T, ORDER>(comp(w[R].p[p]), xm, xp, ym, yp, zm, zp, a.inv_h2);
        }
        const T psi1 = w[R].p[p].x, psi2 = w[R].p[p].y;
        const T pi1 = upi.p[p].x, pi2 = upi.p[p].y;
        const T pot = a.lam_eta2 * ((psi1 * psi1 + psi2 * psi2) - T(1)) + a.a_mass;
        const T kpsi1 = pi1, kpsi2 = pi2;
        const T kpi1 = (lap[0] - psi1 * pot) - a.fric * pi1;
        const T kpi2 = (lap[1] - psi2 * pot) - a.fric * pi2;

        if (MODE == LEAN_S1) {  // U2 = U + adt k   (U = Y)
          o_psi[0].p[p] = mkpair(psi1 + a.adt * kpsi1, psi2 + a.adt * kpsi2);
          o_pi[0].p[p] = mkpair(pi1 + a.adt * kpi1, pi2 + a.adt * kpi2);
        } else if (MODE == LEAN_S23) {  // U' = Y + adt k   (in0 = Y)
          o_psi[0].p[p] = mkpair(in_psi[0].p[p].x + a.adt * kpsi1, in_psi[0].p[p].y + a.adt * kpsi2);
          o_pi[0].p[p] = mkpair(in_pi[0].p[p].x + a.adt * kpi1, in_pi[0].p[p].y + a.adt * kpi2);
        } else if (MODE == LEAN_S4) {  // in0 = Y, in1 = U2, in2 = U3, U = U4, adt = dt/6
          const T third = T(1) / T(3);
          auto comb = [&](T yv, T u2, T u3, T u4, T kk) -> T {
            return (((u2 + T(2) * u3) + u4) - yv) * third + a.adt * kk;
          };
          o_psi[0].p[p] = mkpair(comb(in_psi[0].p[p].x, in_psi[1].p[p].x, in_psi[2].p[p].x, psi1, kpsi1),
                                 comb(in_psi[0].p[p].y, in_psi[1].p[p].y, in_psi[2].p[p].y, psi2, kpsi2));
          o_pi[0].p[p] = mkpair(comb(in_pi[0].p[p].x, in_pi[1].p[p].x, in_pi[2].p[p].x, pi1, kpi1),
                                comb(in_pi[0].p[p].y, in_pi[1].p[p].y, in_pi[2].p[p].y, pi2, kpi2));
        } else if (MODE == CLASSIC_S1) {  // out0 = U + adt k ; out1 (ACC) = U + bdt k
          o_psi[0].p[p] = mkpair(psi1 + a.adt * kpsi1, psi2 + a.adt * kpsi2);
          o_pi[0].p[p] = mkpair(pi1 + a.adt * kpi1, pi2 + a.adt * kpi2);
          o_psi[1].p[p] = mkpair(psi1 + a.bdt * kpsi1, psi2 + a.bdt * kpsi2);
          o_pi[1].p[p] = mkpair(pi1 + a.bdt * kpi1, pi2 + a.bdt * kpi2);
        } else if (MODE == CLASSIC_S23) {  // in0 = Y, in1 = ACC ; out0 = Y + adt k ; out1 = ACC + bdt k
          o_psi[0].p[p] = mkpair(in_psi[0].p[p].x + a.adt * kpsi1, in_psi[0].p[p].y + a.adt * kpsi2);
          o_pi[0].p[p] = mkpair(in_pi[0].p[p].x + a.adt * kpi1, in_pi[0].p[p].y + a.adt * kpi2);
          o_psi[1].p[p] = mkpair(in_psi[1].p[p].x + a.bdt * kpsi1, in_psi[1].p[p].y + a.bdt * kpsi2);
          o_pi[1].p[p] = mkpair(in_pi[1].p[p].x + a.bdt * kpi1, in_pi[1].p[p].y + a.bdt * kpi2);
        } else {  // CLASSIC_S4: in0 = ACC ; out0 = ACC + adt k
          o_psi[0].p[p] = mkpair(in_psi[0].p[p].x + a.adt * kpsi1, in_psi[0].p[p].y + a.adt * kpsi2);
          o_pi[0].p[p] = mkpair(in_pi[0].p[p].x + a.adt * kpi1, in_pi[0].p[p].y + a.adt * kpi2);
        }
      }
#pragma unroll
      for (int q = 0; q < NOUT; ++q) {
        stg16<T>(a.out_psi[q] + off, o_psi[q]);
        stg16<T>(a.out_pi[q] + off, o_pi[q]);
      }
    }
    off += plane;
  }
}

}  // namespace sledge
