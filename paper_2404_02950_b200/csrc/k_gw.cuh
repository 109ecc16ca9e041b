// k_gw.cuh -- K1 for the gravitational-wave auxiliary fields (Eq.16; R25).
//
// With sim.gravitational_waves every cell carries, beside (psi1, psi2, Pi1, Pi2), the six auxiliary fields u_ij and
// their momenta du_ij (ij = xx, yy, zz, xy, xz, yz; L436).  One stage of classic RK4 (L808) of
//   k_u_ij  = du_ij
//   k_du_ij = -(kappa_u / eta_s) du_ij + Lap_h u_ij + c_gw T_ij,      T_ij = sum_c d_i psi_c d_j psi_c
// with Laplacian<order> (L649) and Gradient<order> (L651-658: 3-, 5-, 7-point central first differences), combined in
// the LEAN data-flow of k_rk_pipe.cuh (same buffers as the scalar sector):
//   S1:  U2 = U + dt/2 k        S2/S3: U' = Y + a dt k        S4: Ynew = (U2 + 2 U3 + U4 - Y)/3 + dt/6 k   (U = U4)
// Storage: six pair planes per state buffer, (u_xx,u_yy) (u_zz,u_xy) (u_xz,u_yz) and the same for du, each laid out
// exactly like the (psi1,psi2) plane, so that K2 and K4 serve them unchanged.
//
// Mapping: a CTA owns a 32 x GW_TY column tile of one box and ONE of the three pair planes (blockIdx.y) and marches
// along z; a thread keeps the 2R+1 z-window of its cell of the two differenced planes (psi and its u plane) in
// registers and reads the x/y neighbours of the centre plane through the read-only L1 path (the tile's rows are
// 512-byte runs that the CTA's own threads have just pulled in).  psi is read by all three CTAs of a tile (through
// L2).  Words per cell-stage: 2 (psi) + 12 (U) + 12 per pointwise input state + 12 written.
// (One CTA for all three planes needs four z-windows: 255 registers, one CTA per SM, 39 % of the HBM roofline.)
// No shared-memory staging; the loads that miss L1 (window tops, du, Y of stages 2-3) are issued one plane ahead.
#pragma once
#include "k_rk_pipe.cuh"

namespace sledge {

#ifndef SLEDGE_GW_TY
#define SLEDGE_GW_TY 8
#endif
constexpr int GW_TX = 32, GW_TY = SLEDGE_GW_TY;  // = the fused-sweep tile (sledge.cu asserts it)

template <typename T>
struct GwArgs {
  using P = typename PairOf<T>::type;
  const BoxDev* boxes;
  const TileDev* tiles;   // the level's fused-sweep tiles: (32 * cells per 16 bytes) x 8 columns, z-chunks
  const P* psi;           // (psi1,psi2) of the stage input U, ghosts filled
  const P* u[3];          // u pair planes of U, ghosts filled
  const P* du[3];         // du pair planes of U
  const P* in[3][6];      // S2/S3: in[0] = Y;  S4: in[0] = Y, in[1] = U2, in[2] = U3  (u planes 0..2, du planes 3..5)
  P* out[6];
  int g, ox;
  T inv_h2;    // Laplacian scale, as in PipeArgs
  T inv_h;     // gradient scale: 1/(2h), 1/(12h), 1/(60h) for order 1, 2, 3
  T coupling;  // c_gw
  T fric;      // kappa_u / eta_s
  T adt;       // a_s dt (S1-S3), dt/6 (S4)
};

// Gradient<order> of one component from its neighbours at +-1..+-R along one axis (difference form, as the oracle)
template <typename T, int ORDER>
__device__ __forceinline__ T grad_from(const T* m, const T* p, T inv_h) {
  if (ORDER == 1) return (p[0] - m[0]) * inv_h;
  if (ORDER == 2) return (T(8) * (p[0] - m[0]) - (p[1] - m[1])) * inv_h;
  return ((T(45) * (p[0] - m[0]) - T(9) * (p[1] - m[1])) + (p[2] - m[2])) * inv_h;
}

#ifndef SLEDGE_GW_MINB
#define SLEDGE_GW_MINB 2
#endif
template <typename T, int ORDER, int MODE>
__global__ void __launch_bounds__(GW_TX* GW_TY, (sizeof(T) == 8 && ORDER == 3) ? 1 : SLEDGE_GW_MINB) k_gw_stage(const GwArgs<T> a) {
  using P = typename PairOf<T>::type;
  constexpr int R = ORDER;
  constexpr int CPT = Vec16<T>::CPT;  // the tiles are 32 * CPT cells wide: CPT passes over x
  constexpr int NIN = MODE == LEAN_S1 ? 0 : (MODE == LEAN_S4 ? 3 : 1);
  const TileDev t = a.tiles[blockIdx.x];
  const BoxDev b = a.boxes[t.box];
  const int q = blockIdx.y;  // which u / du pair plane: 0 = (xx,yy), 1 = (zz,xy), 2 = (xz,yz)
  const int tx = threadIdx.x % GW_TX, ty = threadIdx.x / GW_TX;
  const int y = t.y0 + ty;
  if (y >= b.n[1]) return;
  const long long plane = (long long)b.sx * b.sy;
  for (int px = 0; px < CPT; ++px) {
    const int x = t.x0 + px * GW_TX + tx;
    if (x >= b.n[0]) continue;
    const long long off = b.base + (long long)(t.z0 + a.g) * plane + (long long)(y + a.g) * b.sx + (x + a.ox);
    // z-windows of the two differenced planes: w[0] = psi, w[1] = this CTA's u pair plane; w[f][m] = plane z + m - R
    const P* const src[2] = {a.psi, a.u[q]};
    P w[2][2 * R + 1];
#pragma unroll
    for (int f = 0; f < 2; ++f)
#pragma unroll
      for (int m = 0; m < 2 * R; ++m) w[f][m + 1] = __ldg(src[f] + off + (long long)(m - R) * plane);
    // the loads that come from HBM (top of the two z-windows, du, the pointwise stage inputs) are issued one plane
    // ahead: a warp that needs them in the same iteration waits a full memory latency per plane
    P nxt[2], dv_n, yu_n = mkpair(T(0), T(0)), yd_n = mkpair(T(0), T(0));
#pragma unroll
    for (int f = 0; f < 2; ++f) nxt[f] = __ldg(src[f] + off + (long long)R * plane);
    dv_n = __ldg(a.du[q] + off);
    if (MODE == LEAN_S23) {
      yu_n = __ldg(a.in[0][q] + off);
      yd_n = __ldg(a.in[0][3 + q] + off);
    }
    for (int zz = 0; zz < t.nz; ++zz) {
      const long long o = off + (long long)zz * plane;
      const bool more = zz + 1 < t.nz;
#pragma unroll
      for (int f = 0; f < 2; ++f) {
#pragma unroll
        for (int m = 0; m < 2 * R; ++m) w[f][m] = w[f][m + 1];
        w[f][2 * R] = nxt[f];
        if (more) nxt[f] = __ldg(src[f] + o + (long long)(R + 1) * plane);
      }
      const P dv = dv_n;
      const P yu = yu_n, yd = yd_n;
      P yv[NIN > 0 ? NIN : 1][2];
      // S4 inputs: not prefetched (measured: no gain, spills with the 13-point windows); plain loads, because in[1]
      // (U2) is the plane this stage overwrites in place
      if (MODE == LEAN_S4) {
#pragma unroll
        for (int m = 0; m < NIN; ++m) {
          yv[m][0] = a.in[m][q][o];
          yv[m][1] = a.in[m][3 + q][o];
        }
      }
      if (more) {
        dv_n = __ldg(a.du[q] + o + plane);
        if (MODE == LEAN_S23) {
          yu_n = __ldg(a.in[0][q] + o + plane);
          yd_n = __ldg(a.in[0][3 + q] + o + plane);
        }
      }
      // x / y neighbours of the centre plane
      P xm[2][R], xp[2][R], ym[2][R], yp[2][R];
#pragma unroll
      for (int f = 0; f < 2; ++f)
#pragma unroll
        for (int r = 1; r <= R; ++r) {
          xm[f][r - 1] = __ldg(src[f] + o - r);
          xp[f][r - 1] = __ldg(src[f] + o + r);
          ym[f][r - 1] = __ldg(src[f] + o - (long long)r * b.sx);
          yp[f][r - 1] = __ldg(src[f] + o + (long long)r * b.sx);
        }
      // gradients of psi1, psi2 -> T_ij
      T gr[2][3];
#pragma unroll
      for (int c = 0; c < 2; ++c) {
        auto comp = [c](const P& v) -> T { return c == 0 ? v.x : v.y; };
        T m[3], p[3];
#pragma unroll
        for (int r = 0; r < R; ++r) { m[r] = comp(xm[0][r]); p[r] = comp(xp[0][r]); }
        gr[c][0] = grad_from<T, ORDER>(m, p, a.inv_h);
#pragma unroll
        for (int r = 0; r < R; ++r) { m[r] = comp(ym[0][r]); p[r] = comp(yp[0][r]); }
        gr[c][1] = grad_from<T, ORDER>(m, p, a.inv_h);
#pragma unroll
        for (int r = 0; r < R; ++r) { m[r] = comp(w[0][R - 1 - r]); p[r] = comp(w[0][R + 1 + r]); }
        gr[c][2] = grad_from<T, ORDER>(m, p, a.inv_h);
      }
      {  // pair plane q holds components 2q, 2q + 1
        T ku[2], kdu[2], uc[2], duc[2];
#pragma unroll
        for (int c = 0; c < 2; ++c) {
          auto comp = [c](const P& v) -> T { return c == 0 ? v.x : v.y; };
          const int mc = 2 * q + c;
          T xm_[3], xp_[3], ym_[3], yp_[3], zm_[3], zp_[3];
#pragma unroll
          for (int r = 0; r < R; ++r) {
            xm_[r] = comp(xm[1][r]);
            xp_[r] = comp(xp[1][r]);
            ym_[r] = comp(ym[1][r]);
            yp_[r] = comp(yp[1][r]);
            zm_[r] = comp(w[1][R - 1 - r]);
            zp_[r] = comp(w[1][R + 1 + r]);
          }
          uc[c] = comp(w[1][R]);
          duc[c] = comp(dv);
          const T lap = lap_from<T, ORDER>(uc[c], xm_, xp_, ym_, yp_, zm_, zp_, a.inv_h2);
          // (i, j) of component mc in the order xx, yy, zz, xy, xz, yz (L436), one hex digit each
          const int gi = (0x100210 >> (4 * mc)) & 3, gj = (0x221210 >> (4 * mc)) & 3;
          auto pick = [](const T* v, int d) -> T { return d == 0 ? v[0] : (d == 1 ? v[1] : v[2]); };
          const T Tij = pick(gr[0], gi) * pick(gr[0], gj) + pick(gr[1], gi) * pick(gr[1], gj);
          ku[c] = duc[c];
          kdu[c] = (lap + a.coupling * Tij) - a.fric * duc[c];
        }
        P ou, odu;
        if (MODE == LEAN_S1) {
          ou = mkpair(fma(a.adt, ku[0], uc[0]), fma(a.adt, ku[1], uc[1]));
          odu = mkpair(fma(a.adt, kdu[0], duc[0]), fma(a.adt, kdu[1], duc[1]));
        } else if (MODE == LEAN_S23) {
          ou = mkpair(fma(a.adt, ku[0], yu.x), fma(a.adt, ku[1], yu.y));
          odu = mkpair(fma(a.adt, kdu[0], yd.x), fma(a.adt, kdu[1], yd.y));
        } else {  // LEAN_S4: (U2 + 2 U3 + U4 - Y)/3 + dt/6 k
          const T third = T(1) / T(3);
          auto comb = [&](T y0, T u2, T u3, T u4, T kk) -> T { return fma(a.adt, kk, ((fma(T(2), u3, u2) + u4) - y0) * third); };
          ou = mkpair(comb(yv[0][0].x, yv[1][0].x, yv[2][0].x, uc[0], ku[0]), comb(yv[0][0].y, yv[1][0].y, yv[2][0].y, uc[1], ku[1]));
          odu = mkpair(comb(yv[0][1].x, yv[1][1].x, yv[2][1].x, duc[0], kdu[0]), comb(yv[0][1].y, yv[1][1].y, yv[2][1].y, duc[1], kdu[1]));
        }
        a.out[q][o] = ou;
        a.out[3 + q][o] = odu;
      }
    }
  }
}

template <typename T, int ORDER>
int launch_gw(cudaStream_t stream, const GwArgs<T>& a, int grid, int mode) {
  const int nt = GW_TX * GW_TY;
  const dim3 g3(grid, 3);  // y: the three pair planes
  if (mode == LEAN_S1) k_gw_stage<T, ORDER, LEAN_S1><<<g3, nt, 0, stream>>>(a);
  else if (mode == LEAN_S23) k_gw_stage<T, ORDER, LEAN_S23><<<g3, nt, 0, stream>>>(a);
  else if (mode == LEAN_S4) k_gw_stage<T, ORDER, LEAN_S4><<<g3, nt, 0, stream>>>(a);
  else return 1;
  return 0;
}

}  // namespace sledge
