// k_rk_pipe.cuh -- K1: fused Laplacian + Mexican-hat potential + RK4 stage update(s), cp.async-pipelined.
//
// What it computes (Eq.10-11; Laplacian<order> L649; RK4 = integrator.type 4, L808):
//   k_psi_c = Pi_c(U)
//   k_Pi_c  = Lap_h psi_c(U) - psi_c (lambda eta_s^2 (psi1^2 + psi2^2 - 1) + a) - (kappa/eta_s) Pi_c(U)
// for every valid cell of every box of a level in ONE launch, combined into one of the data-flows below.
//
// Data-flows (words = reals moved per cell, R + W):
//   LEAN    (52 words / cell-step)   S1: U2 = Y + dt/2 k                         4R + 4W
//                                    S2: U3 = Y + dt/2 k                         8R + 4W
//                                    S3: U4 = Y + dt k                           8R + 4W
//                                    S4: Ynew = (U2 + 2U3 + U4 - Y)/3 + dt/6 k   16R + 4W
//   CLASSIC (64 words / cell-step)   S1: U2 = Y + dt/2 k ; ACC = Y + dt/6 k      4R + 8W
//                                    S2/S3: U = Y + a dt k ; ACC += dt/3 k       12R + 8W
//                                    S4: Ynew = ACC + dt/6 k                     8R + 4W
//   FUSED   (20 words / cell-step)   two stages per sweep.  Because k_psi = Pi is pointwise, the NEXT stage's psi
//     is known at every neighbour from the current stage's (psi, Pi) there, and the Laplacian is linear:
//       PASS A (stages 1+2):  Lap psi2 = Lap psi_Y + dt/2 Lap Pi_Y              4R + 4W   -> U3
//       PASS B (stages 3+4):  Lap psi4 = Lap psi_Y + dt   Lap Pi3               8R + 4W   -> Ynew
//     PASS B recomputes k1 from Y (same expression as PASS A, same bits) and recovers dt/2 k2 = Pi3 - Pi_Y.
//     Pi is differenced here, so the ghost fill must fill Pi ghosts too (same-level / periodic copies).
//
// Mapping: a CTA owns a TXC x TY column tile of one box and marches along z.  Each thread keeps the 2R+1
// z-window of its own column of every differenced field in registers; only the centre planes go through
// shared memory (double buffered, one __syncthreads per plane) so that x/y neighbours come from on-chip
// memory.  ALL global loads are 16-byte cp.async (LDGSTS) into a D-stage shared-memory ring issued D planes
// ahead, so the bytes in flight do not occupy registers: own-column values of the differenced fields for
// plane z+R, pointwise inputs for plane z, and the x/y halo of plane z.  Outputs go registers -> HBM with
// 16-byte stores.
#pragma once
#include "layout.h"

namespace sledge {

enum StageMode {
  LEAN_S1 = 0,
  LEAN_S23 = 1,
  LEAN_S4 = 2,
  CLASSIC_S1 = 3,
  CLASSIC_S23 = 4,
  CLASSIC_S4 = 5,
  FUSED_A = 6,
  FUSED_B = 7,
  SSP_S23 = 8,  // SSPRK3 (integrator.type 3 / 10, L808) stages 2 and 3: out = wy Y + wu (U + dt k(U)); stage 1 = LEAN_S1
  FUSED_A2 = 10,  // fp64 FUSED sweeps, "W" form (see rk_cell): sweep A stores W = 2 psi_Y + dt Pi_3 in place of Pi_3,
  FUSED_B2 = 11,  // so that sweep B differences two fields (psi_3, W) instead of three (psi_3, Pi_3, psi_Y)
  RKN_ST = 9    // one stage of a user-defined Runge-Kutta-Nystrom scheme (integrator.type 20, L808-815): f = f(Psi_i), and
                // two linear combinations of psi_n, Pi_n, f_1 .. f_4 and f (the stage's f and the next stage field, or
                // the new psi and Pi)
};

template <int MODE> struct ModeInfo;
// NF: differenced (stencil) fields; NP: pointwise inputs (pairs); NOUT: output states (psi + pi each)
template <> struct ModeInfo<LEAN_S1> { static constexpr int NF = 1, NP = 1, NOUT = 1; };
template <> struct ModeInfo<LEAN_S23> { static constexpr int NF = 1, NP = 3, NOUT = 1; };
template <> struct ModeInfo<LEAN_S4> { static constexpr int NF = 1, NP = 7, NOUT = 1; };
template <> struct ModeInfo<CLASSIC_S1> { static constexpr int NF = 1, NP = 1, NOUT = 2; };
template <> struct ModeInfo<CLASSIC_S23> { static constexpr int NF = 1, NP = 5, NOUT = 2; };
template <> struct ModeInfo<CLASSIC_S4> { static constexpr int NF = 1, NP = 3, NOUT = 1; };
template <> struct ModeInfo<SSP_S23> { static constexpr int NF = 1, NP = 3, NOUT = 1; };
template <> struct ModeInfo<RKN_ST> { static constexpr int NF = 1, NP = 6, NOUT = 1; };
template <> struct ModeInfo<FUSED_A> { static constexpr int NF = 2, NP = 0, NOUT = 1; };
template <> struct ModeInfo<FUSED_B> { static constexpr int NF = 3, NP = 1, NOUT = 1; };
template <> struct ModeInfo<FUSED_A2> { static constexpr int NF = 2, NP = 0, NOUT = 1; };
template <> struct ModeInfo<FUSED_B2> { static constexpr int NF = 2, NP = 2, NOUT = 1; };

// Field roles.  Unfused modes: sten[0] = psi(U); pnt[0] = Pi(U); pnt[1+2q], pnt[2+2q] = psi, Pi of input q
// (LEAN: q0 = Y, q1 = U2, q2 = U3; CLASSIC: q0 = Y (S23) or ACC (S4), q1 = ACC).
// FUSED_A: sten = {psi_Y, Pi_Y}.  FUSED_B: sten = {psi_3, Pi_3, psi_Y}, pnt[0] = Pi_Y.
// FUSED_A2: as FUSED_A, second output plane = W.  FUSED_B2: sten = {psi_3, W}, pnt = {psi_Y, Pi_Y}, wu = 1 / dt.
template <typename T>
struct PipeArgs {
  using P = typename PairOf<T>::type;
  const BoxDev* boxes;
  const TileDev* tiles;
  const P* sten[3];
  const void* tmap[3];  // k_rk_tma only: per differenced field, the tensor maps (CUtensorMap, one per box of the level) of
                         // the buffer plane sten[f] points at
  const P* pnt[7];
  P* out_psi[2];
  P* out_pi[2];
  int g, ox;
  int wrap;        // k_rk_plane only: the level is ONE box covering the periodic domain and the kernel wraps its halo /
                   // window addresses itself (L23), so no ghost fill is needed before the sweep
  T inv_h2;        // 1/h^2 (order 1), 1/(12 h^2) (order 2) or 1/(180 h^2) (order 3)
  T lam_eta2[3];   // lambda * eta^2 at t, t + dt/2, t + dt (unfused: [0] = the stage's value)
  T fric[3];       // kappa / eta at the same times
  T a_mass;
  T adt;           // unfused: a_s * dt (S1-S3) or dt/6 (S4);  fused: dt
  T bdt;           // classic: b_s * dt for the accumulator
  T wy, wu;        // SSP_S23: weights of Y and of the forward-Euler step from U (3/4, 1/4 and 1/3, 2/3)
  T rkn_w[2][7];   // RKN_ST: sten[0] = Psi_i; pnt[0] = psi_n, pnt[1] = Pi_n, pnt[2..5] = f_1 .. f_4 (null = absent);
                   // out_psi[0] = sum_q rkn_w[0][q] in_q + rkn_w[0][6] f,  out_pi[0] = the same with rkn_w[1]
  T ko_c[4];       // Kreiss-Oliger (Eq.7): (-1)^(r+1) eps_c / (2^(2r) h) for psi1, psi2, Pi1, Pi2; staged sweeps with
                   // KO != 0 only, where sten[1] = Pi(U) takes the place of pnt[0]
};

__device__ __forceinline__ void cp_async_16(void* smem, const void* gmem) {
  const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
#ifdef SLEDGE_CPASYNC_CA
  asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(s), "l"(gmem) : "memory");
#else
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(s), "l"(gmem) : "memory");
#endif
}
__device__ __forceinline__ void cp_async_pair(double2* smem, const double2* gmem) { cp_async_16(smem, gmem); }
__device__ __forceinline__ void cp_async_pair(float2* smem, const float2* gmem) {
  const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(s), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() {
  asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory");
}

// Laplacian of one component from its 6 (12) neighbours.  The library is compiled with --fmad=false (the tag
// rule needs individually rounded products); K1 is where the fp64 pipe matters, so it contracts explicitly:
// neighbour-sum form s_r = sum_d (u(+r e_d) + u(-r e_d)), then
//   order 1: (s1 - 6u) / h^2      order 2: (16 s1 - s2 - 90u) / (12 h^2)      order 3: (270 s1 - 27 s2 + 2 s3 - 1470u) / (180 h^2)
// 13 fp64 instructions for the 13-point stencil instead of 25 in difference form.  The result differs from the
// difference form sum_d [(u+ - u) + (u- - u)] by rounding only (|err| <~ 1e-15 / h^2 on O(1) fields; R11).
template <typename T, int ORDER>
__device__ __forceinline__ T lap_from(T u, const T* xm, const T* xp, const T* ym, const T* yp, const T* zm,
                                      const T* zp, T inv_h2) {
  const T s1 = ((xp[0] + xm[0]) + (yp[0] + ym[0])) + (zp[0] + zm[0]);
  if (ORDER == 1) return fma(T(-6), u, s1) * inv_h2;
  const T s2 = ((xp[1] + xm[1]) + (yp[1] + ym[1])) + (zp[1] + zm[1]);
  if (ORDER == 2) return fma(T(16), s1, fma(T(-90), u, -s2)) * inv_h2;
  // order 3, 19-point: (270 s1 - 27 s2 + 2 s3 - 1470 u) / (180 h^2)
  const T s3 = ((xp[2] + xm[2]) + (yp[2] + ym[2])) + (zp[2] + zm[2]);
  return fma(T(270), s1, fma(T(-27), s2, fma(T(2), s3, T(-1470) * u))) * inv_h2;
}

// Kreiss-Oliger term of one component (Eq.7, dissipation order r = KO in {2, 3}, p = 2r - 1): the 2r-th
// central differences along x, y, z in neighbour-sum form, s_m as in lap_from:
//   r = 2: s2 - 4 s1 + 18 u        r = 3: s3 - 6 s2 + 15 s1 - 60 u        times coef = (-1)^(r+1) eps / (2^(2r) h)
template <typename T, int KO>
__device__ __forceinline__ T ko_from(T u, const T* xm, const T* xp, const T* ym, const T* yp, const T* zm,
                                     const T* zp, T coef) {
  const T s1 = ((xp[0] + xm[0]) + (yp[0] + ym[0])) + (zp[0] + zm[0]);
  const T s2 = ((xp[1] + xm[1]) + (yp[1] + ym[1])) + (zp[1] + zm[1]);
  if (KO == 2) return fma(T(-4), s1, fma(T(18), u, s2)) * coef;
  const T s3 = ((xp[2] + xm[2]) + (yp[2] + ym[2])) + (zp[2] + zm[2]);
  return fma(T(15), s1, fma(T(-6), s2, fma(T(-60), u, s3))) * coef;
}

// k_Pi of one component (Eq.11 generalised, R2): lap - psi * pot - fric * pi, contracted
template <typename T>
__device__ __forceinline__ T kpi_of(T lap, T psi, T pot, T fric, T pi) {
  return fma(-fric, pi, fma(-psi, pot, lap));
}
// pot = lambda eta^2 (psi1^2 + psi2^2 - 1) + a
template <typename T>
__device__ __forceinline__ T pot_of(T lam_eta2, T a_mass, T p1, T p2) {
  return fma(lam_eta2, fma(p1, p1, fma(p2, p2, T(-1))), a_mass);
}

// One cell of one sweep: from the Laplacians lap[f][c] of the differenced fields, their centre values wc[f] and
// the pointwise inputs pc[q], the new state(s) opsi[q], opi[q] of the mode's data-flow (see the header).
// With HASKO (staged modes only) ko[c] = Q_l u_c of Eq.7 is added to the RHS of every component.
template <typename T, int MODE, bool HASKO = false>
__device__ __forceinline__ void rk_cell(const PipeArgs<T>& a, const T (&lap)[ModeInfo<MODE>::NF][2],
                                        const typename PairOf<T>::type (&wc)[ModeInfo<MODE>::NF],
                                        const typename PairOf<T>::type (&pc)[ModeInfo<MODE>::NP > 0 ? ModeInfo<MODE>::NP : 1],
                                        typename PairOf<T>::type (&opsi)[ModeInfo<MODE>::NOUT],
                                        typename PairOf<T>::type (&opi)[ModeInfo<MODE>::NOUT],
                                        const T* ko = nullptr) {
  using P = typename PairOf<T>::type;
  static_assert(!HASKO || (MODE != FUSED_A && MODE != FUSED_B && MODE != FUSED_A2 && MODE != FUSED_B2),
                "the fused sweeps rely on k_psi = Pi being pointwise");
  constexpr int NP = ModeInfo<MODE>::NP, NOUT = ModeInfo<MODE>::NOUT;
  constexpr int NPA = NP > 0 ? NP : 1;
  if (MODE == FUSED_A || MODE == FUSED_A2) {
    // stages 1 + 2 (O4): U3 = Y + dt/2 k(U2), U2 = Y + dt/2 k(Y); U2 is never stored
    const T hdt = T(0.5) * a.adt;
    const T y1 = wc[0].x, y2 = wc[0].y, q1 = wc[1].x, q2 = wc[1].y;
    const T pot1 = pot_of(a.lam_eta2[0], a.a_mass, y1, y2);
    const T k1a = kpi_of(lap[0][0], y1, pot1, a.fric[0], q1);
    const T k1b = kpi_of(lap[0][1], y2, pot1, a.fric[0], q2);
    const T p2a = fma(hdt, k1a, q1), p2b = fma(hdt, k1b, q2);  // Pi(U2)
    const T u2a = fma(hdt, q1, y1), u2b = fma(hdt, q2, y2);    // psi(U2)
    const T l2a = fma(hdt, lap[1][0], lap[0][0]), l2b = fma(hdt, lap[1][1], lap[0][1]);
    const T pot2 = pot_of(a.lam_eta2[1], a.a_mass, u2a, u2b);
    const T k2a = kpi_of(l2a, u2a, pot2, a.fric[1], p2a);
    const T k2b = kpi_of(l2b, u2b, pot2, a.fric[1], p2b);
    opsi[0] = mkpair(fma(hdt, p2a, y1), fma(hdt, p2b, y2));
    const T p3a = fma(hdt, k2a, q1), p3b = fma(hdt, k2b, q2);  // Pi(U3)
    if (MODE == FUSED_A) opi[0] = mkpair(p3a, p3b);
    else opi[0] = mkpair(fma(a.adt, p3a, T(2) * y1), fma(a.adt, p3b, T(2) * y2));  // W = psi_Y + psi(U4)
  } else if (MODE == FUSED_B2) {
    // Stages 3 + 4 and the final combination from psi_3, W = 2 psi_Y + dt Pi_3 (differenced) and Y (pointwise):
    //   psi(U4) = psi_Y + dt Pi_3 = W - psi_Y,   Pi_3 = (W - 2 psi_Y) / dt  (cancellation: eps |W| / dt absolute, which
    //   enters Ynew with factors <= 2/3: rounding level in fp64; the reason this form is not used in fp32),
    //   k1_Pi + k4_Pi = Lap(psi_Y) + Lap(psi(U4)) + pointwise terms = Lap(W) + ...: Lap psi_Y alone is never needed,
    //   dt/6 2 k2 = 2/3 (U3 - Y) for both components (U3 = Y + dt/2 k2).
    const T dt = a.adt, sixth = a.adt / T(6), inv_dt = a.wu, twothirds = T(2) / T(3);
    const T u3a = wc[0].x, u3b = wc[0].y, wa = wc[1].x, wb = wc[1].y;
    const T y1 = pc[0].x, y2 = pc[0].y, q1 = pc[NPA > 1 ? 1 : 0].x, q2 = pc[NPA > 1 ? 1 : 0].y;
    const T p3a = (wa - T(2) * y1) * inv_dt, p3b = (wb - T(2) * y2) * inv_dt;  // Pi(U3)
    const T u4a = wa - y1, u4b = wb - y2;                                      // psi(U4)
    const T pot3 = pot_of(a.lam_eta2[1], a.a_mass, u3a, u3b);
    const T k3a = kpi_of(lap[0][0], u3a, pot3, a.fric[1], p3a);
    const T k3b = kpi_of(lap[0][1], u3b, pot3, a.fric[1], p3b);
    const T p4a = fma(dt, k3a, q1), p4b = fma(dt, k3b, q2);  // Pi(U4)
    const T pot4 = pot_of(a.lam_eta2[2], a.a_mass, u4a, u4b);
    const T pot1 = pot_of(a.lam_eta2[0], a.a_mass, y1, y2);
    const T k14a = fma(-a.fric[2], p4a, fma(-u4a, pot4, kpi_of(lap[1][0], y1, pot1, a.fric[0], q1)));  // k1 + k4
    const T k14b = fma(-a.fric[2], p4b, fma(-u4b, pot4, kpi_of(lap[1][1], y2, pot1, a.fric[0], q2)));
    opsi[0] = mkpair(fma(sixth, (q1 + p4a) + T(2) * p3a, fma(twothirds, u3a - y1, y1)),
                     fma(sixth, (q2 + p4b) + T(2) * p3b, fma(twothirds, u3b - y2, y2)));
    opi[0] = mkpair(fma(sixth, fma(T(2), k3a, k14a), fma(twothirds, p3a - q1, q1)),
                    fma(sixth, fma(T(2), k3b, k14b), fma(twothirds, p3b - q2, q2)));
  } else if (MODE == FUSED_B) {
    // stages 3 + 4 and the final combination; k1 recomputed from Y (same expression, same bits as in
    // PASS A), dt/2 k2 = Pi3 - Pi_Y
    const T dt = a.adt, hdt = T(0.5) * a.adt, sixth = a.adt / T(6);
    const T u3a = wc[0].x, u3b = wc[0].y, p3a = wc[1].x, p3b = wc[1].y;
    const T y1 = wc[2].x, y2 = wc[2].y, q1 = pc[0].x, q2 = pc[0].y;
    const T pot3 = pot_of(a.lam_eta2[1], a.a_mass, u3a, u3b);
    const T k3a = kpi_of(lap[0][0], u3a, pot3, a.fric[1], p3a);
    const T k3b = kpi_of(lap[0][1], u3b, pot3, a.fric[1], p3b);
    const T u4a = fma(dt, p3a, y1), u4b = fma(dt, p3b, y2);  // psi(U4)
    const T p4a = fma(dt, k3a, q1), p4b = fma(dt, k3b, q2);  // Pi(U4)
    const T l4a = fma(dt, lap[1][0], lap[2][0]), l4b = fma(dt, lap[1][1], lap[2][1]);
    const T pot4 = pot_of(a.lam_eta2[2], a.a_mass, u4a, u4b);
    const T k4a = kpi_of(l4a, u4a, pot4, a.fric[2], p4a);
    const T k4b = kpi_of(l4b, u4b, pot4, a.fric[2], p4b);
    const T pot1 = pot_of(a.lam_eta2[0], a.a_mass, y1, y2);
    const T k1a = kpi_of(lap[2][0], y1, pot1, a.fric[0], q1);
    const T k1b = kpi_of(lap[2][1], y2, pot1, a.fric[0], q2);
    const T p2a = fma(hdt, k1a, q1), p2b = fma(hdt, k1b, q2);  // Pi(U2), same bits as in PASS A
    const T twothirds = T(2) / T(3);
    opsi[0] = mkpair(fma(sixth, (q1 + p4a) + T(2) * (p2a + p3a), y1),
                           fma(sixth, (q2 + p4b) + T(2) * (p2b + p3b), y2));
    opi[0] = mkpair(fma(sixth, fma(T(2), k3a, k1a + k4a), fma(twothirds, p3a - q1, q1)),
                          fma(sixth, fma(T(2), k3b, k1b + k4b), fma(twothirds, p3b - q2, q2)));
  } else if (MODE == RKN_ST) {
    // f = Lap Psi - Psi (lambda eta_s^2 (|Psi|^2 - 1) + a): no first-derivative term in a Nystrom scheme
    const T p1 = wc[0].x, p2 = wc[0].y;
    const T pot = pot_of(a.lam_eta2[0], a.a_mass, p1, p2);
    const T f1 = fma(-p1, pot, lap[0][0]), f2 = fma(-p2, pot, lap[0][1]);
    T o[2][2];
#pragma unroll
    for (int r = 0; r < 2; ++r) {
      T s1 = a.rkn_w[r][6] * f1, s2 = a.rkn_w[r][6] * f2;
#pragma unroll
      for (int q = NPA - 1; q >= 0; --q)
        if (a.pnt[q]) {
          s1 = fma(a.rkn_w[r][q], pc[q].x, s1);
          s2 = fma(a.rkn_w[r][q], pc[q].y, s2);
        }
      o[r][0] = s1;
      o[r][1] = s2;
    }
    opsi[0] = mkpair(o[0][0], o[0][1]);
    opi[0] = mkpair(o[1][0], o[1][1]);
  } else {
    const T psi1 = wc[0].x, psi2 = wc[0].y;
    const T pi1 = pc[0].x, pi2 = pc[0].y;
    const T pot = pot_of(a.lam_eta2[0], a.a_mass, psi1, psi2);
    T kpsi1 = pi1, kpsi2 = pi2;
    T kpi1 = kpi_of(lap[0][0], psi1, pot, a.fric[0], pi1);
    T kpi2 = kpi_of(lap[0][1], psi2, pot, a.fric[0], pi2);
    if (HASKO) {
      kpsi1 += ko[0];
      kpsi2 += ko[1];
      kpi1 += ko[2];
      kpi2 += ko[3];
    }
    // pointwise inputs: in_psi(q) = pv[1 + 2q], in_pi(q) = pv[2 + 2q]
    auto ipsi = [&](int q) -> const P& { return pc[(1 + 2 * q) < NPA ? (1 + 2 * q) : 0]; };
    auto ipi = [&](int q) -> const P& { return pc[(2 + 2 * q) < NPA ? (2 + 2 * q) : 0]; };
    auto axpy = [](T c, T k, T y) -> T { return fma(c, k, y); };
    if (MODE == LEAN_S1) {  // U2 = U + adt k   (U = Y)
      opsi[0] = mkpair(axpy(a.adt, kpsi1, psi1), axpy(a.adt, kpsi2, psi2));
      opi[0] = mkpair(axpy(a.adt, kpi1, pi1), axpy(a.adt, kpi2, pi2));
    } else if (MODE == LEAN_S23) {  // U' = Y + adt k   (in0 = Y)
      opsi[0] = mkpair(axpy(a.adt, kpsi1, ipsi(0).x), axpy(a.adt, kpsi2, ipsi(0).y));
      opi[0] = mkpair(axpy(a.adt, kpi1, ipi(0).x), axpy(a.adt, kpi2, ipi(0).y));
    } else if (MODE == SSP_S23) {  // in0 = Y: out = wy Y + wu (U + adt k), adt = dt
      opsi[0] = mkpair(fma(a.wy, ipsi(0).x, a.wu * axpy(a.adt, kpsi1, psi1)), fma(a.wy, ipsi(0).y, a.wu * axpy(a.adt, kpsi2, psi2)));
      opi[0] = mkpair(fma(a.wy, ipi(0).x, a.wu * axpy(a.adt, kpi1, pi1)), fma(a.wy, ipi(0).y, a.wu * axpy(a.adt, kpi2, pi2)));
    } else if (MODE == LEAN_S4) {  // in0 = Y, in1 = U2, in2 = U3, U = U4, adt = dt/6
      const T third = T(1) / T(3);
      auto comb = [&](T yv, T u2, T u3, T u4, T kk) -> T {
        return fma(a.adt, kk, ((fma(T(2), u3, u2) + u4) - yv) * third);
      };
      opsi[0] = mkpair(comb(ipsi(0).x, ipsi(1).x, ipsi(2).x, psi1, kpsi1),
                             comb(ipsi(0).y, ipsi(1).y, ipsi(2).y, psi2, kpsi2));
      opi[0] = mkpair(comb(ipi(0).x, ipi(1).x, ipi(2).x, pi1, kpi1),
                            comb(ipi(0).y, ipi(1).y, ipi(2).y, pi2, kpi2));
    } else if (MODE == CLASSIC_S1) {  // out0 = U + adt k ; out1 (ACC) = U + bdt k
      opsi[0] = mkpair(axpy(a.adt, kpsi1, psi1), axpy(a.adt, kpsi2, psi2));
      opi[0] = mkpair(axpy(a.adt, kpi1, pi1), axpy(a.adt, kpi2, pi2));
      opsi[NOUT - 1] = mkpair(axpy(a.bdt, kpsi1, psi1), axpy(a.bdt, kpsi2, psi2));
      opi[NOUT - 1] = mkpair(axpy(a.bdt, kpi1, pi1), axpy(a.bdt, kpi2, pi2));
    } else if (MODE == CLASSIC_S23) {  // in0 = Y, in1 = ACC ; out0 = Y + adt k ; out1 = ACC + bdt k
      opsi[0] = mkpair(axpy(a.adt, kpsi1, ipsi(0).x), axpy(a.adt, kpsi2, ipsi(0).y));
      opi[0] = mkpair(axpy(a.adt, kpi1, ipi(0).x), axpy(a.adt, kpi2, ipi(0).y));
      opsi[NOUT - 1] = mkpair(axpy(a.bdt, kpsi1, ipsi(1).x), axpy(a.bdt, kpsi2, ipsi(1).y));
      opi[NOUT - 1] = mkpair(axpy(a.bdt, kpi1, ipi(1).x), axpy(a.bdt, kpi2, ipi(1).y));
    } else {  // CLASSIC_S4: in0 = ACC ; out0 = ACC + adt k
      opsi[0] = mkpair(axpy(a.adt, kpsi1, ipsi(0).x), axpy(a.adt, kpsi2, ipsi(0).y));
      opi[0] = mkpair(axpy(a.adt, kpi1, ipi(0).x), axpy(a.adt, kpi2, ipi(0).y));
    }
  }
}

// KO = 0, or the Kreiss-Oliger dissipation order (2, 3): the window radius is the larger of the two stencils, and
// Pi(U) becomes a second differenced field (it takes the ring slot that pnt[0] had).
template <typename T, int ORDER, int MODE, int TX, int TY, int D, int KO = 0>
struct PipeCfg {
  static constexpr int R = ORDER > KO ? ORDER : KO;
  static constexpr int CPT = Vec16<T>::CPT;
  static constexpr int TXC = TX * CPT;
  static constexpr int SW = TXC + 2 * R;
  static constexpr int SH = TY + 2 * R;
  static constexpr int NT = TX * TY;
  static constexpr int NH = 2 * R * (TXC + TY);  // halo pairs per plane (star stencil: no corners)
  static constexpr int HPT = (NH + NT - 1) / NT;
  static constexpr int P0 = KO ? 1 : 0;  // first pointwise input that is still streamed
  static constexpr int NF = ModeInfo<MODE>::NF + P0;
  static constexpr int NP = ModeInfo<MODE>::NP;
  static constexpr int NOUT = ModeInfo<MODE>::NOUT;
  static constexpr int NOWN = NF + NP - P0;  // ring slots per stage and thread
  static constexpr size_t PAIR = 2 * sizeof(T);
  static constexpr size_t OWN_BYTES = (size_t)D * NOWN * NT * 16;
  static constexpr size_t HALO_BYTES = (size_t)D * NF * NH * PAIR;  // ring slot = NH pairs per field
  static constexpr size_t CTR_BYTES = (size_t)2 * NF * SH * SW * PAIR;
  static constexpr size_t SMEM_BYTES = OWN_BYTES + HALO_BYTES + CTR_BYTES;
};

// Deepest ring (<= dmax stages, >= 2) whose shared memory fits `budget` bytes.
template <typename T, int ORDER, int MODE, int TX, int TY, int KO = 0>
constexpr int pipe_depth(size_t budget, int dmax) {
  int d = 2;
  if (dmax >= 3 && PipeCfg<T, ORDER, MODE, TX, TY, 3, KO>::SMEM_BYTES <= budget) d = 3;
  if (dmax >= 4 && PipeCfg<T, ORDER, MODE, TX, TY, 4, KO>::SMEM_BYTES <= budget) d = 4;
  if (dmax >= 5 && PipeCfg<T, ORDER, MODE, TX, TY, 5, KO>::SMEM_BYTES <= budget) d = 5;
  if (dmax >= 6 && PipeCfg<T, ORDER, MODE, TX, TY, 6, KO>::SMEM_BYTES <= budget) d = 6;
  return d;
}

template <typename T, int ORDER, int MODE, int TX, int TY, int D, int KO = 0>
__global__ void __launch_bounds__(TX* TY) k_rk_pipe(const PipeArgs<T> a) {
  using P = typename PairOf<T>::type;
  using V = Vec16<T>;
  using C = PipeCfg<T, ORDER, MODE, TX, TY, D, KO>;
  constexpr int R = C::R, CPT = C::CPT, TXC = C::TXC, SW = C::SW, SH = C::SH, NT = C::NT, NH = C::NH, HPT = C::HPT;
  constexpr int NF = C::NF, NP = C::NP, NOUT = C::NOUT, P0 = C::P0, NOWN = C::NOWN;
  constexpr int NFM = ModeInfo<MODE>::NF;  // fields the Laplacian is taken of
  constexpr int NPA = NP > 0 ? NP : 1;

  extern __shared__ __align__(16) unsigned char smem_raw[];
  V* const own = reinterpret_cast<V*>(smem_raw);                             // [D][NOWN][NT]
  P* const halo = reinterpret_cast<P*>(smem_raw + C::OWN_BYTES);             // [D][NF][NH]
  P* const ctr = reinterpret_cast<P*>(smem_raw + C::OWN_BYTES + C::HALO_BYTES);  // [2][NF][SH * SW]

  const TileDev t = a.tiles[blockIdx.x];
  const BoxDev b = a.boxes[t.box];
  const int tid = threadIdx.x;
  const int tx = tid % TX, ty = tid / TX;
  const int x = t.x0 + tx * CPT, y = t.y0 + ty;
  const bool active = (x < b.n[0]) && (y < b.n[1]);
  // in a partial tile the columns/rows just past the box edge are ghost cells that the edge cells need as
  // +x / +y neighbours: threads sitting there still stream their own column through shared memory
  const bool loader = (x < b.n[0] + R) && (y < b.n[1] + R);
  const long long plane = (long long)b.sx * b.sy;
  const long long tile_org =
      b.base + (long long)(t.z0 + a.g) * plane + (long long)(t.y0 + a.g) * b.sx + (t.x0 + a.ox);
  long long off = tile_org + (long long)ty * b.sx + tx * CPT;  // this thread's cell in plane z0

  // halo assignment: pair index -> (hx, hy) relative to the tile origin
  int h_goff[HPT];  // global offset relative to tile_org (within a plane)
  int h_soff[HPT];  // offset inside a centre plane, -1 = none
#pragma unroll
  for (int q = 0; q < HPT; ++q) {
    const int idx = tid + q * NT;
    int hx = 0, hy = 0;
    bool ok = idx < NH;
    if (idx < 2 * R * TXC) {  // bottom / top strips, x fastest
      const int row = idx / TXC;
      hx = idx % TXC;
      hy = (row < R) ? (row - R) : (TY + row - R);
    } else {
      const int j = idx - 2 * R * TXC;  // left / right strips
      const int col = j % (2 * R);
      hy = j / (2 * R);
      hx = (col < R) ? (col - R) : (TXC + col - R);
    }
    // stay inside the box's ghosted extent (partial tiles at the high end of a box)
    ok = ok && (t.x0 + hx < b.n[0] + R) && (t.y0 + hy < b.n[1] + R);
    h_goff[q] = hy * b.sx + hx;
    h_soff[q] = ok ? ((hy + R) * SW + (hx + R)) : -1;
  }
  const int s_own = (ty + R) * SW + (tx * CPT + R);

  // one pipeline stage = everything iteration `st` consumes: own-column values of plane z0+st+R of the
  // differenced fields, pointwise inputs of plane z0+st, x/y halo of plane z0+st
  auto issue = [&](int st) {
    const int slot = st % D;
    V* const o = own + (size_t)slot * NOWN * NT + tid;
    const long long po = off + (long long)st * plane;  // `off` is never advanced (see below)
    if (loader) {
#pragma unroll
      for (int f = 0; f < NF; ++f) cp_async_16(o + f * NT, a.sten[f] + po + (long long)R * plane);
    }
    if (active) {
#pragma unroll
      for (int q = P0; q < NP; ++q)
        if (MODE != RKN_ST || a.pnt[q]) cp_async_16(o + (NF + q - P0) * NT, a.pnt[q] + po);
    }
    const long long ho = tile_org + (long long)st * plane;
#pragma unroll
    for (int q = 0; q < HPT; ++q)
      if (h_soff[q] >= 0) {
#pragma unroll
        for (int f = 0; f < NF; ++f)
          cp_async_pair(halo + ((size_t)slot * NF + f) * NH + tid + q * NT, a.sten[f] + ho + h_goff[q]);
      }
  };

  // prologue: fill the ring, then the lower 2R planes of the z-windows straight into registers
#pragma unroll
  for (int st = 0; st < D; ++st) {
    if (st < t.nz) issue(st);
    cp_async_commit();
  }
  V w[NF][2 * R + 1];  // w[f][m] = field f at plane z + m - R
#pragma unroll
  for (int f = 0; f < NF; ++f)
#pragma unroll
    for (int m = 0; m < 2 * R; ++m)
      if (loader) w[f][m + 1] = ldg16_keep<T>(a.sten[f] + off + (long long)(m - R) * plane);

  for (int zz = 0; zz < t.nz; ++zz) {
    const int slot = zz % D;
    P* const cb = ctr + (size_t)(zz & 1) * NF * SH * SW;
    cp_async_wait<D - 1>();  // this thread's copies of stage zz have landed (only this thread reads them)
    const V* const o = own + (size_t)slot * NOWN * NT + tid;
    V pv[NPA];
#pragma unroll
    for (int f = 0; f < NF; ++f) {
#pragma unroll
      for (int m = 0; m < 2 * R; ++m) w[f][m] = w[f][m + 1];
      if (loader) {
        w[f][2 * R] = o[f * NT];
#pragma unroll
        for (int p = 0; p < CPT; ++p) cb[f * SH * SW + s_own + p] = w[f][R].p[p];
      }
    }
    if (active) {
#pragma unroll
      for (int q = P0; q < NP; ++q) pv[q] = o[(NF + q - P0) * NT];
      if (KO) pv[0] = w[NF - 1][R];  // Pi(U) of this plane comes from its own z-window
    }
#pragma unroll
    for (int q = 0; q < HPT; ++q)
      if (h_soff[q] >= 0) {
#pragma unroll
        for (int f = 0; f < NF; ++f)
          cb[f * SH * SW + h_soff[q]] = halo[((size_t)slot * NF + f) * NH + tid + q * NT];
      }
    // refill the slot just drained with stage zz + D
    if (zz + D < t.nz) issue(zz + D);
    cp_async_commit();
    __syncthreads();

    if (active) {
      V o_psi[NOUT], o_pi[NOUT];
#pragma unroll
      for (int p = 0; p < CPT; ++p) {
        const int sc = s_own + p;
        T lap[NFM][2];
        T ko[4] = {T(0), T(0), T(0), T(0)};
#pragma unroll
        for (int f = 0; f < NF; ++f) {
          const P* const s = cb + f * SH * SW;
#pragma unroll
          for (int c = 0; c < 2; ++c) {
            auto comp = [c](const P& v) -> T { return c == 0 ? v.x : v.y; };
            T xm[3], xp[3], ym[3], yp[3], zm[3], zp[3];
#pragma unroll
            for (int r = 1; r <= R; ++r) {
              xm[r - 1] = comp(s[sc - r]);
              xp[r - 1] = comp(s[sc + r]);
              ym[r - 1] = comp(s[sc - r * SW]);
              yp[r - 1] = comp(s[sc + r * SW]);
              zm[r - 1] = comp(w[f][R - r].p[p]);
              zp[r - 1] = comp(w[f][R + r].p[p]);
            }
            if (f < NFM) lap[f < NFM ? f : 0][c] = lap_from<T, ORDER>(comp(w[f][R].p[p]), xm, xp, ym, yp, zm, zp, a.inv_h2);
            if (KO) ko[2 * f + c] = ko_from<T, KO ? KO : 2>(comp(w[f][R].p[p]), xm, xp, ym, yp, zm, zp, a.ko_c[2 * f + c]);
          }
        }
        P wc[NFM], pc[NPA], opsi[NOUT], opi[NOUT];
#pragma unroll
        for (int f = 0; f < NFM; ++f) wc[f] = w[f][R].p[p];
#pragma unroll
        for (int q = 0; q < NPA; ++q) pc[q] = pv[q].p[p];
        rk_cell<T, MODE, KO != 0>(a, lap, wc, pc, opsi, opi, ko);
#pragma unroll
        for (int q = 0; q < NOUT; ++q) {
          o_psi[q].p[p] = opsi[q];
          o_pi[q].p[p] = opi[q];
        }
      }
      const long long oo = off + (long long)zz * plane;
#pragma unroll
      for (int q = 0; q < NOUT; ++q) {
        stg16<T>(a.out_psi[q] + oo, o_psi[q]);
        stg16<T>(a.out_pi[q] + oo, o_pi[q]);
      }
    }
  }
}

}  // namespace sledge
