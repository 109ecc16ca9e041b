// sledge_oracle.cpp -- TEST INFRASTRUCTURE ONLY.
//
// Plain, slow, obviously-correct fp64 CPU implementation of the sledgehamr hot path
// (arXiv 2404.02950), written from the paper text.  Only tests/, __graft_entry__.smoke()
// and bench.py's cpu_baseline / --impl reference legs may build, load or call this file.
// It shares no code, header, table or helper with the CUDA library under
// paper_2404_02950_b200/csrc/ and must never be linked into the product path.
//
// What it computes, and the passage each part follows (PAPER.md line / section):
//   O1 grid        : block-structured levels, ratio 2, periodic domain          L23, L39-53 Eq.1-3
//   O2 Laplacian   : utils::Laplacian<order>, order 1 -> 7-pt, 2 -> 13-pt,
//                    3 -> 19-pt                                                  L207-212, L649 App.A
//                    (coefficients are not printed; they are the unique maximal-order central
//                    stencils on 3 / 5 / 7 points per axis -- pinned by polynomial exactness)
//   O3 RHS         : Eq.10-11 with friction kappa, mass term a, coupling lambda  L178-181, L214-223
//   O4 integrator  : classic RK4 (integrator.type = 4)                           L808 Table V
//   O5 ghost fill  : periodic wrap, same-level copy, coarse->fine trilinear in
//                    space + linear in time                                       L68-74
//   O6 subcycling  : advance l, then l+1 twice, then synchronise                  L66-76, L88 Fig.2
//   O7 average-down: coarse <- mean of 8 fine children                            L74, L88
//   O12 quartic    : quartic polynomial conservative coarse->fine interpolation      L70, L780
//   O11 SSPRK3     : Shu-Osher three-stage scheme (integrator.type 3 / 10)            L808
//   O10 KO term    : Kreiss-Oliger dissipation Q_l added to every component's RHS  L141-146 Eq.7
//   O9 TEE tags    : |coarse - mean of children| > eps at synchronisation         L82-111 Eq.5-6, L373-380 Eq.12
//   O13 GW fields  : auxiliary fields u_ij, du_ij (6 + 6 components) of Eq.16, sourced by
//                    sum_c d_i psi_c d_j psi_c with Gradient<order>                L400-436 Eq.16
//   O14 RKN        : user-defined Runge-Kutta-Nystrom tableau (integrator.type 20)   L808-815 Table V
//   O15 shadow     : level-0 truncation-error tags against a coarsened copy of level 0
//                    evolved for one step of 2 dt                                    L98
//   O8 string tags : plaquette winding number of (psi1,psi2) around 0; rule not printed in the
//                    paper (L349-371 gives only the bool-per-cell hook) -> DESIGN.md reading R8
//   diagnostics    : energies used only by the pins (L678 App.B; Gradient<order> L651-658)
//
// No blocking, fusion or reordering: every loop is the definition written out.  OpenMP pragmas on
// outer box/z loops only change which core executes an iteration, never the arithmetic.
// Build: g++ -O2 -ffp-contract=off -fopenmp -shared -fPIC (see oracle/oracle.py).
//
// Parity pins: tests/test_oracle_pins.py (every function here has at least one pin that is not
// a restatement of its own formula).

#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

constexpr int NCOMP = 4;  // psi1, psi2, pi1, pi2  (L189-190)
constexpr int PSI1 = 0, PSI2 = 1, PI1 = 2, PI2 = 3;
// with sim.gravitational_waves (L404, L436): Gw::u_xx, yy, zz, xy, xz, yz = 4..9, Gw::du_xx .. du_yz = 10..15
constexpr int NCOMP_GW = 16, GW_U = 4, GW_DU = 10;
constexpr int GW_I[6] = {0, 1, 2, 0, 0, 1}, GW_J[6] = {0, 1, 2, 1, 2, 2};  // xx, yy, zz, xy, xz, yz (L436)
constexpr int RKN_MAX = 6;
constexpr int FLAG_BLOCK = 32;  // box-flag reduction granularity (BASELINE.json config 3)

struct Params {
  int32_t n_levels;
  int32_t n0[3];
  int32_t nghost;
  int32_t blocking_factor;
  int32_t lap_order;
  int32_t eta_fixed;
  double h0;
  double lambda;
  double a_mass;
  double friction;
  double ko_strength[4];  // epsilon_KO of Eq.7 per component psi1, psi2, Pi1, Pi2 (L749-750; 0 = off)
  int32_t ko_order;       // sim.dissipation_order = ghost cells the term needs (L751): 2 or 3
  int32_t integrator;     // integrator.type (L808): 0 or 4 = RK4; 3 or 10 = SSPRK3 (10 = its low-storage form)
  int32_t interp;         // coarse->fine ghost interpolation: 0 = cell-centred trilinear (BASELINE.json config 5),
                          // 4 = quartic polynomial conservative (amr.interpolation_type 4, the paper's default)
  int32_t gw;             // sim.gravitational_waves (L404): 1 = evolve the 12 auxiliary components as well
  double gw_coupling;     // Eq.16's 16 pi G (times whatever the project's units absorb), multiplies T_ij
  double gw_friction;     // Eq.16's 3H written like Eq.11's 2/eta: the friction term is (gw_friction / eta) du_ij
  int32_t rkn_stages;     // integrator.type 20: number of stages s of the user's RKN tableau, 1..RKN_MAX
  int32_t pad_;
  double rkn_c[RKN_MAX];     // rkn.nodes (L814)
  double rkn_b[RKN_MAX];     // rkn.weights_b (L812)
  double rkn_bbar[RKN_MAX];  // rkn.weights_bar_b (L813)
  double rkn_a[RKN_MAX * (RKN_MAX + 1) / 2];  // rkn.tableau (L815): rows of the lower triangle incl. the diagonal
};

struct BoxIn {
  int32_t level;
  int32_t lo[3];
  int32_t hi[3];
};

// One box worth of data: NCOMP components, valid region n[0..2] plus g ghost layers.
struct Field {
  int n[3] = {0, 0, 0};
  int g = 0;
  int s[3] = {0, 0, 0};
  int nc = NCOMP;
  std::vector<double> v;
  void init(const int nn[3], int gg, int ncomp = NCOMP) {
    g = gg;
    nc = ncomp;
    for (int d = 0; d < 3; ++d) {
      n[d] = nn[d];
      s[d] = nn[d] + 2 * gg;
    }
    v.assign((size_t)nc * s[0] * s[1] * s[2], 0.0);
  }
  // i,j,k relative to the box's low corner; ghosts are -g..-1 and n..n+g-1.
  inline double& at(int c, int i, int j, int k) {
    return v[(((size_t)c * s[2] + (k + g)) * s[1] + (j + g)) * s[0] + (i + g)];
  }
  inline double at(int c, int i, int j, int k) const {
    return v[(((size_t)c * s[2] + (k + g)) * s[1] + (j + g)) * s[0] + (i + g)];
  }
};

typedef std::vector<Field> LevelState;  // one Field per box of the level

struct Level {
  int n[3];                 // index space extent (n0 * 2^l)
  double h;                 // Eq.1
  std::vector<int> boxes;   // global box ids, in input order
  std::vector<int> owner;   // coarsened (by blocking factor) index space -> local box index or -1
  int no[3];
  LevelState Y;             // current state; after this level's step it is the state at t_new
  LevelState Yold;          // state at t_old, the start of this level's last step (L72)
  double t_old = 0, t_new = 0;
  bool have_pair = false;
  LevelState K[4];          // RK4 slopes (k of the last orc_eval_rhs in K[0])
  std::vector<LevelState> KN;  // O14: f_j of the RKN stages (allocated on first use)
  LevelState U;             // stage state
  // O9: truncation-error tags of this (fine) level, written by average_down when tee_on (L82-111, Eq.5-6, Eq.12)
  bool tee_on = false;
  double tee_eps[4] = {0, 0, 0, 0};  // threshold per component psi1, psi2, Pi1, Pi2 (te_crit_$ScalarField, L781-782)
  uint8_t* tee_tags = nullptr;     // caller's arrays (dense per box, x fastest, boxes back to back)
  uint32_t* tee_counts = nullptr;  // tagged cells per aligned FLAG_BLOCK^3 block of this level
};

struct Oracle {
  Params p;
  std::vector<BoxIn> box;
  std::vector<int> box_local;  // index of the box inside its level
  std::vector<Level> lev;
  std::string err;
};

inline int wrap(int i, int n) {
  int r = i % n;
  return r < 0 ? r + n : r;
}
inline int floordiv2(int i) { return (i >= 0) ? i / 2 : -((-i + 1) / 2); }

// ---- O1: hierarchy ---------------------------------------------------------------------------

int owner_of(const Oracle& o, int l, int i, int j, int k) {  // wrapped indices
  const Level& L = o.lev[l];
  int bf = o.p.blocking_factor;
  return L.owner[((size_t)(k / bf) * L.no[1] + (j / bf)) * L.no[0] + (i / bf)];
}

bool build(Oracle& o, const BoxIn* b, int nbox) {
  const Params& p = o.p;
  char msg[256];
  if (p.n_levels < 1 || p.n_levels > 8) { o.err = "n_levels out of range"; return false; }
  int bf = p.blocking_factor;
  if (bf < 1 || (bf & (bf - 1))) { o.err = "blocking_factor must be a power of 2 (L39)"; return false; }
  if (p.nghost >= bf) { o.err = "nghost must be smaller than blocking_factor (L772)"; return false; }
  if (p.lap_order < 1 || p.lap_order > 3) { o.err = "lap_order must be 1, 2 or 3 (L649)"; return false; }
  if (p.lap_order > p.nghost) { o.err = "lap_order must be <= nghost (L240)"; return false; }
  const bool ko_on = p.ko_strength[0] != 0.0 || p.ko_strength[1] != 0.0 || p.ko_strength[2] != 0.0 || p.ko_strength[3] != 0.0;
  for (int c = 0; c < 4; ++c)
    if (!(p.ko_strength[c] >= 0.0)) { o.err = "dissipation strength must be >= 0 (L749)"; return false; }
  if (ko_on && (p.ko_order < 2 || p.ko_order > 3)) { o.err = "dissipation order must be 2 or 3 (L751)"; return false; }
  if (ko_on && p.ko_order > p.nghost) { o.err = "dissipation order must be <= nghost (L751)"; return false; }
  if (p.integrator != 0 && p.integrator != 4 && p.integrator != 3 && p.integrator != 10 && p.integrator != 20) { o.err = "integrator.type must be 4 (RK4), 3 / 10 (SSPRK3) or 20 (user RKN tableau) (L808)"; return false; }
  if (p.integrator == 20) {  // O14: an explicit Nystrom scheme integrates psi'' = f(psi, eta): no first-derivative terms
    if (p.rkn_stages < 1 || p.rkn_stages > RKN_MAX) { o.err = "rkn: 1..6 stages"; return false; }
    if (p.friction != 0.0 || ko_on) { o.err = "rkn: the scheme needs psi'' = f(psi): friction and dissipation must be 0"; return false; }
    if (p.gw) { o.err = "rkn: gravitational-wave fields are not integrated by the RKN scheme"; return false; }
    for (int i = 0; i < p.rkn_stages; ++i)
      if (p.rkn_a[i * (i + 1) / 2 + i] != 0.0) { o.err = "rkn.tableau: only explicit schemes (zero diagonal) (L815)"; return false; }
  }
  if (p.gw != 0 && p.gw != 1) { o.err = "gw must be 0 or 1 (L404)"; return false; }
  if (p.interp != 0 && p.interp != 4) { o.err = "interp must be 0 (trilinear) or 4 (quartic conservative, L780)"; return false; }
  if (!(p.h0 > 0)) { o.err = "h0 must be positive"; return false; }
  o.lev.resize(p.n_levels);
  for (int l = 0; l < p.n_levels; ++l) {
    Level& L = o.lev[l];
    for (int d = 0; d < 3; ++d) {
      L.n[d] = p.n0[d] << l;
      if (p.n0[d] <= 0 || p.n0[d] % bf) { o.err = "n0 must be a positive multiple of blocking_factor"; return false; }
      L.no[d] = L.n[d] / bf;
    }
    L.h = p.h0 / (double)(1 << l);  // Eq.1
    L.owner.assign((size_t)L.no[0] * L.no[1] * L.no[2], -1);
  }
  o.box.assign(b, b + nbox);
  o.box_local.resize(nbox);
  for (int ib = 0; ib < nbox; ++ib) {
    const BoxIn& B = b[ib];
    if (B.level < 0 || B.level >= p.n_levels) { o.err = "box level out of range"; return false; }
    Level& L = o.lev[B.level];
    for (int d = 0; d < 3; ++d) {
      int n = B.hi[d] - B.lo[d] + 1;
      if (B.lo[d] < 0 || B.hi[d] >= L.n[d] || n <= 0 || B.lo[d] % bf || n % bf) {
        snprintf(msg, sizeof msg, "box %d: not inside the domain / not aligned to the blocking factor (L39)", ib);
        o.err = msg;
        return false;
      }
    }
    int li = (int)L.boxes.size();
    for (int k = B.lo[2] / bf; k <= B.hi[2] / bf; ++k)
      for (int j = B.lo[1] / bf; j <= B.hi[1] / bf; ++j)
        for (int i = B.lo[0] / bf; i <= B.hi[0] / bf; ++i) {
          int& ow = L.owner[((size_t)k * L.no[1] + j) * L.no[0] + i];
          if (ow != -1) {
            snprintf(msg, sizeof msg, "box %d overlaps another box of level %d", ib, B.level);
            o.err = msg;
            return false;
          }
          ow = li;
        }
    o.box_local[ib] = li;
    L.boxes.push_back(ib);
  }
  for (size_t q = 0; q < o.lev[0].owner.size(); ++q)
    if (o.lev[0].owner[q] < 0) { o.err = "level 0 must cover the whole domain (L39)"; return false; }
  // Proper nesting (L70, L137): every fine box grown by one blocking factor of fine cells must lie
  // on valid cells of the next coarser level.
  for (int l = 1; l < p.n_levels; ++l) {
    if (o.lev[l].boxes.empty()) { o.err = "empty refinement level"; return false; }
    for (int ib : o.lev[l].boxes) {
      const BoxIn& B = o.box[ib];
      for (int k = B.lo[2] - bf; k <= B.hi[2] + bf; k += 1)
        for (int j = B.lo[1] - bf; j <= B.hi[1] + bf; j += 1)
          for (int i = B.lo[0] - bf; i <= B.hi[0] + bf; i += 1) {
            int ci = wrap(floordiv2(i), o.lev[l - 1].n[0]);
            int cj = wrap(floordiv2(j), o.lev[l - 1].n[1]);
            int ck = wrap(floordiv2(k), o.lev[l - 1].n[2]);
            if (owner_of(o, l - 1, ci, cj, ck) < 0) {
              snprintf(msg, sizeof msg, "box %d violates proper nesting (gap < blocking factor, L70/L137)", ib);
              o.err = msg;
              return false;
            }
          }
    }
  }
  for (int l = 0; l < p.n_levels; ++l) {
    Level& L = o.lev[l];
    auto alloc = [&](LevelState& S) {
      S.resize(L.boxes.size());
      for (size_t q = 0; q < L.boxes.size(); ++q) {
        const BoxIn& B = o.box[L.boxes[q]];
        int nn[3] = {B.hi[0] - B.lo[0] + 1, B.hi[1] - B.lo[1] + 1, B.hi[2] - B.lo[2] + 1};
        S[q].init(nn, p.nghost, p.gw ? NCOMP_GW : NCOMP);
      }
    };
    alloc(L.Y); alloc(L.Yold); alloc(L.U);
    for (int s = 0; s < 4; ++s) alloc(L.K[s]);
  }
  return true;
}

// value(l, state, comp, i,j,k): periodic wrap, find the owning box, return VALID data (O1).
inline double value(const Oracle& o, int l, const LevelState& S, int c, int i, int j, int k, bool* ok) {
  const Level& L = o.lev[l];
  int wi = wrap(i, L.n[0]), wj = wrap(j, L.n[1]), wk = wrap(k, L.n[2]);
  int ow = owner_of(o, l, wi, wj, wk);
  if (ow < 0) { *ok = false; return 0.0; }
  const BoxIn& B = o.box[L.boxes[ow]];
  return S[ow].at(c, wi - B.lo[0], wj - B.lo[1], wk - B.lo[2]);
}

// ---- O5: ghost fill --------------------------------------------------------------------------
// For each ghost cell of each box of level l in state S (which holds data of time `time`):
//   same-level owner exists -> copy its valid value (periodic wrap included)         L23, L68
//   else (l > 0)            -> trilinear interpolation of the time-interpolated
//                              coarse state c = (1-alpha) old + alpha new             L70-72
// Fine index f = 2c + r sits -1/4 (r=0) or +1/4 (r=1) coarse cell from the centre of c, hence per-axis
// weights 3/4 on c and 1/4 on c-1 (r=0) or c+1 (r=1).
bool fill_ghosts(Oracle& o, int l, LevelState& S, double time) {
  Level& L = o.lev[l];
  const int g = o.p.nghost;
  double alpha = 0.0;
  const LevelState* Cold = nullptr;
  const LevelState* Cnew = nullptr;
  if (l > 0) {
    Level& C = o.lev[l - 1];
    if (C.have_pair && C.t_new != C.t_old) {
      alpha = (time - C.t_old) / (C.t_new - C.t_old);
      Cold = &C.Yold;
      Cnew = &C.Y;
    } else {  // no step taken yet: the coarse level only has its current state
      alpha = 0.0;
      Cold = &C.Y;
      Cnew = &C.Y;
    }
  }
  bool all_ok = true;
#pragma omp parallel for schedule(dynamic)
  for (int q = 0; q < (int)L.boxes.size(); ++q) {
    const BoxIn& B = o.box[L.boxes[q]];
    Field& F = S[q];
    bool ok = true;
    for (int k = -g; k < F.n[2] + g; ++k)
      for (int j = -g; j < F.n[1] + g; ++j)
        for (int i = -g; i < F.n[0] + g; ++i) {
          bool inside = (i >= 0 && i < F.n[0] && j >= 0 && j < F.n[1] && k >= 0 && k < F.n[2]);
          if (inside) continue;
          int gi = B.lo[0] + i, gj = B.lo[1] + j, gk = B.lo[2] + k;  // unwrapped level index
          int wi = wrap(gi, L.n[0]), wj = wrap(gj, L.n[1]), wk = wrap(gk, L.n[2]);
          int ow = owner_of(o, l, wi, wj, wk);
          if (ow >= 0) {
            const BoxIn& Bo = o.box[L.boxes[ow]];
            for (int c = 0; c < F.nc; ++c)
              F.at(c, i, j, k) = S[ow].at(c, wi - Bo.lo[0], wj - Bo.lo[1], wk - Bo.lo[2]);
            continue;
          }
          if (l == 0) { ok = false; continue; }
          int f[3] = {gi, gj, gk};
          int c0[3], c1[3];
          for (int d = 0; d < 3; ++d) {
            c0[d] = floordiv2(f[d]);
            int r = f[d] - 2 * c0[d];
            c1[d] = (r == 0) ? c0[d] - 1 : c0[d] + 1;
          }
          if (o.p.interp == 4) {
            // O12, L70 "fourth-order spatial interpolation", L780 type 4 "quartic polynomial conservative": per axis
            // the quartic whose averages over the coarse cells c0-2 .. c0+2 equal their values, averaged over the
            // fine cell (the left or right half of c0):
            //   r = 0: c0 + (-3 c[-2] + 22 c[-1] - 22 c[+1] + 3 c[+2]) / 128      r = 1: the mirror image
            // (the two children average to c0: conservative); tensor product over the three axes.
            static const double WQ[2][5] = {{-3.0 / 128, 22.0 / 128, 1.0, -22.0 / 128, 3.0 / 128},
                                            {3.0 / 128, -22.0 / 128, 1.0, 22.0 / 128, -3.0 / 128}};
            int r[3];
            for (int d = 0; d < 3; ++d) r[d] = f[d] - 2 * c0[d];
            for (int c = 0; c < F.nc; ++c) {
              double sum = 0.0;
              for (int mz = -2; mz <= 2; ++mz)
                for (int my = -2; my <= 2; ++my)
                  for (int mx = -2; mx <= 2; ++mx) {
                    double vo = value(o, l - 1, *Cold, c, c0[0] + mx, c0[1] + my, c0[2] + mz, &ok);
                    double vn = value(o, l - 1, *Cnew, c, c0[0] + mx, c0[1] + my, c0[2] + mz, &ok);
                    double cv = (1.0 - alpha) * vo + alpha * vn;
                    double wt = (WQ[r[2]][mz + 2] * WQ[r[1]][my + 2]) * WQ[r[0]][mx + 2];
                    sum += wt * cv;
                  }
              F.at(c, i, j, k) = sum;
            }
            continue;
          }
          const double w[2] = {0.75, 0.25};
          for (int c = 0; c < F.nc; ++c) {
            double sum = 0.0;
            for (int dz = 0; dz < 2; ++dz)
              for (int dy = 0; dy < 2; ++dy)
                for (int dx = 0; dx < 2; ++dx) {
                  int ci = dx ? c1[0] : c0[0], cj = dy ? c1[1] : c0[1], ck = dz ? c1[2] : c0[2];
                  double vo = value(o, l - 1, *Cold, c, ci, cj, ck, &ok);
                  double vn = value(o, l - 1, *Cnew, c, ci, cj, ck, &ok);
                  double cv = (1.0 - alpha) * vo + alpha * vn;
                  double wt = (w[dz] * w[dy]) * w[dx];
                  sum += wt * cv;
                }
            F.at(c, i, j, k) = sum;
          }
        }
    if (!ok) {
#pragma omp critical
      all_ok = false;
    }
  }
  if (!all_ok) o.err = "ghost fill: a ghost cell has neither a same-level owner nor coarse data (nesting)";
  return all_ok;
}

// ---- O2: Laplacian ---------------------------------------------------------------------------
// order 1: sum_d [ (u(+e_d) - u) + (u(-e_d) - u) ] / h^2
// order 2: sum_d [ 16 ((u(+e_d) - u) + (u(-e_d) - u)) - ((u(+2e_d) - u) + (u(-2e_d) - u)) ] / (12 h^2)
// (neighbour-minus-centre form of [1,-2,1]/h^2 and [-1,16,-30,16,-1]/(12 h^2); it is exactly zero on
// constants, which the scalar-ODE pin relies on.)
inline double laplacian(const Field& F, int c, int i, int j, int k, int order, double h) {
  const double u = F.at(c, i, j, k);
  if (order == 1) {
    double sx = (F.at(c, i + 1, j, k) - u) + (F.at(c, i - 1, j, k) - u);
    double sy = (F.at(c, i, j + 1, k) - u) + (F.at(c, i, j - 1, k) - u);
    double sz = (F.at(c, i, j, k + 1) - u) + (F.at(c, i, j, k - 1) - u);
    return ((sx + sy) + sz) / (h * h);
  }
  double n1x = (F.at(c, i + 1, j, k) - u) + (F.at(c, i - 1, j, k) - u);
  double n1y = (F.at(c, i, j + 1, k) - u) + (F.at(c, i, j - 1, k) - u);
  double n1z = (F.at(c, i, j, k + 1) - u) + (F.at(c, i, j, k - 1) - u);
  double n2x = (F.at(c, i + 2, j, k) - u) + (F.at(c, i - 2, j, k) - u);
  double n2y = (F.at(c, i, j + 2, k) - u) + (F.at(c, i, j - 2, k) - u);
  double n2z = (F.at(c, i, j, k + 2) - u) + (F.at(c, i, j, k - 2) - u);
  double s1 = (n1x + n1y) + n1z;
  double s2 = (n2x + n2y) + n2z;
  if (order == 2) return (16.0 * s1 - s2) / (12.0 * (h * h));
  // order 3, 19-point (L649): per axis [2, -27, 270, -490, 270, -27, 2] / (180 h^2), the unique 6th-order central
  // stencil on 7 points, in the same neighbour-minus-centre form
  double n3x = (F.at(c, i + 3, j, k) - u) + (F.at(c, i - 3, j, k) - u);
  double n3y = (F.at(c, i, j + 3, k) - u) + (F.at(c, i, j - 3, k) - u);
  double n3z = (F.at(c, i, j, k + 3) - u) + (F.at(c, i, j, k - 3) - u);
  double s3 = (n3x + n3y) + n3z;
  return ((270.0 * s1 - 27.0 * s2) + 2.0 * s3) / (180.0 * (h * h));
}

// ---- O10: Kreiss-Oliger dissipation, Eq.7 (L141-146, L749-751) ---------------------------------
// sim.dissipation_order r in {2, 3} is "the number of ghost cells needed" (L751); Eq.7's p is then 2r - 1 (its
// (p+1)-st derivative is the 2r-th one, and (-1)^((p+3)/2) = (-1)^(r+1) is real only for odd p):
//   Q u = (-1)^(r+1) eps h^(2r-1) / 2^(2r) * sum_d d^(2r)u/dx_d^(2r),
// with the 2r-th derivative as the (2r+1)-point central difference delta^(2r) u / h^(2r):
//   r = 2: [1, -4, 6, -4, 1]        r = 3: [1, -6, 15, -20, 15, -6, 1]      (binomial coefficients, alternating)
// so Q u = (-1)^(r+1) eps / (2^(2r) h) * sum_d delta_d^(2r) u.  On a plane wave its eigenvalue is
// -(eps/h) sum_d sin^(2r)(k_d h / 2) <= 0.  It is added to the evolution of EVERY component, momenta included
// (L146 "each scalar field component"; the listing's Scalar::Pi1, L202, and Table I "for all field components",
// L749-750, make Pi1, Pi2 members of that set), each with its own strength (R22).
inline double ko_term(const Field& F, int c, int i, int j, int k, int r, double eps, double h) {
  static const double C2[5] = {1, -4, 6, -4, 1};
  static const double C3[7] = {1, -6, 15, -20, 15, -6, 1};
  const double* co = (r == 2) ? C2 : C3;
  double sum = 0.0;
  for (int d = 0; d < 3; ++d) {
    double dd = 0.0;
    for (int m = -r; m <= r; ++m)
      dd += co[m + r] * F.at(c, i + (d == 0 ? m : 0), j + (d == 1 ? m : 0), k + (d == 2 ? m : 0));
    sum += dd;
  }
  double sign = (r % 2 == 0) ? -1.0 : 1.0;  // (-1)^(r+1)
  return sign * eps / (std::pow(2.0, 2 * r) * h) * sum;
}

// ---- Gradient<order> (L651-658) ------------------------------------------------------------------
// "three-point, five-point, and seven-point stencil" for order 1, 2, 3; coefficients not printed: the unique
// maximal-order central first-difference stencils,
//   order 1: (u(+1) - u(-1)) / (2h)
//   order 2: (8 (u(+1) - u(-1)) - (u(+2) - u(-2))) / (12h)
//   order 3: (45 (u(+1) - u(-1)) - 9 (u(+2) - u(-2)) + (u(+3) - u(-3))) / (60h)
// (pinned by polynomial exactness up to degree 2 / 4 / 6 and the plane-wave symbols).
inline double gradient(const Field& F, int c, int i, int j, int k, int d, int order, double h) {
  int e[3] = {0, 0, 0};
  e[d] = 1;
  auto u = [&](int m) { return F.at(c, i + m * e[0], j + m * e[1], k + m * e[2]); };
  if (order == 1) return (u(1) - u(-1)) / (2.0 * h);
  if (order == 2) return (8.0 * (u(1) - u(-1)) - (u(2) - u(-2))) / (12.0 * h);
  return ((45.0 * (u(1) - u(-1)) - 9.0 * (u(2) - u(-2))) + (u(3) - u(-3))) / (60.0 * h);
}

// ---- O3: right-hand side, Eq.10-11 ------------------------------------------------------------
//   k_psi_c = Pi_c
//   k_Pi_c  = -(kappa/eta) Pi_c + Lap(psi_c) - lambda eta^2 psi_c (psi1^2 + psi2^2 - 1) - a psi_c
void eval_rhs(const Oracle& o, int l, const LevelState& S, LevelState& K, double eta) {
  const Level& L = o.lev[l];
  const Params& p = o.p;
#pragma omp parallel for schedule(dynamic)
  for (int q = 0; q < (int)L.boxes.size(); ++q) {
    const Field& F = S[q];
    Field& R = K[q];
    for (int k = 0; k < F.n[2]; ++k)
      for (int j = 0; j < F.n[1]; ++j)
        for (int i = 0; i < F.n[0]; ++i) {
          double psi1 = F.at(PSI1, i, j, k), psi2 = F.at(PSI2, i, j, k);
          double pi1 = F.at(PI1, i, j, k), pi2 = F.at(PI2, i, j, k);
          double lap1 = laplacian(F, PSI1, i, j, k, p.lap_order, L.h);
          double lap2 = laplacian(F, PSI2, i, j, k, p.lap_order, L.h);
          double pot = p.lambda * (eta * eta) * ((psi1 * psi1 + psi2 * psi2) - 1.0) + p.a_mass;
          double fr = (p.friction != 0.0) ? p.friction / eta : 0.0;
          R.at(PSI1, i, j, k) = pi1;
          R.at(PSI2, i, j, k) = pi2;
          R.at(PI1, i, j, k) = (lap1 - psi1 * pot) - fr * pi1;
          R.at(PI2, i, j, k) = (lap2 - psi2 * pot) - fr * pi2;
          for (int c = 0; c < NCOMP; ++c)  // Eq.7: Q_l u_c added to the evolution of every component
            if (p.ko_strength[c] != 0.0) R.at(c, i, j, k) += ko_term(F, c, i, j, k, p.ko_order, p.ko_strength[c], L.h);
          if (p.gw) {
            // O13, Eq.16 (L400-436) in the conformal-time form of Eq.9-11 (R25): for the six auxiliary
            // components ij = xx, yy, zz, xy, xz, yz
            //   k_u_ij  = du_ij
            //   k_du_ij = -(kappa_u / eta) du_ij + Lap(u_ij) + c_gw T_ij,   T_ij = sum_c d_i psi_c d_j psi_c
            // with Laplacian<order> and Gradient<order> of the same order (L649-658); the trace part of the scalar
            // stress tensor (delta_ij L) drops out under the TT projection of Eq.13-15 and is not added.
            double gr[2][3];
            for (int c = 0; c < 2; ++c)
              for (int d = 0; d < 3; ++d) gr[c][d] = gradient(F, c, i, j, k, d, p.lap_order, L.h);
            double fru = (p.gw_friction != 0.0) ? p.gw_friction / eta : 0.0;
            for (int m = 0; m < 6; ++m) {
              double T = gr[0][GW_I[m]] * gr[0][GW_J[m]] + gr[1][GW_I[m]] * gr[1][GW_J[m]];
              double lapu = laplacian(F, GW_U + m, i, j, k, p.lap_order, L.h);
              double du = F.at(GW_DU + m, i, j, k);
              R.at(GW_U + m, i, j, k) = du;
              R.at(GW_DU + m, i, j, k) = (lapu + p.gw_coupling * T) - fru * du;
            }
          }
        }
  }
}

// ---- O7: average-down, O9: truncation-error tags ----------------------------------------------
// O9 (self-shadow method, L82-98; Eq.5, Eq.6/12 with f = identity): just before level lf is synchronised onto
// lf-1, both have evolved the same region independently for 2 dt_lf.  For every coarse cell C under fine cells
//   Delta_c(C) = | phi_c^{lf-1}(C) - (1/8) sum_children phi_c^{lf} |,   c = psi1, psi2, Pi1, Pi2 (R21),
// with the coarse value taken BEFORE it is overwritten, and the 8 children of C get the tag byte
//   bit c = Delta_c > eps_c, one threshold per component            (strict >, Eq.12).
// counts: tagged fine cells per aligned FLAG_BLOCK^3 block of level lf.
bool average_down(Oracle& o, int lf) {
  if (lf < 1 || lf >= o.p.n_levels) { o.err = "average_down: bad fine level"; return false; }
  Level& Lf = o.lev[lf];
  Level& Lc = o.lev[lf - 1];
  bool all_ok = true;
  const bool tee = Lf.tee_on;
  int nb[3];
  for (int d = 0; d < 3; ++d) nb[d] = (Lf.n[d] + FLAG_BLOCK - 1) / FLAG_BLOCK;
  if (tee && Lf.tee_counts) memset(Lf.tee_counts, 0, sizeof(uint32_t) * (size_t)nb[0] * nb[1] * nb[2]);
  size_t tag_off = 0;
  for (int q = 0; q < (int)Lf.boxes.size(); ++q) {
    const BoxIn& B = o.box[Lf.boxes[q]];
    const Field& F = Lf.Y[q];
    for (int k = 0; k < F.n[2]; k += 2)
      for (int j = 0; j < F.n[1]; j += 2)
        for (int i = 0; i < F.n[0]; i += 2) {
          int ci = (B.lo[0] + i) / 2, cj = (B.lo[1] + j) / 2, ck = (B.lo[2] + k) / 2;
          int ow = owner_of(o, lf - 1, ci, cj, ck);
          if (ow < 0) { all_ok = false; continue; }
          const BoxIn& Bc = o.box[Lc.boxes[ow]];
          uint8_t tag = 0;
          for (int c = 0; c < F.nc; ++c) {
            double s = 0.0;
            for (int rz = 0; rz < 2; ++rz)
              for (int ry = 0; ry < 2; ++ry)
                for (int rx = 0; rx < 2; ++rx) s += F.at(c, i + rx, j + ry, k + rz);
            double mean = 0.125 * s;
            double& coarse = Lc.Y[ow].at(c, ci - Bc.lo[0], cj - Bc.lo[1], ck - Bc.lo[2]);
            if (tee && c < NCOMP) {  // every scalar component has its own threshold; DBL_MAX (the default) never tags
              double delta = std::fabs(coarse - mean);
              if (delta > Lf.tee_eps[c]) tag |= (uint8_t)(1u << c);
            }
            coarse = mean;
          }
          if (tee) {
            for (int rz = 0; rz < 2; ++rz)
              for (int ry = 0; ry < 2; ++ry)
                for (int rx = 0; rx < 2; ++rx)
                  if (Lf.tee_tags)
                    Lf.tee_tags[tag_off + ((size_t)(k + rz) * F.n[1] + (j + ry)) * F.n[0] + (i + rx)] = tag;
            if (tag && Lf.tee_counts) {
              int bi = (B.lo[0] + i) / FLAG_BLOCK, bj = (B.lo[1] + j) / FLAG_BLOCK, bk = (B.lo[2] + k) / FLAG_BLOCK;
              Lf.tee_counts[((size_t)bk * nb[1] + bj) * nb[0] + bi] += 8;
            }
          }
        }
    tag_off += (size_t)F.n[0] * F.n[1] * F.n[2];
  }
  if (!all_ok) o.err = "average_down: fine cell without a coarse parent";
  return all_ok;
}

// ---- O4 + O6: classic RK4 with recursive time subcycling ---------------------------------------
//   U_1 = Y;  k_s = f(U_s, eta_s), eta_s = t + c_s dt, c = (0, 1/2, 1/2, 1)
//   U_{s+1} = Y + a_s dt k_s, a = (1/2, 1/2, 1);  Y_new = Y + dt/6 (k_1 + 2 k_2 + 2 k_3 + k_4)
bool advance(Oracle& o, int l, double t, double dt, double eta_const);

// ---- O11: SSPRK3 (integrator.type 3 / 10, L808), the Shu-Osher form -----------------------------
//   U1   = Y + dt f(Y, t)
//   U2   = 3/4 Y + 1/4 (U1 + dt f(U1, t + dt))
//   Ynew = 1/3 Y + 2/3 (U2 + dt f(U2, t + dt/2))
// Types 3 and 10 are the same scheme ("smaller memory footprint", L808); ghosts of a stage state are filled at
// that stage's time t + c_s dt, c = (0, 1, 1/2), as for RK4 (L72).
bool advance_ssprk3(Oracle& o, int l, double t, double dt, double eta_const) {
  Level& L = o.lev[l];
  static const double cs[3] = {0.0, 1.0, 0.5};
  static const double wy[3] = {0.0, 0.75, 1.0 / 3.0};  // convex combination of a stage: wy Y + wu (U + dt f(U))
  static const double wu[3] = {1.0, 0.25, 2.0 / 3.0};
  L.Yold = L.Y;
  L.U = L.Y;
  for (int s = 0; s < 3; ++s) {
    double ts = t + cs[s] * dt;
    if (!fill_ghosts(o, l, L.U, ts)) return false;
    double eta_s = o.p.eta_fixed ? eta_const : ts;
    eval_rhs(o, l, L.U, L.K[s], eta_s);
#pragma omp parallel for schedule(dynamic)
    for (int q = 0; q < (int)L.boxes.size(); ++q) {
      Field& U = L.U[q];
      const Field& Y = L.Y[q];
      const Field& K = L.K[s][q];
      for (int c = 0; c < U.nc; ++c)
        for (int k = 0; k < U.n[2]; ++k)
          for (int j = 0; j < U.n[1]; ++j)
            for (int i = 0; i < U.n[0]; ++i) {
              double euler = U.at(c, i, j, k) + dt * K.at(c, i, j, k);  // forward-Euler step from the stage state
              U.at(c, i, j, k) = (s == 0) ? euler : wy[s] * Y.at(c, i, j, k) + wu[s] * euler;
            }
    }
  }
  L.Y = L.U;
  L.t_old = t;
  L.t_new = t + dt;
  L.have_pair = true;
  if (l + 1 < o.p.n_levels) {
    if (!advance(o, l + 1, t, 0.5 * dt, eta_const)) return false;
    if (!advance(o, l + 1, t + 0.5 * dt, 0.5 * dt, eta_const)) return false;
    if (!average_down(o, l + 1)) return false;
  }
  return true;
}

// ---- O14: user-defined Runge-Kutta-Nystrom scheme (integrator.type 20, L808-815) ------------------
// For psi'' = f(psi, eta) (Eq.9-11 without the friction term: f = Lap psi - psi (lambda eta^2 (|psi|^2 - 1) + a)),
// with the user's nodes c, weights b, bar-b and strictly lower-triangular tableau a (R26), s stages:
//   Psi_i   = psi + c_i dt Pi + dt^2 sum_{j<i} a_ij f_j,      f_i = f(Psi_i, t + c_i dt)
//   psi_new = psi + dt Pi + dt^2 sum_i bbar_i f_i,            Pi_new = Pi + dt sum_i b_i f_i
// Ghosts of a stage field are filled at its time t + c_i dt like those of any stage state (L72).  Sums run over
// j (i) ascending, starting from 0.
bool advance_rkn(Oracle& o, int l, double t, double dt, double eta_const) {
  Level& L = o.lev[l];
  const Params& p = o.p;
  const int s = p.rkn_stages;
  if ((int)L.KN.size() < s) {
    L.KN.resize(s);
    for (int i = 0; i < s; ++i) L.KN[i] = L.K[0];
  }
  L.Yold = L.Y;
  for (int i = 0; i < s; ++i) {
    const double* arow = p.rkn_a + i * (i + 1) / 2;
#pragma omp parallel for schedule(dynamic)
    for (int q = 0; q < (int)L.boxes.size(); ++q) {
      Field& U = L.U[q];
      const Field& Y = L.Y[q];
      for (int c = 0; c < 2; ++c)
        for (int k = 0; k < U.n[2]; ++k)
          for (int j = 0; j < U.n[1]; ++j)
            for (int ii = 0; ii < U.n[0]; ++ii) {
              double acc = 0.0;
              for (int m = 0; m < i; ++m) acc += arow[m] * L.KN[m][q].at(PI1 + c, ii, j, k);
              U.at(c, ii, j, k) = (Y.at(c, ii, j, k) + (p.rkn_c[i] * dt) * Y.at(PI1 + c, ii, j, k)) + (dt * dt) * acc;
              U.at(PI1 + c, ii, j, k) = Y.at(PI1 + c, ii, j, k);
            }
    }
    double ts = t + p.rkn_c[i] * dt;
    if (!fill_ghosts(o, l, L.U, ts)) return false;
    double eta_s = p.eta_fixed ? eta_const : ts;
    eval_rhs(o, l, L.U, L.KN[i], eta_s);  // friction = 0, no dissipation: its Pi components are f_i
  }
#pragma omp parallel for schedule(dynamic)
  for (int q = 0; q < (int)L.boxes.size(); ++q) {
    Field& Y = L.Y[q];
    for (int c = 0; c < 2; ++c)
      for (int k = 0; k < Y.n[2]; ++k)
        for (int j = 0; j < Y.n[1]; ++j)
          for (int i = 0; i < Y.n[0]; ++i) {
            double sb = 0.0, sbb = 0.0;
            for (int m = 0; m < s; ++m) {
              double f = L.KN[m][q].at(PI1 + c, i, j, k);
              sb += p.rkn_b[m] * f;
              sbb += p.rkn_bbar[m] * f;
            }
            double y = Y.at(c, i, j, k), yp = Y.at(PI1 + c, i, j, k);
            Y.at(c, i, j, k) = (y + dt * yp) + (dt * dt) * sbb;
            Y.at(PI1 + c, i, j, k) = yp + dt * sb;
          }
  }
  L.t_old = t;
  L.t_new = t + dt;
  L.have_pair = true;
  if (l + 1 < o.p.n_levels) {
    if (!advance(o, l + 1, t, 0.5 * dt, eta_const)) return false;
    if (!advance(o, l + 1, t + 0.5 * dt, 0.5 * dt, eta_const)) return false;
    if (!average_down(o, l + 1)) return false;
  }
  return true;
}

bool advance(Oracle& o, int l, double t, double dt, double eta_const) {
  if (o.p.integrator == 3 || o.p.integrator == 10) return advance_ssprk3(o, l, t, dt, eta_const);
  if (o.p.integrator == 20) return advance_rkn(o, l, t, dt, eta_const);
  Level& L = o.lev[l];
  static const double cs[4] = {0.0, 0.5, 0.5, 1.0};
  static const double as[3] = {0.5, 0.5, 1.0};
  L.Yold = L.Y;
  L.U = L.Y;
  for (int s = 0; s < 4; ++s) {
    double ts = t + cs[s] * dt;
    if (!fill_ghosts(o, l, L.U, ts)) return false;
    double eta_s = o.p.eta_fixed ? eta_const : ts;
    eval_rhs(o, l, L.U, L.K[s], eta_s);
    if (s < 3) {
      double adt = as[s] * dt;
#pragma omp parallel for schedule(dynamic)
      for (int q = 0; q < (int)L.boxes.size(); ++q) {
        Field& U = L.U[q];
        const Field& Y = L.Y[q];
        const Field& K = L.K[s][q];
        for (int c = 0; c < U.nc; ++c)
          for (int k = 0; k < U.n[2]; ++k)
            for (int j = 0; j < U.n[1]; ++j)
              for (int i = 0; i < U.n[0]; ++i) U.at(c, i, j, k) = Y.at(c, i, j, k) + adt * K.at(c, i, j, k);
      }
    }
  }
#pragma omp parallel for schedule(dynamic)
  for (int q = 0; q < (int)L.boxes.size(); ++q) {
    Field& Y = L.Y[q];
    for (int c = 0; c < Y.nc; ++c)
      for (int k = 0; k < Y.n[2]; ++k)
        for (int j = 0; j < Y.n[1]; ++j)
          for (int i = 0; i < Y.n[0]; ++i) {
            double k1 = L.K[0][q].at(c, i, j, k), k2 = L.K[1][q].at(c, i, j, k);
            double k3 = L.K[2][q].at(c, i, j, k), k4 = L.K[3][q].at(c, i, j, k);
            Y.at(c, i, j, k) = Y.at(c, i, j, k) + (dt / 6.0) * (((k1 + 2.0 * k2) + 2.0 * k3) + k4);
          }
  }
  L.t_old = t;
  L.t_new = t + dt;
  L.have_pair = true;
  if (l + 1 < o.p.n_levels) {
    if (!advance(o, l + 1, t, 0.5 * dt, eta_const)) return false;
    if (!advance(o, l + 1, t + 0.5 * dt, 0.5 * dt, eta_const)) return false;
    if (!average_down(o, l + 1)) return false;  // the synchronised state is this level's state at t_new
  }
  return true;
}

// ---- O8: string tags ---------------------------------------------------------------------------
// Winding number of the polygon psi(A)->psi(B)->psi(C)->psi(D)->psi(A) around the origin, counted by
// signed crossings of the positive psi1 axis.  Edge a->b: up = a2<0 && b2>=0, dn = a2>=0 && b2<0,
// cr = a1*b2 - a2*b1 (two products and one subtraction, each rounded; no FMA);
// +1 if up && cr>0, -1 if dn && cr<0.
inline int edge_crossing(double a1, double a2, double b1, double b2) {
  bool up = (a2 < 0.0) && (b2 >= 0.0);
  bool dn = (a2 >= 0.0) && (b2 < 0.0);
  double p = a1 * b2;
  double q = a2 * b1;
  double cr = p - q;
  if (up && cr > 0.0) return 1;
  if (dn && cr < 0.0) return -1;
  return 0;
}
inline int plaquette_winding(const double A[2], const double B[2], const double C[2], const double D[2]) {
  return edge_crossing(A[0], A[1], B[0], B[1]) + edge_crossing(B[0], B[1], C[0], C[1]) +
         edge_crossing(C[0], C[1], D[0], D[1]) + edge_crossing(D[0], D[1], A[0], A[1]);
}

// tags: one byte per valid cell, boxes of the level concatenated in box order, x fastest.
// counts: dense array over aligned FLAG_BLOCK^3 blocks of the level index space, x fastest.
bool tag_strings(Oracle& o, int l, uint8_t* tags, uint32_t* counts) {
  Level& L = o.lev[l];
  // after a coarse step all levels sit at the parent's t_new (alpha = 1: no temporal interpolation, L74)
  double tcur = (l > 0 && o.lev[l - 1].have_pair) ? o.lev[l - 1].t_new : 0.0;
  if (!fill_ghosts(o, l, L.Y, tcur)) return false;
  int nb[3];
  for (int d = 0; d < 3; ++d) nb[d] = (L.n[d] + FLAG_BLOCK - 1) / FLAG_BLOCK;
  if (counts) memset(counts, 0, sizeof(uint32_t) * (size_t)nb[0] * nb[1] * nb[2]);
  size_t off = 0;
  static const int D1[3] = {0, 1, 2};  // (x,y), (y,z), (z,x)
  static const int D2[3] = {1, 2, 0};
  for (int q = 0; q < (int)L.boxes.size(); ++q) {
    const BoxIn& B = o.box[L.boxes[q]];
    const Field& F = L.Y[q];
    for (int k = 0; k < F.n[2]; ++k)
      for (int j = 0; j < F.n[1]; ++j)
        for (int i = 0; i < F.n[0]; ++i) {
          uint8_t tag = 0;
          for (int pl = 0; pl < 3; ++pl) {
            int e1[3] = {0, 0, 0}, e2[3] = {0, 0, 0};
            e1[D1[pl]] = 1;
            e2[D2[pl]] = 1;
            double A[2] = {F.at(PSI1, i, j, k), F.at(PSI2, i, j, k)};
            double Bv[2] = {F.at(PSI1, i + e1[0], j + e1[1], k + e1[2]), F.at(PSI2, i + e1[0], j + e1[1], k + e1[2])};
            double C[2] = {F.at(PSI1, i + e1[0] + e2[0], j + e1[1] + e2[1], k + e1[2] + e2[2]),
                           F.at(PSI2, i + e1[0] + e2[0], j + e1[1] + e2[1], k + e1[2] + e2[2])};
            double Dv[2] = {F.at(PSI1, i + e2[0], j + e2[1], k + e2[2]), F.at(PSI2, i + e2[0], j + e2[1], k + e2[2])};
            int W = plaquette_winding(A, Bv, C, Dv);
            if (W != 0) tag |= (uint8_t)(1u << pl);
          }
          if (tags) tags[off] = tag;
          ++off;
          if (tag && counts) {
            int bi = (B.lo[0] + i) / FLAG_BLOCK, bj = (B.lo[1] + j) / FLAG_BLOCK, bk = (B.lo[2] + k) / FLAG_BLOCK;
            counts[((size_t)bk * nb[1] + bj) * nb[0] + bi] += 1;
          }
        }
  }
  return true;
}

}  // namespace

// =================================================================================================
// C interface for ctypes (tests / smoke / cpu_baseline only)
// =================================================================================================
extern "C" {

typedef struct {
  int32_t n_levels;
  int32_t n0[3];
  int32_t nghost;
  int32_t blocking_factor;
  int32_t lap_order;
  int32_t eta_fixed;
  double h0, lambda, a_mass, friction;
  double ko_strength[4];
  int32_t ko_order;
  int32_t integrator;
  int32_t interp;
  int32_t gw;
  double gw_coupling, gw_friction;
  int32_t rkn_stages;
  int32_t pad_;
  double rkn_c[6], rkn_b[6], rkn_bbar[6], rkn_a[21];
} orc_params;

typedef struct {
  int32_t level;
  int32_t lo[3];
  int32_t hi[3];
} orc_box;

static std::string g_err;

const char* orc_last_error(void* h) {
  if (h) return ((Oracle*)h)->err.c_str();
  return g_err.c_str();
}

void* orc_create(const orc_params* p, const orc_box* b, int nbox) {
  Oracle* o = new Oracle();
  static_assert(sizeof(orc_params) == sizeof(Params), "layout");
  static_assert(sizeof(orc_box) == sizeof(BoxIn), "layout");
  memcpy(&o->p, p, sizeof(Params));
  if (!build(*o, (const BoxIn*)b, nbox)) {
    g_err = o->err;
    delete o;
    return nullptr;
  }
  return o;
}

void orc_destroy(void* h) { delete (Oracle*)h; }

int orc_num_boxes(void* h, int level) { return (int)((Oracle*)h)->lev[level].boxes.size(); }

// src/dst: dense valid region of global box `ib`, x fastest.
int orc_set_state(void* h, int ib, int comp, const double* src) {
  Oracle& o = *(Oracle*)h;
  if (ib < 0 || ib >= (int)o.box.size() || comp < 0 || comp >= (o.p.gw ? NCOMP_GW : NCOMP)) return -1;
  Field& F = o.lev[o.box[ib].level].Y[o.box_local[ib]];
  size_t q = 0;
  for (int k = 0; k < F.n[2]; ++k)
    for (int j = 0; j < F.n[1]; ++j)
      for (int i = 0; i < F.n[0]; ++i) F.at(comp, i, j, k) = src[q++];
  return 0;
}
int orc_get_state(void* h, int ib, int comp, double* dst) {
  Oracle& o = *(Oracle*)h;
  if (ib < 0 || ib >= (int)o.box.size() || comp < 0 || comp >= (o.p.gw ? NCOMP_GW : NCOMP)) return -1;
  const Field& F = o.lev[o.box[ib].level].Y[o.box_local[ib]];
  size_t q = 0;
  for (int k = 0; k < F.n[2]; ++k)
    for (int j = 0; j < F.n[1]; ++j)
      for (int i = 0; i < F.n[0]; ++i) dst[q++] = F.at(comp, i, j, k);
  return 0;
}
// raw access including ghosts (array extent n+2g per axis, x fastest); which: 0 = Y, 1 = last k (K[0])
int orc_set_raw(void* h, int ib, int comp, const double* src) {
  Oracle& o = *(Oracle*)h;
  Field& F = o.lev[o.box[ib].level].Y[o.box_local[ib]];
  size_t q = 0;
  for (int k = -F.g; k < F.n[2] + F.g; ++k)
    for (int j = -F.g; j < F.n[1] + F.g; ++j)
      for (int i = -F.g; i < F.n[0] + F.g; ++i) F.at(comp, i, j, k) = src[q++];
  return 0;
}
int orc_get_raw(void* h, int ib, int comp, int which, double* dst) {
  Oracle& o = *(Oracle*)h;
  Level& L = o.lev[o.box[ib].level];
  const Field& F = (which == 0) ? L.Y[o.box_local[ib]] : L.K[0][o.box_local[ib]];
  size_t q = 0;
  for (int k = -F.g; k < F.n[2] + F.g; ++k)
    for (int j = -F.g; j < F.n[1] + F.g; ++j)
      for (int i = -F.g; i < F.n[0] + F.g; ++i) dst[q++] = F.at(comp, i, j, k);
  return 0;
}

int orc_fill_ghosts(void* h, int level, double time) {
  Oracle& o = *(Oracle*)h;
  if (level < 0 || level >= o.p.n_levels) return -1;
  return fill_ghosts(o, level, o.lev[level].Y, time) ? 0 : -1;
}

// k = f(Y, eta) into K[0] of the level, using whatever the ghosts of Y currently hold
// (do_fill = 1 fills them first at time eta).
int orc_eval_rhs(void* h, int level, double eta, int do_fill) {
  Oracle& o = *(Oracle*)h;
  if (level < 0 || level >= o.p.n_levels) return -1;
  Level& L = o.lev[level];
  if (do_fill && !fill_ghosts(o, level, L.Y, eta)) return -1;
  eval_rhs(o, level, L.Y, L.K[0], eta);
  return 0;
}

// One coarse step of the whole hierarchy from time eta to eta + dt (O6).
int orc_rk_step(void* h, double dt, double eta) {
  Oracle& o = *(Oracle*)h;
  return advance(o, 0, eta, dt, eta) ? 0 : -1;
}

// O9: from now on every synchronisation of `fine_level` also writes truncation-error tags (tags / counts stay owned
// by the caller and must outlive the handle's use; tags == nullptr switches it off)
int orc_tee_enable(void* h, int fine_level, const double* eps4, uint8_t* tags, uint32_t* counts) {
  Oracle& o = *(Oracle*)h;
  if (fine_level < 1 || fine_level >= o.p.n_levels) return -1;
  Level& L = o.lev[fine_level];
  L.tee_on = tags != nullptr || counts != nullptr;
  for (int c = 0; c < NCOMP; ++c) L.tee_eps[c] = eps4[c];
  L.tee_tags = tags;
  L.tee_counts = counts;
  return 0;
}

int orc_average_down(void* h, int fine_level) { return average_down(*(Oracle*)h, fine_level) ? 0 : -1; }

// O15, the shadow level (L98; R27): level 0 has no coarser partner, so "shortly before cell tagging" a
// coarsened copy of it is made -- shadow cell C <- mean of its 8 level-0 children, spacing 2 h_0, ONE box over the
// same periodic domain -- and evolved for a single step of 2 dt while the hierarchy takes two coarse steps of dt; then
//   Delta_c(C) = | shadow_c(C) - (1/8) sum_children phi_c^0 |,  c = psi1, psi2, Pi1, Pi2
// tags the 8 children with bit c iff Delta_c > eps_c (strict, as O9), and the shadow level is discarded.
// tags: one byte per valid level-0 cell, boxes back to back in input order, x fastest; counts: tagged cells per
// aligned 32^3 block of level 0.  The hierarchy ends at eta + 2 dt.
int orc_shadow_tee(void* h, double dt, double eta, const double* eps4, uint8_t* tags, uint32_t* counts) {
  Oracle& o = *(Oracle*)h;
  const Params& p = o.p;
  Oracle sh;
  sh.p = p;
  sh.p.n_levels = 1;
  sh.p.h0 = 2.0 * p.h0;
  int bf = p.blocking_factor;
  for (int d = 0; d < 3; ++d) {
    if (p.n0[d] % 2) { o.err = "shadow level: n0 must be even"; return -1; }
    sh.p.n0[d] = p.n0[d] / 2;
    while (bf > 1 && sh.p.n0[d] % bf) bf /= 2;
  }
  sh.p.blocking_factor = bf;
  BoxIn sb;
  sb.level = 0;
  for (int d = 0; d < 3; ++d) { sb.lo[d] = 0; sb.hi[d] = sh.p.n0[d] - 1; }
  if (!build(sh, &sb, 1)) { o.err = "shadow level: " + sh.err; return -1; }
  Level& L0 = o.lev[0];
  Field& S = sh.lev[0].Y[0];
  auto child = [&](int c, int i, int j, int k) {  // valid level-0 value at level index (i, j, k)
    int ow = owner_of(o, 0, i, j, k);
    const BoxIn& B = o.box[L0.boxes[ow]];
    return L0.Y[ow].at(c, i - B.lo[0], j - B.lo[1], k - B.lo[2]);
  };
  auto mean8 = [&](int c, int I, int J, int K) {
    double s = 0.0;
    for (int rz = 0; rz < 2; ++rz)
      for (int ry = 0; ry < 2; ++ry)
        for (int rx = 0; rx < 2; ++rx) s += child(c, 2 * I + rx, 2 * J + ry, 2 * K + rz);
    return 0.125 * s;
  };
  for (int c = 0; c < S.nc; ++c)
    for (int K = 0; K < S.n[2]; ++K)
      for (int J = 0; J < S.n[1]; ++J)
        for (int I = 0; I < S.n[0]; ++I) S.at(c, I, J, K) = mean8(c, I, J, K);
  if (!advance(sh, 0, eta, 2.0 * dt, eta)) { o.err = "shadow level: " + sh.err; return -1; }
  if (!advance(o, 0, eta, dt, eta)) return -1;
  if (!advance(o, 0, eta + dt, dt, eta + dt)) return -1;
  int nb[3];
  for (int d = 0; d < 3; ++d) nb[d] = (L0.n[d] + FLAG_BLOCK - 1) / FLAG_BLOCK;
  if (counts) memset(counts, 0, sizeof(uint32_t) * (size_t)nb[0] * nb[1] * nb[2]);
  std::vector<size_t> tag_off(L0.boxes.size(), 0);
  for (size_t q = 1; q < L0.boxes.size(); ++q)
    tag_off[q] = tag_off[q - 1] + (size_t)L0.Y[q - 1].n[0] * L0.Y[q - 1].n[1] * L0.Y[q - 1].n[2];
  for (int K = 0; K < S.n[2]; ++K)
    for (int J = 0; J < S.n[1]; ++J)
      for (int I = 0; I < S.n[0]; ++I) {
        uint8_t tag = 0;
        for (int c = 0; c < NCOMP; ++c)
          if (std::fabs(S.at(c, I, J, K) - mean8(c, I, J, K)) > eps4[c]) tag |= (uint8_t)(1u << c);
        int ow = owner_of(o, 0, 2 * I, 2 * J, 2 * K);
        const BoxIn& B = o.box[L0.boxes[ow]];
        const Field& F = L0.Y[ow];
        for (int rz = 0; rz < 2; ++rz)
          for (int ry = 0; ry < 2; ++ry)
            for (int rx = 0; rx < 2; ++rx)
              if (tags)
                tags[tag_off[ow] + ((size_t)(2 * K + rz - B.lo[2]) * F.n[1] + (2 * J + ry - B.lo[1])) * F.n[0] + (2 * I + rx - B.lo[0])] = tag;
        if (tag && counts) counts[((size_t)(2 * K / FLAG_BLOCK) * nb[1] + 2 * J / FLAG_BLOCK) * nb[0] + 2 * I / FLAG_BLOCK] += 8;
      }
  return 0;
}

int orc_tag_strings(void* h, int level, uint8_t* tags, uint32_t* counts) {
  Oracle& o = *(Oracle*)h;
  if (level < 0 || level >= o.p.n_levels) return -1;
  return tag_strings(o, level, tags, counts) ? 0 : -1;
}

// winding number of one plaquette given its four corner values (for brute-force pins)
int orc_plaquette_winding(const double* A, const double* B, const double* C, const double* D) {
  return plaquette_winding(A, B, C, D);
}

// Level-0 energies, summed over valid cells times h^3.  Ghosts of Y are filled first.
//  out[0] = sum 1/2 (Pi1^2 + Pi2^2)
//  out[1] = sum -1/2 (psi1 Lap psi1 + psi2 Lap psi2)          (conserved discrete gradient energy)
//  out[2] = sum lambda eta^2 / 4 (psi1^2 + psi2^2 - 1)^2 + a/2 (psi1^2+psi2^2)
//  out[3] = sum 1/2 |Gradient<order> psi|^2                    (paper's E of App.B)
int orc_energy(void* h, double eta, double* out) {
  Oracle& o = *(Oracle*)h;
  Level& L = o.lev[0];
  if (!fill_ghosts(o, 0, L.Y, eta)) return -1;
  double e[4] = {0, 0, 0, 0};
  double h3 = L.h * L.h * L.h;
  for (size_t q = 0; q < L.boxes.size(); ++q) {
    const Field& F = L.Y[q];
    for (int k = 0; k < F.n[2]; ++k)
      for (int j = 0; j < F.n[1]; ++j)
        for (int i = 0; i < F.n[0]; ++i) {
          double p1 = F.at(PSI1, i, j, k), p2 = F.at(PSI2, i, j, k);
          double q1 = F.at(PI1, i, j, k), q2 = F.at(PI2, i, j, k);
          e[0] += 0.5 * (q1 * q1 + q2 * q2);
          e[1] += -0.5 * (p1 * laplacian(F, PSI1, i, j, k, o.p.lap_order, L.h) +
                          p2 * laplacian(F, PSI2, i, j, k, o.p.lap_order, L.h));
          double m = p1 * p1 + p2 * p2;
          e[2] += 0.25 * o.p.lambda * eta * eta * (m - 1.0) * (m - 1.0) + 0.5 * o.p.a_mass * m;
          double gsum = 0.0;
          for (int c = 0; c < 2; ++c)
            for (int d = 0; d < 3; ++d) {
              double gd = gradient(F, c, i, j, k, d, o.p.lap_order, L.h);
              gsum += gd * gd;
            }
          e[3] += 0.5 * gsum;
        }
  }
  for (int m = 0; m < 4; ++m) out[m] = e[m] * h3;
  return 0;
}

// test / timing infrastructure: number of OpenMP threads the loops over boxes may use (1 = serial)
void orc_set_threads(int n) {
#ifdef _OPENMP
  if (n >= 1) omp_set_num_threads(n);
#else
  (void)n;
#endif
}

int orc_omp_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

}  // extern "C"
