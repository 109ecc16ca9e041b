// sledge.cu -- host side of libsledge.so: hierarchy validation, arena layout, launch logic, C ABI.
//
// Everything the path computes runs in the kernels under csrc/k_*.cuh; this file only validates the box
// list, lays the caller's arena out, builds the device descriptor
// tables and enqueues launches on the caller's stream.  There is no CPU fallback of any step.
#include "../../include/sledge.h"

#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <vector>

#include "k_avgdown.cuh"
#include "k_ghost.cuh"
#include "k_gw.cuh"
#include "k_rk_pipe.cuh"
#include "k_rk_plane.cuh"
#include "k_rk_tma.cuh"
#include "k_tag.cuh"

using namespace sledge;

namespace {

constexpr int NBUF = 4;
constexpr int COUNT_BLOCK = 32;  // box-flag reduction granularity (BASELINE.json config 3)
constexpr int MAX_EVENT_PAIRS = 4096;
constexpr size_t ALIGN = 256;

// K1 tile shape (threads; cells per tile in x = TX * cells-per-16-bytes), z-chunk length and cp.async ring depth
#ifndef SLEDGE_K1_TY
#define SLEDGE_K1_TY 16
#endif
#ifndef SLEDGE_K1_NZ
#define SLEDGE_K1_NZ 128
#endif
#ifndef SLEDGE_K1_DMAX
#define SLEDGE_K1_DMAX 4
#endif
#ifndef SLEDGE_K1_SMEM
#define SLEDGE_K1_SMEM (227 * 1024)
#endif
// The FUSED sweeps load fp64 pipe, shared-memory bandwidth and HBM to within 2x of each other: they want several
// small CTAs per SM so that one CTA's barrier / load phase overlaps another's arithmetic.  Measured on C3
// (profiles/r01_k1_tile_sweep.md): 32x8 tile, two rows per thread (128 threads), prefetch distance 2 (113 KB budget),
// 3 (sweep A) / 2 (sweep B) CTAs per SM.
#ifndef SLEDGE_K1F_TY
#define SLEDGE_K1F_TY 8
#endif
#ifndef SLEDGE_K1F_SMEM
#define SLEDGE_K1F_SMEM (113 * 1024)
#endif
#ifndef SLEDGE_K1F_TX
#define SLEDGE_K1F_TX 32
#endif
constexpr int K1_TX = 32, K1_TY = SLEDGE_K1_TY, K1_NZ = SLEDGE_K1_NZ;
constexpr int K1F_TX = SLEDGE_K1F_TX;  // x vectors per fused tile (k_rk_plane)
constexpr int K1_DMAX = SLEDGE_K1_DMAX;          // cp.async ring: deepest that fits K1_SMEM, at most this
constexpr size_t K1_SMEM = SLEDGE_K1_SMEM;       // shared-memory budget per CTA (227 KB = sm_100a opt-in limit)
constexpr long long K1F_MIN_TILES = 3500;
static_assert(GW_TY == SLEDGE_K1F_TY && GW_TX == SLEDGE_K1F_TX, "k_gw_stage runs over the fused-sweep tiles");
#ifndef SLEDGE_TAG_MIN_NZ
#define SLEDGE_TAG_MIN_NZ 16
#endif
constexpr int TAG_MIN_NZ = SLEDGE_TAG_MIN_NZ;  // shortest z-chunk of a tag tile
constexpr long long TAG_MIN_TILES = 148 * 4 * 6;  // below this many CTAs the tag pass halves its z-chunk (down to TAG_MIN_NZ planes)  // below this many CTAs the fused sweeps halve their z-chunk
constexpr int K1F_TY = SLEDGE_K1F_TY;            // tile rows / budget of the FUSED sweeps
constexpr size_t K1F_SMEM = SLEDGE_K1F_SMEM;
// which on-chip data path a sweep uses: 1 = k_rk_plane (ghosted plane ring), 0 = k_rk_pipe (ring + centre plane)
#ifndef SLEDGE_K1F_PLANE
#define SLEDGE_K1F_PLANE 1
#endif
#ifndef SLEDGE_K1_PLANE
#define SLEDGE_K1_PLANE 0
#endif
#ifndef SLEDGE_K1F_PDMAX
#define SLEDGE_K1F_PDMAX 2
#endif
#ifndef SLEDGE_K1_RY
#define SLEDGE_K1_RY 1
#endif
#ifndef SLEDGE_K1F_RY
#define SLEDGE_K1F_RY 2
#endif
#ifndef SLEDGE_K1F_RY32
#define SLEDGE_K1F_RY32 1  // fp32 sweeps move half the bytes per cell through shared memory: one row per thread is faster
#endif
#ifndef SLEDGE_K1F_MINB_A
#define SLEDGE_K1F_MINB_A 3
#endif
#ifndef SLEDGE_K1F_MINB_B
#define SLEDGE_K1F_MINB_B 2
#endif
#ifndef SLEDGE_K1F_MINB_B2
#define SLEDGE_K1F_MINB_B2 2
#endif
template <int MODE> struct K1Shape {
  static constexpr bool fused = (MODE == FUSED_A || MODE == FUSED_B || MODE == FUSED_A2 || MODE == FUSED_B2);
  static constexpr int TY = fused ? K1F_TY : K1_TY;
  static constexpr size_t SMEM = fused ? K1F_SMEM : K1_SMEM;
  static constexpr bool plane = fused ? (SLEDGE_K1F_PLANE != 0) : (SLEDGE_K1_PLANE != 0);
  static constexpr int PDMAX = fused ? SLEDGE_K1F_PDMAX : 3;
  static constexpr int RY = fused ? SLEDGE_K1F_RY : SLEDGE_K1_RY;  // rows per thread (k_rk_plane)
  static constexpr int MINB = (MODE == FUSED_A || MODE == FUSED_A2) ? SLEDGE_K1F_MINB_A : (MODE == FUSED_B ? SLEDGE_K1F_MINB_B : (MODE == FUSED_B2 ? SLEDGE_K1F_MINB_B2 : 1));
};

// rows per thread of the FUSED sweeps (k_rk_plane / k_rk_tma); the tensor maps' box shape follows from it
template <typename T, int ORDER> struct FusedTile {
  // the 7-plane z-window of the 19-point stencil leaves no registers for a second row
  static constexpr int RY = ORDER == 3 ? 1 : (sizeof(T) == 4 ? SLEDGE_K1F_RY32 : SLEDGE_K1F_RY);
};
#ifndef SLEDGE_K1F_TMA_PDMAX
#define SLEDGE_K1F_TMA_PDMAX 2
#endif

thread_local std::string g_err;

struct LevelHost {
  int n[3], no[3];
  double h;
  std::vector<int> boxes;  // global box ids in input order
  std::vector<BoxDev> boxdev;   // STORAGE boxes: the caller's boxes coalesced into larger rectangles (K1, K2, K4 coarse side)
  std::vector<BoxDev> viewdev;  // the caller's boxes in input order, as windows into their storage box (K3, K4 fine side, copies)
  size_t off_views = 0;
  std::vector<int> owner;
  std::vector<TileDev> tiles, ftiles, tag_tiles;  // K1 staged / K1 fused / K3
  std::vector<int> ghost_prefix, avg_prefix;
  // K3 over storage boxes: per blocking-factor cell the tag offset of its first cell and n0, n1 of the caller's box
  // (k_tag.cuh tag_cells); empty when the tag tiles run over the caller's boxes themselves
  std::vector<int4> tag_cells;
  size_t off_tag_cells = 0;
  std::vector<int> qp_prefix;  // quartic interpolation by coarse parent (k_fill_qparents): CTAs before box b
  size_t off_qp_prefix = 0, off_qp_list = 0, off_qs_list = 0, off_qs_count = 0;
  unsigned n_star_parents = 0;  // read back from the device after the plan
  size_t off_star_list = 0, off_star_count = 0;
  std::vector<uint4> patches, tag_patches;  // star patches / tag patches (k_fill_patches), 2 x uint4 each
  size_t off_patches = 0, off_tag_patches = 0;
  unsigned n_copy_patches = 0;  // the star patch list is sorted: same-level copies first (a copies-only fill launches just those)
  int patch_smem_pairs = 0;    // largest coarse region of an interpolation patch (pairs)
  size_t off_tmaps = 0;        // k_rk_tma: CUtensorMap[NBUF * 2][nbox] of the level's state planes (fused levels only)
  bool has_tmaps = false;
  std::vector<CUtensorMap> tmaps_host;
  // periodic one-box level under the TMA sweeps: star ghost cells (psi and Pi) of buffer b are periodic images of
  // the buffer's current valid data (the sweep that wrote the buffer stored them, or a K2 fill since)
  bool star_ok[4] = {false, false, false, false};
  unsigned n_star = 0;          // GHOST_STAR entries of the ghost list, packed (read back after the plan)
  long long plane_cells = 0;  // pairs per plane (all boxes, ghosts and padding included)
  long long valid_cells = 0;
  long long count_blocks = 0;
  int nb[3];
  bool periodic_box = false;  // ONE box covering the periodic domain: K1 (plane variant) and K3 wrap by themselves
  // arena offsets (bytes)
  size_t off_buf[NBUF][2];
  size_t off_gw[NBUF][6] = {};  // gw: pair planes (u_xx,u_yy) (u_zz,u_xy) (u_xz,u_yz) (du_xx,du_yy) (du_zz,du_xy) (du_xz,du_yz)
  size_t off_boxes, off_tiles, off_ftiles, off_tag_tiles, off_owner, off_ghost_prefix, off_avg_prefix, off_ghost_list;
  // truncation-error tags written at this (fine) level's synchronisations (sledge_tee_enable)
  bool tee_on = false;
  double tee_eps[4] = {0, 0, 0, 0};
  uint8_t* tee_tags = nullptr;
  uint32_t* tee_counts = nullptr;
  // quartic interpolation reads coarse windows through the coarse boxes' ghost cells: true while the whole ghost
  // shell of buffer b (psi and Pi) holds same-level copies of the buffer's current valid data
  int shell_ok[NBUF] = {0, 0, 0, 0};  // 0 = stale, 1 = psi shell valid, 2 = psi and Pi
  // run state
  int cur = 0, old = 0;
  bool have_pair = false;
  double t_old = 0, t_new = 0;
};

struct Plan {
  sledge_params p;
  std::vector<sledge_box> box;
  std::vector<int> box_local;
  std::vector<LevelHost> lev;
  int esz = 8;       // bytes per real
  int cpa = 8;       // cells (pairs) per 128 bytes
  int ox = 8;        // x offset of the first valid cell inside a row
  size_t off_scratch = 0, scratch_bytes = 0, off_err = 0, total = 0;
  bool fine_fused = false;  // FUSED sweeps on levels > 0 too (needs the patch fills' velocity ghosts; set at create)
  // shadow level of level 0 (L98): a nested one-box context inside the same arena
  size_t off_shadow = 0, shadow_bytes = 0;
  sledge_params shadow_p;
  sledge_box shadow_box;
};

}  // namespace

constexpr int N_IN_SLOTS = 2, N_OUT_SLOTS = 4;  // staging slots of the host-buffer copies (one box component each)

struct sledge_ctx {
  Plan plan;
  char* arena = nullptr;
  cudaStream_t stream = nullptr;
  std::string err;
  int64_t launches = 0;
  bool profiling = false;
  bool use_tma = true;  // FUSED sweeps through k_rk_tma (SLEDGE_K1_TMA=0 in the environment selects k_rk_plane)
  bool fill_once = true;  // fine FUSED levels, trilinear: interpolated ghosts of both sweeps in one fill (SLEDGE_FILL_ONCE=0: two)
  bool fused_w = true;  // fp64 FUSED sweeps in the W form (SLEDGE_FUSED_W=0 selects the three-field sweep B)
  bool use_patches = true;  // fills before an RK sweep by region (SLEDGE_K2_PATCHES=0 selects the packed per-cell list)
  sledge_ctx* shadow = nullptr;  // the shadow level's context (shadow_level = 1)
  // host-buffer copies (sledge_set_state_host / get_state_host) run on two streams of their own, double-buffered through
  // the staging slots, so that uploads, repacking kernels and downloads overlap (PCIe is full duplex)
  cudaStream_t s_h2d = nullptr, s_d2h = nullptr;
  // two upload slots; four download slots, so that the repacking kernels of a whole state's downloads never wait on
  // the context stream (ahead of the next step's uploads) for a PCIe copy to drain a slot
  cudaEvent_t ev_in_ready[N_IN_SLOTS] = {}, ev_in_free[N_IN_SLOTS] = {};
  cudaEvent_t ev_out_ready[N_OUT_SLOTS] = {}, ev_out_free[N_OUT_SLOTS] = {};
  bool in_used[N_IN_SLOTS] = {}, out_used[N_OUT_SLOTS] = {};
  unsigned n_in = 0, n_out = 0;
  int device = 0;  // the device the arena lives on: every entry point runs with it current (DeviceGuard)
  std::vector<std::pair<cudaEvent_t, cudaEvent_t>> ev[4];
  size_t ev_used[4] = {0, 0, 0, 0};
};

namespace {

// Kreiss-Oliger dissipation (Eq.7) is on when any component has a non-zero strength (L749)
inline bool ko_on(const sledge_params& p) {
  return p.ko_strength[0] != 0.0 || p.ko_strength[1] != 0.0 || p.ko_strength[2] != 0.0 || p.ko_strength[3] != 0.0;
}
// quartic coarse->fine interpolation evaluated per coarse parent through the coarse boxes' ghost cells (needs two
// coarse ghost layers); with one ghost layer the per-cell entries of k_fill_ghosts<.., QUARTIC> are used
inline bool quartic_by_parent(const sledge_params& p) { return p.interp == SLEDGE_INTERP_QUARTIC && p.nghost >= 2; }
inline bool is_rkn(const sledge_params& p) { return p.integrator == 20; }
inline int stencil_radius(const sledge_params& p) { return ko_on(p) && p.ko_order > p.lap_order ? p.ko_order : p.lap_order; }

int fail(sledge_ctx* ctx, int code, const char* fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof buf, fmt, ap);
  va_end(ap);
  if (ctx) ctx->err = buf; else g_err = buf;
  return code;
}

// Kernel attributes (opt-in shared-memory size) are per device: one flag per device and kernel instantiation.
constexpr int MAX_DEVICES = 64;
struct PerDevice {
  bool done[MAX_DEVICES] = {};
  bool& operator[](int d) { return done[d >= 0 && d < MAX_DEVICES ? d : 0]; }
};
// Makes the context's device current for the duration of an entry point and restores the caller's.
struct DeviceGuard {
  int prev = -1;
  bool switched = false;
  explicit DeviceGuard(int dev) {
    if (cudaGetDevice(&prev) == cudaSuccess && prev != dev) switched = cudaSetDevice(dev) == cudaSuccess;
    else cudaGetLastError();
  }
  ~DeviceGuard() {
    if (switched) cudaSetDevice(prev);
  }
};

inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }
inline int ilog2(int v) {
  int s = 0;
  while ((1 << s) < v) ++s;
  return s;
}
inline int fdiv2(int i) { return i >> 1; }

// Star patches of level l (k_ghost.cuh "star patches"): the six slabs of thickness R = stencil radius around every
// box, cut along the blocking factor; each piece is a same-level copy (periodic wrap included), an interpolation
// whose parents all lie in one coarse box, or a slow patch (parents in several coarse boxes / across the seam).
void plan_patches(Plan& P, int l, bool tagset) {
  LevelHost& L = P.lev[l];
  const sledge_params& p = P.p;
  const int bf = p.blocking_factor, bfs = ilog2(bf), g = p.nghost, R = stencil_radius(p);
  auto wrapi = [](int i, int n) { int r = i % n; return r < 0 ? r + n : r; };
  auto owner_at = [&](const LevelHost& V, int i, int j, int k) {  // wrapped cell index -> local box or -1
    return V.owner[((size_t)(k >> bfs) * V.no[1] + (j >> bfs)) * V.no[0] + (i >> bfs)];
  };
  auto cell_off = [&](const BoxDev& b, int i, int j, int k) {  // box-relative cell -> offset in the level plane
    return b.base + ((long long)(k + g) * b.sy + (j + g)) * b.sx + (i + P.ox);
  };
  std::vector<uint4>& out = tagset ? L.tag_patches : L.patches;
  out.clear();
  if (!tagset) L.patch_smem_pairs = 0;
  for (size_t q = 0; q < L.boxdev.size(); ++q) {
    const BoxDev& b = L.boxdev[q];
    // slabs: star set = six faces of thickness R; tag set (the +1 neighbours the plaquettes of K3 need) = the cells
    // with every coordinate in [0, n] and at least one equal to n: x = n (y, z up to n), y = n (x < n, z up to n),
    // z = n (x, y < n); the extra row / column at n is cut off as pieces one cell wide
    struct Slab { int lo[3], ext[3]; };
    std::vector<Slab> slabs;
    if (!tagset) {
      for (int d = 0; d < 3; ++d)
        for (int side = 0; side < 2; ++side) {
          Slab sl = {{0, 0, 0}, {b.n[0], b.n[1], b.n[2]}};
          sl.lo[d] = side ? b.n[d] : -R;
          sl.ext[d] = R;
          slabs.push_back(sl);
        }
    } else {
      for (int m = 1; m < 8; ++m) {  // bit d of m: coordinate d equals n (one cell), else runs over [0, n)
        Slab sl;
        for (int d = 0; d < 3; ++d) {
          sl.lo[d] = ((m >> d) & 1) ? b.n[d] : 0;
          sl.ext[d] = ((m >> d) & 1) ? 1 : b.n[d];
        }
        slabs.push_back(sl);
      }
    }
    for (const Slab& sl : slabs) {
        int lo[3], ext[3], step[3];
        for (int d = 0; d < 3; ++d) {
          lo[d] = sl.lo[d];
          ext[d] = sl.ext[d];
          step[d] = std::min(bf, sl.ext[d]);  // outside the box a slab is thinner than a blocking cell: one piece
        }
        for (int k0 = lo[2]; k0 < lo[2] + ext[2]; k0 += step[2])
          for (int j0 = lo[1]; j0 < lo[1] + ext[1]; j0 += step[1])
            for (int i0 = lo[0]; i0 < lo[0] + ext[0]; i0 += step[0]) {
              const int e[3] = {step[0], step[1], step[2]};
              const int c[3] = {i0, j0, k0};                                      // box-relative first cell
              const int f[3] = {b.lo[0] + i0, b.lo[1] + j0, b.lo[2] + k0};          // unwrapped level index
              const int w[3] = {wrapi(f[0], L.n[0]), wrapi(f[1], L.n[1]), wrapi(f[2], L.n[2])};
              uint4 A = make_uint4((unsigned)cell_off(b, c[0], c[1], c[2]), 0u, (unsigned)b.sx | ((unsigned)b.sy << 16), 0u);
              uint4 B = make_uint4((unsigned)e[0] | ((unsigned)e[1] << 8) | ((unsigned)e[2] << 16), 0u,
                                   (unsigned)(f[0] + g) | ((unsigned)(f[1] + g) << 16), (unsigned)(f[2] + g));
              // a patch never straddles a blocking-factor cell along the two in-face axes, and along the face normal
              // it is R < bf cells starting or ending on a box face: one owner cell, no periodic seam inside
              const int ow = owner_at(L, w[0], w[1], w[2]);
              if (ow >= 0) {
                const BoxDev& sb = L.boxdev[ow];
                A.y = (unsigned)cell_off(sb, w[0] - sb.lo[0], w[1] - sb.lo[1], w[2] - sb.lo[2]);
                A.w = (unsigned)sb.sx | ((unsigned)sb.sy << 16);
                B.x |= (unsigned)PATCH_COPY << 24;
              } else if (l == 0) {
                continue;  // cannot happen: level 0 covers the domain (checked)
              } else {
                const LevelHost& C = P.lev[l - 1];
                int cmin[3], cmax[3], par = 0;
                bool one = true;
                for (int a2 = 0; a2 < 3; ++a2) {
                  const int fl = f[a2] + e[a2] - 1;
                  const int m0 = fdiv2(f[a2]), m1 = fdiv2(fl);
                  const int p0 = f[a2] - 2 * m0, p1 = fl - 2 * m1;
                  cmin[a2] = p0 ? m0 : m0 - 1;
                  cmax[a2] = p1 ? m1 + 1 : m1;
                  par |= p0 << a2;
                }
                const int wl[3] = {wrapi(cmin[0], C.n[0]), wrapi(cmin[1], C.n[1]), wrapi(cmin[2], C.n[2])};
                const int wh[3] = {wrapi(cmax[0], C.n[0]), wrapi(cmax[1], C.n[1]), wrapi(cmax[2], C.n[2])};
                for (int a2 = 0; a2 < 3; ++a2) one = one && (wh[a2] - wl[a2] == cmax[a2] - cmin[a2]);  // no seam inside
                const int owl = owner_at(C, wl[0], wl[1], wl[2]), owh = owner_at(C, wh[0], wh[1], wh[2]);
                const int ce[3] = {cmax[0] - cmin[0] + 1, cmax[1] - cmin[1] + 1, cmax[2] - cmin[2] + 1};
                if (one && owl >= 0 && owl == owh && ce[0] < 256 && ce[1] < 256 && ce[2] < 256) {  // a box is convex
                  const BoxDev& cb = C.boxdev[owl];
                  A.y = (unsigned)cell_off(cb, wl[0] - cb.lo[0], wl[1] - cb.lo[1], wl[2] - cb.lo[2]);
                  A.w = (unsigned)cb.sx | ((unsigned)cb.sy << 16);
                  B.x |= (unsigned)PATCH_INTERP << 24;
                  B.y = (unsigned)ce[0] | ((unsigned)ce[1] << 8) | ((unsigned)ce[2] << 16) | ((unsigned)par << 24);
                  L.patch_smem_pairs = std::max(L.patch_smem_pairs, ce[0] * ce[1] * ce[2]);  // shared by both sets
                } else {
                  B.x |= (unsigned)PATCH_SLOW << 24;
                }
              }
              out.push_back(A);
              out.push_back(B);
            }
    }
  }
  if (!tagset) {  // same-level copies first
    struct Pair { uint4 A, B; };
    std::vector<Pair> ps(out.size() / 2);
    for (size_t q = 0; q < ps.size(); ++q) ps[q] = Pair{out[2 * q], out[2 * q + 1]};
    const auto mid = std::stable_partition(ps.begin(), ps.end(), [](const Pair& e) { return (e.B.x >> 24) == (unsigned)PATCH_COPY; });
    L.n_copy_patches = (unsigned)(mid - ps.begin());
    for (size_t q = 0; q < ps.size(); ++q) {
      out[2 * q] = ps[q].A;
      out[2 * q + 1] = ps[q].B;
    }
  }
}

// ---- validation + layout (host only; shared by sledge_arena_bytes and sledge_create) --------------
int make_plan(Plan& P, const sledge_params* pp, const sledge_box* boxes, int nbox) {
  if (!pp || !boxes || nbox <= 0) return fail(nullptr, SLEDGE_EINVAL, "null params / empty box list");
  P.p = *pp;
  const sledge_params& p = P.p;
  if (p.n_levels < 1 || p.n_levels > 8) return fail(nullptr, SLEDGE_EINVAL, "n_levels must be 1..8");
  const int bf = p.blocking_factor;
  if (bf < 2 || (bf & (bf - 1))) return fail(nullptr, SLEDGE_EINVAL, "blocking_factor must be a power of 2 >= 2 (L39)");
  if (p.nghost < 1 || p.nghost >= bf) return fail(nullptr, SLEDGE_EINVAL, "need 1 <= nghost < blocking_factor (L772)");
  if (p.lap_order < 1 || p.lap_order > 3) return fail(nullptr, SLEDGE_EINVAL, "lap_order must be 1 (7-point), 2 (13-point) or 3 (19-point) (L649)");
  if (p.lap_order > p.nghost) return fail(nullptr, SLEDGE_EINVAL, "lap_order must be <= nghost (L240)");
  for (int q = 0; q < 4; ++q)
    if (!(p.ko_strength[q] >= 0.0)) return fail(nullptr, SLEDGE_EINVAL, "dissipation strength must be >= 0 (L749)");
  if (ko_on(p)) {
    if (p.ko_order < 2 || p.ko_order > 3) return fail(nullptr, SLEDGE_EINVAL, "dissipation order must be 2 or 3 (L751)");
    if (p.ko_order > p.nghost) return fail(nullptr, SLEDGE_EINVAL, "dissipation order must be <= nghost (L751)");
  }
  if (p.integrator != 0 && p.integrator != 4 && p.integrator != 3 && p.integrator != 10 && p.integrator != 20)
    return fail(nullptr, SLEDGE_EINVAL, "integrator must be 4 (RK4), 3 / 10 (SSPRK3) or 20 (user RKN tableau) (L808)");
  if (p.integrator == 20) {  // explicit Nystrom scheme for psi'' = f(psi, eta) (L808-815)
    if (p.rkn_stages < 1 || p.rkn_stages > SLEDGE_RKN_MAX_STAGES)
      return fail(nullptr, SLEDGE_EINVAL, "rkn_stages must be 1..5 (L812-815)");
    if (p.friction != 0.0 || ko_on(p))
      return fail(nullptr, SLEDGE_EINVAL, "integrator 20 integrates psi'' = f(psi): friction and ko_strength must be 0");
    if (p.gw) return fail(nullptr, SLEDGE_EINVAL, "integrator 20 does not evolve the gravitational-wave fields");
    if (p.rkn_nodes[0] != 0.0) return fail(nullptr, SLEDGE_EINVAL, "rkn_nodes[0] must be 0 (the first stage is the state itself)");
    for (int i = 0; i < p.rkn_stages; ++i)
      if (p.rkn_tableau[i * (i + 1) / 2 + i] != 0.0)
        return fail(nullptr, SLEDGE_EINVAL, "rkn_tableau: only explicit schemes, the diagonal must be 0 (L815)");
  }
  if (p.gw != 0 && p.gw != 1) return fail(nullptr, SLEDGE_EINVAL, "gw must be 0 or 1 (L404)");
  if (p.gw && (p.integrator == 3 || p.integrator == 10))
    return fail(nullptr, SLEDGE_EINVAL, "gw: the auxiliary fields are integrated with classic RK4 (integrator 4) only");
  if (p.gw && p.interp != SLEDGE_INTERP_TRILINEAR)
    return fail(nullptr, SLEDGE_EINVAL, "gw: trilinear coarse->fine interpolation only");
  if (p.shadow_level != 0 && p.shadow_level != 1) return fail(nullptr, SLEDGE_EINVAL, "shadow_level must be 0 or 1 (L98)");
  if (p.interp != SLEDGE_INTERP_TRILINEAR && p.interp != SLEDGE_INTERP_QUARTIC)
    return fail(nullptr, SLEDGE_EINVAL, "interp must be SLEDGE_INTERP_TRILINEAR (0) or SLEDGE_INTERP_QUARTIC (4) (L780)");
  // the 5-cell window around the parent of the outermost ghost cell must stay inside the nesting gap of one
  // blocking factor (L70: "we may not be able to set ghost cells ... because the domain might not extend far enough")
  if (p.interp == SLEDGE_INTERP_QUARTIC && p.n_levels > 1 && (p.nghost + 1) / 2 + 2 > p.blocking_factor / 2)
    return fail(nullptr, SLEDGE_EINVAL, "quartic interpolation: ceil(nghost/2) + 2 coarse cells exceed the nesting gap of blocking_factor/2 (L70)");
  if (p.dtype != SLEDGE_F32 && p.dtype != SLEDGE_F64) return fail(nullptr, SLEDGE_EINVAL, "dtype must be SLEDGE_F32 or SLEDGE_F64");
  if (p.rk_dataflow < SLEDGE_RK_LEAN || p.rk_dataflow > SLEDGE_RK_FUSED3) return fail(nullptr, SLEDGE_EINVAL, "bad rk_dataflow");
  if (!(p.h0 > 0)) return fail(nullptr, SLEDGE_EINVAL, "h0 must be positive");
  for (int d = 0; d < 3; ++d) {
    if (p.n0[d] <= 0 || p.n0[d] % bf) return fail(nullptr, SLEDGE_EINVAL, "n0 must be a positive multiple of blocking_factor (L39)");
    if (((long long)p.n0[d] << (p.n_levels - 1)) > (1 << 24)) return fail(nullptr, SLEDGE_EINVAL, "finest level index space too large");
  }
  P.esz = p.dtype == SLEDGE_F64 ? 8 : 4;
  P.cpa = 128 / (2 * P.esz);
  P.ox = (p.nghost + P.cpa - 1) / P.cpa * P.cpa;
  const int g = p.nghost, bfs = ilog2(bf);
  P.lev.assign(p.n_levels, LevelHost());
  for (int l = 0; l < p.n_levels; ++l) {
    LevelHost& L = P.lev[l];
    for (int d = 0; d < 3; ++d) {
      L.n[d] = p.n0[d] << l;
      L.no[d] = L.n[d] / bf;
      L.nb[d] = (L.n[d] + COUNT_BLOCK - 1) / COUNT_BLOCK;
    }
    L.h = p.h0 / (double)(1 << l);  // Eq.1
    L.owner.assign((size_t)L.no[0] * L.no[1] * L.no[2], -1);
    L.count_blocks = (long long)L.nb[0] * L.nb[1] * L.nb[2];
  }
  P.box.assign(boxes, boxes + nbox);
  P.box_local.assign(nbox, -1);
  size_t max_box_cells = 0;
  for (int ib = 0; ib < nbox; ++ib) {
    const sledge_box& B = boxes[ib];
    if (B.level < 0 || B.level >= p.n_levels) return fail(nullptr, SLEDGE_EINVAL, "box %d: level out of range", ib);
    LevelHost& L = P.lev[B.level];
    BoxDev bd;
    for (int d = 0; d < 3; ++d) {
      const int n = B.hi[d] - B.lo[d] + 1;
      if (B.lo[d] < 0 || B.hi[d] >= L.n[d] || n <= 0 || B.lo[d] % bf || n % bf)
        return fail(nullptr, SLEDGE_EINVAL, "box %d: outside the domain or not aligned to the blocking factor (L39)", ib);
      bd.n[d] = n;
      bd.lo[d] = B.lo[d];
    }
    const int li = (int)L.boxes.size();
    for (int k = B.lo[2] >> bfs; k <= B.hi[2] >> bfs; ++k)
      for (int j = B.lo[1] >> bfs; j <= B.hi[1] >> bfs; ++j)
        for (int i = B.lo[0] >> bfs; i <= B.hi[0] >> bfs; ++i) {
          int& ow = L.owner[((size_t)k * L.no[1] + j) * L.no[0] + i];
          if (ow != -1) return fail(nullptr, SLEDGE_EINVAL, "box %d overlaps box %d of level %d", ib, L.boxes[ow], B.level);
          ow = li;
        }
    bd.sx = bd.sy = 0;  // pitches and base follow from the storage box (below)
    bd.base = 0;
    bd.tag_base = L.valid_cells;
    L.valid_cells += (long long)bd.n[0] * bd.n[1] * bd.n[2];
    max_box_cells = std::max(max_box_cells, (size_t)(bd.n[0] + 2 * g) * (bd.n[1] + 2 * g) * (bd.n[2] + 2 * g));
    P.box_local[ib] = li;
    L.boxes.push_back(ib);
    L.viewdev.push_back(bd);
  }
  for (size_t q = 0; q < P.lev[0].owner.size(); ++q)
    if (P.lev[0].owner[q] < 0) return fail(nullptr, SLEDGE_EINVAL, "level 0 must cover the whole domain (L39)");
  // proper nesting (L70, L137): a fine box grown by one blocking factor (fine cells) lies on valid coarse cells
  for (int l = 1; l < p.n_levels; ++l) {
    const LevelHost& L = P.lev[l];
    const LevelHost& C = P.lev[l - 1];
    if (L.boxes.empty()) return fail(nullptr, SLEDGE_EINVAL, "level %d has no boxes", l);
    for (size_t q = 0; q < L.boxes.size(); ++q) {
      const BoxDev& b = L.viewdev[q];
      // coarse cells touched by the grown box; owner granularity is bf coarse cells
      int clo[3], chi[3];
      for (int d = 0; d < 3; ++d) {
        clo[d] = fdiv2(b.lo[d] - bf);
        chi[d] = fdiv2(b.lo[d] + b.n[d] - 1 + bf);
      }
      for (int k = clo[2] >> bfs; k <= chi[2] >> bfs; ++k)
        for (int j = clo[1] >> bfs; j <= chi[1] >> bfs; ++j)
          for (int i = clo[0] >> bfs; i <= chi[0] >> bfs; ++i) {
            const int wi = ((i % C.no[0]) + C.no[0]) % C.no[0];
            const int wj = ((j % C.no[1]) + C.no[1]) % C.no[1];
            const int wk = ((k % C.no[2]) + C.no[2]) % C.no[2];
            if (C.owner[((size_t)wk * C.no[1] + wj) * C.no[0] + wi] < 0)
              return fail(nullptr, SLEDGE_EINVAL, "box %d violates proper nesting: gap to the level-%d boundary < blocking factor (L70, L137)",
                          L.boxes[q], l - 1);
          }
    }
  }
  // Storage boxes.  Two boxes of a level that share a whole face need no ghost cells between them: the caller's boxes
  // (the granularity the paper's load balancer hands to MPI ranks, L39) are coalesced, greedily along x, then z, then
  // y, into larger rectangles that K1 sweeps and K2 fills as ONE box; every caller's box stays addressable as a view
  // (same pitches, shifted base).  Results do not depend on it: a ghost copy holds the bits of the cell it mirrors.
  // SLEDGE_COALESCE=0 in the environment keeps one storage box per caller's box (diagnostics).
  {
    const char* env = getenv("SLEDGE_COALESCE");
    const bool coalesce = !(env && env[0] == '0');
    int order[3] = {0, 2, 1};  // x, z, y (measured on C5); SLEDGE_COALESCE=zyx (any permutation of xyz) changes it (diagnostics)
    if (env && strlen(env) == 3) {
      int seen = 0, o[3];
      for (int d = 0; d < 3; ++d) {
        o[d] = env[d] - 'x';
        if (o[d] >= 0 && o[d] < 3) seen |= 1 << o[d];
      }
      if (seen == 7)
        for (int d = 0; d < 3; ++d) order[d] = o[d];
    }
    for (int l = 0; l < p.n_levels; ++l) {
      LevelHost& L = P.lev[l];
      struct R3 { int lo[3], hi[3]; };  // inclusive
      std::vector<R3> rs;
      for (const BoxDev& v : L.viewdev) rs.push_back(R3{{v.lo[0], v.lo[1], v.lo[2]}, {v.lo[0] + v.n[0] - 1, v.lo[1] + v.n[1] - 1, v.lo[2] + v.n[2] - 1}});
      // a level that covers the whole domain (level 0 always does, L39) is ONE rectangle whatever the greedy merge
      // below would make of an arbitrary partition
      bool covered = coalesce;
      for (size_t q = 0; covered && q < L.owner.size(); ++q) covered = L.owner[q] >= 0;
      if (covered) rs.assign(1, R3{{0, 0, 0}, {L.n[0] - 1, L.n[1] - 1, L.n[2] - 1}});
      for (bool merged = coalesce && !covered; merged;) {  // until a pass over the three axes merges nothing
        merged = false;
        for (int dd = 0; dd < 3; ++dd) {
          const int d = order[dd], o1 = (d + 1) % 3, o2 = (d + 2) % 3;
          std::sort(rs.begin(), rs.end(), [&](const R3& a, const R3& b) {
            if (a.lo[o1] != b.lo[o1]) return a.lo[o1] < b.lo[o1];
            if (a.lo[o2] != b.lo[o2]) return a.lo[o2] < b.lo[o2];
            if (a.hi[o1] != b.hi[o1]) return a.hi[o1] < b.hi[o1];
            if (a.hi[o2] != b.hi[o2]) return a.hi[o2] < b.hi[o2];
            return a.lo[d] < b.lo[d];
          });
          std::vector<R3> out;
          for (const R3& r : rs) {
            if (!out.empty()) {
              R3& q = out.back();
              // pitches are kept in 16 bits, patch and tile tables in ints: stop well below
              if (q.lo[o1] == r.lo[o1] && q.hi[o1] == r.hi[o1] && q.lo[o2] == r.lo[o2] && q.hi[o2] == r.hi[o2] &&
                  q.hi[d] + 1 == r.lo[d] && r.hi[d] - q.lo[d] + 1 <= 16384) {
                q.hi[d] = r.hi[d];
                merged = true;
                continue;
              }
            }
            out.push_back(r);
          }
          rs.swap(out);
        }
      }
      for (size_t q = 0; q < rs.size(); ++q) {
        const R3& r = rs[q];
        BoxDev bd;
        for (int d = 0; d < 3; ++d) {
          bd.lo[d] = r.lo[d];
          bd.n[d] = r.hi[d] - r.lo[d] + 1;
        }
        // row: [0, ox) left pad + ghosts, [ox, ox+n) valid, then >= g ghosts, pitch a multiple of 128 bytes
        bd.sx = (P.ox + bd.n[0] + g + P.cpa - 1) / P.cpa * P.cpa;
        bd.sy = bd.n[1] + 2 * g;
        bd.base = L.plane_cells;
        bd.tag_base = 0;  // tags are laid out by the caller's boxes (views)
        L.plane_cells += (long long)bd.sx * bd.sy * (bd.n[2] + 2 * g);
        for (int k = r.lo[2] >> bfs; k <= r.hi[2] >> bfs; ++k)
          for (int j = r.lo[1] >> bfs; j <= r.hi[1] >> bfs; ++j)
            for (int i = r.lo[0] >> bfs; i <= r.hi[0] >> bfs; ++i) L.owner[((size_t)k * L.no[1] + j) * L.no[0] + i] = (int)q;
        L.boxdev.push_back(bd);
      }
      for (BoxDev& v : L.viewdev) {
        const BoxDev& sb = L.boxdev[L.owner[((size_t)(v.lo[2] >> bfs) * L.no[1] + (v.lo[1] >> bfs)) * L.no[0] + (v.lo[0] >> bfs)]];
        v.sx = sb.sx;
        v.sy = sb.sy;
        v.base = sb.base + ((long long)(v.lo[2] - sb.lo[2]) * sb.sy + (v.lo[1] - sb.lo[1])) * sb.sx + (v.lo[0] - sb.lo[0]);
      }
    }
  }
  // work tables
  const int cpt = p.dtype == SLEDGE_F64 ? 1 : 2;
  for (int l = 0; l < p.n_levels; ++l) {
    LevelHost& L = P.lev[l];
    L.periodic_box = L.boxdev.size() == 1 && L.boxdev[0].n[0] == L.n[0] && L.boxdev[0].n[1] == L.n[1] &&
                     L.boxdev[0].n[2] == L.n[2];
    L.ghost_prefix.assign(1, 0);
    L.avg_prefix.assign(1, 0);
    L.qp_prefix.assign(1, 0);
    const bool qparents = quartic_by_parent(p) && l > 0;
    // z-chunk of the fused sweeps: long marches amortise the pipeline prologue, but the grid must stay many waves
    // deep (148 SMs x 2-3 CTAs); measured on C2 / C3 (profiles/r01_k1_tile_sweep.md)
    const int txc = K1_TX * cpt, ftxc = K1F_TX * cpt;
    long long ft_long = 0;
    for (const BoxDev& b : L.boxdev)
      ft_long += (long long)((b.n[0] + ftxc - 1) / ftxc) * ((b.n[1] + K1F_TY - 1) / K1F_TY) * ((b.n[2] + K1_NZ - 1) / K1_NZ);
    // measured on C2 / C5 level 0 (256^3: 512 tiles of 128 planes): 64 planes 0.481 ms, 32 planes 0.462 ms per C2 step
    const int fnz = ft_long >= K1F_MIN_TILES ? K1_NZ : (ft_long >= K1F_MIN_TILES / 2 ? K1_NZ / 2 : K1_NZ / 4);
    // z-chunk of the tag pass (K3): a tile costs one extra plane, but the grid should be several waves of 148 SMs x 4 CTAs
    int tnz = K1_NZ;
    for (; tnz > TAG_MIN_NZ; tnz /= 2) {
      long long nt = 0;
      for (const BoxDev& b : (L.viewdev.size() != L.boxdev.size() && bf >= TAG_RY) ? L.boxdev : L.viewdev)
        nt += (long long)((b.n[0] + TAG_TX - 1) / TAG_TX) * ((b.n[1] + TAG_TY - 1) / TAG_TY) * ((b.n[2] + tnz - 1) / tnz);
      if (nt >= TAG_MIN_TILES) break;
    }
    for (size_t q = 0; q < L.boxdev.size(); ++q) {
      const BoxDev& b = L.boxdev[q];
      for (int z0 = 0; z0 < b.n[2]; z0 += K1_NZ)
        for (int y0 = 0; y0 < b.n[1]; y0 += K1_TY)
          for (int x0 = 0; x0 < b.n[0]; x0 += txc) L.tiles.push_back(TileDev{(int)q, x0, y0, z0, std::min(K1_NZ, b.n[2] - z0)});
      for (int z0 = 0; z0 < b.n[2]; z0 += fnz)
        for (int y0 = 0; y0 < b.n[1]; y0 += K1F_TY)
          for (int x0 = 0; x0 < b.n[0]; x0 += ftxc) L.ftiles.push_back(TileDev{(int)q, x0, y0, z0, std::min(fnz, b.n[2] - z0)});
      const long long Gx = b.n[0] + 2 * g, Gy = b.n[1] + 2 * g;
      const long long nghost = Gx * Gy * 2 * g + Gx * 2 * g * b.n[2] + 2LL * g * b.n[1] * b.n[2];
      L.ghost_prefix.push_back(L.ghost_prefix.back() + (int)((nghost + GHOST_THREADS - 1) / GHOST_THREADS));
      if (qparents) {  // parents of the ghost shell: the shell of thickness ceil(g/2) around the coarse footprint
        const long long t = (g + 1) / 2, cx = b.n[0] / 2, cy = b.n[1] / 2, cz = b.n[2] / 2;
        const long long npar = (cx + 2 * t) * (cy + 2 * t) * 2 * t + (cx + 2 * t) * 2 * t * cz + 2 * t * cy * cz;
        L.qp_prefix.push_back(L.qp_prefix.back() + (int)((npar + GHOST_THREADS - 1) / GHOST_THREADS));
      }
    }
    // K3 runs over the storage boxes too where it can find the caller's tag layout per blocking-factor cell (a warp's
    // TAG_RY rows must lie in one such cell); otherwise over the caller's boxes
    const bool tag_lookup = L.viewdev.size() != L.boxdev.size() && bf >= TAG_RY;
    if (tag_lookup) {
      L.tag_cells.assign(L.owner.size(), make_int4(0, 0, 0, 0));
      for (const BoxDev& v : L.viewdev)
        for (int k = v.lo[2] >> bfs; k <= (v.lo[2] + v.n[2] - 1) >> bfs; ++k)
          for (int j = v.lo[1] >> bfs; j <= (v.lo[1] + v.n[1] - 1) >> bfs; ++j)
            for (int i = v.lo[0] >> bfs; i <= (v.lo[0] + v.n[0] - 1) >> bfs; ++i) {
              const long long o = v.tag_base + ((long long)((k << bfs) - v.lo[2]) * v.n[1] + ((j << bfs) - v.lo[1])) * v.n[0] + ((i << bfs) - v.lo[0]);
              L.tag_cells[((size_t)k * L.no[1] + j) * L.no[0] + i] = make_int4((int)(unsigned)(o & 0xffffffffll), (int)(o >> 32), v.n[0], v.n[1]);
            }
    }
    const std::vector<BoxDev>& tagboxes = tag_lookup ? L.boxdev : L.viewdev;
    for (size_t q = 0; q < tagboxes.size(); ++q) {
      const BoxDev& b = tagboxes[q];
      for (int z0 = 0; z0 < b.n[2]; z0 += tnz)
        for (int y0 = 0; y0 < b.n[1]; y0 += TAG_TY)
          for (int x0 = 0; x0 < b.n[0]; x0 += TAG_TX) L.tag_tiles.push_back(TileDev{(int)q, x0, y0, z0, std::min(tnz, b.n[2] - z0)});
    }
    for (size_t q = 0; q < L.viewdev.size(); ++q) {  // the fine side of K4 keeps the caller's box order (tag layout)
      const BoxDev& b = L.viewdev[q];
      const long long ncoarse = (long long)(b.n[0] / 2) * (b.n[1] / 2) * (b.n[2] / 2);
      L.avg_prefix.push_back(L.avg_prefix.back() + (int)((ncoarse + AVG_THREADS - 1) / AVG_THREADS));
    }
  }
  for (int l = 0; l < p.n_levels; ++l)
    if (bf <= 128) {  // patch extents are kept in 8 bits
      plan_patches(P, l, false);
      plan_patches(P, l, true);
    }
  // arena layout
  size_t off = 0;
  auto take = [&](size_t bytes) {
    const size_t o = off;
    off = align_up(off + bytes, ALIGN);
    return o;
  };
  for (int l = 0; l < p.n_levels; ++l) {
    LevelHost& L = P.lev[l];
    const size_t plane_bytes = (size_t)L.plane_cells * 2 * P.esz;
    for (int b = 0; b < NBUF; ++b)
      for (int c = 0; c < 2; ++c) L.off_buf[b][c] = take(plane_bytes);
    if (p.gw)
      for (int b = 0; b < NBUF; ++b)
        for (int c = 0; c < 6; ++c) L.off_gw[b][c] = take(plane_bytes);
    L.off_boxes = take(L.boxdev.size() * sizeof(BoxDev));
    L.off_views = take(L.viewdev.size() * sizeof(BoxDev));
    L.off_tag_cells = take(L.tag_cells.size() * sizeof(int4));
    L.off_tiles = take(L.tiles.size() * sizeof(TileDev));
    L.off_ftiles = take(L.ftiles.size() * sizeof(TileDev));
    L.off_tag_tiles = take(L.tag_tiles.size() * sizeof(TileDev));
    L.off_owner = take(L.owner.size() * sizeof(int));
    L.off_ghost_prefix = take(L.ghost_prefix.size() * sizeof(int));
    L.off_avg_prefix = take(L.avg_prefix.size() * sizeof(int));
    L.off_ghost_list = take((size_t)L.ghost_prefix.back() * GHOST_THREADS * sizeof(GhostEntry));
    L.off_star_list = take((size_t)L.ghost_prefix.back() * GHOST_THREADS * sizeof(GhostEntry));
    L.off_star_count = take(sizeof(unsigned));
    L.off_tmaps = take(L.boxdev.size() * NBUF * 2 * sizeof(CUtensorMap));
    L.off_patches = take(L.patches.size() * sizeof(uint4));
    L.off_tag_patches = take(L.tag_patches.size() * sizeof(uint4));
    L.off_qp_prefix = take(L.qp_prefix.size() * sizeof(int));
    L.off_qp_list = take((size_t)L.qp_prefix.back() * GHOST_THREADS * 2 * sizeof(uint4));
    L.off_qs_list = take((size_t)L.qp_prefix.back() * GHOST_THREADS * 2 * sizeof(uint4));
    L.off_qs_count = take(sizeof(unsigned));
    // the ghost list (k_ghost.cuh) keeps cell offsets in 32 bits and pitches / indices in 16
    if (L.plane_cells >= (1LL << 32)) return fail(nullptr, SLEDGE_EINVAL, "level %d: more than 2^32 stored cells", l);
    for (const BoxDev& b : L.boxdev)
      if (b.sx >= 65536 || b.sy >= 65536) return fail(nullptr, SLEDGE_EINVAL, "level %d: box pitch >= 65536 cells", l);
    for (int d = 0; d < 3; ++d)
      if (L.n[d] + 2 * g >= 65536) return fail(nullptr, SLEDGE_EINVAL, "level %d: more than 65535 cells per axis", l);
  }
  P.scratch_bytes = max_box_cells * P.esz;
  P.off_scratch = take(P.scratch_bytes * 6);  // host copies: staging slots in 0, 1; out 2 .. 5 (N_IN_SLOTS, N_OUT_SLOTS)
  P.off_err = take(sizeof(int));
  if (p.shadow_level) {  // L98: level 0 coarsened by 2, ONE box over the same periodic domain
    sledge_params sp = p;
    sp.n_levels = 1;
    sp.shadow_level = 0;
    sp.h0 = 2.0 * p.h0;
    int sbf = bf;
    for (int d = 0; d < 3; ++d) {
      if (p.n0[d] % 2) return fail(nullptr, SLEDGE_EINVAL, "shadow_level: n0 must be even (L98)");
      sp.n0[d] = p.n0[d] / 2;
      while (sbf > 1 && sp.n0[d] % sbf) sbf /= 2;
    }
    sp.blocking_factor = sbf;
    sledge_box sb;
    sb.level = 0;
    for (int d = 0; d < 3; ++d) {
      sb.lo[d] = 0;
      sb.hi[d] = sp.n0[d] - 1;
    }
    Plan PS;
    const int rc = make_plan(PS, &sp, &sb, 1);
    if (rc) return fail(nullptr, rc, "shadow_level: the coarsened level 0 is not a valid grid (%s)", g_err.c_str());
    P.shadow_p = sp;
    P.shadow_box = sb;
    P.shadow_bytes = PS.total;
    P.off_shadow = take(PS.total);
  }
  P.total = off;
  return SLEDGE_OK;
}

}  // namespace

// ---- launch plumbing ---------------------------------------------------------------------------
namespace {

enum Kind { KIND_STAGE = 0, KIND_GHOST = 1, KIND_TAG = 2, KIND_AVG = 3 };

struct Timed {  // brackets a launch with an event pair while profiling is on
  sledge_ctx* c;
  int kind;
  cudaEvent_t stop = nullptr;
  Timed(sledge_ctx* ctx, int k) : c(ctx), kind(k) {
    ++c->launches;
    if (!c->profiling || c->ev_used[k] >= MAX_EVENT_PAIRS) return;
    if (c->ev_used[k] == c->ev[k].size()) {
      cudaEvent_t a, b;
      cudaEventCreate(&a);
      cudaEventCreate(&b);
      c->ev[k].push_back({a, b});
    }
    cudaEventRecord(c->ev[k][c->ev_used[k]].first, c->stream);
    stop = c->ev[k][c->ev_used[k]].second;
    ++c->ev_used[k];
  }
  ~Timed() {
    if (stop) cudaEventRecord(stop, c->stream);
  }
};

int check_launch(sledge_ctx* c, const char* what) {
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(c, SLEDGE_ECUDA, "%s: %s", what, cudaGetErrorString(e));
  return SLEDGE_OK;
}

// which: 0 = (psi1,psi2), 1 = (Pi1,Pi2); with gw 2..4 = the u pair planes, 5..7 = the du pair planes (component c of
// the state lives in plane c / 2, lane c % 2)
template <typename T> typename PairOf<T>::type* plane_ptr(sledge_ctx* c, int l, int buf, int which) {
  const LevelHost& L = c->plan.lev[l];
  return reinterpret_cast<typename PairOf<T>::type*>(c->arena + (which < 2 ? L.off_buf[buf & 3][which] : L.off_gw[buf & 3][which - 2]));
}
template <typename U> U* tab(sledge_ctx* c, size_t off) { return reinterpret_cast<U*>(c->arena + off); }

LevelGeom geom_of(const Plan& P, int l) {
  const LevelHost& L = P.lev[l];
  LevelGeom gm;
  for (int d = 0; d < 3; ++d) {
    gm.n[d] = L.n[d];
    gm.no[d] = L.no[d];
  }
  gm.bf_shift = ilog2(P.p.blocking_factor);
  gm.g = P.p.nghost;
  gm.ox = P.ox;
  return gm;
}

// K2 arguments for buffer `buf` of level l, whose data is at time `time`
struct VelFill {  // velocity ghosts of the second plane between the times ta and tb (FUSED sweeps on a fine level)
  bool on = false;
  bool w = false;  // the second plane holds W (FUSED_B2): ghost = twice the first plane's
  int buf2 = -1;   // before sweep A: also write the interpolated ghosts of this buffer (U3), see GhostArgs::psi2
  bool w2 = false;
  double half_dt = 0;
  bool copies_only = false;  // before sweep B: the interpolated ghosts are there already
  double ta = 0, tb = 0;
};

template <typename T>
GhostArgs<T> ghost_args(sledge_ctx* c, int l, int buf, double time, int wa = 0, int wb = 1, VelFill vf = VelFill()) {
  Plan& P = c->plan;
  LevelHost& L = P.lev[l];
  GhostArgs<T> a;
  memset(&a, 0, sizeof a);
  a.boxes = tab<BoxDev>(c, L.off_boxes);
  a.blk_prefix = tab<int>(c, L.off_ghost_prefix);
  a.nbox = (int)L.boxdev.size();
  a.psi = plane_ptr<T>(c, l, buf, wa);  // the kernels call their two planes psi and pi; any pair of planes will do
  a.pi = plane_ptr<T>(c, l, buf, wb);
  a.owner = tab<int>(c, L.off_owner);
  a.geom = geom_of(P, l);
  a.err_flag = tab<int>(c, P.off_err);
  a.list = tab<GhostEntry>(c, L.off_ghost_list);
  a.n_entries = (unsigned)L.ghost_prefix.back() * GHOST_THREADS;
  a.star_depth = stencil_radius(P.p);
  a.star_only = 0;
  a.quartic = P.p.interp == SLEDGE_INTERP_QUARTIC ? (quartic_by_parent(P.p) ? 2 : 1) : 0;
  a.copy_only = 0;
  a.qblk_prefix = tab<int>(c, L.off_qp_prefix);
  a.qlist = tab<uint4>(c, L.off_qp_list);
  a.n_qentries = (unsigned)L.qp_prefix.back() * GHOST_THREADS;
  a.star_list = tab<GhostEntry>(c, L.off_star_list);
  a.star_count = tab<unsigned>(c, L.off_star_count);
  a.qstar_list = tab<uint4>(c, L.off_qs_list);
  a.qstar_count = tab<unsigned>(c, L.off_qs_count);
  a.patches = tab<uint4>(c, L.off_patches);
  a.n_patches = (unsigned)(L.patches.size() / 2);
  a.patch_smem_pairs = L.patch_smem_pairs;
  a.has_coarse = l > 0;
  a.alpha = T(0);
  if (l > 0) {
    LevelHost& C = P.lev[l - 1];
    a.cboxes = tab<BoxDev>(c, C.off_boxes);
    a.cowner = tab<int>(c, C.off_owner);
    a.cgeom = geom_of(P, l - 1);
    int bo = C.cur, bn = C.cur;
    double alpha = 0.0;
    if (C.have_pair && C.t_new != C.t_old) {  // linear in time between the coarse old and new states (L72)
      alpha = (time - C.t_old) / (C.t_new - C.t_old);
      bo = C.old;
    }
    a.alpha = (T)alpha;
    // alpha exactly 0 or 1 (first / last stage of a fine step pair, the fill before tagging) or a coarse level
    // with one state only: the blend returns one of the two buffers unchanged, so only that one is read
    if (bo == bn || alpha == 0.0) { bn = bo; a.single = 1; }
    else if (alpha == 1.0) { bo = bn; a.single = 1; }
    if (vf.on) {  // both coarse states are needed whatever alpha is
      const bool pair = C.have_pair && C.t_new != C.t_old;
      bo = pair ? C.old : C.cur;
      bn = C.cur;
      a.single = 0;
      a.vel = vf.w ? 2 : 1;
      if (vf.buf2 >= 0) {
        a.psi2 = plane_ptr<T>(c, l, vf.buf2, wa);
        a.pi2 = plane_ptr<T>(c, l, vf.buf2, wb);
        a.half_dt = (T)vf.half_dt;
        a.w2 = vf.w2 ? 1 : 0;
      }
      a.vel_c = (T)(pair ? 1.0 / (C.t_new - C.t_old) : 0.0);
    }
    a.c_old_psi = plane_ptr<T>(c, l - 1, bo, wa);
    a.c_new_psi = plane_ptr<T>(c, l - 1, bn, wa);
    a.c_old_pi = plane_ptr<T>(c, l - 1, bo, wb);
    a.c_new_pi = plane_ptr<T>(c, l - 1, bn, wb);
  }
  return a;
}

// K2 on buffer `buf` of level l: streams the level's ghost list (built once by plan_ghosts)
// Whole ghost shell of buffer `buf` of level l <- same-level / periodic copies (psi and Pi), no interpolation.
template <typename T>
int fill_shell_copies(sledge_ctx* c, int l, int buf, bool with_pi) {
  LevelHost& L = c->plan.lev[l];
  const int need = with_pi ? 2 : 1;
  if (L.shell_ok[buf & 3] >= need) return SLEDGE_OK;
  GhostArgs<T> a = ghost_args<T>(c, l, buf, 0.0);
  a.copy_only = 1;
  const int grid = (L.ghost_prefix.back() + GHOST_EPT - 1) / GHOST_EPT;
  if (grid > 0) {
    Timed t(c, KIND_GHOST);
    if (with_pi) k_fill_ghosts<T, true><<<grid, GHOST_THREADS, 0, c->stream>>>(a);
    else k_fill_ghosts<T, false><<<grid, GHOST_THREADS, 0, c->stream>>>(a);
  }
  L.shell_ok[buf & 3] = need;
  return check_launch(c, "k_fill_ghosts (coarse shell)");
}

template <typename T>
int launch_ghosts(sledge_ctx* c, int l, int buf, double time, bool fill_pi, bool star_only = false, int wa = 0, int wb = 1,
                  bool tag_only = false, VelFill vf = VelFill()) {
  GhostArgs<T> a = ghost_args<T>(c, l, buf, time, wa, wb, vf);
  // fills before a sweep (star_only) or before K3 (tag_only) go by rectangular patch; with quartic interpolation by
  // coarse parent the patches move the copies only and k_fill_qparents the interpolated cells
  const bool patchable = c->use_patches && (a.quartic == 0 || a.quartic == 2);
  const bool tagp = tag_only && patchable && !c->plan.lev[l].tag_patches.empty();
  if (tagp) {  // only the +1 neighbours of the plaquettes (every coordinate in [0, n], one of them = n)
    a.patches = tab<uint4>(c, c->plan.lev[l].off_tag_patches);
    a.n_patches = (unsigned)(c->plan.lev[l].tag_patches.size() / 2);
  }
  const bool by_patch = patchable && a.n_patches > 0 && (star_only || tagp);
  if (a.quartic == 2 && l > 0 && !vf.copies_only) {  // the coarse windows are read through the coarse boxes' ghost cells
    LevelHost& C = c->plan.lev[l - 1];
    const bool pair = C.have_pair && C.t_new != C.t_old;
    int rc = fill_shell_copies<T>(c, l - 1, C.cur, fill_pi);
    if (rc == SLEDGE_OK && pair) rc = fill_shell_copies<T>(c, l - 1, C.old, fill_pi);
    if (rc) return rc;
  }
  if (by_patch) {  // by rectangular region (k_fill_patches)
    if (a.quartic == 2 || vf.copies_only) a.copy_only = 1;
    if (a.copy_only && !tagp) a.n_patches = c->plan.lev[l].n_copy_patches;  // sorted: the copies come first
    if (a.n_patches > 0) {
      const int pgrid = (int)((a.n_patches + PATCH_WARPS - 1) / PATCH_WARPS);
      // the shared-memory region stages the coarse cells of an interpolation patch: none in a copies-only launch
      const size_t smem = a.copy_only ? 0 : (size_t)PATCH_WARPS * a.patch_smem_pairs * (fill_pi ? 2 : 1) * sizeof(typename PairOf<T>::type);
      if (smem > 48 * 1024) {
        static PerDevice configured2[2];  // per instantiation and device
        bool& cfg = configured2[fill_pi][c->device];
        if (!cfg) {
          if (fill_pi) cudaFuncSetAttribute(k_fill_patches<T, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
          else cudaFuncSetAttribute(k_fill_patches<T, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
          cfg = true;
        }
      }
      Timed t(c, KIND_GHOST);
      if (fill_pi) k_fill_patches<T, true><<<pgrid, PATCH_WARPS * 32, smem, c->stream>>>(a);
      else k_fill_patches<T, false><<<pgrid, PATCH_WARPS * 32, smem, c->stream>>>(a);
      const int prc = check_launch(c, "k_fill_patches");
      if (prc) return prc;
    }
    if (a.quartic == 0) return SLEDGE_OK;
    a.copy_only = 0;
  }
  int grid = (c->plan.lev[l].ghost_prefix.back() + GHOST_EPT - 1) / GHOST_EPT;
  if (star_only) {  // before an RK sweep only the cells its star stencil reaches are needed: the packed list
    a.star_only = 1;
    a.list = a.star_list;
    a.n_entries = c->plan.lev[l].n_star;
    grid = (int)((a.n_entries + GHOST_THREADS * GHOST_EPT - 1) / (GHOST_THREADS * GHOST_EPT));
  }
  if (grid == 0 && !(a.quartic == 2 && l > 0)) return SLEDGE_OK;
  if (grid > 0 && !by_patch) {  // (with by_patch the copies are done and only the parents kernel below is left)
    Timed t(c, KIND_GHOST);
    if (a.quartic == 1 && l > 0) {
      if (fill_pi) k_fill_ghosts<T, true, true><<<grid, GHOST_THREADS, 0, c->stream>>>(a);
      else k_fill_ghosts<T, false, true><<<grid, GHOST_THREADS, 0, c->stream>>>(a);
    } else {
      if (fill_pi) k_fill_ghosts<T, true><<<grid, GHOST_THREADS, 0, c->stream>>>(a);
      else k_fill_ghosts<T, false><<<grid, GHOST_THREADS, 0, c->stream>>>(a);
    }
  }
  int rc = check_launch(c, "k_fill_ghosts");
  if (rc) return rc;
  int qgrid = c->plan.lev[l].qp_prefix.back();
  if (a.quartic == 2 && l > 0 && qgrid > 0 && star_only) {  // only the parents with star children, packed
    a.qlist = a.qstar_list;
    a.n_qentries = c->plan.lev[l].n_star_parents;
  }
  if (a.quartic == 2 && l > 0 && qgrid > 0 && !vf.copies_only) {  // the interpolated cells, one thread per coarse parent
    qgrid = (int)((a.n_qentries + QP_THREADS - 1) / QP_THREADS);
    Timed t(c, KIND_GHOST);
    if (a.single) {
      if (fill_pi) k_fill_qparents<T, true, true><<<qgrid, QP_THREADS, 0, c->stream>>>(a);
      else k_fill_qparents<T, false, true><<<qgrid, QP_THREADS, 0, c->stream>>>(a);
    } else {
      if (fill_pi && a.vel) k_fill_qparents<T, true, false, true><<<qgrid, QP_THREADS, 0, c->stream>>>(a);
      else if (fill_pi) k_fill_qparents<T, true, false><<<qgrid, QP_THREADS, 0, c->stream>>>(a);
      else k_fill_qparents<T, false, false><<<qgrid, QP_THREADS, 0, c->stream>>>(a);
    }
    rc = check_launch(c, "k_fill_qparents");
  }
  return rc;
}

// create-time: resolve every ghost cell of level l into its list entry
template <typename T>
int plan_ghosts(sledge_ctx* c, int l) {
  const GhostArgs<T> a = ghost_args<T>(c, l, 0, 0.0);
  const int grid = c->plan.lev[l].ghost_prefix.back();
  if (grid == 0) return SLEDGE_OK;
  k_plan_ghosts<T><<<grid, GHOST_THREADS, 0, c->stream>>>(a);
  int rc = check_launch(c, "k_plan_ghosts");
  const int qgrid = c->plan.lev[l].qp_prefix.back();
  if (rc == SLEDGE_OK && qgrid > 0) {
    k_plan_qparents<T><<<qgrid, GHOST_THREADS, 0, c->stream>>>(a);
    rc = check_launch(c, "k_plan_qparents");
  }
  return rc;
}

// Tensor maps of the FUSED level's state planes for k_rk_tma: per box and buffer plane a 3-D tensor
// (2 sx reals, sy rows, nz + 2g planes) with the sweep's tile box (2 SW reals, SH rows, 1 plane); out-of-bounds
// elements (high end of a partial tile) are zero-filled.  cuTensorMapEncodeTiled is a host-only driver entry point,
// fetched at run time so that the library keeps loading on machines without a driver.
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
int make_tensor_maps(sledge_ctx* c, int l) {
  Plan& P = c->plan;
  LevelHost& L = P.lev[l];
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult qres;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn ||
      qres != cudaDriverEntryPointSuccess) {
    cudaGetLastError();
    return fail(c, SLEDGE_ECUDA, "cuTensorMapEncodeTiled is not available from this driver");
  }
  const EncodeTiledFn encode = (EncodeTiledFn)fn;
  const int R = P.p.lap_order, g = P.p.nghost;
  const int cpt = P.p.dtype == SLEDGE_F64 ? 1 : 2;
  const int xo = (R + cpt - 1) / cpt * cpt;
  const cuuint32_t sw = (cuuint32_t)(K1F_TX * cpt + 2 * xo), sh = (cuuint32_t)(K1F_TY + 2 * R);
  // L2 promotion of the tile loads: 64 bytes (measured: C5's 32^3 boxes 6.15 -> 5.70 ms of K1 per coarse step against
  // 128 bytes, C3 unchanged); SLEDGE_TMA_L2PROMO = 0 / 128 / 256 selects another size
  CUtensorMapL2promotion promo = CU_TENSOR_MAP_L2_PROMOTION_L2_64B;
  if (const char* ev = getenv("SLEDGE_TMA_L2PROMO")) {
    const int v = atoi(ev);
    promo = v == 0 ? CU_TENSOR_MAP_L2_PROMOTION_NONE : (v == 128 ? CU_TENSOR_MAP_L2_PROMOTION_L2_128B
            : (v == 256 ? CU_TENSOR_MAP_L2_PROMOTION_L2_256B : CU_TENSOR_MAP_L2_PROMOTION_L2_64B));
  }
  const size_t nb = L.boxdev.size();
  L.tmaps_host.assign(nb * NBUF * 2, CUtensorMap());
  for (int buf = 0; buf < NBUF; ++buf)
    for (int which = 0; which < 2; ++which)
      for (size_t q = 0; q < nb; ++q) {
        const BoxDev& b = L.boxdev[q];
        void* base = c->arena + L.off_buf[buf][which] + (size_t)b.base * 2 * P.esz;
        const cuuint64_t dims[3] = {(cuuint64_t)2 * b.sx, (cuuint64_t)b.sy, (cuuint64_t)(b.n[2] + 2 * g)};
        const cuuint64_t strides[2] = {(cuuint64_t)b.sx * 2 * P.esz, (cuuint64_t)b.sx * b.sy * 2 * P.esz};
        const cuuint32_t box[3] = {2 * sw, sh, 1};
        const cuuint32_t estr[3] = {1, 1, 1};
        const CUresult r = encode(&L.tmaps_host[(size_t)(buf * 2 + which) * nb + q],
                                  P.p.dtype == SLEDGE_F64 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3,
                                  base, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                  promo, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) return fail(c, SLEDGE_ECUDA, "cuTensorMapEncodeTiled failed (%d) for box %zu of level %d", (int)r, q, l);
      }
  L.has_tmaps = true;
  return SLEDGE_OK;
}

template <typename T, int ORDER, int MODE, int KO = 0>
cudaError_t launch_pipe_kernel(sledge_ctx* c, const PipeArgs<T>& a, int grid) {
  constexpr int TY = K1Shape<MODE>::TY;
  static PerDevice configured_dev;  // per instantiation and device
  bool& configured = configured_dev[c->device];
  if constexpr (K1Shape<MODE>::fused && KO == 0) {
    if (a.tmap[0]) {  // TMA-staged plane ring (k_rk_tma.cuh); the maps exist on fused levels unless SLEDGE_K1_TMA=0
      constexpr int RY = FusedTile<T, ORDER>::RY;
      constexpr int PD = tma_depth<T, ORDER, MODE, K1F_TX, TY, RY>(K1Shape<MODE>::SMEM, SLEDGE_K1F_TMA_PDMAX);
      using C = TmaCfg<T, ORDER, MODE, K1F_TX, TY, PD, RY>;
      static_assert(C::SMEM_BYTES <= 227 * 1024, "K1 tile does not fit shared memory");
      constexpr int MINB = ORDER == 3 ? 1 : K1Shape<MODE>::MINB;
      auto kern = k_rk_tma<T, ORDER, MODE, K1F_TX, TY, PD, RY, MINB>;
      static PerDevice configured_tma_dev;
      bool& configured_tma = configured_tma_dev[c->device];
      if (!configured_tma) {
        const cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM_BYTES);
        if (e != cudaSuccess) return e;
        configured_tma = true;
      }
      kern<<<grid, C::NT, C::SMEM_BYTES, c->stream>>>(a);
      return cudaSuccess;
    }
  }
  if constexpr (K1Shape<MODE>::plane && KO == 0) {
    constexpr int RY = K1Shape<MODE>::fused ? FusedTile<T, ORDER>::RY : (ORDER == 3 ? 1 : K1Shape<MODE>::RY);
    constexpr int PD = plane_depth<T, ORDER, MODE, K1F_TX, TY, RY>(K1Shape<MODE>::SMEM, K1Shape<MODE>::PDMAX);
    using C = PlaneCfg<T, ORDER, MODE, K1F_TX, TY, PD, RY>;
    static_assert(C::SMEM_BYTES <= 227 * 1024, "K1 tile does not fit shared memory");
    constexpr int MINB = ORDER == 3 ? 1 : K1Shape<MODE>::MINB;
    auto kern = k_rk_plane<T, ORDER, MODE, K1F_TX, TY, PD, RY, MINB>;
    if (!configured) {
      const cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM_BYTES);
      if (e != cudaSuccess) return e;
      configured = true;
    }
    kern<<<grid, C::NT, C::SMEM_BYTES, c->stream>>>(a);
  } else {
    constexpr int D = pipe_depth<T, ORDER, MODE, K1_TX, TY, KO>(K1Shape<MODE>::SMEM, K1_DMAX);
    static_assert(PipeCfg<T, ORDER, MODE, K1_TX, TY, D, KO>::SMEM_BYTES <= 227 * 1024, "K1 tile does not fit shared memory");
    using C = PipeCfg<T, ORDER, MODE, K1_TX, TY, D, KO>;
    auto kern = k_rk_pipe<T, ORDER, MODE, K1_TX, TY, D, KO>;
    if (!configured) {
      const cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM_BYTES);
      if (e != cudaSuccess) return e;
      configured = true;
    }
    kern<<<grid, K1_TX * TY, C::SMEM_BYTES, c->stream>>>(a);
  }
  return cudaSuccess;
}
// staged sweeps with the Kreiss-Oliger term (never the fused ones)
template <typename T, int ORDER, int KO>
cudaError_t launch_pipe_mode_ko(sledge_ctx* c, const PipeArgs<T>& a, int grid, int mode) {
  switch (mode) {
    case LEAN_S1: return launch_pipe_kernel<T, ORDER, LEAN_S1, KO>(c, a, grid);
    case LEAN_S23: return launch_pipe_kernel<T, ORDER, LEAN_S23, KO>(c, a, grid);
    case LEAN_S4: return launch_pipe_kernel<T, ORDER, LEAN_S4, KO>(c, a, grid);
    case CLASSIC_S1: return launch_pipe_kernel<T, ORDER, CLASSIC_S1, KO>(c, a, grid);
    case CLASSIC_S23: return launch_pipe_kernel<T, ORDER, CLASSIC_S23, KO>(c, a, grid);
    case CLASSIC_S4: return launch_pipe_kernel<T, ORDER, CLASSIC_S4, KO>(c, a, grid);
    case SSP_S23: return launch_pipe_kernel<T, ORDER, SSP_S23, KO>(c, a, grid);
    default: return cudaErrorInvalidValue;
  }
}
template <typename T, int ORDER>
cudaError_t launch_pipe_mode(sledge_ctx* c, const PipeArgs<T>& a, int grid, int mode, int ko) {
  if (ko == 2) return launch_pipe_mode_ko<T, ORDER, 2>(c, a, grid, mode);
  if (ko == 3) return launch_pipe_mode_ko<T, ORDER, 3>(c, a, grid, mode);
  switch (mode) {
    case LEAN_S1: return launch_pipe_kernel<T, ORDER, LEAN_S1>(c, a, grid);
    case LEAN_S23: return launch_pipe_kernel<T, ORDER, LEAN_S23>(c, a, grid);
    case LEAN_S4: return launch_pipe_kernel<T, ORDER, LEAN_S4>(c, a, grid);
    case CLASSIC_S1: return launch_pipe_kernel<T, ORDER, CLASSIC_S1>(c, a, grid);
    case CLASSIC_S23: return launch_pipe_kernel<T, ORDER, CLASSIC_S23>(c, a, grid);
    case CLASSIC_S4: return launch_pipe_kernel<T, ORDER, CLASSIC_S4>(c, a, grid);
    case SSP_S23: return launch_pipe_kernel<T, ORDER, SSP_S23>(c, a, grid);
    case RKN_ST: return launch_pipe_kernel<T, ORDER, RKN_ST>(c, a, grid);
    case FUSED_A: return launch_pipe_kernel<T, ORDER, FUSED_A>(c, a, grid);
    case FUSED_A2:
      if constexpr (sizeof(T) == 8) return launch_pipe_kernel<T, ORDER, FUSED_A2>(c, a, grid);
      return cudaErrorInvalidValue;
    case FUSED_B2:
      if constexpr (sizeof(T) == 8) return launch_pipe_kernel<T, ORDER, FUSED_B2>(c, a, grid);
      return cudaErrorInvalidValue;
    default: return launch_pipe_kernel<T, ORDER, FUSED_B>(c, a, grid);
  }
}

template <typename T>
int launch_k1(sledge_ctx* c, int l, int mode, PipeArgs<T>& a) {
  Plan& P = c->plan;
  LevelHost& L = P.lev[l];
  a.boxes = tab<BoxDev>(c, L.off_boxes);
  const bool fused = (mode == FUSED_A || mode == FUSED_B || mode == FUSED_A2 || mode == FUSED_B2);
  a.tiles = tab<TileDev>(c, fused ? L.off_ftiles : L.off_tiles);
  a.g = P.p.nghost;
  a.ox = P.ox;
  const double h2 = L.h * L.h;
  a.inv_h2 = (T)(P.p.lap_order == 1 ? 1.0 / h2 : (P.p.lap_order == 2 ? 1.0 / (12.0 * h2) : 1.0 / (180.0 * h2)));
  a.a_mass = (T)P.p.a_mass;
  for (int b = 0; b < NBUF; ++b) L.shell_ok[b] = 0;  // a sweep rewrites valid cells of this level's buffers
  if (!fused)
    for (int b = 0; b < NBUF; ++b) L.star_ok[b] = false;
  const int ko = ko_on(P.p) ? P.p.ko_order : 0;
  if (ko) {  // Eq.7: (-1)^(r+1) eps / (2^(2r) h_l); Pi(U) is differenced too and moves from pnt[0] to sten[1]
    const double sgn = (ko % 2 == 0) ? -1.0 : 1.0;
    for (int q = 0; q < 4; ++q) a.ko_c[q] = (T)(sgn * P.p.ko_strength[q] / ((double)(1 << (2 * ko)) * L.h));
    a.sten[1] = a.pnt[0];
  }
  const int grid = (int)(fused ? L.ftiles.size() : L.tiles.size());
  cudaError_t e;
  {
    Timed tm(c, KIND_STAGE);
    e = P.p.lap_order == 1 ? launch_pipe_mode<T, 1>(c, a, grid, mode, ko)
        : (P.p.lap_order == 2 ? launch_pipe_mode<T, 2>(c, a, grid, mode, ko) : launch_pipe_mode<T, 3>(c, a, grid, mode, ko));
  }
  if (e != cudaSuccess) return fail(c, SLEDGE_ECUDA, "k_rk_pipe: %s", cudaGetErrorString(e));
  return check_launch(c, "k_rk_pipe");
}

template <typename T>
void set_eta(const Plan& P, PipeArgs<T>& a, int slot, double eta_s) {
  a.lam_eta2[slot] = (T)(P.p.lambda * (eta_s * eta_s));
  a.fric[slot] = (T)(P.p.friction != 0.0 ? P.p.friction / eta_s : 0.0);
}

// The level's new state `nbuf` becomes current; the previous one is kept as `old` (L72).
void finish_step(LevelHost& L, int nbuf, double t, double dt) {
  L.old = L.cur & 3;
  L.cur = nbuf & 3;
  L.t_old = t;
  L.t_new = t + dt;
  L.have_pair = true;
}

// FUSED data-flow (k_rk_pipe.cuh): pass 0 = RK4 stages 1+2 (Y -> U3), pass 1 = stages 3+4 (Y, U3 -> Ynew).
// Buffers: cur = Y, cur+1 = U3, cur+2 = Ynew.  Pi is differenced, so its ghosts are filled too.
template <typename T>
int do_fused_pass(sledge_ctx* c, int l, int pass, double t, double dt, double eta_const) {
  Plan& P = c->plan;
  LevelHost& L = P.lev[l];
  const int cur = L.cur;
  const bool fx = P.p.eta_fixed != 0;
  PipeArgs<T> a;
  memset(&a, 0, sizeof a);
  set_eta(P, a, 0, fx ? eta_const : t);
  set_eta(P, a, 1, fx ? eta_const : t + 0.5 * dt);
  set_eta(P, a, 2, fx ? eta_const : t + dt);
  a.adt = (T)dt;
  // A level that is one box over the periodic domain needs no ghost fill before a sweep: k_rk_plane wraps its own
  // addresses; k_rk_tma (no wrap in a tensor map) stores the periodic images of its results into the star ghost
  // cells of its output instead, so only a state that no such sweep wrote (set_state, average-down) is filled here.
  const bool tma = c->use_tma && L.has_tmaps;
  // fp64: the "W" form of the two sweeps (k_rk_pipe.cuh FUSED_A2 / FUSED_B2): sweep B differences two fields, not three
  const bool use_w = sizeof(T) == 8 && c->fused_w && P.p.rk_dataflow == SLEDGE_RK_FUSED;
  const int R = P.p.lap_order;
  const bool wrap = L.periodic_box && (tma ? (L.n[0] >= 2 * R && L.n[1] >= 2 * R && L.n[2] >= 2 * R) : (SLEDGE_K1F_PLANE != 0));
  a.wrap = wrap ? 1 : 0;
  auto tmaps = [&](int buf, int which) -> const void* {
    return tma ? (const void*)(tab<CUtensorMap>(c, L.off_tmaps) + (size_t)((buf & 3) * 2 + which) * L.boxdev.size()) : nullptr;
  };
  auto ensure_ghosts = [&](int buf, double time) -> int {
    if (l > 0) {  // fine level: Pi ghosts of interpolated cells carry the psi of the sweep's later stage (t + dt/2 or t + dt)
      VelFill vf;
      vf.on = true;
      vf.ta = t;
      vf.tb = pass == 0 ? t + 0.5 * dt : t + dt;
      vf.w = use_w && pass == 1;
      // the fill before sweep A writes the interpolated ghosts of U3 too (they depend on the coarse level only), the
      // fill before sweep B moves the same-level copies only
      if ((P.p.interp == SLEDGE_INTERP_TRILINEAR || quartic_by_parent(P.p)) && c->fill_once) {
        if (pass == 0) {
          vf.buf2 = cur + 1;
          vf.w2 = use_w;
          vf.half_dt = 0.5 * dt;
        } else {
          vf.copies_only = true;
        }
      }
      return launch_ghosts<T>(c, l, buf, time, true, true, 0, 1, false, vf);
    }
    if (!wrap) return launch_ghosts<T>(c, l, buf, time, true, true);
    if (!tma || L.star_ok[buf & 3]) return SLEDGE_OK;
    L.star_ok[buf & 3] = true;
    return launch_ghosts<T>(c, l, buf, time, true, true);
  };
  int rc = SLEDGE_OK;
  if (pass == 0) {
    rc = ensure_ghosts(cur, t);
    if (rc) return rc;
    a.sten[0] = plane_ptr<T>(c, l, cur, 0);
    a.sten[1] = plane_ptr<T>(c, l, cur, 1);
    a.tmap[0] = tmaps(cur, 0);
    a.tmap[1] = tmaps(cur, 1);
    a.out_psi[0] = plane_ptr<T>(c, l, cur + 1, 0);
    a.out_pi[0] = plane_ptr<T>(c, l, cur + 1, 1);
    rc = launch_k1<T>(c, l, use_w ? FUSED_A2 : FUSED_A, a);
    L.star_ok[(cur + 1) & 3] = tma && wrap;
    return rc;
  }
  rc = ensure_ghosts(cur + 1, t + 0.5 * dt);  // Y's ghosts are still valid from pass 0
  if (rc) return rc;
  a.sten[0] = plane_ptr<T>(c, l, cur + 1, 0);
  a.sten[1] = plane_ptr<T>(c, l, cur + 1, 1);  // Pi_3, or W
  a.tmap[0] = tmaps(cur + 1, 0);
  a.tmap[1] = tmaps(cur + 1, 1);
  if (use_w) {
    a.pnt[0] = plane_ptr<T>(c, l, cur, 0);
    a.pnt[1] = plane_ptr<T>(c, l, cur, 1);
    a.wu = (T)(1.0 / dt);
  } else {
    a.sten[2] = plane_ptr<T>(c, l, cur, 0);
    a.tmap[2] = tmaps(cur, 0);
    a.pnt[0] = plane_ptr<T>(c, l, cur, 1);
  }
  a.out_psi[0] = plane_ptr<T>(c, l, cur + 2, 0);
  a.out_pi[0] = plane_ptr<T>(c, l, cur + 2, 1);
  rc = launch_k1<T>(c, l, use_w ? FUSED_B2 : FUSED_B, a);
  if (rc) return rc;
  L.star_ok[(cur + 2) & 3] = tma && wrap;
  finish_step(L, cur + 2, t, dt);
  return SLEDGE_OK;
}

// Fused sweeps need every psi AND Pi ghost to be a copy of a valid cell of the same level, which holds on
// level 0 (it covers the periodic domain, L39); finer levels take their ghosts from time-interpolated coarse
// data at every stage time (L72) and run the LEAN stages.
// With Kreiss-Oliger dissipation k_psi = Pi + Q psi is no longer pointwise: every level runs the staged sweeps.
inline bool is_ssprk3(const sledge_params& p) { return p.integrator == 3 || p.integrator == 10; }
inline bool level_is_fused(const Plan& P, int l) {
  // level 0: its ghosts are copies of valid cells.  Finer levels: the ghosts a sweep forms for the NEXT stage must be
  // the coarse state interpolated at that stage's time (L72), which the patch fills provide as "velocity" ghosts of
  // Pi (k_ghost.cuh: k_fill_patches for trilinear, k_fill_qparents for quartic interpolation by coarse parent)
  const bool lev_ok = l == 0 || (P.fine_fused && (P.p.interp == SLEDGE_INTERP_TRILINEAR || quartic_by_parent(P.p)) && !P.lev[l].patches.empty());
  return (P.p.rk_dataflow == SLEDGE_RK_FUSED || P.p.rk_dataflow == SLEDGE_RK_FUSED3) && lev_ok && !ko_on(P.p) && !is_ssprk3(P.p) && !is_rkn(P.p) && !P.p.gw;
}

// One SSPRK3 stage (integrator.type 3 / 10, L808; Shu-Osher form) of level l, s = 0, 1, 2:
//   U1 = Y + dt f(Y, t);  U2 = 3/4 Y + 1/4 (U1 + dt f(U1, t + dt));  Ynew = 1/3 Y + 2/3 (U2 + dt f(U2, t + dt/2))
// Buffers: cur = Y, cur+1 = U1 (then Ynew), cur+2 = U2: three buffers ("smaller memory footprint", type 10);
// 8 + 12 + 12 = 32 words per cell-step.
template <typename T>
int do_stage_ssp(sledge_ctx* c, int l, int s, double t, double dt, double eta_const) {
  Plan& P = c->plan;
  LevelHost& L = P.lev[l];
  static const double cs[3] = {0.0, 1.0, 0.5};
  static const double wy[3] = {0.0, 0.75, 1.0 / 3.0}, wu[3] = {1.0, 0.25, 2.0 / 3.0};
  const double ts = t + cs[s] * dt;
  const int cur = L.cur;
  const int ubuf = s == 0 ? cur : (s == 1 ? cur + 1 : cur + 2);
  const int obuf = s == 1 ? cur + 2 : cur + 1;
  int rc = launch_ghosts<T>(c, l, ubuf, ts, ko_on(P.p), true);
  if (rc) return rc;
  PipeArgs<T> a;
  memset(&a, 0, sizeof a);
  a.sten[0] = plane_ptr<T>(c, l, ubuf, 0);
  a.pnt[0] = plane_ptr<T>(c, l, ubuf, 1);
  if (s > 0) {
    a.pnt[1] = plane_ptr<T>(c, l, cur, 0);
    a.pnt[2] = plane_ptr<T>(c, l, cur, 1);
  }
  a.out_psi[0] = plane_ptr<T>(c, l, obuf, 0);
  a.out_pi[0] = plane_ptr<T>(c, l, obuf, 1);
  set_eta(P, a, 0, P.p.eta_fixed ? eta_const : ts);
  a.adt = (T)dt;
  a.wy = (T)wy[s];
  a.wu = (T)wu[s];
  rc = launch_k1<T>(c, l, s == 0 ? LEAN_S1 : SSP_S23, a);
  if (rc) return rc;
  if (s == 2) finish_step(L, cur + 1, t, dt);
  return SLEDGE_OK;
}

// Stage s of the gravitational-wave auxiliary fields (Eq.16; R25) in the LEAN data-flow of the
// scalar sector: U = stage input (buffer ubuf, whose psi ghosts the scalar stage has just filled), Y = cur,
// U2 = cur+1 (then the new state), U3 = cur+2, U4 = cur+3.
template <typename T>
int do_stage_gw(sledge_ctx* c, int l, int s, int ubuf, int cur, double ts, double dt, double eta_s) {
  Plan& P = c->plan;
  LevelHost& L = P.lev[l];
  // ghosts of the three u pair planes of the stage input, at the stage time (L72)
  int rc = launch_ghosts<T>(c, l, ubuf, ts, true, true, 2, 3);
  if (rc == SLEDGE_OK) rc = launch_ghosts<T>(c, l, ubuf, ts, false, true, 4, 4);
  if (rc) return rc;
  GwArgs<T> a;
  memset(&a, 0, sizeof a);
  a.boxes = tab<BoxDev>(c, L.off_boxes);
  a.tiles = tab<TileDev>(c, L.off_ftiles);
  a.g = P.p.nghost;
  a.ox = P.ox;
  a.psi = plane_ptr<T>(c, l, ubuf, 0);
  for (int q = 0; q < 3; ++q) {
    a.u[q] = plane_ptr<T>(c, l, ubuf, 2 + q);
    a.du[q] = plane_ptr<T>(c, l, ubuf, 5 + q);
  }
  const int in[3] = {cur, cur + 1, cur + 2};
  const int nin = s == 0 ? 0 : (s == 3 ? 3 : 1);
  for (int m = 0; m < nin; ++m)
    for (int q = 0; q < 6; ++q) a.in[m][q] = plane_ptr<T>(c, l, in[m], 2 + q);
  const int obuf = s == 3 ? cur + 1 : cur + 1 + s;
  for (int q = 0; q < 6; ++q) a.out[q] = plane_ptr<T>(c, l, obuf, 2 + q);
  const double h = L.h, h2 = h * h;
  a.inv_h2 = (T)(P.p.lap_order == 1 ? 1.0 / h2 : (P.p.lap_order == 2 ? 1.0 / (12.0 * h2) : 1.0 / (180.0 * h2)));
  a.inv_h = (T)(P.p.lap_order == 1 ? 1.0 / (2.0 * h) : (P.p.lap_order == 2 ? 1.0 / (12.0 * h) : 1.0 / (60.0 * h)));
  a.coupling = (T)P.p.gw_coupling;
  a.fric = (T)(P.p.gw_friction != 0.0 ? P.p.gw_friction / eta_s : 0.0);
  static const double as[4] = {0.5, 0.5, 1.0, 1.0 / 6.0};
  a.adt = (T)(as[s] * dt);
  const int grid = (int)L.ftiles.size();
  {
    Timed tm(c, KIND_STAGE);
    const int mode = s == 0 ? LEAN_S1 : (s == 3 ? LEAN_S4 : LEAN_S23);
    rc = P.p.lap_order == 1 ? launch_gw<T, 1>(c->stream, a, grid, mode)
         : (P.p.lap_order == 2 ? launch_gw<T, 2>(c->stream, a, grid, mode) : launch_gw<T, 3>(c->stream, a, grid, mode));
  }
  if (rc) return fail(c, SLEDGE_ECUDA, "k_gw_stage: bad mode");
  return check_launch(c, "k_gw_stage");
}

// Stage i of the user-defined Runge-Kutta-Nystrom scheme (integrator.type 20, L808-815; R26).
// Planes: cur = (psi_n, Pi_n); the stage fields Psi_1, Psi_2, ... alternate between (cur+1).psi and (cur+2).psi;
// f_0 .. f_3 are kept in (cur+1).Pi, (cur+2).Pi, (cur+3).psi, (cur+3).Pi, ordered so that the plane the new Pi
// overwrites in place (pointwise) is paired with the plane the new psi goes to: the new state is buffer
// X = cur+1 if the number of stages is odd, else cur+2.
template <typename T>
int do_stage_rkn(sledge_ctx* c, int l, int i, double t, double dt, double eta_const) {
  Plan& P = c->plan;
  LevelHost& L = P.lev[l];
  const sledge_params& p = P.p;
  const int s = p.rkn_stages, cur = L.cur;
  const bool last = i == s - 1;
  using PP = typename PairOf<T>::type;
  auto ping = [&](int k) -> int { return cur + 1 + (k & 1); };  // buffer whose psi plane holds Psi_{k+1}
  PP* const fpl[4] = {plane_ptr<T>(c, l, cur + 1, 1), plane_ptr<T>(c, l, cur + 2, 1), plane_ptr<T>(c, l, cur + 3, 0),
                      plane_ptr<T>(c, l, cur + 3, 1)};
  // f_j lives in fpl[slot(j)]: the in-place target X.Pi must hold a stored f only if one is stored there
  const int X = ping(s - 1);  // buffer of the new state
  auto slot = [&](int j) -> int {  // keep X.Pi for the LAST stored f so that every earlier one is read before the overwrite
    const int xs = (X == cur + 1) ? 0 : 1, other = 1 - xs;
    const int order[4] = {other, 2, 3, xs};
    return order[j];
  };
  const double ts = t + p.rkn_nodes[i] * dt;
  const int ubuf = i == 0 ? cur : ping(i - 1);
  int rc = launch_ghosts<T>(c, l, ubuf, ts, false, true);
  if (rc) return rc;
  PipeArgs<T> a;
  memset(&a, 0, sizeof a);
  a.sten[0] = plane_ptr<T>(c, l, ubuf, 0);
  a.pnt[0] = plane_ptr<T>(c, l, cur, 0);
  a.pnt[1] = plane_ptr<T>(c, l, cur, 1);
  for (int j = 0; j < i; ++j) a.pnt[2 + j] = fpl[slot(j)];
  set_eta(P, a, 0, p.eta_fixed ? eta_const : ts);
  const double* arow = p.rkn_tableau + (i + 1) * (i + 2) / 2;  // row of the NEXT stage
  if (!last) {  // out 0 = f_i, out 1 = Psi_{i+1} = psi_n + c_{i+1} dt Pi_n + dt^2 sum_{j<=i} a_{i+1,j} f_j
    a.rkn_w[0][6] = (T)1;
    a.rkn_w[1][0] = (T)1;
    a.rkn_w[1][1] = (T)(p.rkn_nodes[i + 1] * dt);
    for (int j = 0; j < i; ++j) a.rkn_w[1][2 + j] = (T)(dt * dt * arow[j]);
    a.rkn_w[1][6] = (T)(dt * dt * arow[i]);
    a.out_psi[0] = fpl[slot(i)];
    a.out_pi[0] = plane_ptr<T>(c, l, ping(i), 0);
  } else {  // out 0 = psi_new, out 1 = Pi_new
    a.rkn_w[0][0] = (T)1;
    a.rkn_w[0][1] = (T)dt;
    a.rkn_w[1][1] = (T)1;
    for (int j = 0; j < i; ++j) {
      a.rkn_w[0][2 + j] = (T)(dt * dt * p.rkn_weights_bar_b[j]);
      a.rkn_w[1][2 + j] = (T)(dt * p.rkn_weights_b[j]);
    }
    a.rkn_w[0][6] = (T)(dt * dt * p.rkn_weights_bar_b[i]);
    a.rkn_w[1][6] = (T)(dt * p.rkn_weights_b[i]);
    a.out_psi[0] = plane_ptr<T>(c, l, X, 0);
    a.out_pi[0] = plane_ptr<T>(c, l, X, 1);
  }
  rc = launch_k1<T>(c, l, RKN_ST, a);
  if (rc) return rc;
  if (last) finish_step(L, X, t, dt);
  return SLEDGE_OK;
}

// One RK4 stage of level l: ghost fill of the stage input at its time, then K1.
// t = time at the start of the level's step, eta_const = eta used when eta_fixed.
template <typename T>
int do_stage(sledge_ctx* c, int l, int s, double t, double dt, double eta_const) {
  Plan& P = c->plan;
  LevelHost& L = P.lev[l];
  if (is_ssprk3(P.p)) return s < 3 ? do_stage_ssp<T>(c, l, s, t, dt, eta_const) : SLEDGE_OK;
  if (is_rkn(P.p)) return s < P.p.rkn_stages ? do_stage_rkn<T>(c, l, s, t, dt, eta_const) : SLEDGE_OK;
  if (s > 3) return SLEDGE_OK;
  if (level_is_fused(P, l)) {  // stage calls 1 and 3 run the two sweeps, 0 and 2 are no-ops
    if (s == 1) return do_fused_pass<T>(c, l, 0, t, dt, eta_const);
    if (s == 3) return do_fused_pass<T>(c, l, 1, t, dt, eta_const);
    return SLEDGE_OK;
  }
  static const double cs[4] = {0.0, 0.5, 0.5, 1.0};
  static const double as[4] = {0.5, 0.5, 1.0, 1.0 / 6.0};
  const double ts = t + cs[s] * dt;
  const double eta_s = P.p.eta_fixed ? eta_const : ts;
  const int cur = L.cur;
  const bool lean = P.p.rk_dataflow != SLEDGE_RK_CLASSIC || P.p.gw;  // with gw both sectors share the LEAN buffer roles
  int ubuf, mode, in[3] = {-1, -1, -1}, out[2] = {-1, -1};
  double adt = (s < 3) ? as[s] * dt : dt / 6.0, bdt = 0.0;
  if (lean) {  // buffers: cur = Y, cur+1 = U2 (then Ynew), cur+2 = U3, cur+3 = U4
    if (s == 0) { ubuf = cur; mode = LEAN_S1; out[0] = cur + 1; }
    else if (s == 1) { ubuf = cur + 1; mode = LEAN_S23; in[0] = cur; out[0] = cur + 2; }
    else if (s == 2) { ubuf = cur + 2; mode = LEAN_S23; in[0] = cur; out[0] = cur + 3; }
    else { ubuf = cur + 3; mode = LEAN_S4; in[0] = cur; in[1] = cur + 1; in[2] = cur + 2; out[0] = cur + 1; }
  } else {  // buffers: cur = Y, cur+1 = ACC (then Ynew), cur+2 = Ua, cur+3 = Ub
    if (s == 0) { ubuf = cur; mode = CLASSIC_S1; out[0] = cur + 2; out[1] = cur + 1; bdt = dt / 6.0; }
    else if (s == 1) { ubuf = cur + 2; mode = CLASSIC_S23; in[0] = cur; in[1] = cur + 1; out[0] = cur + 3; out[1] = cur + 1; bdt = dt / 3.0; }
    else if (s == 2) { ubuf = cur + 3; mode = CLASSIC_S23; in[0] = cur; in[1] = cur + 1; out[0] = cur + 2; out[1] = cur + 1; bdt = dt / 3.0; }
    else { ubuf = cur + 2; mode = CLASSIC_S4; in[0] = cur + 1; out[0] = cur + 1; }
  }
  int rc = launch_ghosts<T>(c, l, ubuf, ts, ko_on(P.p), true);  // the dissipation term differences Pi as well
  if (rc) return rc;
  PipeArgs<T> a;
  memset(&a, 0, sizeof a);
  a.sten[0] = plane_ptr<T>(c, l, ubuf, 0);
  a.pnt[0] = plane_ptr<T>(c, l, ubuf, 1);
  for (int q = 0; q < 3; ++q)
    if (in[q] >= 0) {
      a.pnt[1 + 2 * q] = plane_ptr<T>(c, l, in[q], 0);
      a.pnt[2 + 2 * q] = plane_ptr<T>(c, l, in[q], 1);
    }
  for (int q = 0; q < 2; ++q)
    if (out[q] >= 0) {
      a.out_psi[q] = plane_ptr<T>(c, l, out[q], 0);
      a.out_pi[q] = plane_ptr<T>(c, l, out[q], 1);
    }
  set_eta(P, a, 0, eta_s);
  a.adt = (T)adt;
  a.bdt = (T)bdt;
  rc = launch_k1<T>(c, l, mode, a);
  if (rc) return rc;
  if (P.p.gw) {  // the auxiliary fields of Eq.16 take the same stage (LEAN data-flow, same buffers)
    rc = do_stage_gw<T>(c, l, s, ubuf, cur, ts, dt, eta_s);
    if (rc) return rc;
  }
  if (s == 3) finish_step(L, cur + 1, t, dt);
  return SLEDGE_OK;
}

// K4 between level lf of context fc (fine) and level lc of context cc (coarse; the same context for an ordinary
// synchronisation, the shadow context for L98), on the plane pair (wa, wb) of the current states.  With tee the
// truncation-error comparison rides on it (scalar planes only).
template <typename T>
int avg_between(sledge_ctx* fc, int lf, sledge_ctx* cc, int lc, int wa, int wb, bool tee, const double* eps,
                uint8_t* tags, uint32_t* counts) {
  LevelHost& F = fc->plan.lev[lf];
  LevelHost& C = cc->plan.lev[lc];
  AvgArgs<T> a;
  memset(&a, 0, sizeof a);
  a.fboxes = tab<BoxDev>(fc, F.off_views);
  a.blk_prefix = tab<int>(fc, F.off_avg_prefix);
  a.nfbox = (int)F.viewdev.size();
  a.f_psi = plane_ptr<T>(fc, lf, F.cur, wa);
  a.f_pi = plane_ptr<T>(fc, lf, F.cur, wb);
  a.fgeom = geom_of(fc->plan, lf);
  a.cboxes = tab<BoxDev>(cc, C.off_boxes);
  a.cowner = tab<int>(cc, C.off_owner);
  a.cgeom = geom_of(cc->plan, lc);
  a.c_psi = plane_ptr<T>(cc, lc, C.cur, wa);
  a.c_pi = plane_ptr<T>(cc, lc, C.cur, wb);
  a.err_flag = tab<int>(fc, fc->plan.off_err);
  const int grid = F.avg_prefix.back();
  C.shell_ok[C.cur & 3] = 0;  // covered coarse cells change: ghost copies of them are stale
  C.star_ok[C.cur & 3] = false;
  if (tee) {  // truncation-error tags ride on the synchronisation (L98: "just before synchronization")
    for (int q = 0; q < 4; ++q) a.tee_eps[q] = (T)eps[q];
    a.tee_tags = tags;
    a.tee_counts = counts;
    a.nb0 = F.nb[0];
    a.nb1 = F.nb[1];
    if (counts) cudaMemsetAsync(counts, 0, sizeof(uint32_t) * (size_t)F.count_blocks, fc->stream);
  }
  {
    Timed t(fc, KIND_AVG);
    if (tee) k_average_down<T, true><<<grid, AVG_THREADS, 0, fc->stream>>>(a);
    else k_average_down<T, false><<<grid, AVG_THREADS, 0, fc->stream>>>(a);
  }
  return check_launch(fc, "k_average_down");
}

template <typename T>
int do_average_down(sledge_ctx* c, int lf) {
  LevelHost& F = c->plan.lev[lf];
  int rc = avg_between<T>(c, lf, c, lf - 1, 0, 1, F.tee_on, F.tee_eps, F.tee_tags, F.tee_counts);
  if (c->plan.p.gw)  // the auxiliary fields synchronise like every other component (L74)
    for (int w = 2; w < 8 && rc == SLEDGE_OK; w += 2) rc = avg_between<T>(c, lf, c, lf - 1, w, w + 1, false, nullptr, nullptr, nullptr);
  return rc;
}

// O6 / L66-76, Fig.2: level l one step, then level l+1 two half steps, then synchronise.
template <typename T>
int advance(sledge_ctx* c, int l, double t, double dt, double eta_const) {
  const int nst = is_rkn(c->plan.p) ? c->plan.p.rkn_stages : 4;
  for (int s = 0; s < nst; ++s) {
    const int rc = do_stage<T>(c, l, s, t, dt, eta_const);
    if (rc) return rc;
  }
  if (l + 1 < c->plan.p.n_levels) {
    int rc = advance<T>(c, l + 1, t, 0.5 * dt, eta_const);
    if (rc) return rc;
    rc = advance<T>(c, l + 1, t + 0.5 * dt, 0.5 * dt, eta_const);
    if (rc) return rc;
    rc = do_average_down<T>(c, l + 1);
    if (rc) return rc;
  }
  return SLEDGE_OK;
}

template <typename T>
int do_tag(sledge_ctx* c, int l, uint8_t* tags, uint32_t* counts) {
  Plan& P = c->plan;
  LevelHost& L = P.lev[l];
  // after a coarse step every level sits at its parent's t_new: alpha = 1, no temporal interpolation (L74)
  const double tcur = (l > 0 && P.lev[l - 1].have_pair) ? P.lev[l - 1].t_new : 0.0;
  // K3 wraps by itself where its tiles run over ONE box covering the periodic domain (the caller's, or the storage box
  // with the tag layout looked up per blocking-factor cell)
  const bool tag_lookup = !L.tag_cells.empty();
  const bool k3_wraps = L.periodic_box && (L.viewdev.size() == 1 || tag_lookup);
  int rc = k3_wraps ? SLEDGE_OK : launch_ghosts<T>(c, l, L.cur, tcur, false, false, 0, 1, true);
  if (rc) return rc;
  if (counts) cudaMemsetAsync(counts, 0, sizeof(uint32_t) * (size_t)L.count_blocks, c->stream);
  TagArgs<T> a;
  a.boxes = tab<BoxDev>(c, tag_lookup ? L.off_boxes : L.off_views);
  a.tag_cells = tag_lookup ? tab<int4>(c, L.off_tag_cells) : nullptr;
  a.bfs = ilog2(P.p.blocking_factor);
  a.no0 = L.no[0];
  a.no1 = L.no[1];
  a.tiles = tab<TileDev>(c, L.off_tag_tiles);
  a.psi = plane_ptr<T>(c, l, L.cur, 0);
  a.tags = tags;
  a.counts = counts;
  a.g = P.p.nghost;
  a.ox = P.ox;
  a.wrap = k3_wraps ? 1 : 0;
  a.nb0 = L.nb[0];
  a.nb1 = L.nb[1];
  {
    Timed t(c, KIND_TAG);
    static PerDevice configured_dev;  // per instantiation and device
    bool& configured = configured_dev[c->device];
    if (!configured) {
      cudaFuncSetAttribute(k_tag_strings<T, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tag_smem_bytes<T>());
      cudaFuncSetAttribute(k_tag_strings<T, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tag_smem_bytes<T>());
      configured = true;
    }
    if (tag_lookup) k_tag_strings<T, true><<<(int)L.tag_tiles.size(), TAG_THREADS, tag_smem_bytes<T>(), c->stream>>>(a);
    else k_tag_strings<T, false><<<(int)L.tag_tiles.size(), TAG_THREADS, tag_smem_bytes<T>(), c->stream>>>(a);
  }
  return check_launch(c, "k_tag_strings");
}

template <typename T>
int do_copy_comp(sledge_ctx* c, int ib, int comp, void* dense, bool to_state, bool with_ghosts) {
  Plan& P = c->plan;
  const int l = P.box[ib].level;
  LevelHost& L = P.lev[l];
  const BoxDev& b = L.viewdev[P.box_local[ib]];
  const int e = with_ghosts ? P.p.nghost : 0;
  const long long total = (long long)(b.n[0] + 2 * e) * (b.n[1] + 2 * e) * (b.n[2] + 2 * e);
  const int grid = (int)std::min<long long>((total + 255) / 256, 148 * 32);
  auto* pl = plane_ptr<T>(c, l, L.cur, comp >> 1);
  if (to_state) L.shell_ok[L.cur & 3] = 0;
  if (to_state) L.star_ok[L.cur & 3] = false;
  ++c->launches;
  if (to_state) k_copy_comp<T, true><<<grid, 256, 0, c->stream>>>(b, P.p.nghost, P.ox, e, comp, pl, (T*)dense);
  else k_copy_comp<T, false><<<grid, 256, 0, c->stream>>>(b, P.p.nghost, P.ox, e, comp, pl, (T*)dense);
  return check_launch(c, "k_copy_comp");
}

}  // namespace

// =================================================================================================
// sledge_tag_strings_static: K3 on one periodic box with NO allocation (include/sledge.h)
// =================================================================================================
namespace {

// The scratch of the no-allocation entry point: the box / tile tables and the packed pair plane k_tag_strings reads.
// In HOST code this name is only a stand-in for the symbol, not a device address: static_scratch_ptr() asks the
// runtime for the address once per device (with that device current) and the kernels are given that pointer.
static __device__ __align__(256) unsigned char g_static_scratch[SLEDGE_STATIC_SCRATCH_BYTES];

struct StaticLayout {  // byte offsets inside g_static_scratch
  size_t off_box = 0, off_tiles = 256, off_plane = 0, total = 0;
  int sx = 0, sy = 0, ox = 0, tnz = 0, ntx = 0, nty = 0, ntz = 0;
  long long plane_cells = 0;
};

// same row layout as a context with nghost = 1 (make_plan), same z-chunk rule for the tag tiles
StaticLayout static_layout(const int n[3], int esz) {
  StaticLayout S;
  const int g = 1, cpa = 128 / (2 * esz);
  S.ox = (g + cpa - 1) / cpa * cpa;
  S.sx = (S.ox + n[0] + g + cpa - 1) / cpa * cpa;
  S.sy = n[1] + 2 * g;
  S.plane_cells = (long long)S.sx * S.sy * (n[2] + 2 * g);
  S.ntx = (n[0] + TAG_TX - 1) / TAG_TX;
  S.nty = (n[1] + TAG_TY - 1) / TAG_TY;
  int tnz = K1_NZ;
  for (; tnz > TAG_MIN_NZ; tnz /= 2)
    if ((long long)S.ntx * S.nty * ((n[2] + tnz - 1) / tnz) >= TAG_MIN_TILES) break;
  S.tnz = tnz;
  S.ntz = (n[2] + tnz - 1) / tnz;
  S.off_plane = align_up(S.off_tiles + (size_t)S.ntx * S.nty * S.ntz * sizeof(TileDev), ALIGN);
  S.total = S.off_plane + (size_t)S.plane_cells * 2 * esz;
  return S;
}

// Writes everything the tag kernel will read: the BoxDev, the tile table and the valid cells of the pair plane
// (the periodic one-box tag pass reads no ghost cell, k_tag.cuh `wrap`).  Nothing is left over from an earlier call.
template <typename T>
__global__ void k_static_pack(unsigned char* scratch, const StaticLayout S, const int n0, const int n1, const int n2,
                              const T* __restrict__ psi1, const T* __restrict__ psi2) {
  using P = typename PairOf<T>::type;
  const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x, nth = (long long)gridDim.x * blockDim.x;
  BoxDev b;
  b.base = 0;
  b.n[0] = n0; b.n[1] = n1; b.n[2] = n2;
  b.lo[0] = b.lo[1] = b.lo[2] = 0;
  b.sx = S.sx;
  b.sy = S.sy;
  b.tag_base = 0;
  if (tid == 0) *reinterpret_cast<BoxDev*>(scratch + S.off_box) = b;
  TileDev* const tiles = reinterpret_cast<TileDev*>(scratch + S.off_tiles);
  const int ntiles = S.ntx * S.nty * S.ntz;
  for (long long q = tid; q < ntiles; q += nth) {
    const int ix = (int)(q % S.ntx), iy = (int)((q / S.ntx) % S.nty), iz = (int)(q / ((long long)S.ntx * S.nty));
    tiles[q] = TileDev{0, ix * TAG_TX, iy * TAG_TY, iz * S.tnz, min(S.tnz, n2 - iz * S.tnz)};
  }
  P* const plane = reinterpret_cast<P*>(scratch + S.off_plane);
  const long long total = (long long)n0 * n1 * n2;
  for (long long q = tid; q < total; q += nth) {
    const int i = (int)(q % n0), j = (int)((q / n0) % n1), k = (int)(q / ((long long)n0 * n1));
    plane[cell_offset(b, 1, S.ox, i, j, k)] = mkpair(psi1[q], psi2[q]);
  }
}

// device address of g_static_scratch on `dev` (which must be current): asked for once per device
int static_scratch_ptr(int dev, unsigned char** out) {
  static unsigned char* ptr[MAX_DEVICES] = {};
  if (dev < 0 || dev >= MAX_DEVICES) return fail(nullptr, SLEDGE_EINVAL, "device index %d out of range", dev);
  if (!ptr[dev]) {
    void* p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&p, g_static_scratch);
    if (e != cudaSuccess || !p)
      return fail(nullptr, SLEDGE_ECUDA, "cudaGetSymbolAddress(static scratch) on device %d: %s", dev, cudaGetErrorString(e));
    ptr[dev] = static_cast<unsigned char*>(p);
  }
  *out = ptr[dev];
  return SLEDGE_OK;
}

template <typename T>
int do_tag_static(int dev, const void* psi1, const void* psi2, const int n[3], uint8_t* tags, uint32_t* counts,
                  cudaStream_t stream) {
  const StaticLayout S = static_layout(n, (int)sizeof(T));
  unsigned char* scratch = nullptr;
  int rc = static_scratch_ptr(dev, &scratch);
  if (rc) return rc;
  const long long cells = (long long)n[0] * n[1] * n[2];
  const int pgrid = (int)std::min<long long>((cells + 255) / 256, 148 * 16);
  k_static_pack<T><<<pgrid, 256, 0, stream>>>(scratch, S, n[0], n[1], n[2], static_cast<const T*>(psi1), static_cast<const T*>(psi2));
  const int nb[3] = {(n[0] + COUNT_BLOCK - 1) / COUNT_BLOCK, (n[1] + COUNT_BLOCK - 1) / COUNT_BLOCK, (n[2] + COUNT_BLOCK - 1) / COUNT_BLOCK};
  if (counts) cudaMemsetAsync(counts, 0, sizeof(uint32_t) * (size_t)nb[0] * nb[1] * nb[2], stream);
  TagArgs<T> a;
  memset(&a, 0, sizeof a);
  a.boxes = reinterpret_cast<const BoxDev*>(scratch + S.off_box);
  a.tiles = reinterpret_cast<const TileDev*>(scratch + S.off_tiles);
  a.psi = reinterpret_cast<const typename PairOf<T>::type*>(scratch + S.off_plane);
  a.tags = tags;
  a.counts = counts;
  a.g = 1;
  a.ox = S.ox;
  a.wrap = 1;  // one box over the periodic domain: +1 neighbours are read at their wrapped position (L23)
  a.nb0 = nb[0];
  a.nb1 = nb[1];
  a.tag_cells = nullptr;
  static PerDevice configured_dev;  // per instantiation and device (its own flag: the context path keeps its own)
  bool& configured = configured_dev[dev];
  if (!configured) {
    cudaFuncSetAttribute(k_tag_strings<T, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tag_smem_bytes<T>());
    configured = true;
  }
  k_tag_strings<T, false><<<S.ntx * S.nty * S.ntz, TAG_THREADS, tag_smem_bytes<T>(), stream>>>(a);
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(nullptr, SLEDGE_ECUDA, "sledge_tag_strings_static: %s", cudaGetErrorString(e));
  return SLEDGE_OK;
}

}  // namespace

// =================================================================================================
// C ABI (include/sledge.h)
// =================================================================================================
#define DISPATCH(ctx, call_f32, call_f64) ((ctx)->plan.p.dtype == SLEDGE_F64 ? (call_f64) : (call_f32))

extern "C" {

int sledge_arena_bytes(const sledge_params* params, const sledge_box* boxes, int nbox, size_t* bytes) {
  Plan P;
  const int rc = make_plan(P, params, boxes, nbox);
  if (rc) return rc;
  if (bytes) *bytes = P.total;
  return SLEDGE_OK;
}

int sledge_create(sledge_ctx** out, const sledge_params* params, const sledge_box* boxes, int nbox, void* dev_arena,
                  size_t arena_bytes, void* cuda_stream) {
  if (!out) return fail(nullptr, SLEDGE_EINVAL, "ctx output pointer is null");
  *out = nullptr;
  sledge_ctx* c = new sledge_ctx();
  int rc = make_plan(c->plan, params, boxes, nbox);
  if (rc) {
    delete c;
    return rc;
  }
  Plan& P = c->plan;
  if (!dev_arena || ((uintptr_t)dev_arena % ALIGN) || arena_bytes < P.total) {
    rc = fail(nullptr, SLEDGE_ENOMEM, "arena null, not 256-byte aligned or too small (%zu bytes needed, %zu given)", P.total,
              arena_bytes);
    delete c;
    return rc;
  }
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
    cudaGetLastError();
    delete c;
    return fail(nullptr, SLEDGE_ECUDA, "no CUDA device: libsledge has no CPU fallback");
  }
  c->arena = (char*)dev_arena;
  c->stream = (cudaStream_t)cuda_stream;
  {
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, dev_arena) == cudaSuccess && at.type == cudaMemoryTypeDevice) c->device = at.device;
    else {
      cudaGetLastError();
      cudaGetDevice(&c->device);
    }
  }
  DeviceGuard guard(c->device);
  cudaError_t e = cudaMemsetAsync(c->arena, 0, P.total, c->stream);
  auto up = [&](size_t off, const void* src, size_t bytes) {
    if (e == cudaSuccess && bytes) e = cudaMemcpyAsync(c->arena + off, src, bytes, cudaMemcpyHostToDevice, c->stream);
  };
  {
    const char* ev = getenv("SLEDGE_K1_TMA");
    c->use_tma = !(ev && ev[0] == '0');
    const char* eo = getenv("SLEDGE_FILL_ONCE");
    c->fill_once = !(eo && eo[0] == '0');
    const char* ew = getenv("SLEDGE_FUSED_W");
    c->fused_w = !(ew && ew[0] == '0');
    const char* ep = getenv("SLEDGE_K2_PATCHES");
    c->use_patches = !(ep && ep[0] == '0');
    const char* ef = getenv("SLEDGE_FINE_FUSED");
    P.fine_fused = c->use_patches && c->use_tma && !(ef && ef[0] == '0');
  }
  for (int l = 0; l < P.p.n_levels && c->use_tma; ++l)
    if (level_is_fused(P, l) && (rc = make_tensor_maps(c, l)) != SLEDGE_OK) {
      g_err = c->err;
      delete c;
      return rc;
    }
  for (LevelHost& L : P.lev) {
    up(L.off_tmaps, L.tmaps_host.data(), L.tmaps_host.size() * sizeof(CUtensorMap));
    up(L.off_patches, L.patches.data(), L.patches.size() * sizeof(uint4));
    up(L.off_tag_patches, L.tag_patches.data(), L.tag_patches.size() * sizeof(uint4));
    up(L.off_boxes, L.boxdev.data(), L.boxdev.size() * sizeof(BoxDev));
    up(L.off_views, L.viewdev.data(), L.viewdev.size() * sizeof(BoxDev));
    up(L.off_tag_cells, L.tag_cells.data(), L.tag_cells.size() * sizeof(int4));
    up(L.off_tiles, L.tiles.data(), L.tiles.size() * sizeof(TileDev));
    up(L.off_ftiles, L.ftiles.data(), L.ftiles.size() * sizeof(TileDev));
    up(L.off_tag_tiles, L.tag_tiles.data(), L.tag_tiles.size() * sizeof(TileDev));
    up(L.off_owner, L.owner.data(), L.owner.size() * sizeof(int));
    up(L.off_ghost_prefix, L.ghost_prefix.data(), L.ghost_prefix.size() * sizeof(int));
    up(L.off_avg_prefix, L.avg_prefix.data(), L.avg_prefix.size() * sizeof(int));
    up(L.off_qp_prefix, L.qp_prefix.data(), L.qp_prefix.size() * sizeof(int));
  }
  // ghost lists: resolved on the device from the tables just uploaded (the plan kernel of level l reads the
  // tables of l and l-1 only); its launches do not count as hot-path launches
  if (e == cudaSuccess) {
    const int64_t before = c->launches;
    for (int l = 0; l < P.p.n_levels && rc == SLEDGE_OK; ++l)
      rc = DISPATCH(c, plan_ghosts<float>(c, l), plan_ghosts<double>(c, l));
    c->launches = before;
    if (rc != SLEDGE_OK) {
      g_err = c->err;
      delete c;
      return rc;
    }
  }
  // the tables above are pageable host memory: make sure the copies are done before they can go away
  if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
  for (int l = 0; l < P.p.n_levels && e == cudaSuccess; ++l)
    e = cudaMemcpy(&P.lev[l].n_star, c->arena + P.lev[l].off_star_count, sizeof(unsigned), cudaMemcpyDeviceToHost);
  for (int l = 1; l < P.p.n_levels && e == cudaSuccess; ++l)
    if (P.lev[l].qp_prefix.back() > 0)
      e = cudaMemcpy(&P.lev[l].n_star_parents, c->arena + P.lev[l].off_qs_count, sizeof(unsigned), cudaMemcpyDeviceToHost);
  int plan_flag = 0;  // a plan kernel met a ghost or coarse cell that no box provides
  if (e == cudaSuccess) e = cudaMemcpy(&plan_flag, c->arena + P.off_err, sizeof(int), cudaMemcpyDeviceToHost);
  if (e != cudaSuccess) {
    rc = fail(nullptr, SLEDGE_ECUDA, "sledge_create: %s", cudaGetErrorString(e));
    delete c;
    return rc;
  }
  if (plan_flag) {
    rc = fail(nullptr, SLEDGE_ESTATE, "sledge_create: a ghost cell has neither a same-level owner nor coarse data (nesting)");
    delete c;
    return rc;
  }
  if (P.p.shadow_level) {  // the shadow level of level 0 (L98) is a one-box context of its own inside the arena
    rc = sledge_create(&c->shadow, &P.shadow_p, &P.shadow_box, 1, c->arena + P.off_shadow, P.shadow_bytes, cuda_stream);
    if (rc != SLEDGE_OK) {
      sledge_destroy(c);
      return rc;
    }
  }
  *out = c;
  return SLEDGE_OK;
}

int sledge_destroy(sledge_ctx* c) {
  if (!c) return SLEDGE_OK;
  DeviceGuard guard(c->device);
  if (c->shadow) sledge_destroy(c->shadow);
  cudaStreamSynchronize(c->stream);
  if (c->s_h2d) {
    cudaStreamSynchronize(c->s_h2d);
    cudaStreamSynchronize(c->s_d2h);
    for (int k = 0; k < N_IN_SLOTS; ++k) {
      cudaEventDestroy(c->ev_in_ready[k]);
      cudaEventDestroy(c->ev_in_free[k]);
    }
    for (int k = 0; k < N_OUT_SLOTS; ++k) {
      cudaEventDestroy(c->ev_out_ready[k]);
      cudaEventDestroy(c->ev_out_free[k]);
    }
    cudaStreamDestroy(c->s_h2d);
    cudaStreamDestroy(c->s_d2h);
  }
  for (auto& v : c->ev)
    for (auto& pr : v) {
      cudaEventDestroy(pr.first);
      cudaEventDestroy(pr.second);
    }
  delete c;
  return SLEDGE_OK;
}

static int check_box_comp(sledge_ctx* c, int box, int comp, const void* ptr) {
  if (!c) return fail(nullptr, SLEDGE_EINVAL, "null context");
  if (box < 0 || box >= (int)c->plan.box.size()) return fail(c, SLEDGE_EINVAL, "box index %d out of range", box);
  const int ncomp = c->plan.p.gw ? SLEDGE_NCOMP_GW : SLEDGE_NCOMP;
  if (comp < 0 || comp >= ncomp) return fail(c, SLEDGE_EINVAL, "component %d out of range (0..%d)", comp, ncomp - 1);
  if (!ptr) return fail(c, SLEDGE_EINVAL, "null data pointer");
  return SLEDGE_OK;
}

int sledge_set_state(sledge_ctx* c, int box, int comp, const void* dev_src) {
  int rc = check_box_comp(c, box, comp, dev_src);
  if (rc) return rc;
  DeviceGuard guard(c->device);
  c->plan.lev[c->plan.box[box].level].have_pair = false;
  return DISPATCH(c, do_copy_comp<float>(c, box, comp, (void*)dev_src, true, false),
                  do_copy_comp<double>(c, box, comp, (void*)dev_src, true, false));
}

int sledge_get_state(sledge_ctx* c, int box, int comp, void* dev_dst) {
  int rc = check_box_comp(c, box, comp, dev_dst);
  if (rc) return rc;
  DeviceGuard guard(c->device);
  return DISPATCH(c, do_copy_comp<float>(c, box, comp, dev_dst, false, false),
                  do_copy_comp<double>(c, box, comp, dev_dst, false, false));
}

int sledge_get_ghosted(sledge_ctx* c, int box, int comp, void* dev_dst) {
  int rc = check_box_comp(c, box, comp, dev_dst);
  if (rc) return rc;
  DeviceGuard guard(c->device);
  return DISPATCH(c, do_copy_comp<float>(c, box, comp, dev_dst, false, true),
                  do_copy_comp<double>(c, box, comp, dev_dst, false, true));
}

static size_t box_valid_bytes(sledge_ctx* c, int box) {
  const sledge_box& B = c->plan.box[box];
  return (size_t)(B.hi[0] - B.lo[0] + 1) * (B.hi[1] - B.lo[1] + 1) * (B.hi[2] - B.lo[2] + 1) * c->plan.esz;
}

static int host_streams(sledge_ctx* c) {
  if (c->s_h2d) return SLEDGE_OK;
  cudaError_t e = cudaStreamCreateWithFlags(&c->s_h2d, cudaStreamNonBlocking);
  if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&c->s_d2h, cudaStreamNonBlocking);
  for (int k = 0; k < N_IN_SLOTS && e == cudaSuccess; ++k) {
    e = cudaEventCreateWithFlags(&c->ev_in_ready[k], cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->ev_in_free[k], cudaEventDisableTiming);
  }
  for (int k = 0; k < N_OUT_SLOTS && e == cudaSuccess; ++k) {
    e = cudaEventCreateWithFlags(&c->ev_out_ready[k], cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->ev_out_free[k], cudaEventDisableTiming);
  }
  if (e != cudaSuccess) return fail(c, SLEDGE_ECUDA, "host copy streams: %s", cudaGetErrorString(e));
  return SLEDGE_OK;
}

int sledge_set_state_host(sledge_ctx* c, int box, int comp, const void* host_src) {
  int rc = check_box_comp(c, box, comp, host_src);
  if (rc) return rc;
  DeviceGuard guard(c->device);
  if ((rc = host_streams(c)) != SLEDGE_OK) return rc;
  const int k = (int)(c->n_in++ % (unsigned)N_IN_SLOTS);
  void* slot = c->arena + c->plan.off_scratch + (size_t)k * c->plan.scratch_bytes;
  cudaError_t e = cudaSuccess;
  if (c->in_used[k]) e = cudaStreamWaitEvent(c->s_h2d, c->ev_in_free[k], 0);  // the slot's last repack has read it
  if (e == cudaSuccess) e = cudaMemcpyAsync(slot, host_src, box_valid_bytes(c, box), cudaMemcpyHostToDevice, c->s_h2d);
  if (e == cudaSuccess) e = cudaEventRecord(c->ev_in_ready[k], c->s_h2d);
  if (e == cudaSuccess) e = cudaStreamWaitEvent(c->stream, c->ev_in_ready[k], 0);
  if (e != cudaSuccess) return fail(c, SLEDGE_ECUDA, "set_state_host: %s", cudaGetErrorString(e));
  rc = sledge_set_state(c, box, comp, slot);
  if (rc) return rc;
  c->in_used[k] = true;
  e = cudaEventRecord(c->ev_in_free[k], c->stream);
  if (e != cudaSuccess) return fail(c, SLEDGE_ECUDA, "set_state_host: %s", cudaGetErrorString(e));
  return SLEDGE_OK;
}

int sledge_get_state_host(sledge_ctx* c, int box, int comp, void* host_dst) {
  int rc = check_box_comp(c, box, comp, host_dst);
  if (rc) return rc;
  DeviceGuard guard(c->device);
  if ((rc = host_streams(c)) != SLEDGE_OK) return rc;
  const int k = (int)(c->n_out++ % (unsigned)N_OUT_SLOTS);
  void* slot = c->arena + c->plan.off_scratch + (size_t)(N_IN_SLOTS + k) * c->plan.scratch_bytes;
  cudaError_t e = cudaSuccess;
  if (c->out_used[k]) e = cudaStreamWaitEvent(c->stream, c->ev_out_free[k], 0);  // the slot's last download is done
  if (e != cudaSuccess) return fail(c, SLEDGE_ECUDA, "get_state_host: %s", cudaGetErrorString(e));
  rc = sledge_get_state(c, box, comp, slot);
  if (rc) return rc;
  e = cudaEventRecord(c->ev_out_ready[k], c->stream);
  if (e == cudaSuccess) e = cudaStreamWaitEvent(c->s_d2h, c->ev_out_ready[k], 0);
  if (e == cudaSuccess) e = cudaMemcpyAsync(host_dst, slot, box_valid_bytes(c, box), cudaMemcpyDeviceToHost, c->s_d2h);
  if (e == cudaSuccess) e = cudaEventRecord(c->ev_out_free[k], c->s_d2h);
  if (e != cudaSuccess) return fail(c, SLEDGE_ECUDA, "get_state_host: %s", cudaGetErrorString(e));
  c->out_used[k] = true;
  return SLEDGE_OK;
}

int sledge_host_copies_join(sledge_ctx* c) {
  if (!c) return fail(nullptr, SLEDGE_EINVAL, "null context");
  DeviceGuard guard(c->device);
  cudaError_t e = cudaSuccess;
  for (int k = 0; k < N_OUT_SLOTS && e == cudaSuccess; ++k)
    if (c->out_used[k]) e = cudaStreamWaitEvent(c->stream, c->ev_out_free[k], 0);
  for (int k = 0; k < N_IN_SLOTS && e == cudaSuccess; ++k)
    if (c->in_used[k]) e = cudaStreamWaitEvent(c->stream, c->ev_in_free[k], 0);
  if (e != cudaSuccess) return fail(c, SLEDGE_ECUDA, "host_copies_join: %s", cudaGetErrorString(e));
  return SLEDGE_OK;
}

static int check_level(sledge_ctx* c, int level) {
  if (!c) return fail(nullptr, SLEDGE_EINVAL, "null context");
  if (level < 0 || level >= c->plan.p.n_levels) return fail(c, SLEDGE_EINVAL, "level %d out of range", level);
  return SLEDGE_OK;
}

int sledge_fill_ghosts(sledge_ctx* c, int level, double time) {
  int rc = check_level(c, level);
  if (rc) return rc;
  DeviceGuard guard(c->device);
  const int cur = c->plan.lev[level].cur;
  rc = DISPATCH(c, launch_ghosts<float>(c, level, cur, time, true), launch_ghosts<double>(c, level, cur, time, true));
  if (c->plan.p.gw)
    for (int w = 2; w < 8 && rc == SLEDGE_OK; w += 2)
      rc = DISPATCH(c, launch_ghosts<float>(c, level, cur, time, true, false, w, w + 1),
                    launch_ghosts<double>(c, level, cur, time, true, false, w, w + 1));
  return rc;
}

int sledge_rk_stage(sledge_ctx* c, int level, int stage, double dt, double eta) {
  int rc = check_level(c, level);
  if (rc) return rc;
  DeviceGuard guard(c->device);
  if (stage < 0 || stage > 4) return fail(c, SLEDGE_EINVAL, "stage must be 0..3 (0..4 for a five-stage RKN tableau)");
  return DISPATCH(c, do_stage<float>(c, level, stage, eta, dt, eta), do_stage<double>(c, level, stage, eta, dt, eta));
}

int sledge_rk_step(sledge_ctx* c, double dt, double eta) {
  if (!c) return fail(nullptr, SLEDGE_EINVAL, "null context");
  DeviceGuard guard(c->device);
  if (!(dt > 0)) return fail(c, SLEDGE_EINVAL, "dt must be positive");
  return DISPATCH(c, advance<float>(c, 0, eta, dt, eta), advance<double>(c, 0, eta, dt, eta));
}

int sledge_tag_strings(sledge_ctx* c, int level, uint8_t* dev_tags, uint32_t* dev_counts) {
  int rc = check_level(c, level);
  if (rc) return rc;
  DeviceGuard guard(c->device);
  return DISPATCH(c, do_tag<float>(c, level, dev_tags, dev_counts), do_tag<double>(c, level, dev_tags, dev_counts));
}

int sledge_tag_strings_static(const void* dev_psi1, const void* dev_psi2, const int* n, int dtype, uint8_t* dev_tags,
                              uint32_t* dev_counts, void* cuda_stream) {
  if (!dev_psi1 || !dev_psi2 || !n) return fail(nullptr, SLEDGE_EINVAL, "sledge_tag_strings_static: null input");
  if (dtype != SLEDGE_F32 && dtype != SLEDGE_F64) return fail(nullptr, SLEDGE_EINVAL, "dtype must be SLEDGE_F32 or SLEDGE_F64");
  for (int d = 0; d < 3; ++d)
    if (n[d] < 2 || n[d] > 32768) return fail(nullptr, SLEDGE_EINVAL, "sledge_tag_strings_static: n[%d] = %d, need 2..32768", d, n[d]);
  const int esz = dtype == SLEDGE_F64 ? 8 : 4;
  const StaticLayout S = static_layout(n, esz);
  if (S.total > (size_t)SLEDGE_STATIC_SCRATCH_BYTES)
    return fail(nullptr, SLEDGE_EINVAL,
                "sledge_tag_strings_static: a %d x %d x %d %s box needs %zu bytes of scratch, the static array holds %u "
                "(SLEDGE_STATIC_SCRATCH_BYTES; fits 72^3 in fp64, 88^3 in fp32): use a context (sledge_create + sledge_tag_strings)",
                n[0], n[1], n[2], esz == 8 ? "fp64" : "fp32", S.total, (unsigned)SLEDGE_STATIC_SCRATCH_BYTES);
  cudaPointerAttributes at;
  if (cudaPointerGetAttributes(&at, dev_psi1) != cudaSuccess || (at.type != cudaMemoryTypeDevice && at.type != cudaMemoryTypeManaged)) {
    cudaGetLastError();
    return fail(nullptr, SLEDGE_EINVAL, "sledge_tag_strings_static: dev_psi1 is not a device pointer");
  }
  DeviceGuard guard(at.device);
  cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
  return esz == 8 ? do_tag_static<double>(at.device, dev_psi1, dev_psi2, n, dev_tags, dev_counts, stream)
                  : do_tag_static<float>(at.device, dev_psi1, dev_psi2, n, dev_tags, dev_counts, stream);
}

int sledge_average_down(sledge_ctx* c, int fine_level) {
  int rc = check_level(c, fine_level);
  if (rc) return rc;
  DeviceGuard guard(c->device);
  if (fine_level < 1) return fail(c, SLEDGE_EINVAL, "average_down needs fine_level >= 1");
  return DISPATCH(c, do_average_down<float>(c, fine_level), do_average_down<double>(c, fine_level));
}

int sledge_level_cells(const sledge_ctx* c, int level, int64_t* valid_cells, int64_t* count_blocks) {
  if (!c || level < 0 || level >= c->plan.p.n_levels) return SLEDGE_EINVAL;
  if (valid_cells) *valid_cells = c->plan.lev[level].valid_cells;
  if (count_blocks) *count_blocks = c->plan.lev[level].count_blocks;
  return SLEDGE_OK;
}

int sledge_level_storage(const sledge_ctx* c, int level, int* storage_boxes, int64_t* stored_cells) {
  if (!c || level < 0 || level >= c->plan.p.n_levels) return SLEDGE_EINVAL;
  if (storage_boxes) *storage_boxes = (int)c->plan.lev[level].boxdev.size();
  if (stored_cells) *stored_cells = c->plan.lev[level].plane_cells;
  return SLEDGE_OK;
}

int sledge_tee_enable(sledge_ctx* c, int fine_level, const double* eps4, uint8_t* dev_tags, uint32_t* dev_counts) {
  if (!c) return fail(nullptr, SLEDGE_EINVAL, "null context");
  if (fine_level < 1 || fine_level >= c->plan.p.n_levels)
    return fail(c, SLEDGE_EINVAL, "tee_enable: level %d has no coarser level to compare with", fine_level);
  if (!eps4) return fail(c, SLEDGE_EINVAL, "tee_enable: null thresholds");
  for (int q = 0; q < 4; ++q)
    if (!(eps4[q] >= 0)) return fail(c, SLEDGE_EINVAL, "tee_enable: thresholds must be >= 0");
  if (dev_tags && ((uintptr_t)dev_tags & 1)) return fail(c, SLEDGE_EINVAL, "tee_enable: tags must be 2-byte aligned");
  LevelHost& L = c->plan.lev[fine_level];
  L.tee_on = dev_tags != nullptr || dev_counts != nullptr;
  for (int q = 0; q < 4; ++q) L.tee_eps[q] = eps4[q];
  L.tee_tags = dev_tags;
  L.tee_counts = dev_counts;
  return SLEDGE_OK;
}

int sledge_shadow_tee(sledge_ctx* c, double dt, double eta, const double* eps4, uint8_t* dev_tags, uint32_t* dev_counts) {
  if (!c) return fail(nullptr, SLEDGE_EINVAL, "null context");
  DeviceGuard guard(c->device);
  if (!c->shadow) return fail(c, SLEDGE_ESTATE, "shadow_tee: the context was created without shadow_level = 1 (L98)");
  if (!(dt > 0)) return fail(c, SLEDGE_EINVAL, "dt must be positive");
  if (!eps4) return fail(c, SLEDGE_EINVAL, "shadow_tee: null thresholds");
  for (int q = 0; q < 4; ++q)
    if (!(eps4[q] >= 0)) return fail(c, SLEDGE_EINVAL, "shadow_tee: thresholds must be >= 0");
  if (dev_tags && ((uintptr_t)dev_tags & 1)) return fail(c, SLEDGE_EINVAL, "shadow_tee: tags must be 2-byte aligned");
  sledge_ctx* sh = c->shadow;
  const bool gw = c->plan.p.gw != 0;
  // (1) shadow <- mean of the 8 level-0 children (every component)
  sh->plan.lev[0].have_pair = false;
  int rc = SLEDGE_OK;
  for (int w = 0; w < (gw ? 8 : 2) && rc == SLEDGE_OK; w += 2)
    rc = DISPATCH(c, avg_between<float>(c, 0, sh, 0, w, w + 1, false, nullptr, nullptr, nullptr),
                  avg_between<double>(c, 0, sh, 0, w, w + 1, false, nullptr, nullptr, nullptr));
  // (2) one step of 2 dt on the shadow level, two coarse steps of dt on the hierarchy
  if (rc == SLEDGE_OK) rc = sledge_rk_step(sh, 2.0 * dt, eta);
  if (rc != SLEDGE_OK && sh->err.size()) c->err = "shadow level: " + sh->err;
  if (rc == SLEDGE_OK) rc = sledge_rk_step(c, dt, eta);
  if (rc == SLEDGE_OK) rc = sledge_rk_step(c, dt, eta + dt);
  // (3) compare and tag (the K4 TEE kernel with the shadow box on the coarse side)
  if (rc == SLEDGE_OK)
    rc = DISPATCH(c, avg_between<float>(c, 0, sh, 0, 0, 1, true, eps4, dev_tags, dev_counts),
                  avg_between<double>(c, 0, sh, 0, 0, 1, true, eps4, dev_tags, dev_counts));
  c->launches += sh->launches;
  sh->launches = 0;
  return rc;
}

int64_t sledge_launch_count(const sledge_ctx* c) { return c ? c->launches : 0; }

int sledge_level_dataflow(const sledge_ctx* c, int level, int* k1_launches_per_step, int* words_per_cell_step) {
  if (!c || level < 0 || level >= c->plan.p.n_levels) return SLEDGE_EINVAL;
  const Plan& P = c->plan;
  int n = 4, w = P.p.rk_dataflow == SLEDGE_RK_CLASSIC && !P.p.gw ? 64 : 52;
  if (is_ssprk3(P.p)) {
    n = 3;
    w = 32;
  } else if (is_rkn(P.p)) {  // stage i: Psi_i (psi_n itself for i = 0), psi_n, Pi_n, f_0..f_{i-1} in; two planes out
    n = P.p.rkn_stages;
    w = 0;
    for (int i = 0; i < n; ++i) w += (i ? 2 : 0) + 4 + 2 * i + 4;
  } else if (level_is_fused(P, level)) {
    n = 2;
    w = 20;
  }
  if (P.p.gw) {  // psi + U (u, du) in, 12 out, plus Y in stages 2-3 and Y, U2, U3 in stage 4
    n += 4;
    w += (14 + 12) + 2 * (26 + 12) + (50 + 12);
  }
  if (k1_launches_per_step) *k1_launches_per_step = n;
  if (words_per_cell_step) *words_per_cell_step = w;
  return SLEDGE_OK;
}

int sledge_synchronize(sledge_ctx* c) {
  if (!c) return fail(nullptr, SLEDGE_EINVAL, "null context");
  DeviceGuard guard(c->device);
  cudaError_t e = cudaStreamSynchronize(c->stream);
  if (e == cudaSuccess && c->s_d2h) e = cudaStreamSynchronize(c->s_d2h);
  if (e == cudaSuccess && c->s_h2d) e = cudaStreamSynchronize(c->s_h2d);
  int flag = 0;
  if (e == cudaSuccess) e = cudaMemcpy(&flag, c->arena + c->plan.off_err, sizeof(int), cudaMemcpyDeviceToHost);
  if (e != cudaSuccess) return fail(c, SLEDGE_ECUDA, "synchronize: %s", cudaGetErrorString(e));
  if (flag) {  // reported once: cleared so that later calls report later faults only
    cudaMemset(c->arena + c->plan.off_err, 0, sizeof(int));
    return fail(c, SLEDGE_ESTATE, "a kernel found a cell with neither a same-level owner nor coarse data (nesting)");
  }
  return SLEDGE_OK;
}

int sledge_profile_enable(sledge_ctx* c, int on) {
  if (!c) return fail(nullptr, SLEDGE_EINVAL, "null context");
  c->profiling = on != 0;
  for (int k = 0; k < 4; ++k) c->ev_used[k] = 0;
  return SLEDGE_OK;
}

int sledge_profile_read(sledge_ctx* c, int kind, int64_t* launches, double* total_ms) {
  if (!c) return fail(nullptr, SLEDGE_EINVAL, "null context");
  DeviceGuard guard(c->device);
  if (kind < 0 || kind > 3) return fail(c, SLEDGE_EINVAL, "kind must be 0..3");
  const cudaError_t e = cudaStreamSynchronize(c->stream);
  if (e != cudaSuccess) return fail(c, SLEDGE_ECUDA, "profile_read: %s", cudaGetErrorString(e));
  double ms = 0;
  for (size_t q = 0; q < c->ev_used[kind]; ++q) {
    float t = 0;
    cudaEventElapsedTime(&t, c->ev[kind][q].first, c->ev[kind][q].second);
    ms += t;
  }
  if (launches) *launches = (int64_t)c->ev_used[kind];
  if (total_ms) *total_ms = ms;
  return SLEDGE_OK;
}

const char* sledge_last_error(const sledge_ctx* c) { return c ? c->err.c_str() : g_err.c_str(); }

}  // extern "C"
