// k_ghost.cuh -- K2: ghost fill of one stage buffer of one level.
//
// One thread per ghost cell.  For the ghost cell at unwrapped level index f:
//   * wrap f periodically (L23); if a box of the same level owns the wrapped cell, copy its VALID value
//     (same-level copy wins over interpolation, R9);
//   * else (level > 0) trilinear interpolation of the coarse state, itself linearly interpolated in time
//     between the coarse level's old and new states: c = (1-alpha) c_old + alpha c_new (L70-72).
//     f = 2c + r sits -1/4 (r = 0) or +1/4 (r = 1) of a coarse cell from the centre of c: per-axis weights
//     3/4 on c and 1/4 on c-1 (r = 0) or c+1 (r = 1).  Only VALID coarse cells are read, found through the
//     coarse owner table (their existence is what proper nesting guarantees, L70).
// Only valid cells are read and only ghost cells are written, so one launch per level has no hazards.
//
// The box list is static (regridding is outside the library), so WHERE every ghost cell takes its data from
// never changes: k_plan_ghosts resolves it once at create time -- enumeration of the ghost shell, periodic
// wrap, owner lookup, coarse parents -- into one 16-byte GhostEntry per ghost cell, and k_fill_ghosts, which
// runs before every RK stage, only streams that list: one thread per entry, load the entry, move the data.
//   copy   {dst, src}                                  same-level / periodic copy
//   interp {dst, o0, sx | sy << 16, signs}             all 8 coarse parents in ONE coarse box: offset of the
//                                                      (c0,c0,c0) corner, the box's pitches, and per axis
//                                                      whether c1 = c0 + 1 or c0 - 1
//   slow   {dst, (f0+g) | (f1+g) << 16, f2+g}          parents spread over several coarse boxes: the fine index
//                                                      is kept and the parents are looked up on the fly
// Enumeration: the ghost shell of a box is cut into three slab pairs (z-low/high: full ghosted xy-planes;
// y-low/high: full ghosted x-rows; x-low/high), x fastest, so that the wide slabs are written with coalesced
// rows.  A prefix table over boxes (in CTAs) maps the plan kernel's blockIdx.x -> box by bisection.
#pragma once
#include "layout.h"

namespace sledge {

constexpr int GHOST_THREADS = 256;

enum GhostKind { GHOST_COPY = 0, GHOST_INTERP = 1, GHOST_SLOW = 2, GHOST_NONE = 3 };
// x = dst, y / z = see above, w = kind | signs << 2 (bit d of signs: c1 = c0 + 1 along axis d)
typedef uint4 GhostEntry;
constexpr unsigned GHOST_STAR = 32u;  // bit 5 of w

template <typename T>
struct GhostArgs {
  using P = typename PairOf<T>::type;
  const BoxDev* boxes;
  const int* blk_prefix;  // nbox + 1 entries, CTAs before box b
  int nbox;
  P* psi;
  P* pi;             // used only when FILL_PI
  const int* owner;  // this level's owner grid (box index or -1), granularity = blocking factor
  LevelGeom geom;
  // next coarser level (level > 0 only)
  const BoxDev* cboxes;
  const int* cowner;
  LevelGeom cgeom;
  const P* c_old_psi;
  const P* c_new_psi;
  const P* c_old_pi;
  const P* c_new_pi;
  T alpha;
  int single;      // alpha is exactly 0 or 1 (or the coarse level has one state only): c_old == c_new point at the one
                   // buffer that counts; k_fill_qparents then skips the blend (1-alpha) old + alpha new, which would
                   // return it unchanged, together with the second load (the per-cell paths blend as usual: same bits)
  int has_coarse;
  int* err_flag;  // set to 1 if a ghost cell has neither a same-level owner nor coarse data
  GhostEntry* list;  // GHOST_THREADS entries per CTA of the enumeration (written by the plan, read by the fill)
  unsigned n_entries;
  int star_depth;  // plan: the Laplacian's radius R (L649).  Entries of ghost cells that a star stencil of that radius
                   // can reach -- outside the box along exactly ONE axis, by at most R -- carry GHOST_STAR
  int star_only;   // fill: move only GHOST_STAR entries (the fill before an RK sweep); 0 = every ghost cell
  int quartic;     // coarse->fine interpolation: 0 = trilinear (2^3 parents), 1 = quartic conservative (5^3 parents
                   // c0-2 .. c0+2 per axis; amr.interpolation_type 4, L70, L780).  Same entry formats: an INTERP entry
                   // then means "all 5^3 parents in one coarse box", y = offset of the (c0,c0,c0) cell, and the sign
                   // bits are r = f - 2 c0 per axis.
                   // 2 = the same with the window read through the GHOST cells of the coarse box that owns c0 (coarse
                   // nghost >= 2; the host fills the whole coarse shell by same-level copies first): every entry is
                   // an INTERP entry, no owner lookups at fill time
  int copy_only;   // fill: skip INTERP / SLOW entries (the coarse-shell fill that mode 2 needs)
  // quartic mode 2: one 32-byte entry per COARSE parent cell of the ghost shell (k_plan_qparents / k_fill_qparents)
  const int* qblk_prefix;  // nbox + 1 entries, CTAs of the parent enumeration before box b
  uint4* qlist;            // 2 x uint4 per slot
  unsigned n_qentries;
  GhostEntry* star_list;   // plan: the GHOST_STAR entries of `list`, packed; n_star of them (read back by the host)
  unsigned* star_count;
  uint4* qstar_list;       // plan: the parents with star children, packed (order = order of arrival); the fills before
  unsigned* qstar_count;   //       an RK sweep run over this list only, with every lane busy
  // star patches (k_fill_patches): the fills before an RK sweep as rectangular regions, 2 x uint4 per patch
  const uint4* patches;
  unsigned n_patches;
  // "velocity" ghosts of the second plane (k_fill_patches and k_fill_qparents, interpolated cells only; FUSED sweeps on a
  // fine level): the sweep forms the NEXT stage's psi at a ghost cell as psi_g + tau Pi_g, and that must be the coarse
  // state interpolated at the later stage time (L72).  The space-time interpolant I_psi(t) is linear in t between the
  // coarse old and new states, so its time derivative is I[psi_new - psi_old] / (t_new - t_old) whatever the two stage
  // times are: Pi_g <- I[psi_new - psi_old] * vel_c (0 while the coarse level holds one state only).
  int vel;  // 1: velocity ghosts; 2: the second plane holds W = psi_Y + psi(U4) (FUSED_A2 / FUSED_B2 sweeps, fill before
            // sweep B): W_g = I_psi(t) + I_psi(t + dt) = 2 I_psi(t + dt/2) = twice the first plane's ghost value
  T vel_c;  // 1 / (t_new - t_old) of the coarse level
  // k_fill_patches, vel mode before sweep A: the interpolated ghosts of the NEXT sweep's input buffer (U3) are written
  // in the same pass -- they depend on coarse data only, and the interpolant is linear in time:
  // psi2_g = psi_g + half_dt * Pi_g (= I_psi(t + dt/2)); pi2_g = Pi_g (velocity), or 2 psi2_g in the W form (w2 != 0).
  // The fill before sweep B then moves the same-level copies only (copy_only).  Null: off.
  P* psi2;
  P* pi2;
  T half_dt;
  int w2;
  int patch_smem_pairs;    // shared-memory pairs per warp and plane (largest coarse region of an interpolation patch)
};

__device__ __forceinline__ long long cell_offset(const BoxDev& b, int g, int ox, int i, int j, int k) {
  return b.base + ((long long)(k + g) * b.sy + (j + g)) * b.sx + (i + ox);
}

// periodic wrap of an index known to lie in [-n, 2n): ghost cells and their coarse parents are less than one
// ghost width (< blocking factor <= n) outside the domain
__device__ __forceinline__ int wrap1(int i, int n) { return i < 0 ? i + n : (i >= n ? i - n : i); }

__device__ __forceinline__ int owner_lookup(const int* owner, const LevelGeom& gm, int wi, int wj, int wk) {
  return owner[((long long)(wk >> gm.bf_shift) * gm.no[1] + (wj >> gm.bf_shift)) * gm.no[0] + (wi >> gm.bf_shift)];
}

// Offsets of the 8 coarse cells (dz, dy, dx in {0: c0, 1: c1}) inside the coarse level's planes; false if one
// of them is not a valid coarse cell.  Fast path: when c0 and c1 have the same owner box all 8 corners lie in
// it (a box is convex), so one owner pair and one box descriptor serve all of them.
__device__ __forceinline__ bool coarse_offsets(const BoxDev* cboxes, const int* cowner, const LevelGeom& cg,
                                               const int c0[3], const int c1[3], long long o[8]) {
  int w0[3], w1[3];
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    w0[d] = wrap1(c0[d], cg.n[d]);
    w1[d] = wrap1(c1[d], cg.n[d]);
  }
  const int ow0 = owner_lookup(cowner, cg, w0[0], w0[1], w0[2]);
  const int ow1 = owner_lookup(cowner, cg, w1[0], w1[1], w1[2]);
  if (ow0 >= 0 && ow0 == ow1) {
    const BoxDev cb = cboxes[ow0];
    const long long ox0 = w0[0] - cb.lo[0] + cg.ox, ox1 = w1[0] - cb.lo[0] + cg.ox;
    const long long oy0 = (long long)(w0[1] - cb.lo[1] + cg.g) * cb.sx, oy1 = (long long)(w1[1] - cb.lo[1] + cg.g) * cb.sx;
    const long long pl = (long long)cb.sx * cb.sy;
    const long long oz0 = cb.base + (w0[2] - cb.lo[2] + cg.g) * pl, oz1 = cb.base + (w1[2] - cb.lo[2] + cg.g) * pl;
#pragma unroll
    for (int q = 0; q < 8; ++q) o[q] = ((q & 4) ? oz1 : oz0) + ((q & 2) ? oy1 : oy0) + ((q & 1) ? ox1 : ox0);
    return true;
  }
  bool ok = true;
#pragma unroll
  for (int q = 0; q < 8; ++q) {
    const int ci = (q & 1) ? w1[0] : w0[0], cj = (q & 2) ? w1[1] : w0[1], ck = (q & 4) ? w1[2] : w0[2];
    const int ow = owner_lookup(cowner, cg, ci, cj, ck);
    o[q] = 0;
    if (ow < 0) {
      ok = false;
      continue;
    }
    const BoxDev cb = cboxes[ow];
    o[q] = cell_offset(cb, cg.g, cg.ox, ci - cb.lo[0], cj - cb.lo[1], ck - cb.lo[2]);
  }
  return ok;
}

// trilinear x linear-in-time combination (L70-72); q = dz*4 + dy*2 + dx, summed dx fastest from 0
template <typename T>
__device__ __forceinline__ typename PairOf<T>::type interp_coarse(const typename PairOf<T>::type* c_old,
                                                                  const typename PairOf<T>::type* c_new, T alpha,
                                                                  const long long o[8]) {
  using P = typename PairOf<T>::type;
  const T w[2] = {T(0.75), T(0.25)};
  const T oma = T(1) - alpha;
  T s0 = T(0), s1 = T(0);
  P vo[8], vn[8];
#pragma unroll
  for (int q = 0; q < 8; ++q) {
    vo[q] = c_old[o[q]];
    vn[q] = c_new[o[q]];
  }
#pragma unroll
  for (int q = 0; q < 8; ++q) {
    const T cv0 = oma * vo[q].x + alpha * vn[q].x;
    const T cv1 = oma * vo[q].y + alpha * vn[q].y;
    const T wt = (w[(q >> 2) & 1] * w[(q >> 1) & 1]) * w[q & 1];
    s0 += wt * cv0;
    s1 += wt * cv1;
  }
  return mkpair(s0, s1);
}

// the same trilinear combination of the coarse DIFFERENCE new - old (velocity ghosts: I is linear, so
// I[psi_new - psi_old] / (t_new - t_old) is the time derivative of the space-time interpolant)
template <typename T>
__device__ __forceinline__ typename PairOf<T>::type interp_coarse_diff(const typename PairOf<T>::type* c_old,
                                                                       const typename PairOf<T>::type* c_new,
                                                                       const long long o[8]) {
  using P = typename PairOf<T>::type;
  const T w[2] = {T(0.75), T(0.25)};
  T s0 = T(0), s1 = T(0);
  P vo[8], vn[8];
#pragma unroll
  for (int q = 0; q < 8; ++q) {
    vo[q] = c_old[o[q]];
    vn[q] = c_new[o[q]];
  }
#pragma unroll
  for (int q = 0; q < 8; ++q) {
    const T wt = (w[(q >> 2) & 1] * w[(q >> 1) & 1]) * w[q & 1];
    s0 += wt * (vn[q].x - vo[q].x);
    s1 += wt * (vn[q].y - vo[q].y);
  }
  return mkpair(s0, s1);
}

// parents of fine index f along one axis: f = 2 c0 + r sits -1/4 (r = 0) or +1/4 (r = 1) of a coarse cell from
// the centre of c0; the second parent is c0 - 1 (r = 0) or c0 + 1 (r = 1)
__device__ __forceinline__ void parents_of(int f, int& c0, int& c1) {
  c0 = floordiv2(f);
  c1 = (f - 2 * c0) == 0 ? c0 - 1 : c0 + 1;
}

// Create-time pass: one thread per slot of the enumeration, writes a.list[blockIdx.x * GHOST_THREADS + tid].
template <typename T>
__global__ void __launch_bounds__(GHOST_THREADS) k_plan_ghosts(const GhostArgs<T> a) {
  GhostEntry* const out = a.list + (size_t)blockIdx.x * GHOST_THREADS + threadIdx.x;
  // every entry goes to its slot of the full list; those a star stencil reaches are also appended to the packed
  // star list (order of arrival), which is what the fills before an RK sweep stream
  auto emit = [&](const uint4 e) {
    *out = e;
    if ((e.w & GHOST_STAR) && (e.w & 3u) != GHOST_NONE) a.star_list[atomicAdd(a.star_count, 1u)] = e;
  };
  // blockIdx.x -> box
  int lo_b = 0, hi_b = a.nbox;
  const int blk = blockIdx.x;
  while (hi_b - lo_b > 1) {
    const int mid = (lo_b + hi_b) >> 1;
    if (a.blk_prefix[mid] <= blk) lo_b = mid; else hi_b = mid;
  }
  const BoxDev b = a.boxes[lo_b];
  const int g = a.geom.g;
  const int nx = b.n[0], ny = b.n[1], nz = b.n[2];
  const int Gx = nx + 2 * g, Gy = ny + 2 * g;
  // 32-bit arithmetic throughout: a box's ghost shell has far fewer than 2^31 cells (checked at create)
  const unsigned uGx = (unsigned)Gx, uGxy = (unsigned)(Gx * Gy), g2 = (unsigned)(2 * g);
  const unsigned nA = uGxy * g2;                 // z slabs
  const unsigned nB = uGx * g2 * (unsigned)nz;   // y slabs
  const unsigned nC = g2 * (unsigned)ny * (unsigned)nz;  // x slabs
  const unsigned q = (unsigned)(blk - a.blk_prefix[lo_b]) * GHOST_THREADS + threadIdx.x;
  if (q >= nA + nB + nC) {
    emit(make_uint4(0u, 0u, 0u, (unsigned)GHOST_NONE));
    return;
  }
  int i, j, k;
  if (q < nA) {
    const unsigned zz = q / uGxy, r = q - zz * uGxy, jj = r / uGx;
    j = (int)jj - g;
    i = (int)(r - jj * uGx) - g;
    k = (int)zz < g ? (int)zz - g : nz + ((int)zz - g);
  } else if (q < nA + nB) {
    const unsigned p = q - nA, rowlen = uGx * g2;
    const unsigned kk = p / rowlen, r = p - kk * rowlen, yy = r / uGx;
    k = (int)kk;
    i = (int)(r - yy * uGx) - g;
    j = (int)yy < g ? (int)yy - g : ny + ((int)yy - g);
  } else {
    const unsigned p = q - nA - nB, rowlen = g2 * (unsigned)ny;
    const unsigned kk = p / rowlen, r = p - kk * rowlen, jj = r / g2, xx = r - jj * g2;
    k = (int)kk;
    j = (int)jj;
    i = (int)xx < g ? (int)xx - g : nx + ((int)xx - g);
  }
  // how far outside the box, per axis (0 = inside)
  const int dxo = i < 0 ? -i : (i >= nx ? i - nx + 1 : 0), dyo = j < 0 ? -j : (j >= ny ? j - ny + 1 : 0);
  const int dzo = k < 0 ? -k : (k >= nz ? k - nz + 1 : 0);
  const int nout = (dxo > 0) + (dyo > 0) + (dzo > 0);
  const unsigned star = (nout == 1 && dxo + dyo + dzo <= a.star_depth) ? GHOST_STAR : 0u;
  const int f0 = b.lo[0] + i, f1 = b.lo[1] + j, f2 = b.lo[2] + k;  // unwrapped level index
  const int wi = wrap1(f0, a.geom.n[0]), wj = wrap1(f1, a.geom.n[1]), wk = wrap1(f2, a.geom.n[2]);
  const unsigned dst = (unsigned)cell_offset(b, g, a.geom.ox, i, j, k);
  const int ow = owner_lookup(a.owner, a.geom, wi, wj, wk);
  if (ow >= 0) {  // same-level copy wins (R9)
    const BoxDev sb = a.boxes[ow];
    const long long src = cell_offset(sb, g, a.geom.ox, wi - sb.lo[0], wj - sb.lo[1], wk - sb.lo[2]);
    emit(make_uint4(dst, (unsigned)src, 0u, (unsigned)GHOST_COPY | star));
    return;
  }
  if (!a.has_coarse) {
    *a.err_flag = 1;
    emit(make_uint4(0u, 0u, 0u, (unsigned)GHOST_NONE));
    return;
  }
  const int f[3] = {f0, f1, f2};
  if (a.quartic) {
    int c0[3], wl[3], wh[3];
    bool unit = true;
    unsigned rbits = 0u;
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      c0[d] = floordiv2(f[d]);
      rbits |= (unsigned)(f[d] - 2 * c0[d]) << d;
      wl[d] = wrap1(c0[d] - 2, a.cgeom.n[d]);
      wh[d] = wrap1(c0[d] + 2, a.cgeom.n[d]);
      unit = unit && (wh[d] - wl[d] == 4);  // no periodic seam inside the 5-cell window
    }
    if (a.quartic == 2) {  // interpolated by coarse parent (k_fill_qparents), not by this list
      emit(make_uint4(0u, 0u, 0u, (unsigned)GHOST_NONE));
      return;
    }
    const int owl = owner_lookup(a.cowner, a.cgeom, wl[0], wl[1], wl[2]);
    const int owh = owner_lookup(a.cowner, a.cgeom, wh[0], wh[1], wh[2]);
    if (unit && owl >= 0 && owl == owh) {  // a box is convex: the whole window lies in it
      const BoxDev cb = a.cboxes[owl];
      const long long o0 = cell_offset(cb, a.cgeom.g, a.cgeom.ox, wl[0] + 2 - cb.lo[0], wl[1] + 2 - cb.lo[1], wl[2] + 2 - cb.lo[2]);
      emit(make_uint4(dst, (unsigned)o0, (unsigned)cb.sx | ((unsigned)cb.sy << 16), (unsigned)GHOST_INTERP | (rbits << 2) | star));
      return;
    }
    for (int mz = -2; mz <= 2; ++mz)
      for (int my = -2; my <= 2; ++my)
        for (int mx = -2; mx <= 2; ++mx)
          if (owner_lookup(a.cowner, a.cgeom, wrap1(c0[0] + mx, a.cgeom.n[0]), wrap1(c0[1] + my, a.cgeom.n[1]),
                           wrap1(c0[2] + mz, a.cgeom.n[2])) < 0)
            *a.err_flag = 1;
    emit(make_uint4(dst, (unsigned)(f0 + g) | ((unsigned)(f1 + g) << 16), (unsigned)(f2 + g), (unsigned)GHOST_SLOW | star));
    return;
  }
  int c0[3], c1[3], w0[3], w1[3];
  bool unit = true;
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    parents_of(f[d], c0[d], c1[d]);
    w0[d] = wrap1(c0[d], a.cgeom.n[d]);
    w1[d] = wrap1(c1[d], a.cgeom.n[d]);
    unit = unit && (w1[d] - w0[d] == c1[d] - c0[d]);  // no periodic seam between the two parents
  }
  const int ow0 = owner_lookup(a.cowner, a.cgeom, w0[0], w0[1], w0[2]);
  const int ow1 = owner_lookup(a.cowner, a.cgeom, w1[0], w1[1], w1[2]);
  if (unit && ow0 >= 0 && ow0 == ow1) {
    const BoxDev cb = a.cboxes[ow0];
    const long long o0 = cell_offset(cb, a.cgeom.g, a.cgeom.ox, w0[0] - cb.lo[0], w0[1] - cb.lo[1], w0[2] - cb.lo[2]);
    const unsigned signs = (c1[0] > c0[0] ? 1u : 0u) | (c1[1] > c0[1] ? 2u : 0u) | (c1[2] > c0[2] ? 4u : 0u);
    emit(make_uint4(dst, (unsigned)o0, (unsigned)cb.sx | ((unsigned)cb.sy << 16), (unsigned)GHOST_INTERP | (signs << 2) | star));
    return;
  }
  // parents in several coarse boxes (or across the periodic seam of a single one): resolved at fill time
  long long o[8];
  if (!coarse_offsets(a.cboxes, a.cowner, a.cgeom, c0, c1, o)) *a.err_flag = 1;
  emit(make_uint4(dst, (unsigned)(f0 + g) | ((unsigned)(f1 + g) << 16), (unsigned)(f2 + g), (unsigned)GHOST_SLOW | star));
}

// The fill itself: GHOST_EPT entries of the level's list per thread (strided by the CTA size, so that a warp still
// reads consecutive entries).  All entries, then all copy sources, are loaded before anything is stored: the
// dependent chain entry -> source -> store is paid once per thread, not once per ghost cell.
constexpr int GHOST_EPT = 4;

template <typename T, bool FILL_PI>
__device__ __forceinline__ void ghost_interp_entry(const GhostArgs<T>& a, const uint4 en) {
  long long o[8];
  if ((en.w & 3u) == GHOST_INTERP) {
    const long long sx = en.z & 0xffffu, pl = sx * (long long)(en.z >> 16);
    const long long dx = (en.w & 4u) ? 1 : -1, dy = (en.w & 8u) ? sx : -sx, dz = (en.w & 16u) ? pl : -pl;
#pragma unroll
    for (int q = 0; q < 8; ++q) o[q] = (long long)en.y + ((q & 1) ? dx : 0) + ((q & 2) ? dy : 0) + ((q & 4) ? dz : 0);
  } else {
    const int g = a.geom.g;
    const int f[3] = {(int)(en.y & 0xffffu) - g, (int)(en.y >> 16) - g, (int)en.z - g};
    int c0[3], c1[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) parents_of(f[d], c0[d], c1[d]);
    if (!coarse_offsets(a.cboxes, a.cowner, a.cgeom, c0, c1, o)) return;  // reported by the plan
  }
  a.psi[en.x] = interp_coarse<T>(a.c_old_psi, a.c_new_psi, a.alpha, o);
  if (FILL_PI) a.pi[en.x] = interp_coarse<T>(a.c_old_pi, a.c_new_pi, a.alpha, o);
}

// Quartic polynomial conservative interpolation (amr.interpolation_type 4, L70, L780): per axis the quartic whose
// averages over the coarse cells c0-2 .. c0+2 are their values, averaged over the fine cell f = 2 c0 + r:
//   r = 0: c0 + (-3 c[-2] + 22 c[-1] - 22 c[+1] + 3 c[+2]) / 128,   r = 1: the mirror image
// tensor product over the axes, each coarse value linear in time between the coarse old and new states (L72).
// Summed mz, my, mx (x fastest) from 0 with individually rounded operations.
template <typename T>
__device__ __forceinline__ T quartic_weight(int m, int r) {  // m = 0..4 <-> offset m - 2
  const T b = (m == 2) ? T(1) : ((m == 0 || m == 4) ? T(3.0 / 128) : T(22.0 / 128));
  const bool neg = (m == 0 || m == 3) != (r != 0);  // r = 0: -, +, 1, -, +
  return (m != 2 && neg) ? -b : b;
}

template <typename T, bool FILL_PI>
__device__ __forceinline__ void ghost_quartic_entry(const GhostArgs<T>& a, const uint4 en) {
  using P = typename PairOf<T>::type;
  const bool fast = (en.w & 3u) == GHOST_INTERP;
  int r[3], c0[3] = {0, 0, 0};
  long long base = 0, sx = 0, pl = 0;
  if (fast) {
    sx = en.z & 0xffffu;
    pl = sx * (long long)(en.z >> 16);
    base = (long long)en.y;
    r[0] = (en.w >> 2) & 1;
    r[1] = (en.w >> 3) & 1;
    r[2] = (en.w >> 4) & 1;
  } else {
    const int g = a.geom.g;
    const int f[3] = {(int)(en.y & 0xffffu) - g, (int)(en.y >> 16) - g, (int)en.z - g};
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      c0[d] = floordiv2(f[d]);
      r[d] = f[d] - 2 * c0[d];
    }
  }
  const T oma = T(1) - a.alpha;
  T s0 = T(0), s1 = T(0), t0 = T(0), t1 = T(0);
#pragma unroll 1
  for (int mz = 0; mz < 5; ++mz) {
    const T wz = quartic_weight<T>(mz, r[2]);
#pragma unroll 1
    for (int my = 0; my < 5; ++my) {
      const T wzy = wz * quartic_weight<T>(my, r[1]);
      long long o[5];
      if (fast) {
#pragma unroll
        for (int mx = 0; mx < 5; ++mx) o[mx] = base + (mz - 2) * pl + (my - 2) * sx + (mx - 2);
      } else {
        const int cj = wrap1(c0[1] + my - 2, a.cgeom.n[1]), ck = wrap1(c0[2] + mz - 2, a.cgeom.n[2]);
#pragma unroll
        for (int mx = 0; mx < 5; ++mx) {
          const int ci = wrap1(c0[0] + mx - 2, a.cgeom.n[0]);
          const int ow = owner_lookup(a.cowner, a.cgeom, ci, cj, ck);
          if (ow < 0) return;  // reported by the plan
          const BoxDev cb = a.cboxes[ow];
          o[mx] = cell_offset(cb, a.cgeom.g, a.cgeom.ox, ci - cb.lo[0], cj - cb.lo[1], ck - cb.lo[2]);
        }
      }
      P vo[5], vn[5], po[5], pn[5];
#pragma unroll
      for (int mx = 0; mx < 5; ++mx) {
        vo[mx] = a.c_old_psi[o[mx]];
        vn[mx] = a.c_new_psi[o[mx]];
        if (FILL_PI) {
          po[mx] = a.c_old_pi[o[mx]];
          pn[mx] = a.c_new_pi[o[mx]];
        }
      }
#pragma unroll
      for (int mx = 0; mx < 5; ++mx) {
        const T wt = wzy * quartic_weight<T>(mx, r[0]);
        s0 += wt * (oma * vo[mx].x + a.alpha * vn[mx].x);
        s1 += wt * (oma * vo[mx].y + a.alpha * vn[mx].y);
        if (FILL_PI) {
          t0 += wt * (oma * po[mx].x + a.alpha * pn[mx].x);
          t1 += wt * (oma * po[mx].y + a.alpha * pn[mx].y);
        }
      }
    }
  }
  a.psi[en.x] = mkpair(s0, s1);
  if (FILL_PI) a.pi[en.x] = mkpair(t0, t1);
}

template <typename T, bool FILL_PI, bool QUARTIC = false>
__global__ void __launch_bounds__(GHOST_THREADS) k_fill_ghosts(const GhostArgs<T> a) {
  using P = typename PairOf<T>::type;
  const unsigned e0 = blockIdx.x * (GHOST_THREADS * GHOST_EPT) + threadIdx.x;
  uint4 en[GHOST_EPT];
#pragma unroll
  for (int j = 0; j < GHOST_EPT; ++j) {
    const unsigned e = e0 + j * GHOST_THREADS;
    en[j] = e < a.n_entries ? __ldg(reinterpret_cast<const uint4*>(a.list) + e) : make_uint4(0u, 0u, 0u, (unsigned)GHOST_NONE);
    if (a.star_only && !(en[j].w & GHOST_STAR)) en[j].w = (unsigned)GHOST_NONE;  // a star stencil never reads this cell
    if (a.copy_only && (en[j].w & 3u) != GHOST_COPY) en[j].w = (unsigned)GHOST_NONE;
  }
  P v[GHOST_EPT], vp[GHOST_EPT];
#pragma unroll
  for (int j = 0; j < GHOST_EPT; ++j)
    if ((en[j].w & 3u) == GHOST_COPY) {
      v[j] = a.psi[en[j].y];
      if (FILL_PI) vp[j] = a.pi[en[j].y];
    }
#pragma unroll
  for (int j = 0; j < GHOST_EPT; ++j)
    if ((en[j].w & 3u) == GHOST_COPY) {
      a.psi[en[j].x] = v[j];
      if (FILL_PI) a.pi[en[j].x] = vp[j];
    }
#pragma unroll
  for (int j = 0; j < GHOST_EPT; ++j) {
    const unsigned kind = en[j].w & 3u;
    if (kind == GHOST_INTERP || kind == GHOST_SLOW) {
      if (QUARTIC) ghost_quartic_entry<T, FILL_PI>(a, en[j]);
      else ghost_interp_entry<T, FILL_PI>(a, en[j]);
    }
  }
}

// ---- quartic interpolation by coarse parent (mode 2) -------------------------------------------------------------
// The 8 children of a coarse cell share its 5^3 window, and before an RK sweep a whole face layer of parents has all
// 8 children in the star set: one thread per PARENT loads the window once (through the ghost cells of the coarse box
// that owns the parent, which the host has filled with same-level copies), blends old / new in time once, and
// evaluates the 8 children separably (x, then y, then z pass: see k_fill_qparents): 8x fewer loads and ~10x fewer
// operations per ghost cell than the per-cell evaluation, equal to it (and to the oracle's direct triple sum) up to
// rounding order.
// Entry (2 x uint4): a = {offset of child (0,0,0) in the fine planes (mod 2^32: that child may lie outside the stored
// shell), offset of the parent in the coarse planes, coarse sx | sy << 16, fine sx | sy << 16},
// b.x = mask of children that are interpolated ghost cells | (those a star stencil reaches) << 8.
// Enumeration: the parents of the ghost shell of box b are the shell of thickness t = ceil(g/2) around its coarse
// footprint, cut into z / y / x slab pairs like the fine shell.
template <typename T>
__global__ void __launch_bounds__(GHOST_THREADS) k_plan_qparents(const GhostArgs<T> a) {
  uint4* const out = a.qlist + 2 * ((size_t)blockIdx.x * GHOST_THREADS + threadIdx.x);
  out[0] = make_uint4(0u, 0u, 0u, 0u);
  out[1] = make_uint4(0u, 0u, 0u, 0u);
  int lo_b = 0, hi_b = a.nbox;
  const int blk = blockIdx.x;
  while (hi_b - lo_b > 1) {
    const int mid = (lo_b + hi_b) >> 1;
    if (a.qblk_prefix[mid] <= blk) lo_b = mid; else hi_b = mid;
  }
  const BoxDev b = a.boxes[lo_b];
  const int g = a.geom.g, t = (g + 1) / 2;
  const int cx = b.n[0] >> 1, cy = b.n[1] >> 1, cz = b.n[2] >> 1;
  const unsigned Ex = (unsigned)(cx + 2 * t), Ey = (unsigned)(cy + 2 * t), t2 = (unsigned)(2 * t);
  const unsigned nA = Ex * Ey * t2, nB = Ex * t2 * (unsigned)cz, nC = t2 * (unsigned)cy * (unsigned)cz;
  const unsigned q = (unsigned)(blk - a.qblk_prefix[lo_b]) * GHOST_THREADS + threadIdx.x;
  if (q >= nA + nB + nC) return;
  int I, J, K;  // parent relative to the box's coarse footprint
  if (q < nA) {
    const unsigned zz = q / (Ex * Ey), r = q - zz * (Ex * Ey), jj = r / Ex;
    J = (int)jj - t;
    I = (int)(r - jj * Ex) - t;
    K = (int)zz < t ? (int)zz - t : cz + ((int)zz - t);
  } else if (q < nA + nB) {
    const unsigned p = q - nA, rowlen = Ex * t2;
    const unsigned kk = p / rowlen, r = p - kk * rowlen, yy = r / Ex;
    K = (int)kk;
    I = (int)(r - yy * Ex) - t;
    J = (int)yy < t ? (int)yy - t : cy + ((int)yy - t);
  } else {
    const unsigned p = q - nA - nB, rowlen = t2 * (unsigned)cy;
    const unsigned kk = p / rowlen, r = p - kk * rowlen, jj = r / t2, xx = r - jj * t2;
    K = (int)kk;
    J = (int)jj;
    I = (int)xx < t ? (int)xx - t : cx + ((int)xx - t);
  }
  unsigned mask = 0u, smask = 0u;
  for (int c = 0; c < 8; ++c) {
    const int i = 2 * I + (c & 1), j = 2 * J + ((c >> 1) & 1), k = 2 * K + (c >> 2);
    if (i < -g || i >= b.n[0] + g || j < -g || j >= b.n[1] + g || k < -g || k >= b.n[2] + g) continue;
    const int dxo = i < 0 ? -i : (i >= b.n[0] ? i - b.n[0] + 1 : 0), dyo = j < 0 ? -j : (j >= b.n[1] ? j - b.n[1] + 1 : 0);
    const int dzo = k < 0 ? -k : (k >= b.n[2] ? k - b.n[2] + 1 : 0);
    const int nout = (dxo > 0) + (dyo > 0) + (dzo > 0);
    if (nout == 0) continue;  // a valid cell
    const int wi = wrap1(b.lo[0] + i, a.geom.n[0]), wj = wrap1(b.lo[1] + j, a.geom.n[1]), wk = wrap1(b.lo[2] + k, a.geom.n[2]);
    if (owner_lookup(a.owner, a.geom, wi, wj, wk) >= 0) continue;  // same-level copy wins (R9)
    mask |= 1u << c;
    if (nout == 1 && dxo + dyo + dzo <= a.star_depth) smask |= 1u << c;
  }
  if (!mask) return;
  const int C[3] = {(b.lo[0] >> 1) + I, (b.lo[1] >> 1) + J, (b.lo[2] >> 1) + K};  // box corners are even (L39)
  // every window cell must be a valid coarse cell somewhere (nesting, L70): then the ghost cells of the box that
  // owns the parent hold same-level copies of them
  for (int mz = -2; mz <= 2; ++mz)
    for (int my = -2; my <= 2; ++my)
      for (int mx = -2; mx <= 2; ++mx)
        if (owner_lookup(a.cowner, a.cgeom, wrap1(C[0] + mx, a.cgeom.n[0]), wrap1(C[1] + my, a.cgeom.n[1]),
                         wrap1(C[2] + mz, a.cgeom.n[2])) < 0)
          *a.err_flag = 1;
  const int wc[3] = {wrap1(C[0], a.cgeom.n[0]), wrap1(C[1], a.cgeom.n[1]), wrap1(C[2], a.cgeom.n[2])};
  const int owc = owner_lookup(a.cowner, a.cgeom, wc[0], wc[1], wc[2]);
  if (owc < 0) return;
  const BoxDev cb = a.cboxes[owc];
  const long long o0 = cell_offset(cb, a.cgeom.g, a.cgeom.ox, wc[0] - cb.lo[0], wc[1] - cb.lo[1], wc[2] - cb.lo[2]);
  const long long d0 = cell_offset(b, g, a.geom.ox, 2 * I, 2 * J, 2 * K);
  const uint4 ea = make_uint4((unsigned)d0, (unsigned)o0, (unsigned)cb.sx | ((unsigned)cb.sy << 16), (unsigned)b.sx | ((unsigned)b.sy << 16));
  const uint4 eb = make_uint4(mask | (smask << 8), 0u, 0u, 0u);
  out[0] = ea;
  out[1] = eb;
  if (smask) {
    const unsigned idx = atomicAdd(a.qstar_count, 1u);
    a.qstar_list[2 * (size_t)idx] = ea;
    a.qstar_list[2 * (size_t)idx + 1] = eb;
  }
}

#ifndef SLEDGE_QP_MINB
#define SLEDGE_QP_MINB 1
#endif
#ifndef SLEDGE_QP_THREADS
#define SLEDGE_QP_THREADS 64  // ~250 registers per thread (everything unrolled, 125 x 2 loads in flight): measured 256 / 128 / 64 threads = 3.96 / 3.88 / 3.81 ms of C5 ghost time
#endif
constexpr int QP_THREADS = SLEDGE_QP_THREADS;
#ifndef SLEDGE_QP_UZ
#define SLEDGE_QP_UZ 5
#endif
#ifndef SLEDGE_QP_UY
#define SLEDGE_QP_UY 5
#endif
constexpr int QP_UZ = SLEDGE_QP_UZ, QP_UY = SLEDGE_QP_UY;  // unroll factors of the window's z / y loops (5 = fully)
// VEL: the second plane receives velocity ghosts I[psi_new - psi_old] * vel_c (FILL_PI and two coarse states only)
template <typename T, bool FILL_PI, bool SINGLE, bool VEL = false>
__global__ void __launch_bounds__(QP_THREADS, SLEDGE_QP_MINB) k_fill_qparents(const GhostArgs<T> a) {
  using P = typename PairOf<T>::type;
  const unsigned e = blockIdx.x * QP_THREADS + threadIdx.x;
  if (e >= a.n_qentries) return;
  const uint4 eb = __ldg(a.qlist + 2 * (size_t)e + 1);
  const unsigned mask = a.star_only ? ((eb.x >> 8) & 0xffu) : (eb.x & 0xffu);
  if (!mask) return;
  const uint4 ea = __ldg(a.qlist + 2 * (size_t)e);
  const long long csx = ea.z & 0xffffu, cpl = csx * (long long)(ea.z >> 16);
  const unsigned fsx = ea.w & 0xffffu, fpl = fsx * (ea.w >> 16);
  const long long base = (long long)ea.y;
  const T oma = T(1) - a.alpha;
  // Separable evaluation (the interpolant is a tensor product, header of ghost_quartic_entry): along each axis the two
  // children of a parent are  a + b  and  a - b  with a = the centre value and b = the weighted sum of the other four
  // (the r = 1 weights are the mirror image: w(m, 1) = -w(m, 0) for m != 2).  x pass on every row of the window, y pass
  // per z plane, z pass accumulated on the fly: ~230 operations per quantity instead of 1,125 for the direct triple
  // sum; the result differs from the oracle's direct sum by rounding order only (a few 1e-16 relative).
  constexpr int NQ = FILL_PI ? 4 : 2;  // psi1, psi2 and (Pi1, Pi2) or the velocity ghosts
  const T wq[5] = {quartic_weight<T>(0, 0), quartic_weight<T>(1, 0), T(1), quartic_weight<T>(3, 0), quartic_weight<T>(4, 0)};
  T Za[4][NQ], Zb[4][NQ];  // per (y child, x child): centre plane / weighted sum of the other four planes
#pragma unroll
  for (int c = 0; c < 4; ++c)
#pragma unroll
    for (int q = 0; q < NQ; ++q) Za[c][q] = Zb[c][q] = T(0);
#pragma unroll QP_UZ
  for (int mz = 0; mz < 5; ++mz) {
    T Ya[2][NQ], Yb[2][NQ];  // per x child: centre row / weighted sum of the other four rows
#pragma unroll
    for (int c = 0; c < 2; ++c)
#pragma unroll
      for (int q = 0; q < NQ; ++q) Ya[c][q] = Yb[c][q] = T(0);
#pragma unroll QP_UY
    for (int my = 0; my < 5; ++my) {
      const long long row = base + (mz - 2) * cpl + (my - 2) * csx - 2;
      P vo[5], vn[5], po[5], pn[5];
#pragma unroll
      for (int mx = 0; mx < 5; ++mx) {
        vo[mx] = a.c_old_psi[row + mx];
        if (!SINGLE) vn[mx] = a.c_new_psi[row + mx];
        if (FILL_PI && !VEL) {
          po[mx] = a.c_old_pi[row + mx];
          if (!SINGLE) pn[mx] = a.c_new_pi[row + mx];
        }
      }
      T v[5][NQ];  // the row's values, blended in time (L72)
#pragma unroll
      for (int mx = 0; mx < 5; ++mx) {
        v[mx][0] = SINGLE ? vo[mx].x : oma * vo[mx].x + a.alpha * vn[mx].x;
        v[mx][1] = SINGLE ? vo[mx].y : oma * vo[mx].y + a.alpha * vn[mx].y;
        if (FILL_PI) {
          if (VEL) {  // velocity ghosts, or W = twice the first plane (host: never SINGLE)
            v[mx][NQ - 2] = SINGLE ? T(0) : (a.vel == 2 ? T(2) * v[mx][0] : (vn[mx].x - vo[mx].x) * a.vel_c);
            v[mx][NQ - 1] = SINGLE ? T(0) : (a.vel == 2 ? T(2) * v[mx][1] : (vn[mx].y - vo[mx].y) * a.vel_c);
          } else {
            v[mx][NQ - 2] = SINGLE ? po[mx].x : oma * po[mx].x + a.alpha * pn[mx].x;
            v[mx][NQ - 1] = SINGLE ? po[mx].y : oma * po[mx].y + a.alpha * pn[mx].y;
          }
        }
      }
#pragma unroll
      for (int q = 0; q < NQ; ++q) {
        const T xb = (wq[0] * v[0][q] + wq[1] * v[1][q]) + (wq[3] * v[3][q] + wq[4] * v[4][q]);
        const T x0 = v[2][q] + xb, x1 = v[2][q] - xb;  // x children 0 / 1 of this row
        if (my == 2) {
          Ya[0][q] = x0;
          Ya[1][q] = x1;
        } else {
          Yb[0][q] += quartic_weight<T>(my, 0) * x0;
          Yb[1][q] += quartic_weight<T>(my, 0) * x1;
        }
      }
    }
#pragma unroll
    for (int c = 0; c < 4; ++c)  // c = y child * 2 + x child
#pragma unroll
      for (int q = 0; q < NQ; ++q) {
        const T y = (c & 2) ? Ya[c & 1][q] - Yb[c & 1][q] : Ya[c & 1][q] + Yb[c & 1][q];
        if (mz == 2) Za[c][q] = y;
        else Zb[c][q] += quartic_weight<T>(mz, 0) * y;
      }
  }
  T s[8][2], p[8][2];
#pragma unroll
  for (int c = 0; c < 8; ++c) {  // c = z child * 4 + y child * 2 + x child
    s[c][0] = (c & 4) ? Za[c & 3][0] - Zb[c & 3][0] : Za[c & 3][0] + Zb[c & 3][0];
    s[c][1] = (c & 4) ? Za[c & 3][1] - Zb[c & 3][1] : Za[c & 3][1] + Zb[c & 3][1];
    p[c][0] = p[c][1] = T(0);
    if (FILL_PI) {
      p[c][0] = (c & 4) ? Za[c & 3][NQ - 2] - Zb[c & 3][NQ - 2] : Za[c & 3][NQ - 2] + Zb[c & 3][NQ - 2];
      p[c][1] = (c & 4) ? Za[c & 3][NQ - 1] - Zb[c & 3][NQ - 1] : Za[c & 3][NQ - 1] + Zb[c & 3][NQ - 1];
    }
  }
#pragma unroll
  for (int c = 0; c < 8; ++c)
    if (mask & (1u << c)) {
      const unsigned dst = ea.x + (unsigned)(c >> 2) * fpl + (unsigned)((c >> 1) & 1) * fsx + (unsigned)(c & 1);
      a.psi[dst] = mkpair(s[c][0], s[c][1]);
      if (FILL_PI) a.pi[dst] = mkpair(p[c][0], p[c][1]);
      if (VEL && a.psi2 && a.vel == 1) {  // the ghosts of the next sweep's input buffer as well (GhostArgs::psi2)
        const T h0 = fma(a.half_dt, p[c][0], s[c][0]), h1 = fma(a.half_dt, p[c][1], s[c][1]);
        a.psi2[dst] = mkpair(h0, h1);
        a.pi2[dst] = a.w2 ? mkpair(T(2) * h0, T(2) * h1) : mkpair(p[c][0], p[c][1]);
      }
    }
}

// ---- star patches: the fill before an RK sweep, by rectangular region ---------------------------------------------
// The cells a star stencil of radius R reaches outside a box are six slabs R cells thick.  Cut along the blocking
// factor (the granularity of box ownership, L39), every piece -- a patch of R x bf x bf, bf x R x bf or bf x bf x R
// cells -- takes all its data from ONE place, resolved on the host at create time (sledge.cu: plan_patches):
//   COPY    a box of the same level (periodic wrap included): dst / src corner offsets and the two boxes' pitches;
//           16 bytes read + 16 written per cell and plane, no per-cell list entry (2 + 2 words)
//   INTERP  coarse->fine with every parent of the patch in ONE coarse box: the warp stages the coarse region
//           ((bf/2 + 2)^2 x (R/2 + 2) cells or less) in shared memory, blended in time ONCE per coarse cell
//           (c = (1-alpha) old + alpha new, L72), and every fine cell takes its 8 corners from there: ~1.7 coarse
//           loads per fine cell instead of 16, same arithmetic in the same order as interp_coarse (bit-identical)
//   SLOW    parents in several coarse boxes or across the periodic seam: per cell, as ghost_interp_entry
// One warp per patch.  Entry (2 x uint4):
//   A = {dst, src | coarse region base, dst sx | sy << 16, src sx | sy << 16}
//   B = {ex | ey << 8 | ez << 16 | kind << 24, cex | cey << 8 | cez << 16 | parity << 24, (f0+g) | (f1+g) << 16, f2+g}
// parity bit d = (first fine index along d) mod 2; (f0,f1,f2) = unwrapped level index of the first cell.
enum PatchKind { PATCH_COPY = 0, PATCH_INTERP = 1, PATCH_SLOW = 2 };
#ifndef SLEDGE_PATCH_WARPS
#define SLEDGE_PATCH_WARPS 4
#endif
constexpr int PATCH_WARPS = SLEDGE_PATCH_WARPS;

#ifndef SLEDGE_PATCH_MINB
#define SLEDGE_PATCH_MINB 5  // measured on C5: 5 CTAs of 4 warps per SM (102 registers) beats 4 (124) and 6 (85, spills)
#endif
template <typename T, bool FILL_PI>
__global__ void __launch_bounds__(PATCH_WARPS * 32, SLEDGE_PATCH_MINB) k_fill_patches(const GhostArgs<T> a) {
  using P = typename PairOf<T>::type;
  extern __shared__ __align__(16) unsigned char patch_smem[];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const unsigned ip = blockIdx.x * PATCH_WARPS + warp;
  if (ip >= a.n_patches) return;
  const uint4 A = __ldg(a.patches + 2 * (size_t)ip), B = __ldg(a.patches + 2 * (size_t)ip + 1);
  const int ex = B.x & 0xff, ey = (B.x >> 8) & 0xff, ez = (B.x >> 16) & 0xff, kind = B.x >> 24;
  const int dsx = A.z & 0xffff, dpl = dsx * (int)(A.z >> 16);
  const int ncell = ex * ey * ez;
  if (a.copy_only && kind != PATCH_COPY) return;  // quartic interpolation: k_fill_qparents does the rest
  if (kind == PATCH_COPY) {
    const int ssx = A.w & 0xffff, spl = ssx * (int)(A.w >> 16);
    // four cells per lane and pass, every load issued before the first store
    for (int q0 = lane; q0 < ncell; q0 += 128) {
      P v[4], vp[4];
      unsigned d[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int q = q0 + 32 * u;
        if (q < ncell) {
          const int i = q % ex, j = (q / ex) % ey, k = q / (ex * ey);
          const unsigned so = A.y + (unsigned)(k * spl + j * ssx + i);
          d[u] = A.x + (unsigned)(k * dpl + j * dsx + i);
          v[u] = a.psi[so];
          if (FILL_PI) vp[u] = a.pi[so];
        }
      }
#pragma unroll
      for (int u = 0; u < 4; ++u)
        if (q0 + 32 * u < ncell) {
          a.psi[d[u]] = v[u];
          if (FILL_PI) a.pi[d[u]] = vp[u];
        }
    }
    return;
  }
  if (kind == PATCH_INTERP) {
    const int cex = B.y & 0xff, cey = (B.y >> 8) & 0xff, cez = (B.y >> 16) & 0xff, par = B.y >> 24;
    const int csx = A.w & 0xffff, cpl = csx * (int)(A.w >> 16);
    P* const cs = reinterpret_cast<P*>(patch_smem) + (size_t)warp * a.patch_smem_pairs * (FILL_PI ? 2 : 1);
    P* const cp = cs + a.patch_smem_pairs;
    const int ncoarse = cex * cey * cez;
    const T oma = T(1) - a.alpha;
    const bool vel = FILL_PI && a.vel != 0;  // cs = coarse psi blended at alpha, cp = coarse psi NEW - OLD
    if (vel) {
      for (int q0 = lane; q0 < ncoarse; q0 += 128) {
        P vo[4], vn[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          const int q = q0 + 32 * u;
          if (q < ncoarse) {
            const int i = q % cex, j = (q / cex) % cey, k = q / (cex * cey);
            const long long o = (long long)A.y + (k * cpl + j * csx + i);
            vo[u] = a.c_old_psi[o];
            vn[u] = a.c_new_psi[o];
          }
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          const int q = q0 + 32 * u;
          if (q < ncoarse) {
            cs[q] = mkpair(oma * vo[u].x + a.alpha * vn[u].x, oma * vo[u].y + a.alpha * vn[u].y);
            cp[q] = mkpair(vn[u].x - vo[u].x, vn[u].y - vo[u].y);
          }
        }
      }
    } else
    for (int q0 = lane; q0 < ncoarse; q0 += 128) {  // four coarse cells per lane and pass, loads first
      P vo[4], vn[4], po[4], pn[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int q = q0 + 32 * u;
        if (q < ncoarse) {
          const int i = q % cex, j = (q / cex) % cey, k = q / (cex * cey);
          const long long o = (long long)A.y + (k * cpl + j * csx + i);
          vo[u] = a.c_old_psi[o];
          if (!a.single) vn[u] = a.c_new_psi[o];
          if (FILL_PI) {
            po[u] = a.c_old_pi[o];
            if (!a.single) pn[u] = a.c_new_pi[o];
          }
        }
      }
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int q = q0 + 32 * u;
        if (q < ncoarse) {
          if (a.single) {
            cs[q] = vo[u];
            if (FILL_PI) cp[q] = po[u];
          } else {
            cs[q] = mkpair(oma * vo[u].x + a.alpha * vn[u].x, oma * vo[u].y + a.alpha * vn[u].y);
            if (FILL_PI) cp[q] = mkpair(oma * po[u].x + a.alpha * pn[u].x, oma * po[u].y + a.alpha * pn[u].y);
          }
        }
      }
    }
    __syncwarp();
    const T w[2] = {T(0.75), T(0.25)};
    for (int q = lane; q < ncell; q += 32) {
      const int i = q % ex, j = (q / ex) % ey, k = q / (ex * ey);
      // parents of fine index f = 2m + par + i relative to the region's first coarse cell (which is the lowest parent
      // of the patch's first cell: m - 1 if par = 0, else m): c0 = m + ((par + i) >> 1); the second parent is
      // c0 - 1 (even fine index) or c0 + 1 (odd)
      const int px = par & 1, py = (par >> 1) & 1, pz = (par >> 2) & 1;
      const int x0 = ((px + i) >> 1) + 1 - px, y0 = ((py + j) >> 1) + 1 - py, z0 = ((pz + k) >> 1) + 1 - pz;
      const int x1 = ((px + i) & 1) ? x0 + 1 : x0 - 1, y1 = ((py + j) & 1) ? y0 + 1 : y0 - 1, z1 = ((pz + k) & 1) ? z0 + 1 : z0 - 1;
      T s0 = T(0), s1 = T(0), t0 = T(0), t1 = T(0);
#pragma unroll
      for (int c = 0; c < 8; ++c) {
        const int o = (((c & 4) ? z1 : z0) * cey + ((c & 2) ? y1 : y0)) * cex + ((c & 1) ? x1 : x0);
        const T wt = (w[(c >> 2) & 1] * w[(c >> 1) & 1]) * w[c & 1];
        const P cv = cs[o];
        s0 += wt * cv.x;
        s1 += wt * cv.y;
        if (FILL_PI) {
          const P pv = cp[o];
          t0 += wt * pv.x;
          t1 += wt * pv.y;
        }
      }
      const unsigned d = A.x + (unsigned)(k * dpl + j * dsx + i);
      a.psi[d] = mkpair(s0, s1);
      // velocity ghosts: Pi <- I[psi_new - psi_old] / (t_new - t_old) (0 while the coarse level has one state only)
      if (FILL_PI) a.pi[d] = vel ? (a.vel == 2 ? mkpair(T(2) * s0, T(2) * s1) : mkpair(t0 * a.vel_c, t1 * a.vel_c)) : mkpair(t0, t1);
      if (FILL_PI && vel && a.psi2) {  // the ghosts of U3 as well (see GhostArgs::psi2)
        const T v0 = t0 * a.vel_c, v1 = t1 * a.vel_c;
        const T h0 = fma(a.half_dt, v0, s0), h1 = fma(a.half_dt, v1, s1);
        a.psi2[d] = mkpair(h0, h1);
        a.pi2[d] = a.w2 ? mkpair(T(2) * h0, T(2) * h1) : mkpair(v0, v1);
      }
    }
    return;
  }
  // PATCH_SLOW: parents looked up per cell
  const int g = a.geom.g;
  const int f0 = (int)(B.z & 0xffffu) - g, f1 = (int)(B.z >> 16) - g, f2 = (int)B.w - g;
  for (int q = lane; q < ncell; q += 32) {
    const int i = q % ex, j = (q / ex) % ey, k = q / (ex * ey);
    const int f[3] = {f0 + i, f1 + j, f2 + k};
    int c0[3], c1[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) parents_of(f[d], c0[d], c1[d]);
    long long o[8];
    if (!coarse_offsets(a.cboxes, a.cowner, a.cgeom, c0, c1, o)) {
      *a.err_flag = 1;
      continue;
    }
    const unsigned d = A.x + (unsigned)(k * dpl + j * dsx + i);
    a.psi[d] = interp_coarse<T>(a.c_old_psi, a.c_new_psi, a.alpha, o);
    if (FILL_PI) {
      if (a.vel == 2) {
        const P pv = a.psi[d];  // just written by this thread
        a.pi[d] = mkpair(T(2) * pv.x, T(2) * pv.y);
      } else if (a.vel) {
        const P dv = interp_coarse_diff<T>(a.c_old_psi, a.c_new_psi, o);
        const T v0 = dv.x * a.vel_c, v1 = dv.y * a.vel_c;
        a.pi[d] = mkpair(v0, v1);
        if (a.psi2) {
          const P pv = a.psi[d];  // just written by this thread
          const T h0 = fma(a.half_dt, v0, pv.x), h1 = fma(a.half_dt, v1, pv.y);
          a.psi2[d] = mkpair(h0, h1);
          a.pi2[d] = a.w2 ? mkpair(T(2) * h0, T(2) * h1) : mkpair(v0, v1);
        }
      } else {
        a.pi[d] = interp_coarse<T>(a.c_old_pi, a.c_new_pi, a.alpha, o);
      }
    }
  }
}

}  // namespace sledge
