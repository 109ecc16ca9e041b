// k_rk_plane.cuh -- K1, plane-ring variant: the same sweeps as k_rk_pipe.cuh (same modes, same per-cell arithmetic
// rk_cell / lap_from, Eq.10-11), with a different on-chip data path.
//
// k_rk_pipe stages every plane twice in shared memory (cp.async ring -> registers -> centre plane), which makes
// the FUSED sweeps shared-memory-bandwidth bound on B200 (ncu: l1tex throughput 84-92 %, short-scoreboard and
// mio-throttle stalls; profiles/r01_c3_ncu_full_mid.md).  Here cp.async writes each ghosted tile plane (own cells
// AND x/y halo) ONCE, directly in the layout the stencil reads:
//   * ring of S = R + 1 + PD ghosted planes per differenced field; plane p (relative to the tile's z0) lives in
//     slot p % S from the moment its copy is issued (iteration p - R - PD) until it has been the centre plane
//     (iteration p);
//   * iteration zz: wait for plane zz+R, ONE __syncthreads (makes the plane visible and retires plane zz-1, whose
//     slot the copy of plane zz+R+PD issued next overwrites), each thread reads its own cell of plane zz+R into
//     the top of its register z-window (1 LDS per field) and its 4R x/y neighbours from the centre plane zz.
// Shared-memory traffic per cell and field: 4R + 1 vector reads + 1.3-1.6 cp.async writes, against 4R + 2 reads
// + 2.6 writes before; no copy loop.  Pointwise inputs keep their own PD-deep per-thread ring.
#pragma once
#include "k_rk_pipe.cuh"

namespace sledge {

template <typename T, int ORDER, int MODE, int TX, int TY, int PD, int RY = 1>
struct PlaneCfg {
  static constexpr int R = ORDER;
  static constexpr int CPT = Vec16<T>::CPT;
  static constexpr int TXC = TX * CPT;
  static constexpr int XO = (R + CPT - 1) / CPT * CPT;  // column of the first own cell: keeps own vectors 16-byte aligned
  static constexpr int SW = TXC + 2 * XO;
  static constexpr int SH = TY + 2 * R;
  static_assert(TY % RY == 0, "rows per thread must divide the tile height");
  static constexpr int NT = TX * TY / RY;         // threads: each owns RY consecutive rows of one x vector
  static constexpr int NH = 2 * R * (TXC + TY);  // halo pairs per plane (star stencil: no corners)
  static constexpr int HPT = (NH + NT - 1) / NT;
  static constexpr int NF = ModeInfo<MODE>::NF;
  static constexpr int NP = ModeInfo<MODE>::NP;
  static constexpr int NOUT = ModeInfo<MODE>::NOUT;
  static constexpr int S = R + 1 + PD;
  static constexpr size_t PAIR = 2 * sizeof(T);
  static constexpr size_t PLANE_BYTES = (size_t)S * NF * SH * SW * PAIR;
  static constexpr size_t PNT_BYTES = (size_t)PD * NP * RY * NT * 16;
  static constexpr size_t SMEM_BYTES = PLANE_BYTES + PNT_BYTES;
};

// Deepest prefetch distance (<= pdmax, >= 1) whose shared memory fits `budget` bytes.
template <typename T, int ORDER, int MODE, int TX, int TY, int RY = 1>
constexpr int plane_depth(size_t budget, int pdmax) {
  int d = 1;
  if (pdmax >= 2 && PlaneCfg<T, ORDER, MODE, TX, TY, 2, RY>::SMEM_BYTES <= budget) d = 2;
  if (pdmax >= 3 && PlaneCfg<T, ORDER, MODE, TX, TY, 3, RY>::SMEM_BYTES <= budget) d = 3;
  if (pdmax >= 4 && PlaneCfg<T, ORDER, MODE, TX, TY, 4, RY>::SMEM_BYTES <= budget) d = 4;
  return d;
}


// RY = rows per thread: a thread owns the same x vector of RY consecutive rows, so that the y neighbours of one
// of its cells that are its own other cells come from registers (4R + 1 -> 2R + 2R/RY + 1 vector reads per cell).
template <typename T, int ORDER, int MODE, int TX, int TY, int PD, int RY, int MINB>
__global__ void __launch_bounds__(TX* TY / RY, MINB) k_rk_plane(const PipeArgs<T> a) {
  using P = typename PairOf<T>::type;
  using V = Vec16<T>;
  using C = PlaneCfg<T, ORDER, MODE, TX, TY, PD, RY>;
  constexpr int R = C::R, CPT = C::CPT, TXC = C::TXC, XO = C::XO, SW = C::SW, SH = C::SH, NT = C::NT, NH = C::NH;
  constexpr int HPT = C::HPT, NF = C::NF, NP = C::NP, NOUT = C::NOUT, S = C::S;
  constexpr int NPA = NP > 0 ? NP : 1;
  constexpr int PSZ = SH * SW;  // pairs per field plane

  extern __shared__ __align__(16) unsigned char smem_raw[];
  P* const planes = reinterpret_cast<P*>(smem_raw);                  // [S][NF][SH * SW]
  V* const pring = reinterpret_cast<V*>(smem_raw + C::PLANE_BYTES);  // [PD][NP][RY][NT]

  const TileDev t = a.tiles[blockIdx.x];
  const BoxDev b = a.boxes[t.box];
  const int tid = threadIdx.x;
  const int tx = tid % TX, ty = (tid / TX) * RY;  // ty = first of this thread's rows
  const int x = t.x0 + tx * CPT, y = t.y0 + ty;
  // in a partial tile the columns/rows just past the box edge are ghost cells that the edge cells need as
  // +x / +y neighbours: threads sitting there still copy their own cells ("loader")
  bool active[RY], loader[RY];
#pragma unroll
  for (int j = 0; j < RY; ++j) {
    active[j] = (x < b.n[0]) && (y + j < b.n[1]);
    loader[j] = (x < b.n[0] + R) && (y + j < b.n[1] + R);
  }
  const long long plane = (long long)b.sx * b.sy;
  const long long tile_org =
      b.base + (long long)(t.z0 + a.g) * plane + (long long)(t.y0 + a.g) * b.sx + (t.x0 + a.ox);
  const long long off = tile_org + (long long)ty * b.sx + tx * CPT;  // this thread's first cell in plane z0
  // periodic single-box level (a.wrap): anything outside [0, n) is read at its wrapped position instead of from
  // the ghost layers (L23).  wofs(c, n) = displacement that brings coordinate c into the box.
  const bool wr = a.wrap != 0;
  auto wofs = [wr](int c, int n) -> int { return !wr ? 0 : (c < 0 ? n : (c >= n ? -n : 0)); };
  long long offl[RY];  // load address of row j (== off + j * sx unless the row / column lies past the box edge)
#pragma unroll
  for (int j = 0; j < RY; ++j) offl[j] = off + (long long)(j + wofs(y + j, b.n[1])) * b.sx + wofs(x, b.n[0]);
  auto zofs = [&](int p) -> long long { return (long long)(p + wofs(t.z0 + p, b.n[2])) * plane; };

  // halo assignment: pair index -> (hx, hy) relative to the tile origin
  int h_goff[HPT];  // global offset relative to tile_org (within a plane)
  int h_soff[HPT];  // offset inside a shared-memory plane, -1 = none
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
    h_goff[q] = (hy + wofs(t.y0 + hy, b.n[1])) * b.sx + hx + wofs(t.x0 + hx, b.n[0]);
    h_soff[q] = ok ? ((hy + R) * SW + (hx + XO)) : -1;
  }
  const int s_own = (ty + R) * SW + (tx * CPT + XO);  // row j of this thread: s_own + j * SW

  // copy of the ghosted plane p (relative to z0) of every differenced field into `slot`
  auto issue_plane = [&](int p, int slot) {
    P* const dst = planes + (size_t)slot * NF * PSZ;
    const long long po = zofs(p);
#pragma unroll
    for (int j = 0; j < RY; ++j)
      if (loader[j]) {
#pragma unroll
        for (int f = 0; f < NF; ++f) cp_async_16(dst + f * PSZ + s_own + j * SW, a.sten[f] + offl[j] + po);
      }
#pragma unroll
    for (int q = 0; q < HPT; ++q)
      if (h_soff[q] >= 0) {
#pragma unroll
        for (int f = 0; f < NF; ++f) cp_async_pair(dst + f * PSZ + h_soff[q], a.sten[f] + tile_org + po + h_goff[q]);
      }
  };
  // pointwise inputs of plane st into this thread's ring entries st % PD
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

  // prologue: centre planes 0..R-1, then stages 0..PD-1 (stage st = plane st+R and pointwise inputs of plane st);
  // planes above z0+nz+R-1 are never needed
  const int np = t.nz + R;  // planes 0 .. np-1 are copied
#pragma unroll
  for (int p = 0; p < R; ++p) issue_plane(p, p);
#pragma unroll
  for (int st = 0; st < PD; ++st) {
    if (st + R < np) issue_plane(st + R, (st + R) % S);
    if (st < t.nz) issue_pnt(st);
    cp_async_commit();
  }
  // lower 2R planes of the z-windows straight into registers
  V w[NF][RY][2 * R + 1];  // w[f][j][m] = field f, row j, plane z + m - R
#pragma unroll
  for (int f = 0; f < NF; ++f)
#pragma unroll
    for (int j = 0; j < RY; ++j)
#pragma unroll
      for (int m = 0; m < 2 * R; ++m)
        if (loader[j]) w[f][j][m + 1] = ldg16_keep<T>(a.sten[f] + offl[j] + zofs(m - R));

  int slot_c = 0;             // slot of the centre plane zz
  int slot_t = R % S;         // slot of plane zz + R
  int slot_n = (R + PD) % S;  // slot of plane zz + R + PD
  for (int zz = 0; zz < t.nz; ++zz) {
    cp_async_wait<PD - 1>();  // this thread's part of stage zz has landed ...
    __syncthreads();          // ... and everybody's; plane zz-1 is retired
    const P* const cb = planes + (size_t)slot_c * NF * PSZ;
    const P* const tb = planes + (size_t)slot_t * NF * PSZ;
    V pv[RY][NPA];
#pragma unroll
    for (int f = 0; f < NF; ++f)
#pragma unroll
      for (int j = 0; j < RY; ++j) {
#pragma unroll
        for (int m = 0; m < 2 * R; ++m) w[f][j][m] = w[f][j][m + 1];
        if (loader[j]) w[f][j][2 * R] = *reinterpret_cast<const V*>(tb + f * PSZ + s_own + j * SW);
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
    if (zz + PD + R < np) issue_plane(zz + PD + R, slot_n);
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
            if (i >= R && i < R + RY) col[i] = w[f][i - R][R].p[p];
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
                zm[r - 1] = comp(w[f][j][R - r].p[p]);
                zp[r - 1] = comp(w[f][j][R + r].p[p]);
              }
              lap[j][f][c] = lap_from<T, ORDER>(comp(w[f][j][R].p[p]), xm, xp, ym, yp, zm, zp, a.inv_h2);
            }
          }
        }
#pragma unroll
        for (int j = 0; j < RY; ++j) {
          P wc[NF], pc[NPA], opsi[NOUT], opi[NOUT];
#pragma unroll
          for (int f = 0; f < NF; ++f) wc[f] = w[f][j][R].p[p];
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
#pragma unroll
      for (int j = 0; j < RY; ++j)
        if (active[j]) {
          const long long oo = off + (long long)zz * plane + (long long)j * b.sx;
#pragma unroll
          for (int q = 0; q < NOUT; ++q) {
            stg16<T>(a.out_psi[q] + oo, o_psi[j][q]);
            stg16<T>(a.out_pi[q] + oo, o_pi[j][q]);
          }
        }
    }
    slot_c = slot_c + 1 == S ? 0 : slot_c + 1;
    slot_t = slot_t + 1 == S ? 0 : slot_t + 1;
    slot_n = slot_n + 1 == S ? 0 : slot_n + 1;
  }
}

}  // namespace sledge
