// Fused single-pass time step (the in-kernel analogue of the paper's enlarged-ghost idea,
// PAPER.md P:42): one launch reads p, vx, vy, vz of step n once and writes all four of step n+1 once
// (32 B/pt instead of the 48 B/pt of the two-kernel step), producing the same bits as update_v_tiled followed by
// update_p_tiled because every point goes through the same stag_diff / cpml_apply / upd sequence.
//
// The new pressure at a node needs the NEW velocities of its 8 neighbours per axis ("a pressure-to-velocity
// stencil update followed by a velocity-to-pressure stencil update"), and those need the OLD pressure 4 further out:
// a ghost of 2r = 8 cells per full step, exactly the paper's count.  Inside one GPU that ghost is
//   x, y : recomputed.  A 64x16 tile computes vx_new on 72x16 and vy_new on 64x23 points; the extra strips are done
//          by four "halo" warps, the tile itself by eight "main" warps, and the values meet in a double-buffered
//          shared-memory exchange (E) guarded by full/empty mbarriers;
//   z    : streamed.  Each main thread keeps p_old[m-7..m] and vz_new[k-4..k+3] of its four x-points in registers.
// Because neighbouring tiles re-read old values that the owner is about to overwrite, the step is out of place:
// state "in" -> state "out" (fields and psi), swapped by the host after every launch.
//
// Stage of ring iteration m (k = m-7 is the output plane, kz = m-4 the vz plane), all by TMA, OOB = 0 = wall (R4):
//   [ p box (TX+16)x(TY+14) of plane k | p tile of plane m | vz tile of plane kz | vx x-halo tile of plane k |
//     vy y-halo tile of plane k | Kc tile of plane k ]
#pragma once
#include "fdtd_kernels.cuh"

namespace fdtd {

constexpr int FW_MAIN = NT / 32;                 // 8 main warps: one float4 of the 64x16 tile per thread
constexpr int FW_HALO = 4;                       // one warpgroup: vy_new on rows y0-4..y0-1 and y0+TY..y0+TY+2 (7 x 16 float4
                                                 // units, two rows per warp) and, by its last warp, vx_new on the two 4-wide
                                                 // strips left/right of the tile (2 x 16 units)
constexpr int FNW = FW_MAIN + FW_HALO;           // 12 warps = 3 per SM sub-partition
constexpr int FNT = FNW * 32;                    // 384 threads
constexpr int F_REGS_MAIN = 216, F_REGS_HALO = 72;   // setmaxnreg split of the 3 x 168 registers per sub-partition lane
constexpr int FNS = 4;                           // TMA ring stages
constexpr int BW = TX + 16;                      // p box: columns x0-8 .. x0+TX+7
constexpr int BH = TY + 14;                      // p box: rows    y0-7 .. y0+TY+6
constexpr int EVY_ROWS = TY + 8;                 // vy_new exchange rows y0-4 .. y0+TY+3 (the last one is never read)
constexpr int F_PB_FLOATS = BW * BH;
constexpr int F_VX_FLOATS = HW * TY;
constexpr int F_VY_FLOATS = TX * PH;
constexpr int F_OFF_PT = F_PB_FLOATS;
constexpr int F_OFF_VZ = F_OFF_PT + TILE_FLOATS;
constexpr int F_OFF_VX = F_OFF_VZ + TILE_FLOATS;
constexpr int F_OFF_VY = F_OFF_VX + F_VX_FLOATS;
constexpr int F_OFF_KC = F_OFF_VY + F_VY_FLOATS;
constexpr int F_STAGE_FLOATS = F_OFF_KC + TILE_FLOATS;
constexpr int E_OFF_VY = F_VX_FLOATS;            // exchange buffer: [vx_new 16 x 72 | vy_new 24 x 64]
constexpr int E_FLOATS = F_VX_FLOATS + TX * EVY_ROWS;
constexpr int F_SMEM_BYTES = (FNS * F_STAGE_FLOATS + 2 * E_FLOATS) * 4;
static_assert((F_PB_FLOATS * 4) % 128 == 0 && (F_VX_FLOATS * 4) % 128 == 0 && (F_VY_FLOATS * 4) % 128 == 0 && (E_FLOATS * 4) % 128 == 0,
              "TMA destinations must stay 128-B aligned");

// The "out" state of a fused step (same layout as the DomainView's own arrays, which are the "in" state).
struct OutSet {
  float* f[4];
  float* psi[2][3][2];
};

struct FusedBars {
  uint64_t* full;     // [FNS] TMA stage landed
  uint64_t* empty;    // [FNS] every warp has read the stage
  uint64_t* efull;    // [2]   every warp has written its part of the exchange buffer
  uint64_t* eempty;   // [2]   every main warp has read the exchange buffer
};

__device__ __forceinline__ void warp_arrive(uint64_t* bar) {
  __syncwarp();
  if ((threadIdx.x & 31) == 0) mbar_arrive(bar);
}

__device__ __forceinline__ void fused_issue(const TMaps& tm, float* smem, uint64_t* full, unsigned slot, int m, int x0, int y0, int z0,
                                            bool has_kc) {
  const int k = m - 7;
  const bool vz = m >= z0, out = k >= z0;
  uint64_t* bar = &full[slot];
  float* st = smem + slot * F_STAGE_FLOATS;
  mbar_expect_tx(bar, TILE_BYTES + (vz ? TILE_BYTES : 0) +
                          (out ? (F_PB_FLOATS + F_VX_FLOATS + F_VY_FLOATS) * 4 + (has_kc ? TILE_BYTES : 0) : 0));
  tma_load_3d(st + F_OFF_PT, &tm.tile[0], bar, x0, y0, m);
  if (vz) tma_load_3d(st + F_OFF_VZ, &tm.tile[3], bar, x0, y0, m - 4);
  if (out) {
    tma_load_3d(st, &tm.p_box, bar, x0 - 8, y0 - 7, k);
    tma_load_3d(st + F_OFF_VX, &tm.vx_halo, bar, x0 - 4, y0, k);
    tma_load_3d(st + F_OFF_VY, &tm.vy_halo, bar, x0, y0 - 4, k);
    if (has_kc) tma_load_3d(st + F_OFF_KC, &tm.tile[4], bar, x0, y0, k);
  }
}

// ---- main warps: the tile's own points ------------------------------------------------------------------
__device__ __forceinline__ void fused_main(const DomainView& D, const OutSet& O, const float* smem, float* ebuf, const FusedBars& Q,
                                           unsigned it, unsigned eit, int x0, int y0, int z0, int z1) {
  const int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;
  const int i = x0 + 4 * tx, j = y0 + ty;
  const bool has_kc = D.kc != nullptr;
  const bool active = (i < D.nx) && (j < D.ny);
  const float B = D.b0;
  const float Bxy = active ? B : 0.f;
  const float Bx3 = (i + 3 + D.ox) == D.gn[0] - 1 ? 0.f : Bxy;           // pinned last half node (R3)
  const float By = (j + D.oy) == D.gn[1] - 1 ? 0.f : Bxy;
  const long long rowoff = (long long)j * D.pitch + i;
  long long goff = rowoff + (long long)z0 * D.plane;                     // plane k  (vx, vy, p)
  long long goffz = rowoff + (long long)(z0 - 4) * D.plane;              // plane kz (vz); first used at kz = z0-4
  const int boff = (ty + 7) * BW + 4 * tx + 8;                           // own float4 in the p box
  const int toff = ty * TX + 4 * tx;                                     // own float4 in a plain tile
  const int exo = ty * HW + 4 * tx + 4;                                  // own float4 in E.vx
  const int eyo = E_OFF_VY + (ty + 4) * TX + 4 * tx;                     // own float4 in E.vy
  const bool any_x = touches(D, 0, x0, x0 + TX), any_y = touches(D, 1, y0, y0 + TY);
  const int sx = (any_x && active) ? slab_side(D, 0, i) : -1;
  const int sy = (any_y && active) ? slab_side(D, 1, j) : -1;
  long long pox = sx >= 0 ? psi_index(D, 0, sx, i, j, z0) : 0;           // same offset in psi_v / psi_p, in / out
  long long poy = sy >= 0 ? psi_index(D, 1, sy, i, j, z0) : 0;
  const long long stride_px = sx >= 0 ? (long long)D.ny * D.ln[0][sx] : 0;
  const long long stride_py = sy >= 0 ? (long long)D.ln[1][sy] * D.pitch : 0;
  const int gi = i + D.ox, gj = j + D.oy;

  V4 q0 = zero4(), q1 = zero4(), q2 = zero4(), q3 = zero4(), q4 = zero4(), q5 = zero4(), q6 = zero4(), q7 = zero4();   // p_old[m-7 .. m]
  V4 w0 = zero4(), w1 = zero4(), w2 = zero4(), w3 = zero4(), w4 = zero4(), w5 = zero4(), w6 = zero4(), w7 = zero4();   // vz_new[kz-7 .. kz]

  for (int m = z0 - 7; m < z1 + 7; ++m, ++it) {
    const unsigned slot = it % FNS;
    const int k = m - 7, kz = m - 4;
    const bool out = k >= z0, hvz = m >= z0;
    const float* st = smem + slot * F_STAGE_FLOATS;
    // psi of the velocity family: issue the global loads before waiting on the tile
    V4 psx, psy, psz;
    const int szv = (hvz && active && kz >= 0 && kz < D.nz) ? slab_side(D, 2, kz) : -1;
    long long poz = 0;
    if (out && sx >= 0) psx = ldg4(D.psi[0][0][sx] + pox);
    if (out && sy >= 0) psy = ldg4(D.psi[0][1][sy] + poy);
    if (szv >= 0) { poz = psi_index(D, 2, szv, i, j, kz); psz = ldg4(D.psi[0][2][szv] + poz); }
    // ... and of the pressure family at plane k
    const int szp = (out && active) ? slab_side(D, 2, k) : -1;
    V4 ppx, ppy, ppz;
    long long pozp = 0;
    if (out && sx >= 0) ppx = ldg4(D.psi[1][0][sx] + pox);
    if (out && sy >= 0) ppy = ldg4(D.psi[1][1][sy] + poy);
    if (szp >= 0) { pozp = psi_index(D, 2, szp, i, j, k); ppz = ldg4(D.psi[1][2][szp] + pozp); }

    mbar_wait(&Q.full[slot], (it / FNS) & 1);
    q0 = q1; q1 = q2; q2 = q3; q3 = q4; q4 = q5; q5 = q6; q6 = q7; q7 = ld4(st + F_OFF_PT + toff);
    V4 dxv, dyv, vx4, vy4, vz4, kc4;
    if (out) {
      const float* row = st + boff;
      const V4 c = ld4(row);
      dxv = diff_x<true>(ld4(row - 4), c, ld4(row + 4));
      dyv = diff_8(ld4(row + BW), c, ld4(row + 2 * BW), ld4(row - BW), ld4(row + 3 * BW), ld4(row - 2 * BW), ld4(row + 4 * BW),
                   ld4(row - 3 * BW));
      vx4 = ld4(st + F_OFF_VX + exo);
      vy4 = ld4(st + F_OFF_VY + (ty + 4) * TX + 4 * tx);
      kc4 = has_kc ? ld4(st + F_OFF_KC + toff) : splat4(D.kc0);
    }
    if (hvz) vz4 = ld4(st + F_OFF_VZ + toff);
    warp_arrive(&Q.empty[slot]);

    const unsigned eb = eit & 1, eu = eit >> 1;
    float* E = ebuf + eb * E_FLOATS;
    if (out) {
      // ---- velocity sub-update at plane k
      if (any_x) {
        if (sx >= 0) {
          cpml4(dxv, psx, ldg4(D.tab[0][0][0] + gi), ldg4(D.tab[0][0][1] + gi), ldg4(D.tab[0][0][2] + gi));
          st4(O.psi[0][0][sx] + pox, psx);
        }
      }
      if (any_y) {
        if (sy >= 0) {
          cpml4s(dyv, psy, __ldg(D.tab[0][1][0] + gj), __ldg(D.tab[0][1][1] + gj), __ldg(D.tab[0][1][2] + gj));
          st4(O.psi[0][1][sy] + poy, psy);
        }
      }
      vx4.v[0] = upd(vx4.v[0], Bxy, dxv.v[0]); vx4.v[1] = upd(vx4.v[1], Bxy, dxv.v[1]);
      vx4.v[2] = upd(vx4.v[2], Bxy, dxv.v[2]); vx4.v[3] = upd(vx4.v[3], Bx3, dxv.v[3]);
#pragma unroll
      for (int e = 0; e < 4; ++e) vy4.v[e] = upd(vy4.v[e], By, dyv.v[e]);
      if (active) { st4(O.f[1] + goff, vx4); st4(O.f[2] + goff, vy4); }
      mbar_wait(&Q.eempty[eb], (eu & 1) ^ 1);            // the readers of two planes ago are done with this buffer
      st4(E + exo, vx4);
      st4(E + eyo, vy4);
      warp_arrive(&Q.efull[eb]);
    }
    if (hvz) {
      // ---- vz_new at kz+1/2 from p_old[kz-3 .. kz+4] = q0..q7
      V4 dzv = diff_8(q4, q3, q5, q2, q6, q1, q7, q0);
      const int gk = kz + D.oz;
      if (szv >= 0) {
        cpml4s(dzv, psz, __ldg(D.tab[0][2][0] + gk), __ldg(D.tab[0][2][1] + gk), __ldg(D.tab[0][2][2] + gk));
        if (kz >= z0 && kz < z1) st4(O.psi[0][2][szv] + poz, psz);      // lead-in / tail planes belong to another item
      }
      const float Bz = (kz < 0 || kz >= D.nz || gk == D.gn[2] - 1) ? 0.f : Bxy;
#pragma unroll
      for (int e = 0; e < 4; ++e) vz4.v[e] = upd(vz4.v[e], Bz, dzv.v[e]);
      if (active && kz >= z0 && kz < z1) st4(O.f[3] + goffz, vz4);
      w0 = w1; w1 = w2; w2 = w3; w3 = w4; w4 = w5; w5 = w6; w6 = w7; w7 = vz4;
      goffz += D.plane;
    }
    if (out) {
      // ---- pressure sub-update at plane k: vz_new[k-4 .. k+3] = w0..w7
      V4 dzp = diff_8(w4, w3, w5, w2, w6, w1, w7, w0);
      mbar_wait(&Q.efull[eb], eu & 1);
      const float* xr = E + exo;
      V4 dxp = diff_x<false>(ld4(xr - 4), vx4, ld4(xr + 4));
      const float* col = E + E_OFF_VY + ty * TX + 4 * tx;                 // row ty of E.vy <-> y = j-4
      V4 dyp = diff_8(vy4, ld4(col + 3 * TX), ld4(col + 5 * TX), ld4(col + 2 * TX), ld4(col + 6 * TX), ld4(col + TX), ld4(col + 7 * TX),
                      ld4(col));
      warp_arrive(&Q.eempty[eb]);
      if (any_x) {
        if (sx >= 0) {
          cpml4(dxp, ppx, ldg4(D.tab[1][0][0] + gi), ldg4(D.tab[1][0][1] + gi), ldg4(D.tab[1][0][2] + gi));
          st4(O.psi[1][0][sx] + pox, ppx);
          pox += stride_px;
        }
      }
      if (any_y) {
        if (sy >= 0) {
          cpml4s(dyp, ppy, __ldg(D.tab[1][1][0] + gj), __ldg(D.tab[1][1][1] + gj), __ldg(D.tab[1][1][2] + gj));
          st4(O.psi[1][1][sy] + poy, ppy);
          poy += stride_py;
        }
      }
      if (szp >= 0) {
        const int gk = k + D.oz;
        cpml4s(dzp, ppz, __ldg(D.tab[1][2][0] + gk), __ldg(D.tab[1][2][1] + gk), __ldg(D.tab[1][2][2] + gk));
        st4(O.psi[1][2][szp] + pozp, ppz);
      }
      V4 p4;
#pragma unroll
      for (int e = 0; e < 4; ++e) p4.v[e] = upd(q0.v[e], kc4.v[e], __fadd_rn(__fadd_rn(dxp.v[e], dyp.v[e]), dzp.v[e]));
      if (active) st4(O.f[0] + goff, p4);
      goff += D.plane;
      ++eit;
    }
  }
}

// ---- halo warps: the redundantly computed ghost of the tile, never stored to global memory ----------------
// Warp hw (0..3) computes vy_new on two of the rows y0-4..y0-1, y0+TY..y0+TY+2 (16 float4 units per row; the eighth
// row slot is idle); warp 3 also computes vx_new on the strips x0-4..x0-1 and x0+TX..x0+TX+3 (rows y0..y0+TY-1).
// Lane 0 of warp 0 is the TMA producer of the CTA.
__device__ __forceinline__ void fused_halo(const TMaps& tm, const DomainView& D, float* smem, float* ebuf, const FusedBars& Q, unsigned it,
                                           unsigned eit, int hw, int x0, int y0, int z0, int z1) {
  const int lane = threadIdx.x & 31;
  const bool has_kc = D.kc != nullptr;
  // vy unit of this lane
  const int r = 2 * hw + (lane >> 4), c = lane & 15;
  const int jy = r < 4 ? y0 - 4 + r : y0 + TY + (r - 4), iy = x0 + 4 * c;
  const bool used = r < 7;                                   // the row y0+TY+3 is never read
  const bool valid_y = used && jy >= 0 && jy < D.ny && iy < D.nx;
  const float Bvy = valid_y ? D.b0 : 0.f;
  const float By = (jy + D.oy) == D.gn[1] - 1 ? 0.f : Bvy;   // pinned last half node (R3)
  const int brow = r < 4 ? r + 3 : TY + 3 + r;               // row of y = jy in the p box
  const int boff_y = (used ? brow : 3) * BW + 4 * c + 8;
  const int rr = r < 4 ? r : TY + r;                         // row of y = jy in E.vy and in the vy y-halo tile
  const int eyo = rr * TX + 4 * c;
  const int sy = valid_y ? slab_side(D, 1, jy) : -1;
  long long poy = sy >= 0 ? psi_index(D, 1, sy, iy, jy, z0) : 0;
  const long long stride_py = sy >= 0 ? (long long)D.ln[1][sy] * D.pitch : 0;
  const int gj = jy + D.oy;
  // vx unit of this lane (warp 3 only)
  const bool do_x = hw == FW_HALO - 1;
  const int row = lane >> 1, side = lane & 1;
  const int xx = side ? x0 + TX : x0 - 4, jx = y0 + row;
  const bool valid_x = do_x && xx >= 0 && xx < D.nx && jx < D.ny;
  const float Bvx = valid_x ? D.b0 : 0.f;
  const float Bx3 = (xx + 3 + D.ox) == D.gn[0] - 1 ? 0.f : Bvx;
  const int boff_x = (row + 7) * BW + (side ? TX + 8 : 4);
  const int exo = row * HW + (side ? TX + 4 : 0);
  const int sx = valid_x ? slab_side(D, 0, xx) : -1;
  long long pox = sx >= 0 ? psi_index(D, 0, sx, xx, jx, z0) : 0;
  const long long stride_px = sx >= 0 ? (long long)D.ny * D.ln[0][sx] : 0;
  const int gi = xx + D.ox;
  const int m_begin = z0 - 7, m_end = z1 + 7;

  for (int m = m_begin; m < m_end; ++m, ++it) {
    const unsigned slot = it % FNS;
    const bool out = (m - 7) >= z0;
    // producer duty: refill the stage every warp released in the previous iteration
    if (hw == 0) {
      if (lane == 0 && m > m_begin && (m - 1 + FNS) < m_end) {
        const unsigned ps = (it - 1) % FNS;
        mbar_wait(&Q.empty[ps], ((it - 1) / FNS) & 1);
        fused_issue(tm, smem, Q.full, ps, m - 1 + FNS, x0, y0, z0, has_kc);
      }
      __syncwarp();
    }
    V4 psy, psx;
    if (out && sy >= 0) psy = ldg4(D.psi[0][1][sy] + poy);
    if (out && sx >= 0) psx = ldg4(D.psi[0][0][sx] + pox);
    const float* st = smem + slot * F_STAGE_FLOATS;
    mbar_wait(&Q.full[slot], (it / FNS) & 1);
    V4 dyv, vy4, dxv, vx4;
    if (out) {
      const float* rw = st + boff_y;
      dyv = diff_8(ld4(rw + BW), ld4(rw), ld4(rw + 2 * BW), ld4(rw - BW), ld4(rw + 3 * BW), ld4(rw - 2 * BW), ld4(rw + 4 * BW),
                   ld4(rw - 3 * BW));
      vy4 = ld4(st + F_OFF_VY + eyo);
      if (do_x) {
        const float* rx = st + boff_x;
        dxv = diff_x<true>(ld4(rx - 4), ld4(rx), ld4(rx + 4));
        vx4 = ld4(st + F_OFF_VX + exo);
      }
    }
    warp_arrive(&Q.empty[slot]);
    if (out) {
      if (sy >= 0) {
        cpml4s(dyv, psy, __ldg(D.tab[0][1][0] + gj), __ldg(D.tab[0][1][1] + gj), __ldg(D.tab[0][1][2] + gj));
        poy += stride_py;
      }
#pragma unroll
      for (int e = 0; e < 4; ++e) vy4.v[e] = upd(vy4.v[e], By, dyv.v[e]);
      if (do_x) {
        if (sx >= 0) {
          cpml4(dxv, psx, ldg4(D.tab[0][0][0] + gi), ldg4(D.tab[0][0][1] + gi), ldg4(D.tab[0][0][2] + gi));
          pox += stride_px;
        }
        vx4.v[0] = upd(vx4.v[0], Bvx, dxv.v[0]); vx4.v[1] = upd(vx4.v[1], Bvx, dxv.v[1]);
        vx4.v[2] = upd(vx4.v[2], Bvx, dxv.v[2]); vx4.v[3] = upd(vx4.v[3], Bx3, dxv.v[3]);
      }
      const unsigned eb = eit & 1, eu = eit >> 1;
      float* E = ebuf + eb * E_FLOATS;
      mbar_wait(&Q.eempty[eb], (eu & 1) ^ 1);
      st4(E + E_OFF_VY + eyo, vy4);
      if (do_x) st4(E + exo, vx4);
      warp_arrive(&Q.efull[eb]);
      ++eit;
    }
  }
}

__global__ void __launch_bounds__(FNT, 1) step_fused(const __grid_constant__ TMaps tm, const __grid_constant__ DomainView D,
                                                     const __grid_constant__ OutSet O, const __grid_constant__ Sched S) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  float* smem = reinterpret_cast<float*>(smem_raw);
  float* ebuf = smem + FNS * F_STAGE_FLOATS;
  __shared__ __align__(8) uint64_t bars[2 * FNS + 4];
  __shared__ int s_item;
  const FusedBars Q{bars, bars + FNS, bars + 2 * FNS, bars + 2 * FNS + 2};
  if (threadIdx.x == 0) {
#pragma unroll
    for (int s = 0; s < FNS; ++s) { mbar_init(&Q.full[s], 1); mbar_init(&Q.empty[s], FNW); }
    mbar_init(&Q.efull[0], FNW); mbar_init(&Q.efull[1], FNW);
    mbar_init(&Q.eempty[0], FW_MAIN); mbar_init(&Q.eempty[1], FW_MAIN);
    fence_barrier_init();
    if (blockIdx.x == 0) *S.other = 0u;
  }
  const int warp = threadIdx.x >> 5;
  unsigned it = 0, eit = 0;
  int x0, y0, z0, z1;
  // The two roles never share code after this point, so each is compiled against its own register budget: the two main
  // warpgroups take the registers the halo warpgroup gives up (3 warps per SM sub-partition: 2 x 216 + 72 <= 512).
  if (warp < FW_MAIN) {
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(F_REGS_MAIN));
    while (next_item(S, &s_item, x0, y0, z0, z1, D.nz)) {
      fused_main(D, O, smem, ebuf, Q, it, eit, x0, y0, z0, z1);
      it += z1 - z0 + 14;
      eit += z1 - z0;
    }
  } else {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(F_REGS_HALO));
    const bool has_kc = D.kc != nullptr;
    while (next_item(S, &s_item, x0, y0, z0, z1, D.nz)) {
      const int niter = z1 - z0 + 14;
      if (threadIdx.x == FW_MAIN * 32) {
#pragma unroll
        for (int s = 0; s < FNS; ++s)
          if (s < niter) fused_issue(tm, smem, Q.full, (it + s) % FNS, z0 - 7 + s, x0, y0, z0, has_kc);
      }
      fused_halo(tm, D, smem, ebuf, Q, it, eit, warp - FW_MAIN, x0, y0, z0, z1);
      it += niter;
      eit += z1 - z0;
    }
  }
}

}  // namespace fdtd
