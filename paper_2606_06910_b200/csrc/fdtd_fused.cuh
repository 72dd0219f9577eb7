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
//          shared-memory exchange (E, three buffers) guarded by one mbarrier per buffer;
//   z    : streamed.  Each main thread keeps p_old[k..k+7] and vz_new[k-4..k+3] of its four x-points in registers.
// Because neighbouring tiles re-read old values that the owner is about to overwrite, the step is out of place:
// state "in" -> state "out" (fields and psi), swapped by the host after every launch.
//
// Stage of ring iteration m (k = m-7 is the output plane, kz = m-4 the vz plane), all by TMA, OOB = 0 = wall (R4):
//   [ p box (TX+16)x(TY+14) of plane k | p tile of plane m | vz tile of plane kz | vx x-halo tile of plane k |
//     vy y-halo tile of plane k | Kc tile of plane k | HB: bx x-halo tile, by y-halo tile of plane k, bz tile of plane kz ]
// (HB = heterogeneous density: dt/(rho_bar dx) per half node, FDTD_DENSITY_ARRAY, reading R6.)
//
// Roles (one CTA of 512 threads per SM, registers redistributed with setmaxnreg):
//   warps 0-7   main     one float4 of the tile per thread; planes that cannot touch a z slab run an instantiation of the
//                        plane body without any z-slab code, items that touch no x / y slab one without x / y slab code
//   warps 8-11  halo     the recomputed ghost strips (never stored to global memory)
//   warps 12-15 producer lane 0 of warp 12 issues every TMA load and does nothing else (a lane that has just issued
//                        tensor copies sees its own shared-memory loads stall for about a thousand cycles)
#pragma once
#include "fdtd_kernels.cuh"

namespace fdtd {

constexpr int FW_MAIN = NT / 32;                 // 8 main warps
constexpr int FW_HALO = 4;                       // vy_new on rows y0-4..y0-1 and y0+TY..y0+TY+2 (7 x 16 float4 units, two rows
                                                 // per warp); the last warp also does vx_new on the two 4-wide strips
constexpr int FW_PROD = 4;                       // producer warpgroup (one working lane)
constexpr int FNW = FW_MAIN + FW_HALO;           // 12 consumer warps
constexpr int FNT = (FNW + FW_PROD) * 32;        // 512 threads = 4 warps per SM sub-partition
constexpr int F_REGS_MAIN = 200, F_REGS_HALO = 80, F_REGS_PROD = 32;   // 2 x 200 + 80 + 32 = 512 registers per sub-partition lane
constexpr int FNS = 4;                           // TMA ring stages
// Lead-in of an item (tile x z-chunk): before the first output plane z0 the rings need p_old[z0-7 .. z0+6] and
// vz_new[z0-4 .. z0+2].  A lead-in plane carries one or two 4-KB tiles, far less than a stage holds, and with one plane per
// stage the lead-in ran at the latency of four TMA round trips per four planes (980 cycles per plane, measured).  So the
// lead-in planes are batched: stage 0 of an item holds the seven p tiles of planes z0-7 .. z0-1, the next L2S stages hold L2P
// planes each of (p tile of plane m, vz tile of plane m-4 [, dt/(rho_bar dx) of vz]) for m = z0 .. z0+6.
template <int V> __host__ __device__ constexpr int f_lead2_planes() { return V == 1 ? 3 : 4; }      // planes per lead-in-2 stage
template <int V> __host__ __device__ constexpr int f_lead2_stages() { return V == 1 ? 3 : 2; }      // 3+3+1 or 4+3 planes
template <int V> __host__ __device__ constexpr int f_lead2_tiles() { return V == 1 ? 3 : 2; }       // tiles per lead-in-2 plane
template <int V> __host__ __device__ constexpr int f_lead() { return 1 + f_lead2_stages<V>(); } // stages before the first output plane
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
constexpr int F_OFF_BX = F_OFF_KC + TILE_FLOATS; // HB only
constexpr int F_OFF_BY = F_OFF_BX + F_VX_FLOATS;
constexpr int F_OFF_BZ = F_OFF_BY + F_VY_FLOATS;
// x / y slab psi of plane k through the stage (uniform density only: the density-array stage has no room for it):
// [psi_vx box PXW x TY | psi_px | psi_vy tile | psi_py tile] behind the 8 tiles a lead-in-2 stage holds
constexpr int F_OFF_PSXV = 8 * TILE_FLOATS, F_OFF_PSXP = F_OFF_PSXV + PXW * TY, F_OFF_PSYV = F_OFF_PSXP + PXW * TY, F_OFF_PSYP = F_OFF_PSYV + TILE_FLOATS;
static_assert(F_OFF_BX <= 8 * TILE_FLOATS && (PXW * TY * 4) % 128 == 0, "stage layout");
// kernel variant V: 0 = uniform density, x / y slab psi by global loads; 1 = density arrays (HB); 2 = uniform density, x / y
// slab psi through the stage (PT)
template <int V> __host__ __device__ constexpr int f_stage_floats() { return V == 1 ? F_OFF_BZ + TILE_FLOATS : (V == 2 ? F_OFF_PSYP + TILE_FLOATS : 8 * TILE_FLOATS); }
static_assert(8 * TILE_FLOATS <= f_stage_floats<0>() && 9 * TILE_FLOATS <= f_stage_floats<1>() && 8 * TILE_FLOATS <= f_stage_floats<2>(), "lead-in batches must fit a stage");
constexpr int E_OFF_VY = F_VX_FLOATS;            // exchange buffer: [vx_new 16 x 72 | vy_new 24 x 64]
constexpr int E_FLOATS = F_VX_FLOATS + TX * EVY_ROWS;
constexpr int E_BUFS = 3;                        // three exchange buffers: the halo warps may run two planes ahead of the main warps
template <int V> __host__ __device__ constexpr int f_smem_bytes() { return (FNS * f_stage_floats<V>() + E_BUFS * E_FLOATS) * 4; }
static_assert((F_PB_FLOATS * 4) % 128 == 0 && (F_VX_FLOATS * 4) % 128 == 0 && (F_VY_FLOATS * 4) % 128 == 0 && (E_FLOATS * 4) % 128 == 0,
              "TMA destinations must stay 128-B aligned");
static_assert(f_smem_bytes<1>() <= 227 * 1024 - 4096 && f_smem_bytes<2>() <= 227 * 1024 - 4096, "stage ring + exchange buffers + static shared memory must fit one SM");

// The "out" state of a fused step (same layout as the DomainView's own arrays, which are the "in" state).
struct OutSet {
  float* f[4];
  float* psi[2][3][2];
};

// CPML tables of the item's columns x0-4 .. x0+TX+3 and rows y0-4 .. y0+TY+3 in shared memory ([family][a, b, 1/kappa]).
constexpr int TCX = HW, TCY = TY + 8;
struct TabCache {
  float x[2][3][TCX];
  float y[2][3][TCY];
};
// filled by all consumer threads of the CTA after next_item, then a named barrier among them (the producer group is not in it)
__device__ __forceinline__ void fill_tab_cache(const DomainView& D, TabCache& T, int x0, int y0) {
  // block-uniform: nothing to do unless the tile or its ghost strips reach an x or y slab
  if (!(touches(D, 0, x0 - 4, x0 + TX + 4) || touches(D, 1, y0 - 4, y0 + TY + 4))) return;
  for (int t = threadIdx.x; t < 6 * TCX; t += FNW * 32) {
    const int col = t % TCX, ft = t / TCX;
    const int g = min(max(x0 - 4 + col + D.ox, 0), D.gn[0] - 1);
    T.x[ft / 3][ft % 3][col] = __ldg(D.tab[ft / 3][0][ft % 3] + g);
  }
  for (int t = threadIdx.x; t < 6 * TCY; t += FNW * 32) {
    const int row = t % TCY, ft = t / TCY;
    const int g = min(max(y0 - 4 + row + D.oy, 0), D.gn[1] - 1);
    T.y[ft / 3][ft % 3][row] = __ldg(D.tab[ft / 3][1][ft % 3] + g);
  }
  asm volatile("bar.sync 1, %0;" ::"n"(FNW * 32) : "memory");
}
struct FusedBars {
  uint64_t* full;     // [FNS] TMA stage landed
  uint64_t* empty;    // [FNS] every warp has read the stage
  uint64_t* efull;    // [E_BUFS] every warp has written its part of the exchange buffer
};

__device__ __forceinline__ void warp_arrive(uint64_t* bar) {
  __syncwarp();
  if ((threadIdx.x & 31) == 0) mbar_arrive(bar);
}

// Stage s of an item: s = 0 and 1 .. L2S are the batched lead-in stages, s >= f_lead() carries output plane k = z0 + s - f_lead().
template <int V>
__device__ __forceinline__ void fused_issue(const TMaps& tm, float* smem, uint64_t* full, unsigned slot, int s, int x0, int y0, int z0,
                                            bool has_kc, const DomainView& D) {
  constexpr bool HB = V == 1;
  constexpr int L2P = f_lead2_planes<V>(), L2S = f_lead2_stages<V>(), TPP = f_lead2_tiles<V>();
  uint64_t* bar = &full[slot];
  float* st = smem + slot * f_stage_floats<V>();
  if (s == 0) {
    mbar_expect_tx(bar, 7 * TILE_BYTES);
#pragma unroll
    for (int j = 0; j < 7; ++j) tma_load_3d(st + j * TILE_FLOATS, &tm.tile[0], bar, x0, y0, z0 - 7 + j);
    return;
  }
  if (s <= L2S) {
    const int m0 = z0 + (s - 1) * L2P, np = min(L2P, z0 + 7 - m0);
    mbar_expect_tx(bar, np * TPP * TILE_BYTES);
    for (int j = 0; j < np; ++j) {
      tma_load_3d(st + (TPP * j) * TILE_FLOATS, &tm.tile[0], bar, x0, y0, m0 + j);
      tma_load_3d(st + (TPP * j + 1) * TILE_FLOATS, &tm.tile[3], bar, x0, y0, m0 + j - 4);
      if (HB) tma_load_3d(st + (TPP * j + 2) * TILE_FLOATS, &tm.bq_tile, bar, x0, y0, m0 + j - 4);
    }
    return;
  }
  const int k = z0 + s - f_lead<V>(), m = k + 7;
  // the x / y slab this tile touches, if its psi goes through the stage (recomputed per stage from the kernel parameters: the
  // producer lane has 32 registers, and whatever it spills it reloads behind a tensor copy, at a thousand cycles a load)
  int sxt = -1, syt = -1;
  if (V == 2) {
#pragma unroll
    for (int side = 0; side < 2; ++side) {
      if (D.ln[0][side] > 0 && x0 < D.ls[0][side] + D.ln[0][side] && x0 + TX > D.ls[0][side]) sxt = side;
      if (D.ln[1][side] > 0 && y0 < D.ls[1][side] + D.ln[1][side] && y0 + TY > D.ls[1][side]) syt = side;
    }
  }
  mbar_expect_tx(bar, (HB ? 3 : 2) * TILE_BYTES + (F_PB_FLOATS + (HB ? 2 : 1) * (F_VX_FLOATS + F_VY_FLOATS)) * 4 + (has_kc ? TILE_BYTES : 0) +
                          (sxt >= 0 ? 2 * PXW * TY * 4 : 0) + (syt >= 0 ? 2 * TILE_BYTES : 0));
  if (V == 2 && sxt >= 0) {         // psi_vx, psi_px of plane k: the slab's columns from the tile's first one on, this tile's rows
    const int cx0 = max(x0, D.ls[0][sxt]) - D.ls[0][sxt];
    tma_load_3d(st + F_OFF_PSXV, &tm.psi_x[0][sxt], bar, cx0, y0, k);
    tma_load_3d(st + F_OFF_PSXP, &tm.psi_x[1][sxt], bar, cx0, y0, k);
  }
  if (V == 2 && syt >= 0) {         // psi_vy, psi_py of plane k: this tile's columns, 16 slab rows from the tile's first row (outside the slab: zero fill)
    const int cy0 = y0 - D.ls[1][syt];
    tma_load_3d(st + F_OFF_PSYV, &tm.psi_y[0][syt], bar, x0, cy0, k);
    tma_load_3d(st + F_OFF_PSYP, &tm.psi_y[1][syt], bar, x0, cy0, k);
  }
  tma_load_3d(st + F_OFF_PT, &tm.tile[0], bar, x0, y0, m);
  tma_load_3d(st + F_OFF_VZ, &tm.tile[3], bar, x0, y0, m - 4);
  if (HB) tma_load_3d(st + F_OFF_BZ, &tm.bq_tile, bar, x0, y0, m - 4);
  tma_load_3d(st, &tm.p_box, bar, x0 - 8, y0 - 7, k);
  tma_load_3d(st + F_OFF_VX, &tm.vx_halo, bar, x0 - 4, y0, k);
  tma_load_3d(st + F_OFF_VY, &tm.vy_halo, bar, x0, y0 - 4, k);
  if (has_kc) tma_load_3d(st + F_OFF_KC, &tm.tile[4], bar, x0, y0, k);
  if (HB) {
    tma_load_3d(st + F_OFF_BX, &tm.bq_halo[0], bar, x0 - 4, y0, k);
    tma_load_3d(st + F_OFF_BY, &tm.bq_halo[1], bar, x0, y0 - 4, k);
  }
}

// ---- main warps: the tile's own points ------------------------------------------------------------------
// Everything a main thread keeps over one item.  The two z queues are arrays that are only ever indexed with
// compile-time constants, so they live in registers.
// XS / YS: 0 = the item touches no x / y slab, 1 = psi by global loads one plane ahead, 2 = psi through the TMA stage
template <int XS, int YS>
struct MainState {
  V4 pq[8];                 // p_old ring:  logical entry n (after the push of plane k) = p_old[k+n]
  V4 wq[8];                 // vz_new ring: logical entry n (after the push of plane k) = vz_new[k-4+n]
  long long goff;           // element offset of this thread's float4 in plane k of a field
  long long pox, poy;       // element offsets of plane k in the x / y slab psi arrays
  V4 nvx, npx, nvy, npy;    // psi_v / psi_p of plane k, loaded one iteration ahead (XS / YS items)
  V4 nvz, npz;              // psi_vz of plane k+3 and psi_pz of plane k, loaded one iteration ahead (planes in a z slab)
  unsigned it, eit;
  bool pre;                 // the next stage's "full" phase was already seen complete by an early probe
};

// per-item constants of a main thread
struct MainK {
  int boff, toff, exo;      // own float4 (float offsets) in the p box, in a plain tile, in an x-halo tile (vx, E.vx, bx)
  int tx, ty;
  int z1, zv_end;           // last output plane + 1; vz planes >= zv_end belong to the next z chunk
  int zl, zh;               // z slabs: local planes [0, zl) and [zh, nz)
  int kz_pin;               // vz planes >= kz_pin take a zero update coefficient (pinned last half node R3, and planes above the grid)
  float B, By, kc0;
  int pinx;                 // element of this thread's float4 that is the pinned last half node of x (R3), 4: none
  int psxo;                 // own float4 in the staged x-slab psi box (XS == 2)
  bool active, in_x, in_y, has_kc;
  int sxs, sys;             // slab side (0 / 1) of this thread's columns / row when in_x / in_y
  long long stride_px, stride_py, zrow;
  const float* psi_in[2][2];   // [family][0 = x slab, 1 = y slab] of the slab side this thread lies in (in state)
  float* psi_out[2][2];
};

// vz_new[kz] from the p ring (a0..a7 = p_old[kz-3 .. kz+4]); CPML in the z slabs; stored if this item owns the plane.
// z slab planes of local index v (0 <= v < nz): [0, zl) and [zh, nz)
__device__ __forceinline__ bool in_z_slab(const DomainView& D, const MainK& K, int v) {
  return (unsigned)(v - K.zl) >= (unsigned)(K.zh - K.zl) && (unsigned)v < (unsigned)D.nz;
}
// psi of the z slab (family fam) at plane v for this thread's float4, or zeros outside the slabs / for inactive threads
__device__ __forceinline__ V4 load_psi_z(const DomainView& D, const MainK& K, int fam, int v) {
  if (!(in_z_slab(D, K, v) && K.active)) return zero4();
  const int sz = v < K.zl ? 0 : 1;
  return ldg4(D.psi[fam][2][sz] + (long long)(v - D.ls[2][sz]) * D.plane + K.zrow);
}
constexpr int F_ZPF = 3;   // planes ahead of the register load that the z-slab psi lines are pulled into L2 (0.4 - 0.9 % of the step)
__device__ __forceinline__ void prefetch_psi_z(const DomainView& D, const MainK& K, int fam, int v) {
  if (!(in_z_slab(D, K, v) && K.active)) return;
  const int sz = v < K.zl ? 0 : 1;
  prefetch_l2(D.psi[fam][2][sz] + (long long)(v - D.ls[2][sz]) * D.plane + K.zrow);
}
template <int V, bool ZS, bool PRE>
__device__ __forceinline__ V4 fused_vz(const DomainView& D, const OutSet& O, const MainK& K, const V4& a0, const V4& a1, const V4& a2,
                                       const V4& a3, const V4& a4, const V4& a5, const V4& a6, const V4& a7, V4 vz4, const V4& bz4, int kz,
                                       long long goff_kz, bool own, const V4& psz_pre) {
  constexpr bool HB = V == 1;
  V4 dzv = diff_8(a4, a3, a5, a2, a6, a1, a7, a0);
  if (ZS && (unsigned)(kz - K.zl) >= (unsigned)(K.zh - K.zl) && (unsigned)kz < (unsigned)D.nz) {   // block-uniform: z slab
    const int sz = kz < K.zl ? 0 : 1;
    const long long poz = (long long)(kz - D.ls[2][sz]) * D.plane + K.zrow;
    const int gk = kz + D.oz;
    const float ta = __ldg(D.tab[0][2][0] + gk), tb = __ldg(D.tab[0][2][1] + gk), tk = __ldg(D.tab[0][2][2] + gk);
    V4 psz = PRE ? psz_pre : (K.active ? ldg4(D.psi[0][2][sz] + poz) : zero4());
    cpml4s(dzv, psz, ta, tb, tk);
    if (own) st4(O.psi[0][2][sz] + poz, psz);
  }
  if (HB) {
    const bool pin = (unsigned)kz >= (unsigned)K.kz_pin;             // also planes below the grid (kz < 0): v outside is 0 (R4)
#pragma unroll
    for (int e = 0; e < 4; ++e) vz4.v[e] = upd(vz4.v[e], pin ? 0.f : bz4.v[e], dzv.v[e]);
  } else {
    const float Bz = (unsigned)kz >= (unsigned)K.kz_pin ? 0.f : K.B;
    vz4 = upd4(vz4, Bz, Bz, Bz, dzv);
  }
  if (own) st4(O.f[3] + goff_kz, vz4);
  return vz4;
}

// One steady-state iteration: output plane k (m = k+7, kz = k+3).  R = position of the oldest ring entry on entry.
// ZS = this plane or its vz plane may lie in a z slab (the lean instantiation carries no z-slab code at all).
template <int R, bool ZS, int XS, int YS, int V>
__device__ __forceinline__ void fused_plane(const DomainView& D, const OutSet& O, const float* smem, float* ebuf, const FusedBars& Q,
                                            const TabCache& T, const MainK& K, MainState<XS, YS>& C, int k) {
  constexpr bool HB = V == 1;
#define PQ(n) C.pq[(R + 1 + (n)) & 7]
#define WQ(n) C.wq[(R + 1 + (n)) & 7]
  const unsigned slot = C.it % FNS;
  const float* st = smem + slot * f_stage_floats<V>();
  // psi of plane k arrived during the previous iteration; start the loads of plane k+1 now
  V4 psx, psy, ppx, ppy;
  if (XS == 1) {
    psx = C.nvx; ppx = C.npx;
    if (K.in_x && k + 1 < K.z1) { C.nvx = ldg4(K.psi_in[0][0] + C.pox + K.stride_px); C.npx = ldg4(K.psi_in[1][0] + C.pox + K.stride_px); }
  }
  if (YS == 1) {
    psy = C.nvy; ppy = C.npy;
    if (K.in_y && k + 1 < K.z1) { C.nvy = ldg4(K.psi_in[0][1] + C.poy + K.stride_py); C.npy = ldg4(K.psi_in[1][1] + C.poy + K.stride_py); }
  }
  // z slabs: psi_vz of plane k+3 and psi_pz of plane k arrived during the previous iteration; start those of the next plane
  V4 psz, ppz;
  if (ZS) {
    psz = C.nvz; ppz = C.npz;
    C.nvz = load_psi_z(D, K, 0, k + 4);
    C.npz = load_psi_z(D, K, 1, k + 1);
    prefetch_psi_z(D, K, 0, k + 4 + F_ZPF);      // ... and pull the lines of a few planes further on into L2
    prefetch_psi_z(D, K, 1, k + 1 + F_ZPF);
  }
  if (!C.pre) mbar_wait(&Q.full[slot], (C.it / FNS) & 1);
  C.pq[R] = ld4(st + F_OFF_PT + K.toff);                         // newest p_old plane k+7 replaces p_old[k-1]
  const float* row = st + K.boff;
  const V4 c = ld4(row);
  V4 dxv = diff_x<true>(ld4(row - 4), c, ld4(row + 4));
  V4 dyv = diff_8(ld4(row + BW), c, ld4(row + 2 * BW), ld4(row - BW), ld4(row + 3 * BW), ld4(row - 2 * BW), ld4(row + 4 * BW),
                  ld4(row - 3 * BW));
  V4 vx4 = ld4(st + F_OFF_VX + K.exo);
  V4 vy4 = ld4(st + F_OFF_VY + 4 * TX + K.toff);
  V4 vz4 = ld4(st + F_OFF_VZ + K.toff);
  const V4 kc4 = K.has_kc ? ld4(st + F_OFF_KC + K.toff) : splat4(K.kc0);
  V4 bx4, by4, bz4;
  if (HB) { bx4 = ld4(st + F_OFF_BX + K.exo); by4 = ld4(st + F_OFF_BY + 4 * TX + K.toff); bz4 = ld4(st + F_OFF_BZ + K.toff); }
  if (XS == 2 && K.in_x) { psx = ld4(st + F_OFF_PSXV + K.psxo); ppx = ld4(st + F_OFF_PSXP + K.psxo); }
  if (YS == 2 && K.in_y) { psy = ld4(st + F_OFF_PSYV + K.toff); ppy = ld4(st + F_OFF_PSYP + K.toff); }
  warp_arrive(&Q.empty[slot]);

  // ---- velocity sub-update at plane k
  if (XS) {
    if (K.in_x) {
      cpml4(dxv, psx, ld4(T.x[0][0] + 4 + 4 * K.tx), ld4(T.x[0][1] + 4 + 4 * K.tx), ld4(T.x[0][2] + 4 + 4 * K.tx));
      st4(K.psi_out[0][0] + C.pox, psx);
    }
  }
  if (YS) {
    if (K.in_y) {
      cpml4s(dyv, psy, T.y[0][0][4 + K.ty], T.y[0][1][4 + K.ty], T.y[0][2][4 + K.ty]);
      st4(K.psi_out[0][1] + C.poy, psy);
    }
  }
  if (HB) {
#pragma unroll
    for (int e = 0; e < 4; ++e) {
      vx4.v[e] = upd(vx4.v[e], e >= K.pinx ? 0.f : bx4.v[e], dxv.v[e]);
      vy4.v[e] = upd(vy4.v[e], K.By == 0.f ? 0.f : by4.v[e], dyv.v[e]);
    }
  } else {
    vx4 = upd4_pin(vx4, K.B, K.pinx, dxv);
    vy4 = upd4(vy4, K.By, K.By, K.By, dyv);
  }
  if (K.active) { st4(O.f[1] + C.goff, vx4); st4(O.f[2] + C.goff, vy4); }
  const unsigned eb = C.eit % E_BUFS;
  float* E = ebuf + eb * E_FLOATS;
  // this buffer was last read for plane eit-3, and every main warp is at most one plane away from this one
  st4(E + K.exo, vx4);
  st4(E + E_OFF_VY + 4 * TX + K.toff, vy4);
  warp_arrive(&Q.efull[eb]);

  // ---- vz_new at kz+1/2 from p_old[kz-3 .. kz+4], then D-_z of the new vz ring
  C.wq[R] = fused_vz<V, ZS, true>(D, O, K, PQ(0), PQ(1), PQ(2), PQ(3), PQ(4), PQ(5), PQ(6), PQ(7), vz4, bz4, k + 3, C.goff + 3 * D.plane,
                               K.active && k < K.zv_end, psz);
  V4 dzp = diff_8(WQ(4), WQ(3), WQ(5), WQ(2), WQ(6), WQ(1), WQ(7), WQ(0));
  const bool pz = ZS && (unsigned)(k - K.zl) >= (unsigned)(K.zh - K.zl);    // block-uniform: plane k lies in a z slab
  const int szp = k < K.zl ? 0 : 1;
  const long long pozp = pz ? (long long)(k - D.ls[2][szp]) * D.plane + K.zrow : 0;

  // ---- pressure sub-update at plane k
  C.pre = mbar_test(&Q.full[(C.it + 1) % FNS], ((C.it + 1) / FNS) & 1);      // probe the next stage now, use the answer next iteration
  mbar_wait(&Q.efull[eb], (C.eit / E_BUFS) & 1);
  const float* xr = E + K.exo;
  V4 dxp = diff_x<false>(ld4(xr - 4), vx4, ld4(xr + 4));
  const float* col = E + E_OFF_VY + K.toff;                       // row ty of E.vy <-> y = j-4
  V4 dyp = diff_8(vy4, ld4(col + 3 * TX), ld4(col + 5 * TX), ld4(col + 2 * TX), ld4(col + 6 * TX), ld4(col + TX), ld4(col + 7 * TX),
                  ld4(col));
  if (XS) {
    if (K.in_x) {
      cpml4(dxp, ppx, ld4(T.x[1][0] + 4 + 4 * K.tx), ld4(T.x[1][1] + 4 + 4 * K.tx), ld4(T.x[1][2] + 4 + 4 * K.tx));
      st4(K.psi_out[1][0] + C.pox, ppx);
      C.pox += K.stride_px;
    }
  }
  if (YS) {
    if (K.in_y) {
      cpml4s(dyp, ppy, T.y[1][0][4 + K.ty], T.y[1][1][4 + K.ty], T.y[1][2][4 + K.ty]);
      st4(K.psi_out[1][1] + C.poy, ppy);
      C.poy += K.stride_py;
    }
  }
  if (pz) {
    const int gk = k + D.oz;
    cpml4s(dzp, ppz, __ldg(D.tab[1][2][0] + gk), __ldg(D.tab[1][2][1] + gk), __ldg(D.tab[1][2][2] + gk));
    if (K.active) st4(O.psi[1][2][szp] + pozp, ppz);
  }
  const float2 s0 = __fadd2_rn(__fadd2_rn(lo2(dxp), lo2(dyp)), lo2(dzp)), s1 = __fadd2_rn(__fadd2_rn(hi2(dxp), hi2(dyp)), hi2(dzp));
  const V4 p4 = join2(mad2(pk(-kc4.v[0], -kc4.v[1]), s0, lo2(PQ(0))), mad2(pk(-kc4.v[2], -kc4.v[3]), s1, hi2(PQ(0))));
  if (K.active) st4(O.f[0] + C.goff, p4);
  C.goff += D.plane;
  ++C.it; ++C.eit;
#undef PQ
#undef WQ
}

// Planes [k, kend) of an item.  Both rings stay in canonical order (oldest entry at index 0): they are shifted by one entry
// per plane (56 register moves).  Renaming instead of moving needs the body unrolled 8x (or 4x / 2x with a rotation per
// group), and every unrolled form measured slower than this one (8x: 2.06 instead of 1.44 ms at 552^3, 4x: 1.51, 2x: 1.50):
// the body must stay resident in the instruction cache, and the kernel is not bound by issue slots.  Re-measured on the final
// build of round 2: the 2x form has 8.6 % fewer instructions per plane and is 6 % slower at 1600^3 (profiles/r02_ncu_step_fused.md).
template <bool ZS, int XS, int YS, int V>
__device__ __forceinline__ void fused_run(const DomainView& D, const OutSet& O, const float* smem, float* ebuf, const FusedBars& Q,
                                          const TabCache& T, const MainK& K, MainState<XS, YS>& C, int k, int kend) {
  if (ZS && k < kend) { C.nvz = load_psi_z(D, K, 0, k + 3); C.npz = load_psi_z(D, K, 1, k); }
  for (; k < kend; ++k) {
#pragma unroll
    for (int n = 0; n < 7; ++n) { C.pq[n] = C.pq[n + 1]; C.wq[n] = C.wq[n + 1]; }
    fused_plane<7, ZS, XS, YS, V>(D, O, smem, ebuf, Q, T, K, C, k);       // writes the newest entries at index 7
  }
}

template <int XS, int YS, int V>
__device__ __forceinline__ void fused_main_item(const DomainView& D, const OutSet& O, const float* smem, float* ebuf, const FusedBars& Q,
                                             const TabCache& T, unsigned& it_io, unsigned& eit_io, int x0, int y0, int z0, int z1) {
  constexpr bool HB = V == 1;
  const int tid = threadIdx.x;
  MainK K;
  K.tx = tid & 15; K.ty = tid >> 4;
  const int i = x0 + 4 * K.tx, j = y0 + K.ty;
  K.z1 = z1; K.zv_end = z1 - 3;
  K.has_kc = D.kc != nullptr;
  K.kc0 = D.kc0;
  K.active = (i < D.nx) && (j < D.ny);
  K.B = K.active ? D.b0 : 0.f;
  K.pinx = pinned_x_element(i + D.ox, D.gn[0]);
  K.By = (j + D.oy) == D.gn[1] - 1 ? 0.f : (HB ? 1.f : K.B);
  K.kz_pin = min(D.gn[2] - 1 - D.oz, D.nz);
  K.zrow = (long long)j * D.pitch + i;
  K.boff = (K.ty + 7) * BW + 4 * K.tx + 8;
  K.toff = K.ty * TX + 4 * K.tx;
  K.exo = K.ty * HW + 4 * K.tx + 4;
  K.zl = D.ln[2][0];                                                // low z slab = local planes [0, zl)
  K.zh = D.ln[2][1] > 0 ? D.ls[2][1] : 0x3fffffff;                  // high z slab = local planes [zh, nz)
  const int sx = (XS && K.active) ? slab_side(D, 0, i) : -1;
  const int sy = (YS && K.active) ? slab_side(D, 1, j) : -1;
  K.in_x = sx >= 0; K.in_y = sy >= 0;
  K.sxs = max(sx, 0); K.sys = max(sy, 0);
  K.psxo = K.in_x ? K.ty * PXW + (i - max(x0, D.ls[0][K.sxs])) : 0;
  K.stride_px = K.in_x ? (long long)D.ny * D.ln[0][K.sxs] : 0;
  K.stride_py = K.in_y ? (long long)D.ln[1][K.sys] * D.pitch : 0;
#pragma unroll
  for (int fam = 0; fam < 2; ++fam) {
    K.psi_in[fam][0] = D.psi[fam][0][K.sxs]; K.psi_out[fam][0] = O.psi[fam][0][K.sxs];
    K.psi_in[fam][1] = D.psi[fam][1][K.sys]; K.psi_out[fam][1] = O.psi[fam][1][K.sys];
  }
  MainState<XS, YS> C;
  C.it = it_io; C.eit = eit_io; C.pre = false;
  C.pox = K.in_x ? psi_index(D, 0, K.sxs, i, j, z0) : 0;
  C.poy = K.in_y ? psi_index(D, 1, K.sys, i, j, z0) : 0;
  C.goff = K.zrow + (long long)z0 * D.plane;
#pragma unroll
  for (int n = 0; n < 8; ++n) { C.pq[n] = zero4(); C.wq[n] = zero4(); }
  constexpr int SF = f_stage_floats<V>();
  // lead-in stage 0: the seven p tiles of planes z0-7 .. z0-1 fill the ring (entry 0 stays zero: it is the one shifted out first)
  {
    const unsigned slot = C.it % FNS;
    mbar_wait(&Q.full[slot], (C.it / FNS) & 1);
    const float* st = smem + slot * SF + K.toff;
#pragma unroll
    for (int j = 0; j < 7; ++j) C.pq[j + 1] = ld4(st + j * TILE_FLOATS);
    warp_arrive(&Q.empty[slot]);
    ++C.it;
  }
  // lead-in stages 1 .. L2S: planes m = z0 .. z0+6 also produce vz_new[z0-4 .. z0+2] (the first four belong to the z chunk below)
  {
    constexpr int L2P = f_lead2_planes<V>(), L2S = f_lead2_stages<V>(), TPP = f_lead2_tiles<V>();
    int m = z0;
    for (int b = 0; b < L2S; ++b, ++C.it) {
      const unsigned slot = C.it % FNS;
      mbar_wait(&Q.full[slot], (C.it / FNS) & 1);
      const float* st = smem + slot * SF + K.toff;
#pragma unroll
      for (int j = 0; j < L2P; ++j) {
        if (m < z0 + 7) {                                              // block-uniform
          const V4 v = ld4(st + (TPP * j) * TILE_FLOATS);
          V4 vz4 = ld4(st + (TPP * j + 1) * TILE_FLOATS);
          V4 bz4;
          if (HB) bz4 = ld4(st + (TPP * j + 2) * TILE_FLOATS);
#pragma unroll
          for (int n = 0; n < 7; ++n) C.pq[n] = C.pq[n + 1];
          C.pq[7] = v;
          const int kz = m - 4;                                        // planes z0 .. z0+2 are this item's own
          vz4 = fused_vz<V, true, false>(D, O, K, C.pq[0], C.pq[1], C.pq[2], C.pq[3], C.pq[4], C.pq[5], C.pq[6], C.pq[7], vz4, bz4, kz,
                                    K.zrow + (long long)kz * D.plane, K.active && kz >= z0 && kz < z1, vz4);
#pragma unroll
          for (int n = 0; n < 7; ++n) C.wq[n] = C.wq[n + 1];
          C.wq[7] = vz4;
          ++m;
        }
      }
      warp_arrive(&Q.empty[slot]);
    }
    C.pre = false;
  }
  // now pq[n] = p_old[z0-1+n], wq[n] = vz_new[z0-5+n]: entry 0 of both rings is the oldest
  if (XS == 1 && K.in_x) { C.nvx = ldg4(K.psi_in[0][0] + C.pox); C.npx = ldg4(K.psi_in[1][0] + C.pox); }
  if (YS == 1 && K.in_y) { C.nvy = ldg4(K.psi_in[0][1] + C.poy); C.npy = ldg4(K.psi_in[1][1] + C.poy); }
  // z range of the item = [z0, za) + [za, zb) + [zb, z1): only the outer two can touch a z slab (plane k or vz plane k+3)
  const int za = min(max(K.zl, z0), z1), zb = min(max(K.zh - 3, za), z1);
  fused_run<true, XS, YS, V>(D, O, smem, ebuf, Q, T, K, C, z0, za);
  fused_run<false, XS, YS, V>(D, O, smem, ebuf, Q, T, K, C, za, zb);
  fused_run<true, XS, YS, V>(D, O, smem, ebuf, Q, T, K, C, zb, z1);
  it_io = C.it; eit_io = C.eit;
}

// ---- halo warps: the redundantly computed ghost of the tile, never stored to global memory ----------------
// Warp hw (0..3) computes vy_new on two of the rows y0-4..y0-1, y0+TY..y0+TY+2 (16 float4 units per row; the eighth
// row slot is idle); warp 3 also computes vx_new on the strips x0-4..x0-1 and x0+TX..x0+TX+3 (rows y0..y0+TY-1).
template <int V>
__device__ __forceinline__ void fused_halo(const DomainView& D, float* smem, float* ebuf, const FusedBars& Q, const TabCache& T, unsigned it,
                                           unsigned eit, int hw, int x0, int y0, int z0, int z1) {
  constexpr bool HB = V == 1;
  const int lane = threadIdx.x & 31;
  constexpr int SF = f_stage_floats<V>();
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
  // vx unit of this lane (warp 3 only)
  const bool do_x = hw == FW_HALO - 1;
  const int row = lane >> 1, side = lane & 1;
  const int xx = side ? x0 + TX : x0 - 4, jx = y0 + row;
  const bool valid_x = do_x && xx >= 0 && xx < D.nx && jx < D.ny;
  const float Bvx = valid_x ? D.b0 : 0.f;
  const int pinx = pinned_x_element(xx + D.ox, D.gn[0]);
  const int boff_x = (row + 7) * BW + (side ? TX + 8 : 4);
  const int exo = row * HW + (side ? TX + 4 : 0);
  const int sx = valid_x ? slab_side(D, 0, xx) : -1;
  long long pox = sx >= 0 ? psi_index(D, 0, sx, xx, jx, z0) : 0;
  const long long stride_px = sx >= 0 ? (long long)D.ny * D.ln[0][sx] : 0;
  const int xcol = side ? TX + 4 : 0;                        // the strip's first column in the table cache
  const int m_begin = z0 + 7 - f_lead<V>(), m_end = z1 + 7;      // the first f_lead() stages are the batched lead-in: wait and release only
  V4 npsy = zero4(), npsx = zero4();
  if (sy >= 0) npsy = ldg4(D.psi[0][1][sy] + poy);
  if (sx >= 0) npsx = ldg4(D.psi[0][0][sx] + pox);

  for (int m = m_begin; m < m_end; ++m, ++it) {
    const unsigned slot = it % FNS;
    const bool out = (m - 7) >= z0;
    // psi of the ghost strips, loaded one plane ahead (the halo warps have about one plane of slack, which an unhidden
    // DRAM latency per plane would use up in every slab item)
    V4 psy = npsy, psx = npsx;
    if (out && (m - 7) + 1 < z1) {
      if (sy >= 0) npsy = ldg4(D.psi[0][1][sy] + poy + stride_py);
      if (sx >= 0) npsx = ldg4(D.psi[0][0][sx] + pox + stride_px);
    }
    const float* st = smem + slot * SF;
    mbar_wait(&Q.full[slot], (it / FNS) & 1);
    V4 dyv, vy4, dxv, vx4, by4, bx4;
    if (out) {
      const float* rw = st + boff_y;
      dyv = diff_8(ld4(rw + BW), ld4(rw), ld4(rw + 2 * BW), ld4(rw - BW), ld4(rw + 3 * BW), ld4(rw - 2 * BW), ld4(rw + 4 * BW),
                   ld4(rw - 3 * BW));
      vy4 = ld4(st + F_OFF_VY + eyo);
      if (HB) by4 = ld4(st + F_OFF_BY + eyo);
      if (do_x) {
        const float* rx = st + boff_x;
        dxv = diff_x<true>(ld4(rx - 4), ld4(rx), ld4(rx + 4));
        vx4 = ld4(st + F_OFF_VX + exo);
        if (HB) bx4 = ld4(st + F_OFF_BX + exo);
      }
    }
    warp_arrive(&Q.empty[slot]);
    if (out) {
      if (sy >= 0) {
        cpml4s(dyv, psy, T.y[0][0][rr], T.y[0][1][rr], T.y[0][2][rr]);
        poy += stride_py;
      }
      if (HB) {
#pragma unroll
        for (int e = 0; e < 4; ++e) vy4.v[e] = upd(vy4.v[e], By == 0.f ? 0.f : by4.v[e], dyv.v[e]);
      } else {
        vy4 = upd4(vy4, By, By, By, dyv);
      }
      if (do_x) {
        if (sx >= 0) {
          cpml4(dxv, psx, ld4(T.x[0][0] + xcol), ld4(T.x[0][1] + xcol), ld4(T.x[0][2] + xcol));
          pox += stride_px;
        }
        if (HB) {
#pragma unroll
          for (int e = 0; e < 4; ++e) vx4.v[e] = upd(vx4.v[e], (Bvx == 0.f || e >= pinx) ? 0.f : bx4.v[e], dxv.v[e]);
        } else {
          vx4 = upd4_pin(vx4, Bvx, pinx, dxv);
        }
      }
      const unsigned eb = eit % E_BUFS;
      float* E = ebuf + eb * E_FLOATS;
      // this buffer was last read for plane eit-3; every main warp is past that once the efull phase of plane eit-2 is
      // complete (a main warp arrives there only after it has finished reading the plane before), so the halo warps can
      // run up to two planes ahead and their psi / stage latencies stay off the main warps' critical path
      if (eit > 1) mbar_wait(&Q.efull[(eit - 2) % E_BUFS], ((eit - 2) / E_BUFS) & 1);
      st4(E + E_OFF_VY + eyo, vy4);
      if (do_x) st4(E + exo, vx4);
      warp_arrive(&Q.efull[eb]);
      ++eit;
    }
  }
}

template <int V>
__global__ void __launch_bounds__(FNT, 1) step_fused(const __grid_constant__ TMaps tm, const __grid_constant__ DomainView D,
                                                     const __grid_constant__ OutSet O, const __grid_constant__ Sched S) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  float* smem = reinterpret_cast<float*>(smem_raw);
  float* ebuf = smem + FNS * f_stage_floats<V>();
  __shared__ __align__(8) uint64_t bars[2 * FNS + E_BUFS];
  __shared__ int s_item;
  __shared__ __align__(16) TabCache tabc;
  const FusedBars Q{bars, bars + FNS, bars + 2 * FNS};
  if (threadIdx.x == 0) {
#pragma unroll
    for (int s = 0; s < FNS; ++s) { mbar_init(&Q.full[s], 1); mbar_init(&Q.empty[s], FNW); }
#pragma unroll
    for (int b = 0; b < E_BUFS; ++b) mbar_init(&Q.efull[b], FNW);
    fence_barrier_init();
    if (blockIdx.x == 0) *S.other = 0u;
  }
  const int warp = threadIdx.x >> 5;
  unsigned it = 0, eit = 0;
  int x0, y0, z0, z1;
  // The roles never share code after this point, so each is compiled against its own register budget: the two main
  // warpgroups take the registers the halo and producer warpgroups give up (2 x 200 + 80 + 32 <= 512 per sub-partition lane).
  if (warp < FW_MAIN) {
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(F_REGS_MAIN));
    while (next_item(S, &s_item, x0, y0, z0, z1, D.nz)) {
      fill_tab_cache(D, tabc, x0, y0);
      const bool xs = touches(D, 0, x0, x0 + TX), ys = touches(D, 1, y0, y0 + TY);      // block-uniform
      // Few instantiations per kernel: with seven plane-body variants in one kernel ptxas spilled 1.3 KB in the main warps
      // (with two, nothing).  Variant 2 runs every slab item through one instantiation; a tile that touches only an x slab
      // has in_y false in every thread and skips the y code by a uniform branch.
      if (!xs && !ys) fused_main_item<0, 0, V>(D, O, smem, ebuf, Q, tabc, it, eit, x0, y0, z0, z1);
      else if constexpr (V == 2) fused_main_item<2, 2, V>(D, O, smem, ebuf, Q, tabc, it, eit, x0, y0, z0, z1);
      else if (xs && !ys) fused_main_item<1, 0, V>(D, O, smem, ebuf, Q, tabc, it, eit, x0, y0, z0, z1);
      else if (!xs) fused_main_item<0, 1, V>(D, O, smem, ebuf, Q, tabc, it, eit, x0, y0, z0, z1);
      else fused_main_item<1, 1, V>(D, O, smem, ebuf, Q, tabc, it, eit, x0, y0, z0, z1);
    }
  } else if (warp < FNW) {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(F_REGS_HALO));
    while (next_item(S, &s_item, x0, y0, z0, z1, D.nz)) {
      fill_tab_cache(D, tabc, x0, y0);
      fused_halo<V>(D, smem, ebuf, Q, tabc, it, eit, warp - FW_MAIN, x0, y0, z0, z1);
      it += z1 - z0 + f_lead<V>();
      eit += z1 - z0;
    }
  } else {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(F_REGS_PROD));
    const bool has_kc = D.kc != nullptr;
    const bool producer = threadIdx.x == FNW * 32;
    while (next_item(S, &s_item, x0, y0, z0, z1, D.nz)) {
      const int niter = z1 - z0 + f_lead<V>();
      if (producer) {
        for (int s = 0; s < niter; ++s) {
          const unsigned slot = (it + s) % FNS;
          if (s >= FNS) mbar_wait(&Q.empty[slot], ((it + s - FNS) / FNS) & 1);      // every consumer warp released the stage
          fused_issue<V>(tm, smem, Q.full, slot, s, x0, y0, z0, has_kc, D);
        }
      }
      it += niter;
    }
  }
}

}  // namespace fdtd
