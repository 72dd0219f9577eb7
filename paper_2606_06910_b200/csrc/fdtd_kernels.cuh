// Device code of the B200 FDTD + CPML time step (sm_100a).
//
// Two kernel families implement the two sub-updates of PAPER.md P:40 (with the CPML terms of P:46-56):
//   *_ref   : one thread per point, global loads only (cross-check; the only path for periodic boundaries)
//   *_tiled : the product path — 64x16 (x,y) tiles streamed along z.  The halo-bearing operand (p for the
//             velocity update, vy for the pressure update) is staged in shared memory by TMA
//             (cp.async.bulk.tensor, completion on an mbarrier, out-of-bounds = zero fill = the wall rule R4),
//             the z neighbours live in a register queue, everything else is 128-bit global traffic.
// Arithmetic is pinned with explicit intrinsics so that every launch shape (monolithic, subdomain, tiled, ref)
// produces the same bits for the same point (needed by BASELINE config 5's bit-identity).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace fdtd {

// Staggered 8th-order weights 1225/1024, -245/3072, 49/5120, -5/7168 (BASELINE.json config 1; the a_l of P:38, R1).
#define FDTD_C1 1.1962890625f
#define FDTD_C2 (-245.0f / 3072.0f)
#define FDTD_C3 (49.0f / 5120.0f)
#define FDTD_C4 (-5.0f / 7168.0f)

// One domain (the whole grid, or one in-HBM subdomain with its ghost cells) as the kernels see it.
struct DomainView {
  int nx, ny, nz;          // local extents (ghost cells included)
  int pitch;               // floats per x row (multiple of 8; columns >= nx are kept zero)
  long long plane;         // pitch * ny
  int ox, oy, oz;          // global index of local (0,0,0)
  int gn[3];               // global total-grid extents
  int periodic;
  float* f[4];             // p, vx, vy, vz
  const float* kc;         // K dt/dx per node (local layout) or nullptr -> kc0
  float kc0, b0;           // homogeneous K dt/dx and dt/(rho dx)
  int ls[3][2], ln[3][2];  // CPML storage slabs in LOCAL indices: [axis][side] start, count (0 = none)
  float* psi[2][3][2];     // [family 0 = psi_v, 1 = psi_p][axis][side], slab-local
  const float* tab[2][3][3];  // [family][axis][a, b, 1/kappa], indexed by GLOBAL index along the axis
};

// ---------------------------------------------------------------- arithmetic (identical in every kernel)
// D = sum_l c_l (hi_l - lo_l), accumulated l = 1..4 (P:38 in the staggered reading R1).
__device__ __forceinline__ float stag_diff(float h1, float l1, float h2, float l2, float h3, float l3, float h4, float l4) {
  float d = __fmul_rn(FDTD_C1, __fsub_rn(h1, l1));
  d = __fmaf_rn(FDTD_C2, __fsub_rn(h2, l2), d);
  d = __fmaf_rn(FDTD_C3, __fsub_rn(h3, l3), d);
  d = __fmaf_rn(FDTD_C4, __fsub_rn(h4, l4), d);
  return d;
}
// psi <- b psi + a d ; returns d/kappa + psi (update-then-use R10).
__device__ __forceinline__ float cpml_apply(float d, float& psi, float a, float b, float ik) {
  psi = __fmaf_rn(b, psi, __fmul_rn(a, d));
  return __fmaf_rn(d, ik, psi);
}
__device__ __forceinline__ float upd(float f, float coef, float d) { return __fmaf_rn(-coef, d, f); }

// psi slab addressing (slab-local storage).
__device__ __forceinline__ long long psi_index(const DomainView& D, int axis, int side, int i, int j, int k) {
  if (axis == 0) return ((long long)k * D.ny + j) * D.ln[0][side] + (i - D.ls[0][side]);
  if (axis == 1) return ((long long)k * D.ln[1][side] + (j - D.ls[1][side])) * D.pitch + i;
  return ((long long)(k - D.ls[2][side]) * D.ny + j) * D.pitch + i;
}
// which storage slab (0 low, 1 high, -1 none) holds local index v of this axis
__device__ __forceinline__ int slab_side(const DomainView& D, int axis, int v) {
  if (D.ln[axis][0] > 0 && v >= D.ls[axis][0] && v < D.ls[axis][0] + D.ln[axis][0]) return 0;
  if (D.ln[axis][1] > 0 && v >= D.ls[axis][1] && v < D.ls[axis][1] + D.ln[axis][1]) return 1;
  return -1;
}

// ---------------------------------------------------------------- reference kernels (one thread per point)
__device__ __forceinline__ float rd_ref(const DomainView& D, const float* __restrict__ a, int i, int j, int k) {
  if (D.periodic) {
    i = (i % D.nx + D.nx) % D.nx; j = (j % D.ny + D.ny) % D.ny; k = (k % D.nz + D.nz) % D.nz;
  } else if (i < 0 || i >= D.nx || j < 0 || j >= D.ny || k < 0 || k >= D.nz) {
    return 0.0f;
  }
  return a[(long long)k * D.plane + (long long)j * D.pitch + i];
}

__global__ void __launch_bounds__(256) update_v_ref(DomainView D) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y * blockDim.y + threadIdx.y;
  const int k = blockIdx.z;
  if (i >= D.nx || j >= D.ny || k >= D.nz) return;
  const long long q = (long long)k * D.plane + (long long)j * D.pitch + i;
  const float* p = D.f[0];
  const int g[3] = {i + D.ox, j + D.oy, k + D.oz};
  const int loc[3] = {i, j, k};
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    if (!D.periodic && g[a] == D.gn[a] - 1) continue;   // pinned last half node (R3)
    const int ex = a == 0, ey = a == 1, ez = a == 2;
    float d = stag_diff(rd_ref(D, p, i + ex, j + ey, k + ez), rd_ref(D, p, i, j, k),
                        rd_ref(D, p, i + 2 * ex, j + 2 * ey, k + 2 * ez), rd_ref(D, p, i - ex, j - ey, k - ez),
                        rd_ref(D, p, i + 3 * ex, j + 3 * ey, k + 3 * ez), rd_ref(D, p, i - 2 * ex, j - 2 * ey, k - 2 * ez),
                        rd_ref(D, p, i + 4 * ex, j + 4 * ey, k + 4 * ez), rd_ref(D, p, i - 3 * ex, j - 3 * ey, k - 3 * ez));
    const int side = slab_side(D, a, loc[a]);
    if (side >= 0) {
      float* ps = D.psi[0][a][side] + psi_index(D, a, side, i, j, k);
      float s = *ps;
      d = cpml_apply(d, s, D.tab[0][a][0][g[a]], D.tab[0][a][1][g[a]], D.tab[0][a][2][g[a]]);
      *ps = s;
    }
    D.f[1 + a][q] = upd(D.f[1 + a][q], D.b0, d);
  }
}

__global__ void __launch_bounds__(256) update_p_ref(DomainView D) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y * blockDim.y + threadIdx.y;
  const int k = blockIdx.z;
  if (i >= D.nx || j >= D.ny || k >= D.nz) return;
  const long long q = (long long)k * D.plane + (long long)j * D.pitch + i;
  const int g[3] = {i + D.ox, j + D.oy, k + D.oz};
  const int loc[3] = {i, j, k};
  float dd[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    const float* v = D.f[1 + a];
    const int ex = a == 0, ey = a == 1, ez = a == 2;
    float d = stag_diff(rd_ref(D, v, i, j, k), rd_ref(D, v, i - ex, j - ey, k - ez),
                        rd_ref(D, v, i + ex, j + ey, k + ez), rd_ref(D, v, i - 2 * ex, j - 2 * ey, k - 2 * ez),
                        rd_ref(D, v, i + 2 * ex, j + 2 * ey, k + 2 * ez), rd_ref(D, v, i - 3 * ex, j - 3 * ey, k - 3 * ez),
                        rd_ref(D, v, i + 3 * ex, j + 3 * ey, k + 3 * ez), rd_ref(D, v, i - 4 * ex, j - 4 * ey, k - 4 * ez));
    const int side = slab_side(D, a, loc[a]);
    if (side >= 0) {
      float* ps = D.psi[1][a][side] + psi_index(D, a, side, i, j, k);
      float s = *ps;
      d = cpml_apply(d, s, D.tab[1][a][0][g[a]], D.tab[1][a][1][g[a]], D.tab[1][a][2][g[a]]);
      *ps = s;
    }
    dd[a] = d;
  }
  const float kc = D.kc ? D.kc[q] : D.kc0;
  D.f[0][q] = upd(D.f[0][q], kc, __fadd_rn(__fadd_rn(dd[0], dd[1]), dd[2]));
}

// ---------------------------------------------------------------- TMA / mbarrier primitives (inline PTX)
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred P1;\n"
      "WAIT_LOOP:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
      "@P1 bra DONE;\n"
      "bra WAIT_LOOP;\n"
      "DONE:\n"
      "}\n" ::"r"(smem_u32(bar)),
      "r"(parity)
      : "memory");
}
__device__ __forceinline__ void tma_load_3d(void* dst, const CUtensorMap* map, uint64_t* bar, int c0, int c1, int c2) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];" ::"r"(smem_u32(dst)),
      "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2)
      : "memory");
}
__device__ __forceinline__ void fence_barrier_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// ---------------------------------------------------------------- tiled kernels
constexpr int TX = 64;            // tile width in x (floats); 16 lanes x V4
constexpr int TY = 16;            // tile height in y (rows)
constexpr int NT = 256;           // threads per CTA
constexpr int VW = TX + 8;        // p tile for update_v: columns x0-4 .. x0+TX+3
constexpr int VH = TY + 7;        //                      rows    y0-3 .. y0+TY+3
constexpr int VSTAGES = 4;
constexpr int PW = TX;            // vy tile for update_p: columns x0 .. x0+TX-1
constexpr int PH = TY + 8;        //                       rows    y0-4 .. y0+TY+3
constexpr int PSTAGES = 4;
constexpr int V_TILE_BYTES = VW * VH * 4;                       // bytes one TMA box delivers
constexpr int P_TILE_BYTES = PW * PH * 4;
constexpr int V_STAGE_FLOATS = ((V_TILE_BYTES + 127) / 128) * 32;  // stage stride: TMA destinations stay 128-B aligned
constexpr int P_STAGE_FLOATS = ((P_TILE_BYTES + 127) / 128) * 32;
constexpr int V_SMEM_BYTES = VSTAGES * V_STAGE_FLOATS * 4;
constexpr int P_SMEM_BYTES = PSTAGES * P_STAGE_FLOATS * 4;

// Four consecutive x values held in registers; moved as one 128-bit access.
struct V4 { float v[4]; };
__device__ __forceinline__ V4 from4(float4 f) { V4 r; r.v[0] = f.x; r.v[1] = f.y; r.v[2] = f.z; r.v[3] = f.w; return r; }
__device__ __forceinline__ V4 ldg4(const float* p) { return from4(__ldg(reinterpret_cast<const float4*>(p))); }
__device__ __forceinline__ V4 ld4(const float* p) { return from4(*reinterpret_cast<const float4*>(p)); }
__device__ __forceinline__ void st4(float* p, const V4& a) { *reinterpret_cast<float4*>(p) = make_float4(a.v[0], a.v[1], a.v[2], a.v[3]); }
__device__ __forceinline__ V4 splat4(float x) { V4 r; r.v[0] = r.v[1] = r.v[2] = r.v[3] = x; return r; }
__device__ __forceinline__ V4 zero4() { return splat4(0.f); }
#define F4(a, e) ((a).v[e])

// Velocity sub-update: v_a <- v_a - B [(1/kappa_a) D+_a p + psi_va] on planes [z0, z1) of one tile.
// On arrival of p plane m: vx, vy of plane m are updated from the shared-memory tile, p[m] enters the register
// queue, and vz of plane m-4 is updated from the queue (D+_z at k+1/2 reads p[k-3 .. k+4]).
__global__ void __launch_bounds__(NT) update_v_tiled(const __grid_constant__ CUtensorMap tm_p, DomainView D, int zchunk) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  float* tiles = reinterpret_cast<float*>(smem_raw);
  __shared__ __align__(8) uint64_t full[VSTAGES];

  const int z0 = blockIdx.z * zchunk;
  if (z0 >= D.nz) return;
  const int z1 = min(z0 + zchunk, D.nz);
  const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
  const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY;
  const int i = x0 + 4 * tx, j = y0 + ty;
  const bool active = (i < D.nx) && (j < D.ny);
  const int gj = j + D.oy;

  if (threadIdx.x == 0) {
#pragma unroll
    for (int s = 0; s < VSTAGES; ++s) mbar_init(&full[s], 1);
    fence_barrier_init();
  }
  __syncthreads();

  const int m_begin = z0 - 3, m_end = z1 + 4;       // p planes m_begin .. m_end-1 are consumed
  if (threadIdx.x == 0) {
#pragma unroll
    for (int s = 0; s < VSTAGES; ++s)
      if (m_begin + s < m_end) {
        mbar_expect_tx(&full[s], V_TILE_BYTES);
        tma_load_3d(tiles + s * V_STAGE_FLOATS, &tm_p, &full[s], x0 - 4, y0 - 3, m_begin + s);
      }
  }

  // per-thread invariants
  const long long rowoff = (long long)j * D.pitch + i;
  float* __restrict__ vx = D.f[1];
  float* __restrict__ vy = D.f[2];
  float* __restrict__ vz = D.f[3];
  const float B = D.b0;
  // keep-masks: component e is written only if it is a real column and not the pinned last half node (R3)
  bool wx[4], wc[4];
#pragma unroll
  for (int e = 0; e < 4; ++e) {
    wc[e] = (i + e) < D.nx;
    wx[e] = wc[e] && (D.periodic || (i + e + D.ox) != D.gn[0] - 1);
  }
  const bool wy_row = gj != D.gn[1] - 1;
  // CPML x / y slabs touched by this thread (x: the V4 lies wholly inside or outside a storage slab)
  const int sx = active ? slab_side(D, 0, i) : -1;
  const int sy = active ? slab_side(D, 1, j) : -1;
  V4 ax = zero4(), bx = zero4(), ikx = zero4();
  float ay = 0.f, by = 0.f, iky = 1.f;
  if (sx >= 0) {
    ax = ldg4(D.tab[0][0][0] + i + D.ox); bx = ldg4(D.tab[0][0][1] + i + D.ox); ikx = ldg4(D.tab[0][0][2] + i + D.ox);
  }
  if (sy >= 0) { ay = __ldg(D.tab[0][1][0] + gj); by = __ldg(D.tab[0][1][1] + gj); iky = __ldg(D.tab[0][1][2] + gj); }

  V4 q0 = zero4(), q1 = zero4(), q2 = zero4(), q3 = zero4(), q4 = zero4(), q5 = zero4(), q6 = zero4(), q7 = zero4();

  int it = 0;
  for (int m = m_begin; m < m_end; ++m, ++it) {
    const int s = it % VSTAGES;
    const uint32_t parity = (it / VSTAGES) & 1;
    const bool do_xy = active && m >= z0 && m < z1;
    const int kz = m - 4;
    const bool do_z = active && kz >= z0 && kz < z1 && (D.periodic || (kz + D.oz) != D.gn[2] - 1);
    // issue the streaming loads before waiting on the tile
    V4 vx4 = zero4(), vy4 = zero4(), vz4 = zero4(), psx = zero4(), psy = zero4(), psz = zero4();
    const long long qxy = (long long)m * D.plane + rowoff;
    const long long qz = (long long)kz * D.plane + rowoff;
    int sz = -1;
    if (do_xy) {
      vx4 = ld4(vx + qxy);
      vy4 = ld4(vy + qxy);
      if (sx >= 0) psx = ld4(D.psi[0][0][sx] + psi_index(D, 0, sx, i, j, m));
      if (sy >= 0) psy = ld4(D.psi[0][1][sy] + psi_index(D, 1, sy, i, j, m));
    }
    if (do_z) {
      vz4 = ld4(vz + qz);
      sz = slab_side(D, 2, kz);
      if (sz >= 0) psz = ld4(D.psi[0][2][sz] + psi_index(D, 2, sz, i, j, kz));
    }

    mbar_wait(&full[s], parity);
    const float* row = tiles + s * V_STAGE_FLOATS + (ty + 3) * VW + 4 * tx + 4;
    const V4 c = ld4(row);
    V4 dxv, dyv;
    {
      const V4 l = ld4(row - 4), r = ld4(row + 4);
      const float w[12] = {l.v[0], l.v[1], l.v[2], l.v[3], c.v[0], c.v[1], c.v[2], c.v[3], r.v[0], r.v[1], r.v[2], r.v[3]};   // p[i-4+n]
#pragma unroll
      for (int e = 0; e < 4; ++e)
        F4(dxv, e) = stag_diff(w[5 + e], w[4 + e], w[6 + e], w[3 + e], w[7 + e], w[2 + e], w[8 + e], w[1 + e]);
      const V4 yp1 = ld4(row + VW), yp2 = ld4(row + 2 * VW), yp3 = ld4(row + 3 * VW), yp4 = ld4(row + 4 * VW);
      const V4 ym1 = ld4(row - VW), ym2 = ld4(row - 2 * VW), ym3 = ld4(row - 3 * VW);
#pragma unroll
      for (int e = 0; e < 4; ++e)
        F4(dyv, e) = stag_diff(F4(yp1, e), F4(c, e), F4(yp2, e), F4(ym1, e), F4(yp3, e), F4(ym2, e), F4(yp4, e), F4(ym3, e));
    }
    q0 = q1; q1 = q2; q2 = q3; q3 = q4; q4 = q5; q5 = q6; q6 = q7; q7 = c;    // q7 = p[m], q0 = p[m-7]
    __syncthreads();                                                            // every thread is done with stage s
    if (threadIdx.x == 0 && m + VSTAGES < m_end) {
      mbar_expect_tx(&full[s], V_TILE_BYTES);
      tma_load_3d(tiles + s * V_STAGE_FLOATS, &tm_p, &full[s], x0 - 4, y0 - 3, m + VSTAGES);
    }

    if (do_xy) {
      if (sx >= 0) {
#pragma unroll
        for (int e = 0; e < 4; ++e) {
          const float old = F4(psx, e);
          F4(dxv, e) = cpml_apply(F4(dxv, e), F4(psx, e), F4(ax, e), F4(bx, e), F4(ikx, e));
          if (!wx[e]) F4(psx, e) = old;          // the pinned half node keeps its psi too (R3)
        }
        st4(D.psi[0][0][sx] + psi_index(D, 0, sx, i, j, m), psx);
      }
      if (sy >= 0 && wy_row) {
#pragma unroll
        for (int e = 0; e < 4; ++e) F4(dyv, e) = cpml_apply(F4(dyv, e), F4(psy, e), ay, by, iky);
        st4(D.psi[0][1][sy] + psi_index(D, 1, sy, i, j, m), psy);
      }
#pragma unroll
      for (int e = 0; e < 4; ++e) {
        const float nvx = upd(F4(vx4, e), B, F4(dxv, e));
        F4(vx4, e) = wx[e] ? nvx : (wc[e] ? F4(vx4, e) : 0.f);
        const float nvy = upd(F4(vy4, e), B, F4(dyv, e));
        F4(vy4, e) = wc[e] ? ((D.periodic || wy_row) ? nvy : F4(vy4, e)) : 0.f;
      }
      st4(vx + qxy, vx4);
      st4(vy + qxy, vy4);
    }
    if (do_z) {
      V4 dzv;
#pragma unroll
      for (int e = 0; e < 4; ++e)   // D+_z at kz+1/2: p[kz+l] = q(3+l), p[kz-l+1] = q(4-l)
        F4(dzv, e) = stag_diff(F4(q4, e), F4(q3, e), F4(q5, e), F4(q2, e), F4(q6, e), F4(q1, e), F4(q7, e), F4(q0, e));
      if (sz >= 0) {
        const int gk = kz + D.oz;
        const float az = __ldg(D.tab[0][2][0] + gk), bz = __ldg(D.tab[0][2][1] + gk), ikz = __ldg(D.tab[0][2][2] + gk);
#pragma unroll
        for (int e = 0; e < 4; ++e) F4(dzv, e) = cpml_apply(F4(dzv, e), F4(psz, e), az, bz, ikz);
        st4(D.psi[0][2][sz] + psi_index(D, 2, sz, i, j, kz), psz);
      }
#pragma unroll
      for (int e = 0; e < 4; ++e) F4(vz4, e) = wc[e] ? upd(F4(vz4, e), B, F4(dzv, e)) : 0.f;
      st4(vz + qz, vz4);
    }
  }
}

// Pressure sub-update: p <- p - Kc [sum_a (1/kappa_a) D-_a v_a + psi_pa] on planes [z0, z1).
// vx: own V4 + left/right neighbours by 128-bit loads; vy: TMA-staged tile (rows y0-4 .. y0+TY+3);
// vz: register queue along z (D-_z at node k reads vz[k-4 .. k+3]).
__global__ void __launch_bounds__(NT) update_p_tiled(const __grid_constant__ CUtensorMap tm_vy, DomainView D, int zchunk) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  float* tiles = reinterpret_cast<float*>(smem_raw);
  __shared__ __align__(8) uint64_t full[PSTAGES];

  const int z0 = blockIdx.z * zchunk;
  if (z0 >= D.nz) return;
  const int z1 = min(z0 + zchunk, D.nz);
  const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
  const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY;
  const int i = x0 + 4 * tx, j = y0 + ty;
  const bool active = (i < D.nx) && (j < D.ny);
  const int gj = j + D.oy;

  if (threadIdx.x == 0) {
#pragma unroll
    for (int s = 0; s < PSTAGES; ++s) mbar_init(&full[s], 1);
    fence_barrier_init();
  }
  __syncthreads();
  if (threadIdx.x == 0) {
#pragma unroll
    for (int s = 0; s < PSTAGES; ++s)
      if (z0 + s < z1) {
        mbar_expect_tx(&full[s], P_TILE_BYTES);
        tma_load_3d(tiles + s * P_STAGE_FLOATS, &tm_vy, &full[s], x0, y0 - 4, z0 + s);
      }
  }

  const long long rowoff = (long long)j * D.pitch + i;
  float* __restrict__ p = D.f[0];
  const float* __restrict__ vx = D.f[1];
  const float* __restrict__ vz = D.f[3];
  bool wc[4];
#pragma unroll
  for (int e = 0; e < 4; ++e) wc[e] = (i + e) < D.nx;
  const bool has_l = i >= 4, has_r = (i + 4) < D.pitch;
  const int sx = active ? slab_side(D, 0, i) : -1;
  const int sy = active ? slab_side(D, 1, j) : -1;
  V4 ax = zero4(), bx = zero4(), ikx = zero4();
  float ay = 0.f, by = 0.f, iky = 1.f;
  if (sx >= 0) {
    ax = ldg4(D.tab[1][0][0] + i + D.ox); bx = ldg4(D.tab[1][0][1] + i + D.ox); ikx = ldg4(D.tab[1][0][2] + i + D.ox);
  }
  if (sy >= 0) { ay = __ldg(D.tab[1][1][0] + gj); by = __ldg(D.tab[1][1][1] + gj); iky = __ldg(D.tab[1][1][2] + gj); }

  // vz queue: q0 = vz[k-4] ... q7 = vz[k+3]; before the first iteration q1..q7 = vz[z0-4 .. z0+2]
  V4 q0 = zero4(), q1 = zero4(), q2 = zero4(), q3 = zero4(), q4 = zero4(), q5 = zero4(), q6 = zero4(), q7 = zero4();
  if (active) {
    auto ldz = [&](int kk) -> V4 { return (kk >= 0 && kk < D.nz) ? ld4(vz + (long long)kk * D.plane + rowoff) : zero4(); };
    q1 = ldz(z0 - 4); q2 = ldz(z0 - 3); q3 = ldz(z0 - 2); q4 = ldz(z0 - 1); q5 = ldz(z0); q6 = ldz(z0 + 1); q7 = ldz(z0 + 2);
  }

  int it = 0;
  for (int k = z0; k < z1; ++k, ++it) {
    const int s = it % PSTAGES;
    const uint32_t parity = (it / PSTAGES) & 1;
    const long long qk = (long long)k * D.plane + rowoff;
    V4 vzn = zero4(), vxc = zero4(), vxl = zero4(), vxr = zero4(), p4 = zero4(), kc4 = zero4();
    V4 psx = zero4(), psy = zero4(), psz = zero4();
    int sz = -1;
    if (active) {
      if (k + 3 < D.nz) vzn = ld4(vz + qk + 3 * D.plane);
      vxc = ld4(vx + qk);
      if (has_l) vxl = ld4(vx + qk - 4);
      if (has_r) vxr = ld4(vx + qk + 4);
      p4 = ld4(p + qk);
      if (D.kc) kc4 = ldg4(D.kc + qk);
      else kc4 = splat4(D.kc0);
      if (sx >= 0) psx = ld4(D.psi[1][0][sx] + psi_index(D, 0, sx, i, j, k));
      if (sy >= 0) psy = ld4(D.psi[1][1][sy] + psi_index(D, 1, sy, i, j, k));
      sz = slab_side(D, 2, k);
      if (sz >= 0) psz = ld4(D.psi[1][2][sz] + psi_index(D, 2, sz, i, j, k));
    }
    q0 = q1; q1 = q2; q2 = q3; q3 = q4; q4 = q5; q5 = q6; q6 = q7; q7 = vzn;

    mbar_wait(&full[s], parity);
    V4 dyv;
    {
      const float* col = tiles + s * P_STAGE_FLOATS + ty * PW + 4 * tx;     // tile row r <-> y = y0-4+r
      const V4 r0 = ld4(col), r1 = ld4(col + PW), r2 = ld4(col + 2 * PW), r3 = ld4(col + 3 * PW);
      const V4 r4 = ld4(col + 4 * PW), r5 = ld4(col + 5 * PW), r6 = ld4(col + 6 * PW), r7 = ld4(col + 7 * PW);
#pragma unroll
      for (int e = 0; e < 4; ++e)   // D-_y at node j: vy[j+l-1] = row(ty+3+l), vy[j-l] = row(ty+4-l)
        F4(dyv, e) = stag_diff(F4(r4, e), F4(r3, e), F4(r5, e), F4(r2, e), F4(r6, e), F4(r1, e), F4(r7, e), F4(r0, e));
    }
    __syncthreads();
    if (threadIdx.x == 0 && k + PSTAGES < z1) {
      mbar_expect_tx(&full[s], P_TILE_BYTES);
      tma_load_3d(tiles + s * P_STAGE_FLOATS, &tm_vy, &full[s], x0, y0 - 4, k + PSTAGES);
    }
    if (!active) continue;

    V4 dxv, dzv;
    {
      const float w[12] = {vxl.v[0], vxl.v[1], vxl.v[2], vxl.v[3], vxc.v[0], vxc.v[1], vxc.v[2], vxc.v[3], vxr.v[0], vxr.v[1], vxr.v[2], vxr.v[3]};  // vx[i-4+n]
#pragma unroll
      for (int e = 0; e < 4; ++e)   // D-_x at node i+e: vx[i+e+l-1] = w(3+e+l), vx[i+e-l] = w(4+e-l)
        F4(dxv, e) = stag_diff(w[4 + e], w[3 + e], w[5 + e], w[2 + e], w[6 + e], w[1 + e], w[7 + e], w[e]);
#pragma unroll
      for (int e = 0; e < 4; ++e)   // D-_z at node k: vz[k+l-1] = q(3+l), vz[k-l] = q(4-l)
        F4(dzv, e) = stag_diff(F4(q4, e), F4(q3, e), F4(q5, e), F4(q2, e), F4(q6, e), F4(q1, e), F4(q7, e), F4(q0, e));
    }
    if (sx >= 0) {
#pragma unroll
      for (int e = 0; e < 4; ++e) F4(dxv, e) = cpml_apply(F4(dxv, e), F4(psx, e), F4(ax, e), F4(bx, e), F4(ikx, e));
      st4(D.psi[1][0][sx] + psi_index(D, 0, sx, i, j, k), psx);
    }
    if (sy >= 0) {
#pragma unroll
      for (int e = 0; e < 4; ++e) F4(dyv, e) = cpml_apply(F4(dyv, e), F4(psy, e), ay, by, iky);
      st4(D.psi[1][1][sy] + psi_index(D, 1, sy, i, j, k), psy);
    }
    if (sz >= 0) {
      const int gk = k + D.oz;
      const float az = __ldg(D.tab[1][2][0] + gk), bz = __ldg(D.tab[1][2][1] + gk), ikz = __ldg(D.tab[1][2][2] + gk);
#pragma unroll
      for (int e = 0; e < 4; ++e) F4(dzv, e) = cpml_apply(F4(dzv, e), F4(psz, e), az, bz, ikz);
      st4(D.psi[1][2][sz] + psi_index(D, 2, sz, i, j, k), psz);
    }
#pragma unroll
    for (int e = 0; e < 4; ++e)
      F4(p4, e) = wc[e] ? upd(F4(p4, e), F4(kc4, e), __fadd_rn(__fadd_rn(F4(dxv, e), F4(dyv, e)), F4(dzv, e))) : 0.f;
    st4(p + qk, p4);
  }
}

// ---------------------------------------------------------------- small kernels
// p[src_s] += w_s[n] for every source, then n <- n + 1 (R14).  One block; the step counter lives on the device so
// that a time step is a fixed launch sequence.
struct SourceView {
  int n, len;
  const long long* offset;   // flat element offset of each source in its domain's p array, or -1 if not held
  float* p;
  const float* wav;
  long long* step;           // device step counter (shared by all domains; advanced by the launch with advance = 1)
};
__global__ void inject_sources(SourceView S, int advance) {
  const long long n = *S.step;
  __syncthreads();
  for (int s = threadIdx.x; s < S.n; s += blockDim.x)
    if (n < S.len && S.offset[s] >= 0) S.p[S.offset[s]] = __fadd_rn(S.p[S.offset[s]], S.wav[(long long)s * S.len + n]);
  if (advance && threadIdx.x == 0) *S.step = n + 1;
}

// In place: wave speed c (fp32) -> K dt/dx = rho c^2 dt/dx in double, rounded once to fp32 (R6).  Padding columns stay 0.
__global__ void speed_to_kc_kernel(float* a, long long n, int pitch, int nx, double rho, double dt, double dx, int* bad) {
  for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += (long long)gridDim.x * blockDim.x) {
    if ((int)(t % pitch) >= nx) { a[t] = 0.f; continue; }
    const double c = (double)a[t];
    if (!(c > 0.0) || c > 1e30) atomicAdd(bad, 1);
    a[t] = (float)(rho * c * c * dt / dx);
  }
}

__device__ __forceinline__ uint64_t splitmix64(uint64_t x) {
  x += 0x9E3779B97F4A7C15ull;
  x = (x ^ (x >> 30)) * 0xBF58476D1CE4E5B9ull;
  x = (x ^ (x >> 27)) * 0x94D049BB133111EBull;
  return x ^ (x >> 31);
}
// Counter-based synthetic initial state: value depends on the GLOBAL index only.
__global__ void fill_hash_kernel(DomainView D, int which, uint64_t seed, float scale) {
  const long long n = (long long)D.nx * D.ny * D.nz;
  for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += (long long)gridDim.x * blockDim.x) {
    const int i = (int)(t % D.nx);
    const long long r = t / D.nx;
    const int j = (int)(r % D.ny), k = (int)(r / D.ny);
    const uint64_t g = (uint64_t)(i + D.ox) + (uint64_t)D.gn[0] * ((uint64_t)(j + D.oy) + (uint64_t)D.gn[1] * (uint64_t)(k + D.oz));
    const uint64_t h = splitmix64(seed + ((uint64_t)which << 56) + g);
    const float u = __fsub_rn(__fmul_rn((float)(int)(uint32_t)(h >> 40), 1.0f / 8388608.0f), 1.0f);
    D.f[which][(long long)k * D.plane + (long long)j * D.pitch + i] = __fmul_rn(scale, u);
  }
}

__global__ void absmax_kernel(DomainView D, int which, int lx, int ly, int lz, int sx, int sy, int sz, unsigned int* out) {
  const long long n = (long long)sx * sy * sz;
  float m = 0.f;
  for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += (long long)gridDim.x * blockDim.x) {
    const int i = (int)(t % sx);
    const long long r = t / sx;
    const int j = (int)(r % sy), k = (int)(r / sy);
    m = fmaxf(m, fabsf(D.f[which][(long long)(k + lz) * D.plane + (long long)(j + ly) * D.pitch + (i + lx)]));
  }
  for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
  if ((threadIdx.x & 31) == 0) atomicMax(out, __float_as_uint(m));   // non-negative floats order like unsigned ints
}

// Expand one slab-local psi array into a full-volume scratch array (debug / parity of the recursion).
__global__ void expand_psi_kernel(DomainView D, int fam, int axis, float* out /* nx*ny*nz packed */) {
  const long long n = (long long)D.nx * D.ny * D.nz;
  for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += (long long)gridDim.x * blockDim.x) {
    const int i = (int)(t % D.nx);
    const long long r = t / D.nx;
    const int j = (int)(r % D.ny), k = (int)(r / D.ny);
    const int loc[3] = {i, j, k};
    const int side = slab_side(D, axis, loc[axis]);
    out[t] = side >= 0 ? D.psi[fam][axis][side][psi_index(D, axis, side, i, j, k)] : 0.f;
  }
}

}  // namespace fdtd
