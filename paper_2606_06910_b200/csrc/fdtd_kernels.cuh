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

// One domain (the whole grid, or one in-HBM subdomain with its ghost cells) as the kernels see it.  T = float is the
// product path; T = double is the verification precision: state and arithmetic in double, every coefficient
// (weights, CPML tables, K dt/dx, dt/(rho_bar dx), wavelets) the same fp32 number as in the fp32 path.
template <class T>
struct DomainViewT {
  typedef T real;
  int nx, ny, nz;          // local extents (ghost cells included)
  int pitch;               // elements per x row (multiple of 8; columns >= nx are kept zero)
  long long plane;         // pitch * ny
  int ox, oy, oz;          // global index of local (0,0,0)
  int gn[3];               // global total-grid extents
  int periodic;
  T* f[4];                 // p, vx, vy, vz
  const float* kc;         // K dt/dx per node (local layout) or nullptr -> kc0
  float kc0, b0;           // homogeneous K dt/dx and dt/(rho dx)
  const float* bq[3];      // dt/(rho_bar dx) at the half nodes of vx, vy, vz (local layout) or nullptr -> b0 (R6)
  int ls[3][2], ln[3][2];  // CPML storage slabs in LOCAL indices: [axis][side] start, count (0 = none)
  T* psi[2][3][2];         // [family 0 = psi_v, 1 = psi_p][axis][side], slab-local
  const float* tab[2][3][3];  // [family][axis][a, b, 1/kappa], indexed by GLOBAL index along the axis
};
typedef DomainViewT<float> DomainView;

// ---------------------------------------------------------------- arithmetic (identical in every kernel)
// D = sum_l c_l (hi_l - lo_l), accumulated l = 1..4 (P:38 in the staggered reading R1).
// Every product and every sum is rounded on its own, in the order of the recurrence as written:
// no fused multiply-add.  The result therefore has the bits of the plain evaluation — the fp32 oracle's — and parity is
// exact instead of "within rounding" (an FMA chain drifts from it by 1e-4 of the final field over 500 steps near a point
// source, where the velocity has cancelled from 300 times its final size; measured cost of the separate roundings: 2 %,
// the kernels are bound by shared-memory and HBM bandwidth, not by arithmetic issue).
__device__ __forceinline__ float mad(float a, float b, float c) { return __fadd_rn(__fmul_rn(a, b), c); }
// Packed fp32x2 (sm_100a FADD2 / FMUL2): two independent IEEE operations per instruction.  ptxas contracts a packed
// multiply into a packed add that consumes it (FFMA2) whatever the rounding modifiers say, so every product that feeds a
// sum is formed by two scalar FMULs; only the sums and differences are packed.
__device__ __forceinline__ float2 mul2(float2 a, float2 b) { return make_float2(__fmul_rn(a.x, b.x), __fmul_rn(a.y, b.y)); }
__device__ __forceinline__ float2 mad2(float2 a, float2 b, float2 c) { return __fadd2_rn(mul2(a, b), c); }
__device__ __forceinline__ float stag_diff(float h1, float l1, float h2, float l2, float h3, float l3, float h4, float l4) {
  float d = __fmul_rn(FDTD_C1, __fsub_rn(h1, l1));
  d = mad(FDTD_C2, __fsub_rn(h2, l2), d);
  d = mad(FDTD_C3, __fsub_rn(h3, l3), d);
  d = mad(FDTD_C4, __fsub_rn(h4, l4), d);
  return d;
}
// psi <- b psi + a d ; returns d/kappa + psi (update-then-use R10).
__device__ __forceinline__ float cpml_apply(float d, float& psi, float a, float b, float ik) {
  psi = mad(b, psi, __fmul_rn(a, d));
  return mad(d, ik, psi);
}
__device__ __forceinline__ float upd(float f, float coef, float d) { return mad(-coef, d, f); }
// the same sequences in double (verification precision): products and sums rounded separately here too
__device__ __forceinline__ double mad(double a, double b, double c) { return __dadd_rn(__dmul_rn(a, b), c); }
__device__ __forceinline__ double stag_diff(double h1, double l1, double h2, double l2, double h3, double l3, double h4, double l4) {
  double d = __dmul_rn((double)FDTD_C1, __dsub_rn(h1, l1));
  d = mad((double)FDTD_C2, __dsub_rn(h2, l2), d);
  d = mad((double)FDTD_C3, __dsub_rn(h3, l3), d);
  d = mad((double)FDTD_C4, __dsub_rn(h4, l4), d);
  return d;
}
__device__ __forceinline__ double cpml_apply(double d, double& psi, double a, double b, double ik) {
  psi = mad(b, psi, __dmul_rn(a, d));
  return mad(d, ik, psi);
}
__device__ __forceinline__ double upd(double f, double coef, double d) { return mad(-coef, d, f); }
__device__ __forceinline__ float add3(float a, float b, float c) { return __fadd_rn(__fadd_rn(a, b), c); }
__device__ __forceinline__ double add3(double a, double b, double c) { return __dadd_rn(__dadd_rn(a, b), c); }

// psi slab addressing (slab-local storage).
template <class V>
__device__ __forceinline__ long long psi_index(const V& D, int axis, int side, int i, int j, int k) {
  if (axis == 0) return ((long long)k * D.ny + j) * D.ln[0][side] + (i - D.ls[0][side]);
  if (axis == 1) return ((long long)k * D.ln[1][side] + (j - D.ls[1][side])) * D.pitch + i;
  return ((long long)(k - D.ls[2][side]) * D.ny + j) * D.pitch + i;
}
// which storage slab (0 low, 1 high, -1 none) holds local index v of this axis
template <class V>
__device__ __forceinline__ int slab_side(const V& D, int axis, int v) {
  if (D.ln[axis][0] > 0 && v >= D.ls[axis][0] && v < D.ls[axis][0] + D.ln[axis][0]) return 0;
  if (D.ln[axis][1] > 0 && v >= D.ls[axis][1] && v < D.ls[axis][1] + D.ln[axis][1]) return 1;
  return -1;
}

// ---------------------------------------------------------------- reference kernels (one thread per point)
template <class V>
__device__ __forceinline__ typename V::real rd_ref(const V& D, const typename V::real* __restrict__ a, int i, int j, int k) {
  if (D.periodic) {
    i = (i % D.nx + D.nx) % D.nx; j = (j % D.ny + D.ny) % D.ny; k = (k % D.nz + D.nz) % D.nz;
  } else if (i < 0 || i >= D.nx || j < 0 || j >= D.ny || k < 0 || k >= D.nz) {
    return 0;
  }
  return a[(long long)k * D.plane + (long long)j * D.pitch + i];
}

template <class V>
__global__ void __launch_bounds__(256) update_v_ref(V D) {
  typedef typename V::real T;
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y * blockDim.y + threadIdx.y;
  const int k = blockIdx.z;
  if (i >= D.nx || j >= D.ny || k >= D.nz) return;
  const long long q = (long long)k * D.plane + (long long)j * D.pitch + i;
  const T* p = D.f[0];
  const int g[3] = {i + D.ox, j + D.oy, k + D.oz};
  const int loc[3] = {i, j, k};
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    if (!D.periodic && g[a] == D.gn[a] - 1) continue;   // pinned last half node (R3)
    const int ex = a == 0, ey = a == 1, ez = a == 2;
    T d = stag_diff(rd_ref(D, p, i + ex, j + ey, k + ez), rd_ref(D, p, i, j, k),
                    rd_ref(D, p, i + 2 * ex, j + 2 * ey, k + 2 * ez), rd_ref(D, p, i - ex, j - ey, k - ez),
                    rd_ref(D, p, i + 3 * ex, j + 3 * ey, k + 3 * ez), rd_ref(D, p, i - 2 * ex, j - 2 * ey, k - 2 * ez),
                    rd_ref(D, p, i + 4 * ex, j + 4 * ey, k + 4 * ez), rd_ref(D, p, i - 3 * ex, j - 3 * ey, k - 3 * ez));
    const int side = slab_side(D, a, loc[a]);
    if (side >= 0) {
      T* ps = D.psi[0][a][side] + psi_index(D, a, side, i, j, k);
      T s = *ps;
      d = cpml_apply(d, s, (T)D.tab[0][a][0][g[a]], (T)D.tab[0][a][1][g[a]], (T)D.tab[0][a][2][g[a]]);
      *ps = s;
    }
    D.f[1 + a][q] = upd(D.f[1 + a][q], (T)(D.bq[a] ? D.bq[a][q] : D.b0), d);
  }
}

template <class V>
__global__ void __launch_bounds__(256) update_p_ref(V D) {
  typedef typename V::real T;
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y * blockDim.y + threadIdx.y;
  const int k = blockIdx.z;
  if (i >= D.nx || j >= D.ny || k >= D.nz) return;
  const long long q = (long long)k * D.plane + (long long)j * D.pitch + i;
  const int g[3] = {i + D.ox, j + D.oy, k + D.oz};
  const int loc[3] = {i, j, k};
  T dd[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    const T* v = D.f[1 + a];
    const int ex = a == 0, ey = a == 1, ez = a == 2;
    T d = stag_diff(rd_ref(D, v, i, j, k), rd_ref(D, v, i - ex, j - ey, k - ez),
                    rd_ref(D, v, i + ex, j + ey, k + ez), rd_ref(D, v, i - 2 * ex, j - 2 * ey, k - 2 * ez),
                    rd_ref(D, v, i + 2 * ex, j + 2 * ey, k + 2 * ez), rd_ref(D, v, i - 3 * ex, j - 3 * ey, k - 3 * ez),
                    rd_ref(D, v, i + 3 * ex, j + 3 * ey, k + 3 * ez), rd_ref(D, v, i - 4 * ex, j - 4 * ey, k - 4 * ez));
    const int side = slab_side(D, a, loc[a]);
    if (side >= 0) {
      T* ps = D.psi[1][a][side] + psi_index(D, a, side, i, j, k);
      T s = *ps;
      d = cpml_apply(d, s, (T)D.tab[1][a][0][g[a]], (T)D.tab[1][a][1][g[a]], (T)D.tab[1][a][2][g[a]]);
      *ps = s;
    }
    dd[a] = d;
  }
  const T kc = (T)(D.kc ? D.kc[q] : D.kc0);
  D.f[0][q] = upd(D.f[0][q], kc, add3(dd[0], dd[1], dd[2]));
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
      "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1, %2;\n"
      "@P1 bra DONE;\n"
      "bra WAIT_LOOP;\n"
      "DONE:\n"
      "}\n" ::"r"(smem_u32(bar)),
      "r"(parity), "r"(0x989680)   // suspend-time hint: the warp sleeps in hardware instead of spinning on the issue port
      : "memory");
}
// non-blocking probe of a phase (used one iteration early, so that its latency overlaps with arithmetic)
__device__ __forceinline__ bool mbar_test(uint64_t* bar, uint32_t parity) {
  uint32_t done;
  asm volatile(
      "{\n"
      ".reg .pred P1;\n"
      "mbarrier.test_wait.parity.shared::cta.b64 P1, [%1], %2;\n"
      "selp.u32 %0, 1, 0, P1;\n"
      "}\n"
      : "=r"(done)
      : "r"(smem_u32(bar)), "r"(parity)
      : "memory");
  return done != 0;
}
__device__ __forceinline__ void tma_load_3d(void* dst, const CUtensorMap* map, uint64_t* bar, int c0, int c1, int c2) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];" ::"r"(smem_u32(dst)),
      "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2)
      : "memory");
}
// non-binding prefetch of one 128-B line into L2 (psi of a later plane: streamed once, so only latency matters)
__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }
__device__ __forceinline__ void fence_barrier_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// ---------------------------------------------------------------- tiled kernels
// Persistent CTAs (grid = resident CTAs of the whole GPU) pull work items from an atomic counter.  One item is a
// 64x16 (x,y) tile over a chunk of z planes.  Every streamed operand of an item arrives in shared memory through TMA
// into an NS-stage ring: a "full" mbarrier per stage is armed with the stage's byte count, an "empty" mbarrier
// collects one arrival per warp once the warp has read the stage, and one elected thread refills the stage used in
// the previous iteration — no CTA-wide barrier inside the plane loop.  Results leave through 128-bit stores; the
// z neighbours live in a register queue.  CPML slabs are handled by block-uniform branches (x / y per item, z per
// plane) with slab-local psi arrays read and written directly.
constexpr int TX = 64;             // tile width in x (floats): 16 lanes x 4
constexpr int TY = 16;             // tile height in y (rows)
constexpr int NT = 256;            // threads per CTA
constexpr int NW = NT / 32;        // warps per CTA
constexpr int NS = 4;              // ring stages
constexpr int PSI_AHEAD = 3;       // planes of psi prefetched into L2 ahead of their use in the x / y slabs
constexpr int HW = TX + 8;         // x-halo tile width: columns x0-4 .. x0+TX+3
constexpr int VH = TY + 7;         // p rows for update_v: y0-3 .. y0+TY+3
constexpr int PH = TY + 8;         // vy rows for update_p: y0-4 .. y0+TY+3
constexpr int TILE_FLOATS = TX * TY;
constexpr int TILE_BYTES = TILE_FLOATS * 4;
// update_v stage: [p halo tile | vx | vy | vz]
constexpr int V_P_BYTES = HW * VH * 4;
constexpr int V_P_FLOATS = ((V_P_BYTES + 127) / 128) * 32;     // keep every TMA destination 128-B aligned
constexpr int V_OFF_VX = V_P_FLOATS, V_OFF_VY = V_OFF_VX + TILE_FLOATS, V_OFF_VZ = V_OFF_VY + TILE_FLOATS;
constexpr int V_STAGE_FLOATS = V_OFF_VZ + TILE_FLOATS;
constexpr int V_SMEM_BYTES = NS * V_STAGE_FLOATS * 4;
// update_p stage: [vx x-halo tile | vy y-halo tile | vz | p | kc]
constexpr int P_VX_BYTES = HW * TY * 4;
constexpr int P_VY_BYTES = TX * PH * 4;
constexpr int P_OFF_VY = P_VX_BYTES / 4, P_OFF_VZ = P_OFF_VY + P_VY_BYTES / 4, P_OFF_P = P_OFF_VZ + TILE_FLOATS, P_OFF_KC = P_OFF_P + TILE_FLOATS;
constexpr int P_STAGE_FLOATS = P_OFF_KC + TILE_FLOATS;
constexpr int P_SMEM_BYTES = NS * P_STAGE_FLOATS * 4;
static_assert(P_VX_BYTES % 128 == 0 && P_VY_BYTES % 128 == 0 && TILE_BYTES % 128 == 0, "TMA destinations must stay 128-B aligned");

struct TMaps {
  CUtensorMap p_halo;     // p,  box HW x VH   (update_v)
  CUtensorMap vx_halo;    // vx, box HW x TY   (update_p)
  CUtensorMap vy_halo;    // vy, box TX x PH   (update_p)
  CUtensorMap tile[5];    // p, vx, vy, vz, kc with box TX x TY
  CUtensorMap p_box;      // p,  box (TX+16) x (TY+14)   (step_fused)
  CUtensorMap bq_halo[2]; // dt/(rho_bar dx) of vx, box HW x TY; of vy, box TX x PH   (step_fused<true>)
  CUtensorMap bq_tile;    // dt/(rho_bar dx) of vz, box TX x TY                         (step_fused<true>)
  CUtensorMap psi_x[2][2]; // x-slab psi [family][side] as (w, ny, nz), box PXW x TY   (step_fused<false>, psi through the stage)
  CUtensorMap psi_y[2][2]; // y-slab psi [family][side] as (nx, rows, nz), box TX x TY (step_fused<false>, psi through the stage)
};
constexpr int PXW = 40;    // widest x slab (columns, multiple of 4) whose psi goes through the TMA stage

// Work decomposition of one launch (same for both sub-updates of a domain).
struct Sched {
  int ntx, nty, nzc, zchunk;   // tiles in x, y; chunks in z; planes per chunk
  int nitems;
  unsigned int* counter;       // this launch's work counter
  unsigned int* other;         // the counter of the next launch on this domain: reset here
  const int4* table;           // optional: item -> (x0, y0, z0, z1) in the order they are handed out (nullptr: tile-major decode)
  int psi_tma;                 // step_fused: the x / y slab psi of the main warps arrives through the TMA stage (host-checked: slabs
                               // at most PXW columns wide, no tile touches both slabs of an axis, no density arrays)
};

// Four consecutive x values held in registers; moved as one 128-bit access.
struct V4 { float v[4]; };
__device__ __forceinline__ V4 from4(float4 f) { V4 r; r.v[0] = f.x; r.v[1] = f.y; r.v[2] = f.z; r.v[3] = f.w; return r; }
__device__ __forceinline__ V4 ldg4(const float* p) { return from4(__ldg(reinterpret_cast<const float4*>(p))); }
__device__ __forceinline__ V4 ld4(const float* p) { return from4(*reinterpret_cast<const float4*>(p)); }
__device__ __forceinline__ void st4(float* p, const V4& a) { *reinterpret_cast<float4*>(p) = make_float4(a.v[0], a.v[1], a.v[2], a.v[3]); }
__device__ __forceinline__ V4 splat4(float x) { V4 r; r.v[0] = r.v[1] = r.v[2] = r.v[3] = x; return r; }
__device__ __forceinline__ V4 zero4() { return splat4(0.f); }

// D along x for four consecutive outputs from the 12 values w[n] = f[i-4+n]:
//   FWD (D+ at i+e+1/2): f[i+e+l] - f[i+e-l+1];  BWD (D- at node i+e): f[i+e+l-1] - f[i+e-l]
template <bool FWD>
__device__ __forceinline__ V4 diff_x(const V4& l, const V4& c, const V4& r) {
  const float w[12] = {l.v[0], l.v[1], l.v[2], l.v[3], c.v[0], c.v[1], c.v[2], c.v[3], r.v[0], r.v[1], r.v[2], r.v[3]};
  V4 d;
#pragma unroll
  for (int e = 0; e < 4; ++e) {
    const int o = FWD ? 4 + e : 3 + e;
    d.v[e] = stag_diff(w[o + 1], w[o], w[o + 2], w[o - 1], w[o + 3], w[o - 2], w[o + 4], w[o - 3]);
  }
  return d;
}
__device__ __forceinline__ float2 pk(float a, float b) { return make_float2(a, b); }
__device__ __forceinline__ float2 sub2(float2 a, float2 b) { return __fadd2_rn(a, make_float2(-b.x, -b.y)); }
__device__ __forceinline__ float2 stag_diff2(float2 h1, float2 l1, float2 h2, float2 l2, float2 h3, float2 l3, float2 h4, float2 l4) {
  float2 d = mul2(pk(FDTD_C1, FDTD_C1), sub2(h1, l1));
  d = mad2(pk(FDTD_C2, FDTD_C2), sub2(h2, l2), d);
  d = mad2(pk(FDTD_C3, FDTD_C3), sub2(h3, l3), d);
  d = mad2(pk(FDTD_C4, FDTD_C4), sub2(h4, l4), d);
  return d;
}
__device__ __forceinline__ float2 lo2(const V4& a) { return make_float2(a.v[0], a.v[1]); }
__device__ __forceinline__ float2 hi2(const V4& a) { return make_float2(a.v[2], a.v[3]); }
__device__ __forceinline__ V4 join2(float2 a, float2 b) { V4 r; r.v[0] = a.x; r.v[1] = a.y; r.v[2] = b.x; r.v[3] = b.y; return r; }
__device__ __forceinline__ V4 diff_8(const V4& h1, const V4& l1, const V4& h2, const V4& l2, const V4& h3, const V4& l3, const V4& h4,
                                     const V4& l4) {
  return join2(stag_diff2(lo2(h1), lo2(l1), lo2(h2), lo2(l2), lo2(h3), lo2(l3), lo2(h4), lo2(l4)),
               stag_diff2(hi2(h1), hi2(l1), hi2(h2), hi2(l2), hi2(h3), hi2(l3), hi2(h4), hi2(l4)));
}
// f - coef d for four points, coefficients (c01, c01, c2, c3)
__device__ __forceinline__ V4 upd4(const V4& f, float c01, float c2, float c3, const V4& d) {
  return join2(mad2(pk(-c01, -c01), lo2(d), lo2(f)), mad2(pk(-c2, -c3), hi2(d), hi2(f)));
}
// The pinned last half node of the x axis (R3) inside a float4 that starts at global column g: its element index, or 4
// if the float4 does not hold it.  When Nx is a multiple of 4 it is always element 3 (the fast path of the callers).
__device__ __forceinline__ int pinned_x_element(int g, int gnx) {
  const unsigned e = (unsigned)(gnx - 1 - g);
  return e < 4u ? (int)e : 4;
}
// f - c d for four points with the coefficient zeroed from element `pin` on (4: none): the pinned half node keeps its
// value, and the elements behind it lie outside the grid, where v is 0 (R4) — they arrive as zeros (TMA bounds) and must stay
// zeros, because the single-pass step hands vx_new to the neighbouring columns through shared memory.
__device__ __forceinline__ V4 upd4_pin(const V4& f, float c, int pin, const V4& d) {
  return join2(mad2(pk(pin <= 0 ? -0.f : -c, pin <= 1 ? -0.f : -c), lo2(d), lo2(f)), mad2(pk(pin <= 2 ? -0.f : -c, pin <= 3 ? -0.f : -c), hi2(d), hi2(f)));
}
// An exact packed product for the CPML terms: fma(a, b, -0) is the rounded product bit for bit (signed zeros, subnormals,
// infinities and NaNs included), and an FFMA2 cannot be folded into the FADD2 that consumes it the way ptxas folds a packed
// multiply.  The -0 comes from constant memory, so that the compiler cannot see its value and turn the fma back into a
// multiply.  Used in the slab code only: it halves the multiplies of a CPML term (three products per point), which is what a
// slab plane pays on top of an interior one; in the stencil sums it changed no measured time (profiles/r02_ncu_step_fused.md).
__constant__ float2 c_negzero2 = {-0.0f, -0.0f};
__device__ __forceinline__ float2 mul2x(float2 a, float2 b) { return __ffma2_rn(a, b, c_negzero2); }
__device__ __forceinline__ float2 mad2x(float2 a, float2 b, float2 c) { return __fadd2_rn(mul2x(a, b), c); }
__device__ __forceinline__ void cpml4(V4& d, V4& ps, const V4& a, const V4& b, const V4& ik) {
  const float2 p0 = mad2x(lo2(b), lo2(ps), mul2x(lo2(a), lo2(d))), p1 = mad2x(hi2(b), hi2(ps), mul2x(hi2(a), hi2(d)));
  d = join2(mad2x(lo2(d), lo2(ik), p0), mad2x(hi2(d), hi2(ik), p1));
  ps = join2(p0, p1);
}
__device__ __forceinline__ void cpml4s(V4& d, V4& ps, float a, float b, float ik) {
  const float2 a2 = pk(a, a), b2 = pk(b, b), k2 = pk(ik, ik);
  const float2 p0 = mad2x(b2, lo2(ps), mul2x(a2, lo2(d))), p1 = mad2x(b2, hi2(ps), mul2x(a2, hi2(d)));
  d = join2(mad2x(lo2(d), k2, p0), mad2x(hi2(d), k2, p1));
  ps = join2(p0, p1);
}

// ring bookkeeping shared by both kernels
struct Ring {
  uint64_t* full;
  uint64_t* empty;
};
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// the warp has finished reading stage `slot`
__device__ __forceinline__ void release_stage(const Ring& R, unsigned slot) {
  __syncwarp();
  if ((threadIdx.x & 31) == 0) mbar_arrive(&R.empty[slot]);
}

__device__ __forceinline__ bool touches(const DomainView& D, int axis, int lo, int hi) {
  return (D.ln[axis][0] > 0 && lo < D.ls[axis][0] + D.ln[axis][0] && hi > D.ls[axis][0]) ||
         (D.ln[axis][1] > 0 && lo < D.ls[axis][1] + D.ln[axis][1] && hi > D.ls[axis][1]);
}

// CPML tables [a, b, 1/kappa] of the item's 64 columns and 16 rows in shared memory: the per-plane global table loads sat
// right before their use in the slab items (long-scoreboard stalls in the ncu source view of step_fused and of these).
struct TabCache1 {
  float x[3][TX];
  float y[3][TY];
};
__device__ __forceinline__ void fill_tab_cache1(const DomainView& D, TabCache1& T, int fam, int x0, int y0) {
  for (int t = threadIdx.x; t < 3 * TX; t += NT) T.x[t / TX][t % TX] = __ldg(D.tab[fam][0][t / TX] + min(x0 + t % TX + D.ox, D.gn[0] - 1));
  for (int t = threadIdx.x; t < 3 * TY; t += NT) T.y[t / TY][t % TY] = __ldg(D.tab[fam][1][t / TY] + min(y0 + t % TY + D.oy, D.gn[1] - 1));
  __syncthreads();
}

// ---- velocity sub-update: v_a <- v_a - B [(1/kappa_a) D+_a p + psi_va] for one item.
// On arrival of stage "p plane m": vx, vy of plane m are updated from the tile, p[m] enters the register queue and
// vz of plane m-4 is updated from the queue (D+_z at k+1/2 reads p[k-3 .. k+4]).  The pinned last half node of each
// axis (R3) is kept by a zero update coefficient (its psi stays 0 through a zero `a` in the device table).
template <bool HB>
__device__ __forceinline__ void v_item(const TMaps& tm, const DomainView& D, float* smem, const Ring& R, TabCache1& T, unsigned& it, int x0,
                                       int y0, int z0, int z1) {
  const int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;
  const int i = x0 + 4 * tx, j = y0 + ty;
  const int m_begin = z0 - 3, m_end = z1 + 4;

  auto issue = [&](unsigned slot, int m) {
    const bool xy = m >= z0 && m < z1, zz = (m - 4) >= z0 && (m - 4) < z1;
    uint64_t* bar = &R.full[slot];
    float* st = smem + slot * V_STAGE_FLOATS;
    mbar_expect_tx(bar, V_P_BYTES + (xy ? 2 * TILE_BYTES : 0) + (zz ? TILE_BYTES : 0));
    tma_load_3d(st, &tm.p_halo, bar, x0 - 4, y0 - 3, m);
    if (xy) {
      tma_load_3d(st + V_OFF_VX, &tm.tile[1], bar, x0, y0, m);
      tma_load_3d(st + V_OFF_VY, &tm.tile[2], bar, x0, y0, m);
    }
    if (zz) tma_load_3d(st + V_OFF_VZ, &tm.tile[3], bar, x0, y0, m - 4);
  };
  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < NS; ++s)
      if (m_begin + s < m_end) issue((it + s) % NS, m_begin + s);
  }

  const bool active = (i < D.nx) && (j < D.ny);
  const float B = D.b0;
  const long long rowoff = (long long)j * D.pitch + i;
  float* gvx = D.f[1] + rowoff + (long long)z0 * D.plane;
  float* gvy = D.f[2] + rowoff + (long long)z0 * D.plane;
  float* gvz = D.f[3] + rowoff + (long long)z0 * D.plane;
  // heterogeneous density (HB): dt/(rho_bar dx) per half node, read straight from global memory (one reader per value)
  const float* gbx = HB ? D.bq[0] + rowoff + (long long)z0 * D.plane : nullptr;
  const float* gby = HB ? D.bq[1] + rowoff + (long long)z0 * D.plane : nullptr;
  const float* gbz = HB ? D.bq[2] + rowoff + (long long)z0 * D.plane : nullptr;
  const int poff = (ty + 3) * HW + 4 * tx + 4;      // own float4 inside the p halo tile
  const int toff = ty * TX + 4 * tx;                // own float4 inside a plain tile
  // pinned last half nodes: zero coefficient
  const int pinx = pinned_x_element(i + D.ox, D.gn[0]);
  const float By = (j + D.oy) == D.gn[1] - 1 ? 0.f : B;
  // CPML: block-uniform "does this item touch an x / y slab", per-thread "is my float4 / row inside one"
  const bool any_x = touches(D, 0, x0, x0 + TX), any_y = touches(D, 1, y0, y0 + TY);
  if (any_x || any_y) fill_tab_cache1(D, T, 0, x0, y0);          // block-uniform
  const int sx = (any_x && active) ? slab_side(D, 0, i) : -1;
  const int sy = (any_y && active) ? slab_side(D, 1, j) : -1;
  float* ppx = sx >= 0 ? D.psi[0][0][sx] + psi_index(D, 0, sx, i, j, z0) : nullptr;
  float* ppy = sy >= 0 ? D.psi[0][1][sy] + psi_index(D, 1, sy, i, j, z0) : nullptr;
  const long long stride_px = sx >= 0 ? (long long)D.ny * D.ln[0][sx] : 0;
  const long long stride_py = sy >= 0 ? (long long)D.ln[1][sy] * D.pitch : 0;

  V4 q0 = zero4(), q1 = zero4(), q2 = zero4(), q3 = zero4(), q4 = zero4(), q5 = zero4(), q6 = zero4(), q7 = zero4();
  bool pre = false;   // the next stage's barrier was already seen complete by a non-blocking probe (a blocking wait costs ~300 cycles even then)

  for (int m = m_begin; m < m_end; ++m, ++it) {
    const unsigned slot = it % NS;
    const bool xy = m >= z0 && m < z1;
    const int kz = m - 4;
    const bool zz = kz >= z0 && kz < z1;
    // psi of this iteration: issue the loads before waiting on the tile
    V4 psx, psy, psz;
    const int sz = zz ? slab_side(D, 2, kz) : -1;
    float* ppz = nullptr;
    if (xy && sx >= 0) { psx = ld4(ppx); prefetch_l2(ppx + PSI_AHEAD * stride_px); }
    if (xy && sy >= 0) { psy = ld4(ppy); prefetch_l2(ppy + PSI_AHEAD * stride_py); }
    if (sz >= 0 && active) { ppz = D.psi[0][2][sz] + psi_index(D, 2, sz, i, j, kz); psz = ld4(ppz); }
    V4 bx4, by4, bz4;
    if (HB) {
      if (xy && active) { bx4 = ldg4(gbx); by4 = ldg4(gby); }
      if (zz && active) bz4 = ldg4(gbz);
    }
    const float* st = smem + slot * V_STAGE_FLOATS;
    if (!pre) mbar_wait(&R.full[slot], (it / NS) & 1);

    const float* row = st + poff;
    const V4 c = ld4(row);
    V4 dxv, dyv, vx4, vy4, vz4;
    if (xy) {
      dxv = diff_x<true>(ld4(row - 4), c, ld4(row + 4));
      dyv = diff_8(ld4(row + HW), c, ld4(row + 2 * HW), ld4(row - HW), ld4(row + 3 * HW), ld4(row - 2 * HW), ld4(row + 4 * HW),
                   ld4(row - 3 * HW));
      vx4 = ld4(st + V_OFF_VX + toff);
      vy4 = ld4(st + V_OFF_VY + toff);
    }
    if (zz) vz4 = ld4(st + V_OFF_VZ + toff);
    release_stage(R, slot);
    pre = mbar_test(&R.full[(it + 1) % NS], ((it + 1) / NS) & 1);
    // producer duty, after this thread's own shared-memory loads of the iteration: a lane that has just issued tensor
    // copies sees its next shared-memory loads stall for about a thousand cycles (traced on step_fused).  Refill the stage
    // every warp released in the previous iteration.
    if (tid == 0 && m > m_begin && (m - 1 + NS) < m_end) {
      const unsigned ps = (it - 1) % NS;
      mbar_wait(&R.empty[ps], ((it - 1) / NS) & 1);
      issue(ps, m - 1 + NS);
    }
    q0 = q1; q1 = q2; q2 = q3; q3 = q4; q4 = q5; q5 = q6; q6 = q7; q7 = c;     // q7 = p[m] ... q0 = p[m-7]

    if (xy) {
      if (any_x) {
        if (sx >= 0) {
          cpml4(dxv, psx, ld4(T.x[0] + 4 * tx), ld4(T.x[1] + 4 * tx), ld4(T.x[2] + 4 * tx));
          st4(ppx, psx);
          ppx += stride_px;
        }
      }
      if (any_y) {
        if (sy >= 0) {
          cpml4s(dyv, psy, T.y[0][ty], T.y[1][ty], T.y[2][ty]);
          st4(ppy, psy);
          ppy += stride_py;
        }
      }
      if (HB) {
        const bool lasty = (j + D.oy) == D.gn[1] - 1;
#pragma unroll
        for (int e = 0; e < 4; ++e) {
          vx4.v[e] = upd(vx4.v[e], e >= pinx ? 0.f : bx4.v[e], dxv.v[e]);
          vy4.v[e] = upd(vy4.v[e], lasty ? 0.f : by4.v[e], dyv.v[e]);
        }
        gbx += D.plane;
        gby += D.plane;
      } else {
#pragma unroll
        for (int e = 0; e < 4; ++e) vx4.v[e] = upd(vx4.v[e], e >= pinx ? 0.f : B, dxv.v[e]);
#pragma unroll
        for (int e = 0; e < 4; ++e) vy4.v[e] = upd(vy4.v[e], By, dyv.v[e]);
      }
      if (active) { st4(gvx, vx4); st4(gvy, vy4); }
      gvx += D.plane;
      gvy += D.plane;
    }
    if (zz) {
      // D+_z at kz+1/2: p[kz+l] = q(3+l), p[kz-l+1] = q(4-l)
      V4 dzv = diff_8(q4, q3, q5, q2, q6, q1, q7, q0);
      const int gk = kz + D.oz;
      if (sz >= 0 && active) {
        cpml4s(dzv, psz, __ldg(D.tab[0][2][0] + gk), __ldg(D.tab[0][2][1] + gk), __ldg(D.tab[0][2][2] + gk));
        st4(ppz, psz);
      }
      const float Bz = gk == D.gn[2] - 1 ? 0.f : B;
#pragma unroll
      for (int e = 0; e < 4; ++e) vz4.v[e] = upd(vz4.v[e], HB ? (gk == D.gn[2] - 1 ? 0.f : bz4.v[e]) : Bz, dzv.v[e]);
      if (active) st4(gvz, vz4);
      gvz += D.plane;
      if (HB) gbz += D.plane;
    }
  }
}

__device__ __forceinline__ bool next_item(const Sched& S, int* s_item, int& x0, int& y0, int& z0, int& z1, int nz) {
  __syncthreads();                                   // previous item fully consumed (all stages released, s_item read)
  if (threadIdx.x == 0) *s_item = (int)atomicAdd(S.counter, 1u);
  __syncthreads();
  const int item = *s_item;
  if (item >= S.nitems) return false;
  if (S.table) {
    const int4 t = __ldg(S.table + item);
    x0 = t.x; y0 = t.y; z0 = t.z; z1 = t.w;
    return true;
  }
  const int txi = item % S.ntx, r = item / S.ntx;
  const int tyi = r % S.nty, zc = r / S.nty;
  x0 = txi * TX; y0 = tyi * TY; z0 = zc * S.zchunk; z1 = min(z0 + S.zchunk, nz);
  return true;
}

__device__ __forceinline__ void ring_init(uint64_t* full, uint64_t* empty, unsigned int* other) {
  if (threadIdx.x == 0) {
#pragma unroll
    for (int s = 0; s < NS; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], NW); }
    fence_barrier_init();
    if (blockIdx.x == 0) *other = 0u;                // arm the next launch's work counter
  }
}

template <bool HB>
__global__ void __launch_bounds__(NT, 2) update_v_tiled(const __grid_constant__ TMaps tm, const __grid_constant__ DomainView D,
                                                        const __grid_constant__ Sched S) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  float* smem = reinterpret_cast<float*>(smem_raw);
  __shared__ __align__(8) uint64_t full[NS];
  __shared__ __align__(8) uint64_t empty[NS];
  __shared__ int s_item;
  ring_init(full, empty, S.other);
  const Ring R{full, empty};
  unsigned it = 0;
  int x0, y0, z0, z1;
  __shared__ __align__(16) TabCache1 tabc;
  while (next_item(S, &s_item, x0, y0, z0, z1, D.nz)) v_item<HB>(tm, D, smem, R, tabc, it, x0, y0, z0, z1);
}

// ---- pressure sub-update: p <- p - Kc [sum_a (1/kappa_a) D-_a v_a + psi_pa] for one item.
// Stage "vz plane m" also carries vx (x-halo tile), vy (y-halo tile), p and Kc of plane k = m-3; vz[m] enters the
// register queue and p[k] is updated (D-_z at node k reads vz[k-4 .. k+3]).
__device__ __forceinline__ void p_item(const TMaps& tm, const DomainView& D, float* smem, const Ring& R, TabCache1& T, unsigned& it, int x0,
                                       int y0, int z0, int z1) {
  const int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;
  const int i = x0 + 4 * tx, j = y0 + ty;
  const int m_begin = z0 - 4, m_end = z1 + 3;
  const bool has_kc = D.kc != nullptr;

  auto issue = [&](unsigned slot, int m) {
    const int k = m - 3;
    const bool out = k >= z0;                        // k < z1 always holds for m < m_end
    uint64_t* bar = &R.full[slot];
    float* st = smem + slot * P_STAGE_FLOATS;
    mbar_expect_tx(bar, TILE_BYTES + (out ? P_VX_BYTES + P_VY_BYTES + TILE_BYTES + (has_kc ? TILE_BYTES : 0) : 0));
    tma_load_3d(st + P_OFF_VZ, &tm.tile[3], bar, x0, y0, m);
    if (out) {
      tma_load_3d(st, &tm.vx_halo, bar, x0 - 4, y0, k);
      tma_load_3d(st + P_OFF_VY, &tm.vy_halo, bar, x0, y0 - 4, k);
      tma_load_3d(st + P_OFF_P, &tm.tile[0], bar, x0, y0, k);
      if (has_kc) tma_load_3d(st + P_OFF_KC, &tm.tile[4], bar, x0, y0, k);
    }
  };
  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < NS; ++s)
      if (m_begin + s < m_end) issue((it + s) % NS, m_begin + s);
  }

  const bool active = (i < D.nx) && (j < D.ny);
  const long long rowoff = (long long)j * D.pitch + i;
  float* gp = D.f[0] + rowoff + (long long)z0 * D.plane;
  const int xoff = ty * HW + 4 * tx + 4;             // own float4 inside the vx x-halo tile
  const int toff = ty * TX + 4 * tx;                 // own float4 in a plain tile; row ty of the vy tile <-> y = y0-4+ty
  const float kc0 = D.kc0;
  const bool any_x = touches(D, 0, x0, x0 + TX), any_y = touches(D, 1, y0, y0 + TY);
  if (any_x || any_y) fill_tab_cache1(D, T, 1, x0, y0);          // block-uniform
  const int sx = (any_x && active) ? slab_side(D, 0, i) : -1;
  const int sy = (any_y && active) ? slab_side(D, 1, j) : -1;
  float* ppx = sx >= 0 ? D.psi[1][0][sx] + psi_index(D, 0, sx, i, j, z0) : nullptr;
  float* ppy = sy >= 0 ? D.psi[1][1][sy] + psi_index(D, 1, sy, i, j, z0) : nullptr;
  const long long stride_px = sx >= 0 ? (long long)D.ny * D.ln[0][sx] : 0;
  const long long stride_py = sy >= 0 ? (long long)D.ln[1][sy] * D.pitch : 0;

  V4 q0 = zero4(), q1 = zero4(), q2 = zero4(), q3 = zero4(), q4 = zero4(), q5 = zero4(), q6 = zero4(), q7 = zero4();
  bool pre = false;   // the next stage's barrier was already seen complete by a non-blocking probe (a blocking wait costs ~300 cycles even then)

  for (int m = m_begin; m < m_end; ++m, ++it) {
    const unsigned slot = it % NS;
    const int k = m - 3;
    const bool out = k >= z0;
    V4 psx, psy, psz;
    const int sz = out ? slab_side(D, 2, k) : -1;
    float* ppz = nullptr;
    if (out && sx >= 0) { psx = ld4(ppx); prefetch_l2(ppx + PSI_AHEAD * stride_px); }
    if (out && sy >= 0) { psy = ld4(ppy); prefetch_l2(ppy + PSI_AHEAD * stride_py); }
    if (sz >= 0 && active) { ppz = D.psi[1][2][sz] + psi_index(D, 2, sz, i, j, k); psz = ld4(ppz); }
    // producer duty before the wait (measured: here the early refill is worth more than the stall it causes, unlike update_v)
    if (tid == 0 && m > m_begin && (m - 1 + NS) < m_end) {
      const unsigned ps = (it - 1) % NS;
      mbar_wait(&R.empty[ps], ((it - 1) / NS) & 1);
      issue(ps, m - 1 + NS);
    }
    const float* st = smem + slot * P_STAGE_FLOATS;
    if (!pre) mbar_wait(&R.full[slot], (it / NS) & 1);

    q0 = q1; q1 = q2; q2 = q3; q3 = q4; q4 = q5; q5 = q6; q6 = q7; q7 = ld4(st + P_OFF_VZ + toff);   // q7 = vz[m] = vz[k+3]
    V4 dxv, dyv, p4, kc4;
    if (out) {
      const float* xr = st + xoff;
      dxv = diff_x<false>(ld4(xr - 4), ld4(xr), ld4(xr + 4));
      const float* col = st + P_OFF_VY + toff;
      // D-_y at node j: vy[j+l-1] = row(ty+3+l), vy[j-l] = row(ty+4-l)
      dyv = diff_8(ld4(col + 4 * TX), ld4(col + 3 * TX), ld4(col + 5 * TX), ld4(col + 2 * TX), ld4(col + 6 * TX), ld4(col + TX),
                   ld4(col + 7 * TX), ld4(col));
      p4 = ld4(st + P_OFF_P + toff);
      kc4 = has_kc ? ld4(st + P_OFF_KC + toff) : splat4(kc0);
    }
    release_stage(R, slot);
    pre = mbar_test(&R.full[(it + 1) % NS], ((it + 1) / NS) & 1);

    if (out) {
      // D-_z at node k: vz[k+l-1] = q(3+l), vz[k-l] = q(4-l)
      V4 dzv = diff_8(q4, q3, q5, q2, q6, q1, q7, q0);
      if (any_x) {
        if (sx >= 0) {
          cpml4(dxv, psx, ld4(T.x[0] + 4 * tx), ld4(T.x[1] + 4 * tx), ld4(T.x[2] + 4 * tx));
          st4(ppx, psx);
          ppx += stride_px;
        }
      }
      if (any_y) {
        if (sy >= 0) {
          cpml4s(dyv, psy, T.y[0][ty], T.y[1][ty], T.y[2][ty]);
          st4(ppy, psy);
          ppy += stride_py;
        }
      }
      if (sz >= 0 && active) {
        const int gk = k + D.oz;
        cpml4s(dzv, psz, __ldg(D.tab[1][2][0] + gk), __ldg(D.tab[1][2][1] + gk), __ldg(D.tab[1][2][2] + gk));
        st4(ppz, psz);
      }
#pragma unroll
      for (int e = 0; e < 4; ++e) p4.v[e] = upd(p4.v[e], kc4.v[e], __fadd_rn(__fadd_rn(dxv.v[e], dyv.v[e]), dzv.v[e]));
      if (active) st4(gp, p4);
      gp += D.plane;
    }
  }
}

__global__ void __launch_bounds__(NT, 2) update_p_tiled(const __grid_constant__ TMaps tm, const __grid_constant__ DomainView D,
                                                        const __grid_constant__ Sched S) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  float* smem = reinterpret_cast<float*>(smem_raw);
  __shared__ __align__(8) uint64_t full[NS];
  __shared__ __align__(8) uint64_t empty[NS];
  __shared__ int s_item;
  ring_init(full, empty, S.other);
  const Ring R{full, empty};
  unsigned it = 0;
  int x0, y0, z0, z1;
  __shared__ __align__(16) TabCache1 tabc;
  while (next_item(S, &s_item, x0, y0, z0, z1, D.nz)) p_item(tm, D, smem, R, tabc, it, x0, y0, z0, z1);
}


// ---------------------------------------------------------------- small kernels
// p[src_s] += w_s[n] for every source (R14).  The step index n is kept on the host and passed in, so steps taken
// before fdtd_set_sources count too.  Sources that share a node are added by the first of them, one after the other in
// source order — the order of the recurrence (oracle: a plain loop over the sources), and no lost update.
template <class T>
struct SourceViewT {
  int n, len;
  const long long* offset;   // flat element offset of each source in its domain's p array, or -1 if not held
  T* p;
  const float* wav;
  long long lo, hi;          // only sources whose offset lies in [lo, hi) (a plane range; everything: 0, LLONG_MAX)
};
typedef SourceViewT<float> SourceView;
template <class T>
__global__ void inject_sources(SourceViewT<T> S, long long n) {
  if (n >= S.len) return;
  for (int s = threadIdx.x; s < S.n; s += blockDim.x) {
    const long long off = S.offset[s];
    if (off < S.lo || off >= S.hi) continue;              // not held by this domain (-1), or outside the plane range
    bool first = true;
    for (int t = 0; t < s; ++t) first = first && S.offset[t] != off;
    if (!first) continue;
    T v = S.p[off];
    for (int t = s; t < S.n; ++t)
      if (S.offset[t] == off) v = v + (T)S.wav[(long long)t * S.len + n];      // one rounded addition per source
    S.p[off] = v;
  }
}

// In place: wave speed c (fp32) -> K dt/dx = rho c^2 dt/dx in double, rounded once to fp32 (R6).  Padding columns stay 0.
__global__ void speed_to_kc_kernel(float* a, long long n, int pitch, int nx, double rho, double dt, double dx) {
  for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += (long long)gridDim.x * blockDim.x) {
    if ((int)(t % pitch) >= nx) { a[t] = 0.f; continue; }
    const double c = (double)a[t];
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
template <class V>
__global__ void fill_hash_kernel(V D, int which, uint64_t seed, float scale) {
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

template <class V>
__global__ void absmax_kernel(V D, int which, int lx, int ly, int lz, int sx, int sy, int sz, unsigned int* out) {
  const long long n = (long long)sx * sy * sz;
  float m = 0.f;
  for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += (long long)gridDim.x * blockDim.x) {
    const int i = (int)(t % sx);
    const long long r = t / sx;
    const int j = (int)(r % sy), k = (int)(r / sy);
    m = fmaxf(m, fabsf((float)D.f[which][(long long)(k + lz) * D.plane + (long long)(j + ly) * D.pitch + (i + lx)]));
  }
  for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
  if ((threadIdx.x & 31) == 0) atomicMax(out, __float_as_uint(m));   // non-negative floats order like unsigned ints
}

// Expand one slab-local psi array into a full-volume scratch array (debug / parity of the recursion).
template <class V>
__global__ void expand_psi_kernel(V D, int fam, int axis, typename V::real* out /* nx*ny*nz packed */) {
  const long long n = (long long)D.nx * D.ny * D.nz;
  for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += (long long)gridDim.x * blockDim.x) {
    const int i = (int)(t % D.nx);
    const long long r = t / D.nx;
    const int j = (int)(r % D.ny), k = (int)(r / D.ny);
    const int loc[3] = {i, j, k};
    const int side = slab_side(D, axis, loc[axis]);
    out[t] = side >= 0 ? D.psi[fam][axis][side][psi_index(D, axis, side, i, j, k)] : 0;
  }
}

}  // namespace fdtd
