// Host side of the C ABI declared in include/fdtd_b200.h: workspace layout, CPML coefficient setup,
// TMA descriptors, launch orchestration of one time step, halo exchange of the in-HBM subdomain mode
// (P:76-82).  No CPU fallback: every compute entry point needs a CUDA device.
#include "../../include/fdtd_b200.h"
#include "fdtd_kernels.cuh"
#include "fdtd_fused.cuh"

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <string>
#include <thread>
#include <algorithm>
#include <vector>

using namespace fdtd;

namespace {

thread_local std::string g_err;
void set_err(const std::string& s) { g_err = s; }

#define CK(call)                                                                                   \
  do {                                                                                             \
    cudaError_t e_ = (call);                                                                       \
    if (e_ != cudaSuccess) {                                                                       \
      set_err(std::string(#call) + ": " + cudaGetErrorString(e_));                                 \
      return FDTD_ECUDA;                                                                           \
    }                                                                                              \
  } while (0)

inline uint64_t align_up(uint64_t v, uint64_t a) { return (v + a - 1) / a * a; }
inline int round_up(int v, int a) { return (v + a - 1) / a * a; }

// ---- CPML tables (readings R7-R9) -------------------------------------------------------------
struct AxisTable { std::vector<float> a, b, ik; };

AxisTable make_axis_table(int N, int L0, int L1, bool half, const fdtd_params& P) {
  AxisTable t;
  const int len = round_up(N, 4) + 4;
  t.a.assign(len, 0.0f); t.b.assign(len, 1.0f); t.ik.assign(len, 1.0f);
  const double q = (double)P.cpml_order;
  for (int i = 0; i < N; ++i) {
    const double pos = i + (half ? 0.5 : 0.0);
    double rho = 0.0; int L = 0;
    if (L0 > 0 && L0 - pos > 0.0) { rho = (L0 - pos) / L0; L = L0; }                              // low face
    else if (L1 > 0 && pos - (N - 1 - L1) > 0.0) { rho = (pos - (N - 1 - L1)) / L1; L = L1; }     // high face
    if (L == 0) continue;
    const double smax = -(q + 1.0) * P.cpml_c_ref * std::log(P.cpml_R0) / (2.0 * L * P.dx);
    const double rq = std::pow(rho, q);
    const double sig = smax * rq;
    const double kap = 1.0 + (P.cpml_kappa_max - 1.0) * rq;
    const double alp = P.cpml_alpha_max * std::fmax(0.0, 1.0 - rho);
    const double bb = std::exp(-(sig / kap + alp) * P.dt);
    const double den = kap * (sig + kap * alp);
    t.a[i] = (float)(den == 0.0 ? 0.0 : sig * (bb - 1.0) / den);
    t.b[i] = (float)bb;
    t.ik[i] = (float)(1.0 / kap);
  }
  return t;
}

// ---- geometry ------------------------------------------------------------------------------------------
struct Geometry {
  int gn[3];                 // global total grid
  int nd[3];                 // subdomain grid
  int ghost, msub;
  // global CPML storage slabs per axis: low [0, gs0), high [gh, gn) (x rounded to multiples of 4)
  int gs0[3], gh[3];
  bool valid = false;
  std::string why;
};

Geometry make_geometry(const fdtd_params& P) {
  Geometry G;
  auto bad = [&](const char* w) { G.valid = false; G.why = w; return G; };
  for (int a = 0; a < 3; ++a) {
    if (P.n_interior[a] <= 0) return bad("n_interior must be positive");
    if (P.cpml[2 * a] < 0 || P.cpml[2 * a + 1] < 0) return bad("cpml thickness must be >= 0");
    long long n = (long long)P.n_interior[a] + P.cpml[2 * a] + P.cpml[2 * a + 1];
    if (n > 100000) return bad("axis too long");
    G.gn[a] = (int)n;
    G.nd[a] = P.decomp[a] <= 0 ? 1 : P.decomp[a];
  }
  if (!(P.dx > 0.0) || !(P.dt > 0.0)) return bad("dx and dt must be positive");
  if (P.boundary != FDTD_WALL && P.boundary != FDTD_PERIODIC) return bad("unknown boundary");
  if (P.kernel < FDTD_KERNEL_AUTO || P.kernel > FDTD_KERNEL_FUSED) return bad("unknown kernel selector");
  if (P.kernel == FDTD_KERNEL_FUSED && P.boundary == FDTD_PERIODIC) return bad("FDTD_KERNEL_FUSED needs WALL boundaries");
  if (P.density != FDTD_DENSITY_UNIFORM && P.density != FDTD_DENSITY_ARRAY) return bad("unknown density selector");
  if (P.medium != FDTD_MEDIUM_ARRAY && P.medium != FDTD_MEDIUM_UNIFORM) return bad("unknown medium selector");
  if (P.precision != FDTD_PRECISION_FP32 && P.precision != FDTD_PRECISION_FP64) return bad("unknown precision selector");
  if (P.time_block < 0 || P.time_block > 8 || P.time_block_planes < 0) return bad("time_block must be 0 .. 8 and time_block_planes >= 0");
  if (P.time_block > 1 && P.kernel != FDTD_KERNEL_FUSED) return bad("time_block needs FDTD_KERNEL_FUSED");
  if (P.precision == FDTD_PRECISION_FP64 && P.kernel == FDTD_KERNEL_FUSED)
    return bad("the fp64 verification precision runs the one-thread-per-point kernels only (FDTD_KERNEL_AUTO or FDTD_KERNEL_REF)");
  if (P.boundary == FDTD_PERIODIC)
    for (int f = 0; f < 6; ++f) if (P.cpml[f]) return bad("PERIODIC excludes CPML");
  for (int f = 0; f < 6; ++f)
    if (P.cpml[f] > 0 && (!(P.cpml_R0 > 0.0) || P.cpml_order < 1 || !(P.cpml_kappa_max >= 1.0) || P.cpml_alpha_max < 0.0 || !(P.cpml_c_ref > 0.0)))
      return bad("bad CPML parameters");
  const bool sub = G.nd[0] * G.nd[1] * G.nd[2] > 1;
  if (sub && P.precision == FDTD_PRECISION_FP64) return bad("the fp64 verification precision is monolithic only");
  if (sub && P.time_block > 1) return bad("time_block is monolithic only");
  G.ghost = sub ? P.ghost : 0;
  G.msub = sub ? P.substeps_per_exchange : 0;
  if (sub) {
    if (P.boundary == FDTD_PERIODIC) return bad("subdomain mode needs WALL boundaries");
    if (G.msub < 1 || G.ghost < 4 * G.msub) return bad("ghost must be >= 4 * substeps_per_exchange");
    if (P.kernel == FDTD_KERNEL_FUSED && (G.msub % 2)) return bad("the fused step advances two sub-updates: substeps_per_exchange must be even");
    if (P.kernel == FDTD_KERNEL_FUSED && (G.gn[0] % 4)) return bad("FDTD_KERNEL_FUSED in subdomain mode needs a total Nx that is a multiple of 4");
    for (int a = 0; a < 3; ++a) {
      if (G.gn[a] % G.nd[a]) return bad("total grid not divisible by decomp");
      if (G.gn[a] / G.nd[a] < G.ghost) return bad("ghost deeper than a subdomain");
    }
    // an x cut (block-xy) keeps every subdomain's rows float4-aligned, and its ghost columns clear of the x layers
    if (G.nd[0] > 1) {
      const int own = G.gn[0] / G.nd[0];
      if ((own % 4) || (G.ghost % 4)) return bad("an x cut needs subdomain widths and a ghost depth that are multiples of 4");
      if (own - G.ghost < round_up(P.cpml[0], 4) + 4 || own - G.ghost < P.cpml[1] + 8) return bad("an x cut needs subdomains wider than ghost + CPML layer");
    }
  }
  for (int a = 0; a < 3; ++a) {
    const int L0 = P.cpml[2 * a], L1 = P.cpml[2 * a + 1];
    int s0 = L0, h = L1 > 0 ? G.gn[a] - 1 - L1 : G.gn[a];
    if (a == 0) { s0 = std::min(round_up(s0, 4), round_up(G.gn[a], 4)); h = h / 4 * 4; }
    if (h < 0) h = 0;
    if (L0 > 0 && L1 > 0 && s0 > h) return bad("grid smaller than its CPML layers");
    G.gs0[a] = s0; G.gh[a] = h;
  }
  G.valid = true;
  return G;
}

// One domain on the host: its view plus what the launches need.
struct Domain {
  DomainView v;
  DomainViewT<double> v64;     // FDTD_PRECISION_FP64: the same geometry with double fields and psi (v.f / v.psi then alias them)
  int own_lo[3], own_hi[3];    // owned cells in local indices
  int cx, cy, cz;              // position in the subdomain grid
  TMaps tm;
  OutSet alt;                  // fused mode: the other state (fields + psi); swapped with v.f / v.psi after every launch
  TMaps tm_alt;                // its tensor maps
  unsigned int* counters = nullptr;  // device: [0] update_v, [1] update_p, [2], [3] step_fused (alternating) work counters
  Sched sched;
  Sched sched_f;               // work decomposition of step_fused
  int fused_parity = 0;
  // time_block >= 2: scratch states and the launch list of one block of k steps (slab by slab, step by step)
  OutSet xs[2];
  TMaps tm_xs[2];
  struct TbLaunch { int zlo, zhi, in_state, out_state, step; const int4* table; int nitems; };   // states: 0 current, 1 out, 2 X, 3 Y
  std::vector<TbLaunch> tb;
  long long* src_offset = nullptr;   // device, per source
};

struct Layout {
  uint64_t total = 0;
  struct Dom {
    int n[3], o[3], pitch;
    int ls[3][2], ln[3][2];
    uint64_t f[4], kc, psi[2][3][2], src_off, counters;
    uint64_t f2[4], psi2[2][3][2];   // fused mode: second state
    uint64_t bq[3];                  // FDTD_DENSITY_ARRAY: dt/(rho_bar dx) at the half nodes of vx, vy, vz
    uint64_t items, items_cap;       // fused mode: item table of step_fused (int4 per item)
    uint64_t fx[2][4], psix[2][2][3][2];   // time_block >= 2: scratch states X, Y (intermediate steps of a z slab)
    uint64_t tb_items, tb_items_cap;       // ... and the item tables of its per-slab launches
    int tb_planes;                         // ... slab thickness
  };
  std::vector<Dom> doms;
  uint64_t tab[2][3][3];
  int tablen[3];
  uint64_t wav, absmax;
  bool has_kc = true;
};

constexpr int MAX_SRC = 64;
constexpr int MAX_WAV_FLOATS = 1 << 22;

Layout make_layout(const fdtd_params& P, const Geometry& G) {
  Layout L;
  L.has_kc = P.medium == FDTD_MEDIUM_ARRAY || P.density == FDTD_DENSITY_ARRAY;   // the K dt/dx array is optional (16.4 GB at 1600^3)
  uint64_t off = 0;
  auto take = [&](uint64_t bytes) { uint64_t o = off; off = align_up(off + bytes, 256); return o; };
  for (int cz = 0; cz < G.nd[2]; ++cz)
    for (int cy = 0; cy < G.nd[1]; ++cy)
     for (int cx = 0; cx < G.nd[0]; ++cx) {
      Layout::Dom d{};
      const int c[3] = {cx, cy, cz};
      for (int a = 0; a < 3; ++a) {
        const int own = G.gn[a] / G.nd[a];
        const int glo = c[a] > 0 ? G.ghost : 0, ghi = c[a] < G.nd[a] - 1 ? G.ghost : 0;
        d.n[a] = own + glo + ghi;
        d.o[a] = c[a] * own - glo;
        // local parts of the global storage slabs
        const int lo_end = std::min(G.gs0[a], d.o[a] + d.n[a]);       // global end of the low slab inside this domain
        d.ls[a][0] = 0; d.ln[a][0] = (P.cpml[2 * a] > 0 && d.o[a] < G.gs0[a]) ? std::max(0, lo_end - d.o[a]) : 0;
        const int hi_beg = std::max(G.gh[a], d.o[a]);
        d.ls[a][1] = hi_beg - d.o[a];
        d.ln[a][1] = (P.cpml[2 * a + 1] > 0 && d.o[a] + d.n[a] > G.gh[a]) ? std::max(0, d.o[a] + d.n[a] - hi_beg) : 0;
        if (d.ln[a][1] == 0) d.ls[a][1] = 0;
      }
      if (d.ln[0][0] > 0) d.ln[0][0] = round_up(d.ln[0][0], 4);
      if (d.ln[0][1] > 0) d.ln[0][1] = round_up(d.n[0] - d.ls[0][1], 4);
      d.pitch = round_up(d.n[0], 8);
      const uint64_t es = P.precision == FDTD_PRECISION_FP64 ? 8 : 4;          // bytes per field / psi element
      const uint64_t vol = (uint64_t)d.pitch * d.n[1] * d.n[2] * 4;            // one fp32 array (K dt/dx, dt/(rho_bar dx))
      for (int f = 0; f < 4; ++f) d.f[f] = take(vol / 4 * es);
      d.kc = L.has_kc ? take(vol) : 0;
      for (int fam = 0; fam < 2; ++fam)
        for (int s = 0; s < 2; ++s) {
          d.psi[fam][0][s] = take((uint64_t)d.ln[0][s] * d.n[1] * d.n[2] * es + 16);
          d.psi[fam][1][s] = take((uint64_t)d.pitch * d.ln[1][s] * d.n[2] * es + 16);
          d.psi[fam][2][s] = take((uint64_t)d.pitch * d.n[1] * d.ln[2][s] * es + 16);
        }
      if (P.kernel == FDTD_KERNEL_FUSED) {
        d.items_cap = (uint64_t)((d.n[0] + TX - 1) / TX) * ((d.n[1] + TY - 1) / TY) * (d.n[2] / 16 + 8);
        d.items = take(d.items_cap * 16);
        for (int f = 0; f < 4; ++f) d.f2[f] = take(vol);
        for (int fam = 0; fam < 2; ++fam)
          for (int s = 0; s < 2; ++s) {
            d.psi2[fam][0][s] = take((uint64_t)d.ln[0][s] * d.n[1] * d.n[2] * 4 + 16);
            d.psi2[fam][1][s] = take((uint64_t)d.pitch * d.ln[1][s] * d.n[2] * 4 + 16);
            d.psi2[fam][2][s] = take((uint64_t)d.pitch * d.n[1] * d.ln[2][s] * 4 + 16);
          }
      }
      if (P.kernel == FDTD_KERNEL_FUSED && P.time_block > 1) {
        for (int x = 0; x < (P.time_block > 2 ? 2 : 1); ++x) {
          for (int f = 0; f < 4; ++f) d.fx[x][f] = take(vol);
          for (int fam = 0; fam < 2; ++fam)
            for (int s = 0; s < 2; ++s) {
              d.psix[x][fam][0][s] = take((uint64_t)d.ln[0][s] * d.n[1] * d.n[2] * 4 + 16);
              d.psix[x][fam][1][s] = take((uint64_t)d.pitch * d.ln[1][s] * d.n[2] * 4 + 16);
              d.psix[x][fam][2][s] = take((uint64_t)d.pitch * d.n[1] * d.ln[2][s] * 4 + 16);
            }
        }
        // slab thickness: given, or such that the planes one slab touches (fields in + out, all its steps) stay near 64 MB
        // of the 126 MB L2; never thinner than the 8 planes of ghost one extra step costs on each side
        int zs = P.time_block_planes;
        if (zs <= 0) {
          const double per_plane = (double)d.pitch * d.n[1] * 4 * 8;
          zs = (int)(64e6 / per_plane) - 16 * (P.time_block - 1);
        }
        d.tb_planes = std::max(8, std::min(zs, d.n[2]));
        const uint64_t tiles = (uint64_t)((d.n[0] + TX - 1) / TX) * ((d.n[1] + TY - 1) / TY);
        const uint64_t nslab = (d.n[2] + d.tb_planes - 1) / d.tb_planes;
        d.tb_items_cap = tiles * nslab * P.time_block * (1 + (d.tb_planes + 16 * P.time_block) / 64) + 16;
        d.tb_items = take(d.tb_items_cap * 16);
      }
      if (P.density == FDTD_DENSITY_ARRAY)
        for (int a = 0; a < 3; ++a) d.bq[a] = take(vol);
      d.src_off = take(MAX_SRC * sizeof(long long));
      d.counters = take(64);
      L.doms.push_back(d);
    }
  for (int a = 0; a < 3; ++a) {
    L.tablen[a] = round_up(G.gn[a], 4) + 4;
    for (int fam = 0; fam < 2; ++fam)
      for (int t = 0; t < 3; ++t) L.tab[fam][a][t] = take((uint64_t)L.tablen[a] * 4);
  }
  L.absmax = take(64);
  L.wav = take((uint64_t)MAX_WAV_FLOATS * 4);
  L.total = off;
  return L;
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

}  // namespace

struct fdtd_ctx {
  fdtd_params P;
  Geometry G;
  Layout L;
  char* ws;
  cudaStream_t stream;
  std::vector<Domain> doms;
  AxisTable tabs[2][3];
  std::vector<float> dev_a[2][3];
  bool use_ref;
  bool fp64 = false;
  size_t es = 4;                // bytes per field / psi element
  bool fused = false;
  int grid_f = 0;
  int nsrc = 0, wlen = 0;
  long long step_index = 0;      // time steps taken since fdtd_create (the wavelet index of the next injection, R14)
  float* d_wav;
  int64_t launches = 0;
  int64_t substeps_done = 0;    // sub-updates since the last halo exchange (subdomain mode)
  int time_block = 1;           // steps advanced per z-slab pass (FDTD_KERNEL_FUSED)
  int64_t plane_steps_computed = 0, plane_steps_owned = 0;   // time_block: redundant-compute counters (planes x steps)
  int grid_v = 0, grid_p = 0;       // resident CTAs of the whole GPU for each tiled kernel
};

namespace {

int make_tmap(EncodeTiledFn enc, CUtensorMap* m, float* base, const DomainView& v, int bw, int bh) {
  cuuint64_t dims[3] = {(cuuint64_t)v.nx, (cuuint64_t)v.ny, (cuuint64_t)v.nz};
  cuuint64_t strides[2] = {(cuuint64_t)v.pitch * 4, (cuuint64_t)v.plane * 4};
  cuuint32_t box[3] = {(cuuint32_t)bw, (cuuint32_t)bh, 1};
  cuuint32_t estr[3] = {1, 1, 1};
  CUresult r = enc(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, base, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                   CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) { set_err("cuTensorMapEncodeTiled failed with CUresult " + std::to_string((int)r)); return FDTD_ECUDA; }
  return FDTD_OK;
}

// x / y slab psi as tensors for the single-pass step's stage: the x slab [nz][ny][w] with a PXW x TY box, the y slab
// [nz][rows][pitch] with a TX x TY box.
int make_tmap_psi(EncodeTiledFn enc, CUtensorMap* m, float* base, int d0, int d1, int d2, long long row_stride, int bw) {
  cuuint64_t dims[3] = {(cuuint64_t)d0, (cuuint64_t)d1, (cuuint64_t)d2};
  cuuint64_t strides[2] = {(cuuint64_t)row_stride * 4, (cuuint64_t)row_stride * 4 * (cuuint64_t)d1};
  cuuint32_t box[3] = {(cuuint32_t)bw, (cuuint32_t)TY, 1};
  cuuint32_t estr[3] = {1, 1, 1};
  CUresult r = enc(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, base, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                   CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) { set_err("cuTensorMapEncodeTiled (psi) failed with CUresult " + std::to_string((int)r)); return FDTD_ECUDA; }
  return FDTD_OK;
}

// Can the x / y slab psi of this domain go through the TMA stage of step_fused?  The x slabs must fit the staged box and no
// tile may touch both slabs of an axis (a tile's box comes from one slab array).
bool psi_tma_ok(const DomainView& v) {
  for (int s = 0; s < 2; ++s) if (v.ln[0][s] > PXW) return false;
  const int tile[2] = {TX, TY}, n[2] = {v.nx, v.ny};
  for (int a = 0; a < 2; ++a) {
    if (v.ln[a][0] == 0 || v.ln[a][1] == 0) continue;
    for (int t0 = 0; t0 < n[a]; t0 += tile[a])
      if (t0 < v.ls[a][0] + v.ln[a][0] && t0 + tile[a] > v.ls[a][1]) return false;
  }
  return true;
}

// Persistent launch plan: grid = resident CTAs; items = tiles x z-chunks with enough items per CTA for balance.
int plan_launch(fdtd_ctx* c, const void* kernel, int smem, int* grid, int threads = NT) {
  int per_sm = 0, sms = 148;
  CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, threads, smem));
  CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, c->P.device));
  if (per_sm < 1) { set_err("tiled kernel does not fit on an SM"); return FDTD_ECUDA; }
  *grid = per_sm * sms;
  return FDTD_OK;
}

void plan_items(Domain& d, int grid) {
  const DomainView& v = d.v;
  Sched& S = d.sched;
  S.ntx = (v.nx + TX - 1) / TX;
  S.nty = (v.ny + TY - 1) / TY;
  const long long tiles = (long long)S.ntx * S.nty;
  // about 8 items per resident CTA, chunks of 16..64 planes (each chunk re-reads 7 planes of the z-halo operand)
  long long zc = (long long)v.nz * tiles / (8LL * std::max(grid, 1));
  zc = std::max(16LL, std::min(64LL, zc));
  int n = (int)((v.nz + zc - 1) / zc);
  S.zchunk = (v.nz + n - 1) / n;
  S.nzc = (v.nz + S.zchunk - 1) / S.zchunk;
  S.nitems = (int)(tiles * S.nzc);
  S.table = nullptr;
  S.psi_tma = 0;
}

// step_fused items: every item pays a lead-in of 14 planes (batched into 3 - 4 pipeline stages), so chunks are long.
// Items are handed out from a table, most expensive first (a tile x z-chunk that touches an x / y slab costs about 1.5x
// an interior one per plane), with z-chunks that shrink from round to round, so that the CTAs finish together; within one
// cost class the order stays x-fastest, so that concurrently running items are neighbours and share their halos in L2.
void plan_items_fused(Domain& d, int grid, std::vector<int4>& table) {
  const DomainView& v = d.v;
  Sched& S = d.sched_f;
  S.ntx = (v.nx + TX - 1) / TX;
  S.nty = (v.ny + TY - 1) / TY;
  const long long tiles = (long long)S.ntx * S.nty;
  long long zc = (long long)v.nz * tiles / (12LL * std::max(grid, 1));
  zc = std::max(32LL, std::min(256LL, zc));
  // z-chunk boundaries: the first rounds take 1.5 zc planes, later ones shrink towards 32
  std::vector<int> zb{0};
  double sz = 1.5 * (double)zc;
  while (zb.back() < v.nz) {
    int take = (int)std::max(32.0, sz);
    if (v.nz - zb.back() - take < 24) take = v.nz - zb.back();          // no tiny last chunk: every chunk pays a 14-plane lead-in
    zb.push_back(std::min(v.nz, zb.back() + take));
    sz *= 0.8;
  }
  auto touches_slab = [&](int axis, int lo, int hi) {
    return (v.ln[axis][0] > 0 && lo < v.ls[axis][0] + v.ln[axis][0] && hi > v.ls[axis][0]) ||
           (v.ln[axis][1] > 0 && lo < v.ls[axis][1] + v.ln[axis][1] && hi > v.ls[axis][1]);
  };
  struct Item { double cost; int4 t; };
  std::vector<Item> items;
  // Inside one cost class the order is x fastest.  On wide grids (16 or more tiles per row) the rows go in pairs, y fastest
  // inside a pair, so that a tile's y neighbour is its neighbour in the list as well and its y halo is found in L2 (DRAM
  // reads of a 1600^3 step: 97.6 -> 88 GB with bands of 4 rows; 0.6 % of the capped step with pairs, which cost narrow grids
  // 1 %: there the rows are close in the list anyway).
  const int band = S.ntx >= 16 ? 2 : 1;
  for (size_t c = 0; c + 1 < zb.size(); ++c)
    for (int b0 = 0; b0 < S.nty; b0 += band)
      for (int tx = 0; tx < S.ntx; ++tx)
        for (int ty = b0; ty < std::min(S.nty, b0 + band); ++ty) {
        const int x0 = tx * TX, y0 = ty * TY;
        const bool slab = touches_slab(0, x0, x0 + TX) || touches_slab(1, y0, y0 + TY);
        items.push_back({(zb[c + 1] - zb[c] + 4) * (slab ? 1.5 : 1.0), make_int4(x0, y0, zb[c], zb[c + 1])});
      }
  std::stable_sort(items.begin(), items.end(), [](const Item& a, const Item& b) { return a.cost > b.cost; });
  table.clear();
  for (auto& it : items) table.push_back(it.t);
  S.zchunk = (int)zc;
  S.nzc = (int)zb.size() - 1;
  S.nitems = (int)table.size();
  S.psi_tma = (v.bq[0] == nullptr && psi_tma_ok(v)) ? 1 : 0;
}

// The three builds of the single-pass step: 1 = density arrays, 2 = uniform density with the x / y slab psi through the TMA
// stage (when the domain's slabs allow it, psi_tma_ok), 0 = uniform density with psi by global loads.
void launch_step_fused(int grid, cudaStream_t stream, const TMaps& tm, const DomainView& vin, const OutSet& O, const Sched& S) {
  if (vin.bq[0]) step_fused<1><<<grid, FNT, f_smem_bytes<1>(), stream>>>(tm, vin, O, S);
  else if (S.psi_tma) step_fused<2><<<grid, FNT, f_smem_bytes<2>(), stream>>>(tm, vin, O, S);
  else step_fused<0><<<grid, FNT, f_smem_bytes<0>(), stream>>>(tm, vin, O, S);
}

// One fused time step of one domain: state v.f / v.psi -> d.alt, then the two are swapped.
int launch_fused(fdtd_ctx* c, Domain& d) {
  Sched S = d.sched_f;
  S.counter = d.counters + 2 + d.fused_parity;
  S.other = d.counters + 2 + (1 - d.fused_parity);
  launch_step_fused(std::min(c->grid_f, S.nitems), c->stream, d.tm, d.v, d.alt, S);
  c->launches++;
  CK(cudaGetLastError());
  d.fused_parity ^= 1;
  for (int f = 0; f < 4; ++f) std::swap(d.v.f[f], d.alt.f[f]);
  for (int fam = 0; fam < 2; ++fam)
    for (int a = 0; a < 3; ++a)
      for (int s = 0; s < 2; ++s) std::swap(d.v.psi[fam][a][s], d.alt.psi[fam][a][s]);
  std::swap(d.tm, d.tm_alt);
  return FDTD_OK;
}

// Items of step_fused for the planes [zlo, zhi) only (one z slab of the time-blocked mode): chunks of at most 64 planes,
// slab-touching tiles first.
void plan_items_range(const Domain& d, int zlo, int zhi, std::vector<int4>& table) {
  const DomainView& v = d.v;
  const int ntx = (v.nx + TX - 1) / TX, nty = (v.ny + TY - 1) / TY;
  const int nch = std::max(1, (zhi - zlo + 63) / 64);
  auto touches_slab = [&](int axis, int lo, int hi) {
    return (v.ln[axis][0] > 0 && lo < v.ls[axis][0] + v.ln[axis][0] && hi > v.ls[axis][0]) ||
           (v.ln[axis][1] > 0 && lo < v.ls[axis][1] + v.ln[axis][1] && hi > v.ls[axis][1]);
  };
  std::vector<int4> rest;
  for (int c = 0; c < nch; ++c) {
    const int z0 = zlo + (int)((long long)(zhi - zlo) * c / nch), z1 = zlo + (int)((long long)(zhi - zlo) * (c + 1) / nch);
    for (int ty = 0; ty < nty; ++ty)
      for (int tx = 0; tx < ntx; ++tx) {
        const int x0 = tx * TX, y0 = ty * TY;
        (touches_slab(0, x0, x0 + TX) || touches_slab(1, y0, y0 + TY) ? table : rest).push_back(make_int4(x0, y0, z0, z1));
      }
  }
  table.insert(table.end(), rest.begin(), rest.end());
}

int launch_inject_range(fdtd_ctx* c, Domain& d, float* p, long long n, int zlo, int zhi);

// k time steps in one pass over the z slabs (the single-device form of the paper's enlarged ghost, P:42, P:82,
// blocked along z): for every slab [a, b) step j = 1..k is computed on [a - 8(k-j), b + 8(k-j)) — a ghost of 2r = 8 planes
// per remaining step on each side, recomputed by the neighbouring slabs as well — so that the slab's planes can stay in L2
// between its k launches.  Intermediate steps live in the scratch states X / Y, the last one goes to the out state, which
// then becomes the current state.  Same arithmetic per point as k single steps: same bits.
int do_time_block(fdtd_ctx* c) {
  Domain& d = c->doms[0];
  for (const auto& L : d.tb) {
    DomainView vin = d.v;
    const TMaps* tm = &d.tm;
    if (L.in_state >= 2) {
      const OutSet& I = d.xs[L.in_state - 2];
      for (int f = 0; f < 4; ++f) vin.f[f] = I.f[f];
      for (int fam = 0; fam < 2; ++fam)
        for (int a = 0; a < 3; ++a)
          for (int s = 0; s < 2; ++s) vin.psi[fam][a][s] = I.psi[fam][a][s];
      tm = &d.tm_xs[L.in_state - 2];
    }
    const OutSet& O = L.out_state == 1 ? d.alt : d.xs[L.out_state - 2];
    Sched S = d.sched_f;
    S.table = L.table;
    S.nitems = L.nitems;
    S.counter = d.counters + 2 + d.fused_parity;
    S.other = d.counters + 2 + (1 - d.fused_parity);
    launch_step_fused(std::min(c->grid_f, S.nitems), c->stream, *tm, vin, O, S);
    c->launches++;
    CK(cudaGetLastError());
    d.fused_parity ^= 1;
    c->plane_steps_computed += L.zhi - L.zlo;
    int r = launch_inject_range(c, d, O.f[0], c->step_index + L.step, L.zlo, L.zhi);
    if (r) return r;
  }
  c->plane_steps_owned += (int64_t)d.v.nz * c->time_block;
  c->step_index += c->time_block;
  for (int f = 0; f < 4; ++f) std::swap(d.v.f[f], d.alt.f[f]);
  for (int fam = 0; fam < 2; ++fam)
    for (int a = 0; a < 3; ++a)
      for (int s = 0; s < 2; ++s) std::swap(d.v.psi[fam][a][s], d.alt.psi[fam][a][s]);
  std::swap(d.tm, d.tm_alt);
  return FDTD_OK;
}

int launch_substep(fdtd_ctx* c, Domain& d, int which /*0 = v, 1 = p*/) {
  const DomainView& v = d.v;
  if (c->use_ref) {
    dim3 b(64, 4, 1), g((v.nx + 63) / 64, (v.ny + 3) / 4, v.nz);
    if (c->fp64) {
      if (which == 0) update_v_ref<<<g, b, 0, c->stream>>>(d.v64);
      else update_p_ref<<<g, b, 0, c->stream>>>(d.v64);
    } else {
      if (which == 0) update_v_ref<<<g, b, 0, c->stream>>>(v);
      else update_p_ref<<<g, b, 0, c->stream>>>(v);
    }
  } else {
    Sched S = d.sched;
    S.counter = d.counters + which;
    S.other = d.counters + (1 - which);
    if (which == 0 && v.bq[0]) update_v_tiled<true><<<std::min(c->grid_v, S.nitems), NT, V_SMEM_BYTES, c->stream>>>(d.tm, v, S);
    else if (which == 0) update_v_tiled<false><<<std::min(c->grid_v, S.nitems), NT, V_SMEM_BYTES, c->stream>>>(d.tm, v, S);
    else update_p_tiled<<<std::min(c->grid_p, S.nitems), NT, P_SMEM_BYTES, c->stream>>>(d.tm, v, S);
  }
  c->launches++;
  CK(cudaGetLastError());
  return FDTD_OK;
}

// Source injection of time step number c->step_index (R14), then the step index advances — with or without sources.
int launch_inject(fdtd_ctx* c) {
  const long long n = c->step_index++;
  if (c->nsrc == 0 || n >= c->wlen) return FDTD_OK;
  for (size_t k = 0; k < c->doms.size(); ++k) {
    if (c->fp64) {
      SourceViewT<double> S{c->nsrc, c->wlen, c->doms[k].src_offset, c->doms[k].v64.f[0], c->d_wav, 0, 0x7fffffffffffffffLL};
      inject_sources<<<1, 64, 0, c->stream>>>(S, n);
    } else {
      SourceView S{c->nsrc, c->wlen, c->doms[k].src_offset, c->doms[k].v.f[0], c->d_wav, 0, 0x7fffffffffffffffLL};
      inject_sources<<<1, 64, 0, c->stream>>>(S, n);
    }
    c->launches++;
  }
  CK(cudaGetLastError());
  return FDTD_OK;
}

// the sources whose plane lies in [zlo, zhi) into the pressure array p of a state that is not the current one (time_block)
int launch_inject_range(fdtd_ctx* c, Domain& d, float* p, long long n, int zlo, int zhi) {
  if (c->nsrc == 0 || n >= c->wlen) return FDTD_OK;
  SourceView S{c->nsrc, c->wlen, d.src_offset, p, c->d_wav, (long long)zlo * d.v.plane, (long long)zhi * d.v.plane};
  inject_sources<<<1, 64, 0, c->stream>>>(S, n);
  c->launches++;
  CK(cudaGetLastError());
  return FDTD_OK;
}

// ---- halo exchange between in-HBM subdomains (pack -> copy -> unpack; here one fused copy kernel per
// phase because source and destination share one address space) --------------------------------------
struct CopyJob {
  const float* src; float* dst;
  long long sp, sr, dp, dr;   // plane / row strides (floats) of source and destination
  int w, h, d;                // box size: w floats per row (multiple of 4), h rows, d planes
};
constexpr int MAX_JOBS = 24;
struct CopyBatch { CopyJob job[MAX_JOBS]; int n; };

__global__ void __launch_bounds__(256) halo_copy_kernel(const __grid_constant__ CopyBatch B) {
  const CopyJob& J = B.job[blockIdx.y];
  const int w4 = J.w >> 2;
  const long long n = (long long)w4 * J.h * J.d;
  for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += (long long)gridDim.x * blockDim.x) {
    const int x = (int)(t % w4);
    const long long r = t / w4;
    const int y = (int)(r % J.h), z = (int)(r / J.h);
    const float4 val = *reinterpret_cast<const float4*>(J.src + z * J.sp + y * J.sr + 4 * x);
    *reinterpret_cast<float4*>(J.dst + z * J.dp + y * J.dr + 4 * x) = val;
  }
}

int run_batch(fdtd_ctx* c, const CopyBatch& B) {
  if (B.n == 0) return FDTD_OK;
  long long mx = 0;
  for (int i = 0; i < B.n; ++i) mx = std::max(mx, (long long)(B.job[i].w / 4) * B.job[i].h * B.job[i].d);
  const int bx = (int)std::min<long long>(std::max<long long>((mx + 255) / 256, 1), 148 * 4);
  halo_copy_kernel<<<dim3(bx, B.n), 256, 0, c->stream>>>(B);
  c->launches++;
  CK(cudaGetLastError());
  return FDTD_OK;
}

// Adds the jobs that refresh `dst`'s ghost cells on its low/high side of `axis` (0 = x, 1 = y, 2 = z) from the owner.
// The phases run x, then y, then z; a phase copies the ghost range along its own axis, the whole local extent (ghost cells
// included) along the axes already exchanged and the owned range along the axes still to come, which carries the edges and
// corners (R21).  An x cut moves g-wide column blocks — the strided access that makes block-xy the slow layout.
void add_face_jobs(fdtd_ctx* c, std::vector<CopyJob>& jobs, Domain& dst, Domain& src, int axis, int side) {
  const DomainView &dv = dst.v, &sv = src.v;
  const int g = c->G.ghost;
  const int dn[3] = {dv.nx, dv.ny, dv.nz};
  const int dofs[3] = {dv.ox, dv.oy, dv.oz}, sofs[3] = {sv.ox, sv.oy, sv.oz};
  int b0[3], b1[3];                                       // the box in dst-local indices
  for (int a = 0; a < 3; ++a) {
    if (a == axis) { b0[a] = side == 0 ? 0 : dst.own_hi[a]; b1[a] = b0[a] + g; }
    else if (a < axis) { b0[a] = 0; b1[a] = dn[a]; }
    else { b0[a] = dst.own_lo[a]; b1[a] = dst.own_hi[a]; }
  }
  int s0[3];                                              // the same cells in src-local indices
  for (int a = 0; a < 3; ++a) s0[a] = b0[a] + dofs[a] - sofs[a];
  const int w = axis == 0 ? g : dv.pitch;                 // phases y, z move whole rows (both pitches are equal)
  const int dx0 = axis == 0 ? b0[0] : 0, sx0 = axis == 0 ? s0[0] : 0;
  auto push = [&](const float* sb, float* db, long long sp, long long sr, long long dp, long long dr, int ww, int h, int d,
                  long long soff, long long doff) {
    if (ww <= 0 || h <= 0 || d <= 0) return;
    jobs.push_back(CopyJob{sb + soff, db + doff, sp, sr, dp, dr, ww, h, d});
  };
  const int dy0 = b0[1], dy1 = b1[1], dz0 = b0[2], dz1 = b1[2], sy0 = s0[1], sz0 = s0[2];
  for (int f = 0; f < 4; ++f)
    push(sv.f[f], dv.f[f], sv.plane, sv.pitch, dv.plane, dv.pitch, w, dy1 - dy0, dz1 - dz0,
         (long long)sz0 * sv.plane + (long long)sy0 * sv.pitch + sx0, (long long)dz0 * dv.plane + (long long)dy0 * dv.pitch + dx0);
  // psi pieces that live in the ghost box (R21): x slabs (all j,k), y slabs (rows in slab), z slabs (planes in slab)
  for (int fam = 0; fam < 2; ++fam) {
    for (int s = 0; s < 2; ++s) {
      // x slabs: whole slab width; an x-phase box never meets an x layer (make_geometry)
      if (axis != 0 && dv.ln[0][s] > 0 && sv.ln[0][s] == dv.ln[0][s]) {
        const int wx = dv.ln[0][s];
        push(sv.psi[fam][0][s], dv.psi[fam][0][s], (long long)sv.ny * wx, wx, (long long)dv.ny * wx, wx, wx, dy1 - dy0, dz1 - dz0,
             ((long long)sz0 * sv.ny + sy0) * wx, ((long long)dz0 * dv.ny + dy0) * wx);
      }
      // y-slab rows inside the box
      if (dv.ln[1][s] > 0) {
        const int a0 = std::max(dy0, dv.ls[1][s]), a1 = std::min(dy1, dv.ls[1][s] + dv.ln[1][s]);
        if (a1 > a0 && sv.ln[1][s] > 0) {
          const int sa0 = a0 + dv.oy - sv.oy;
          if (sa0 >= sv.ls[1][s] && sa0 + (a1 - a0) <= sv.ls[1][s] + sv.ln[1][s])
            push(sv.psi[fam][1][s], dv.psi[fam][1][s], (long long)sv.ln[1][s] * sv.pitch, sv.pitch, (long long)dv.ln[1][s] * dv.pitch,
                 dv.pitch, w, a1 - a0, dz1 - dz0, ((long long)sz0 * sv.ln[1][s] + (sa0 - sv.ls[1][s])) * sv.pitch + sx0,
                 ((long long)dz0 * dv.ln[1][s] + (a0 - dv.ls[1][s])) * dv.pitch + dx0);
        }
      }
      // z-slab planes inside the box
      if (dv.ln[2][s] > 0) {
        const int a0 = std::max(dz0, dv.ls[2][s]), a1 = std::min(dz1, dv.ls[2][s] + dv.ln[2][s]);
        if (a1 > a0 && sv.ln[2][s] > 0) {
          const int sa0 = a0 + dv.oz - sv.oz;
          if (sa0 >= sv.ls[2][s] && sa0 + (a1 - a0) <= sv.ls[2][s] + sv.ln[2][s])
            push(sv.psi[fam][2][s], dv.psi[fam][2][s], (long long)sv.ny * sv.pitch, sv.pitch, (long long)dv.ny * dv.pitch, dv.pitch, w,
                 dy1 - dy0, a1 - a0, ((long long)(sa0 - sv.ls[2][s]) * sv.ny + sy0) * sv.pitch + sx0,
                 ((long long)(a0 - dv.ls[2][s]) * dv.ny + dy0) * dv.pitch + dx0);
        }
      }
    }
  }
}

int exchange_halos(fdtd_ctx* c) {
  if (c->doms.size() <= 1) return FDTD_OK;
  const int nd[3] = {c->G.nd[0], c->G.nd[1], c->G.nd[2]};
  for (int axis = 0; axis <= 2; ++axis) {
    if (nd[axis] == 1) continue;
    std::vector<CopyJob> jobs;
    for (auto& d : c->doms) {
      const int pos[3] = {d.cx, d.cy, d.cz};
      for (int side = 0; side < 2; ++side) {
        int np[3] = {pos[0], pos[1], pos[2]};
        np[axis] += side == 0 ? -1 : 1;
        if (np[axis] < 0 || np[axis] >= nd[axis]) continue;
        Domain& src = c->doms[((size_t)np[2] * nd[1] + np[1]) * nd[0] + np[0]];
        add_face_jobs(c, jobs, d, src, axis, side);
      }
    }
    for (size_t b = 0; b < jobs.size(); b += MAX_JOBS) {
      CopyBatch B{};
      B.n = (int)std::min<size_t>(MAX_JOBS, jobs.size() - b);
      for (int i = 0; i < B.n; ++i) B.job[i] = jobs[b + i];
      int r = run_batch(c, B);
      if (r) return r;
    }
  }
  return FDTD_OK;
}

int do_fused_step(fdtd_ctx* c) {
  if (c->doms.size() > 1 && c->substeps_done % c->G.msub == 0) {
    int r = exchange_halos(c);
    if (r) return r;
  }
  for (auto& d : c->doms) {
    int r = launch_fused(c, d);
    if (r) return r;
  }
  c->substeps_done += 2;
  return FDTD_OK;
}

int do_substep(fdtd_ctx* c, int which) {
  if (c->doms.size() > 1 && c->substeps_done % c->G.msub == 0) {
    int r = exchange_halos(c);
    if (r) return r;
  }
  for (auto& d : c->doms) {
    int r = launch_substep(c, d, which);
    if (r) return r;
  }
  c->substeps_done++;
  return FDTD_OK;
}

// every value > 0 and finite (NaN fails the first test); split over a few host threads: 4e9 values at config 4
bool all_positive_finite(const float* a, size_t n) {
  const unsigned nt = (unsigned)std::max<size_t>(1, std::min<size_t>(std::min<size_t>(16, std::thread::hardware_concurrency()), n >> 20));
  std::vector<char> ok(nt, 1);
  std::vector<std::thread> th;
  for (unsigned t = 0; t < nt; ++t)
    th.emplace_back([&, t] {
      const size_t lo = n * t / nt, hi = n * (t + 1) / nt;
      bool good = true;
      for (size_t q = lo; q < hi; ++q) good = good && (a[q] > 0.0f) && (a[q] <= 3.0e38f);
      ok[t] = good;
    });
  for (auto& x : th) x.join();
  return std::all_of(ok.begin(), ok.end(), [](char v) { return v != 0; });
}

// gather / scatter between a packed host total-grid array and the domains
int copy_field(fdtd_ctx* c, float* const* dom_base_f, float* host_f, bool to_host, bool owned_only, size_t es = 4) {
  const int gnx = c->G.gn[0], gny = c->G.gn[1];
  char* host = (char*)host_f;
  for (auto& d : c->doms) {
    const DomainView& v = d.v;
    const int il = owned_only ? d.own_lo[0] : 0, ih = owned_only ? d.own_hi[0] : v.nx;
    const int jl = owned_only ? d.own_lo[1] : 0, jh = owned_only ? d.own_hi[1] : v.ny;
    const int kl = owned_only ? d.own_lo[2] : 0, kh = owned_only ? d.own_hi[2] : v.nz;
    char* base = (char*)dom_base_f[&d - &c->doms[0]];
    if (jl == 0 && jh == v.ny && v.ny == gny && v.oy == 0) {
      // whole planes: rows of consecutive planes are consecutive on both sides -> one 2-D copy
      char* dev = base + ((long long)kl * v.plane + il) * es;
      char* h = host + ((long long)(kl + v.oz) * gny * gnx + (il + v.ox)) * es;
      const size_t rows = (size_t)(kh - kl) * v.ny;
      if (to_host) CK(cudaMemcpy2DAsync(h, (size_t)gnx * es, dev, (size_t)v.pitch * es, (size_t)(ih - il) * es, rows, cudaMemcpyDeviceToHost, c->stream));
      else CK(cudaMemcpy2DAsync(dev, (size_t)v.pitch * es, h, (size_t)gnx * es, (size_t)(ih - il) * es, rows, cudaMemcpyHostToDevice, c->stream));
      continue;
    }
    for (int k = kl; k < kh; ++k) {
      char* dev = base + ((long long)k * v.plane + (long long)jl * v.pitch + il) * es;
      char* h = host + (((long long)(k + v.oz) * gny + (jl + v.oy)) * gnx + (il + v.ox)) * es;
      if (to_host) CK(cudaMemcpy2DAsync(h, (size_t)gnx * es, dev, (size_t)v.pitch * es, (size_t)(ih - il) * es, jh - jl, cudaMemcpyDeviceToHost, c->stream));
      else CK(cudaMemcpy2DAsync(dev, (size_t)v.pitch * es, h, (size_t)gnx * es, (size_t)(ih - il) * es, jh - jl, cudaMemcpyHostToDevice, c->stream));
    }
  }
  CK(cudaStreamSynchronize(c->stream));
  return FDTD_OK;
}

}  // namespace

template <class V>
static int get_psi_impl(fdtd_ctx* c, Domain& d, const V& v, int fam, int axis, typename V::real* dst) {
  typedef typename V::real T;
  const int gnx = c->G.gn[0], gny = c->G.gn[1];
  const size_t n = (size_t)v.nx * v.ny * v.nz;
  T* tmp = nullptr;
  CK(cudaMalloc(&tmp, n * sizeof(T)));                 // debug-only scratch, not field storage
  expand_psi_kernel<<<148 * 8, 256, 0, c->stream>>>(v, fam, axis, tmp);
  c->launches++;
  for (int k = d.own_lo[2]; k < d.own_hi[2]; ++k) {
    const T* dev = tmp + ((size_t)k * v.ny + d.own_lo[1]) * v.nx + d.own_lo[0];
    T* h = dst + ((size_t)(k + v.oz) * gny + (d.own_lo[1] + v.oy)) * gnx + (d.own_lo[0] + v.ox);
    cudaMemcpy2DAsync(h, (size_t)gnx * sizeof(T), dev, (size_t)v.nx * sizeof(T), (size_t)(d.own_hi[0] - d.own_lo[0]) * sizeof(T),
                      d.own_hi[1] - d.own_lo[1], cudaMemcpyDeviceToHost, c->stream);
  }
  cudaError_t e = cudaStreamSynchronize(c->stream);
  cudaFree(tmp);
  CK(e);
  return FDTD_OK;
}

// =========================================================================================== C ABI
extern "C" {

const char* fdtd_last_error(void) { return g_err.c_str(); }

int fdtd_coeffs(float out[4]) {
  if (!out) return FDTD_EINVAL;
  out[0] = FDTD_C1; out[1] = FDTD_C2; out[2] = FDTD_C3; out[3] = FDTD_C4;
  return FDTD_OK;
}

uint64_t fdtd_workspace_bytes(const fdtd_params* P) {
  if (!P) return 0;
  Geometry G = make_geometry(*P);
  if (!G.valid) { set_err(G.why); return 0; }
  return make_layout(*P, G).total;
}

fdtd_ctx* fdtd_create(const fdtd_params* P) {
  if (!P) { set_err("params is NULL"); return nullptr; }
  Geometry G = make_geometry(*P);
  if (!G.valid) { set_err(G.why); return nullptr; }
  Layout L = make_layout(*P, G);
  if (!P->workspace || ((uintptr_t)P->workspace & 255) || P->workspace_bytes < L.total) {
    set_err("workspace NULL, misaligned or too small (need " + std::to_string(L.total) + " bytes)");
    return nullptr;
  }
  auto fail = [&](fdtd_ctx* c, cudaError_t e, const char* what) -> fdtd_ctx* {
    set_err(std::string(what) + ": " + cudaGetErrorString(e));
    delete c;
    return nullptr;
  };
  fdtd_ctx* c = new fdtd_ctx();
  c->P = *P; c->G = G; c->L = L;
  c->ws = (char*)P->workspace;
  c->stream = (cudaStream_t)P->stream;
  // The tiled kernels move whole float4s.  A monolithic grid of any Nx takes them (the last float4 of a row reaches into the
  // row's padding, which nothing reads: TMA bounds are the grid's); the halo copies of the subdomain mode need Nx % 4 == 0.
  c->fp64 = P->precision == FDTD_PRECISION_FP64;
  c->es = c->fp64 ? 8 : 4;
  const bool subdomains = G.nd[0] * G.nd[1] * G.nd[2] > 1;
  c->use_ref = P->kernel == FDTD_KERNEL_REF || P->boundary == FDTD_PERIODIC || (subdomains && (G.gn[0] % 4) != 0) || c->fp64;
  c->fused = P->kernel == FDTD_KERNEL_FUSED;      // make_geometry has checked that the tiled path applies
  cudaError_t e;
  if ((e = cudaSetDevice(P->device)) != cudaSuccess) return fail(c, e, "cudaSetDevice");
  if ((e = cudaMemsetAsync(c->ws, 0, L.total, c->stream)) != cudaSuccess) return fail(c, e, "cudaMemsetAsync(workspace)");

  // CPML tables: double on the host, rounded once to fp32 (a6)
  for (int a = 0; a < 3; ++a)
    for (int fam = 0; fam < 2; ++fam) {
      c->tabs[fam][a] = make_axis_table(G.gn[a], P->cpml[2 * a], P->cpml[2 * a + 1], fam == 0, *P);
      const AxisTable& t = c->tabs[fam][a];
      // device copy of the half-node `a`: 0 at the pinned last half node (R3), so its psi stays 0 as in the
      // recurrence, which never updates that node; fdtd_cpml_table returns the plain formula values
      c->dev_a[fam][a] = t.a;
      if (fam == 0 && P->boundary == FDTD_WALL) c->dev_a[fam][a][G.gn[a] - 1] = 0.0f;
      const float* src[3] = {c->dev_a[fam][a].data(), t.b.data(), t.ik.data()};
      for (int k = 0; k < 3; ++k)
        if ((e = cudaMemcpyAsync(c->ws + L.tab[fam][a][k], src[k], (size_t)L.tablen[a] * 4, cudaMemcpyHostToDevice, c->stream)) != cudaSuccess)
          return fail(c, e, "cudaMemcpyAsync(tables)");
    }
  if ((e = cudaStreamSynchronize(c->stream)) != cudaSuccess) return fail(c, e, "cudaStreamSynchronize");

  c->d_wav = (float*)(c->ws + L.wav);

  EncodeTiledFn enc = nullptr;
  if (!c->use_ref) {
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qr;
    if ((e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qr)) != cudaSuccess || !fn)
      return fail(c, e, "cudaGetDriverEntryPoint(cuTensorMapEncodeTiled)");
    enc = (EncodeTiledFn)fn;
  }

  size_t di = 0;
  for (int cz = 0; cz < G.nd[2]; ++cz)
    for (int cy = 0; cy < G.nd[1]; ++cy)
     for (int cx = 0; cx < G.nd[0]; ++cx, ++di) {
      const Layout::Dom& ld = L.doms[di];
      Domain d{};
      DomainView& v = d.v;
      v.nx = ld.n[0]; v.ny = ld.n[1]; v.nz = ld.n[2];
      v.pitch = ld.pitch; v.plane = (long long)ld.pitch * ld.n[1];
      v.ox = ld.o[0]; v.oy = ld.o[1]; v.oz = ld.o[2];
      for (int a = 0; a < 3; ++a) v.gn[a] = G.gn[a];
      v.periodic = P->boundary == FDTD_PERIODIC;
      for (int f = 0; f < 4; ++f) v.f[f] = (float*)(c->ws + ld.f[f]);
      v.kc = nullptr;
      for (int a = 0; a < 3; ++a) v.bq[a] = nullptr;
      v.kc0 = (float)(1.0 * 1.0 * 1.0 * P->dt / P->dx);
      v.b0 = (float)(P->dt / (1.0 * P->dx));
      for (int a = 0; a < 3; ++a)
        for (int s = 0; s < 2; ++s) {
          v.ls[a][s] = ld.ls[a][s]; v.ln[a][s] = ld.ln[a][s];
          for (int fam = 0; fam < 2; ++fam) v.psi[fam][a][s] = (float*)(c->ws + ld.psi[fam][a][s]);
        }
      for (int fam = 0; fam < 2; ++fam)
        for (int a = 0; a < 3; ++a)
          for (int k = 0; k < 3; ++k) v.tab[fam][a][k] = (const float*)(c->ws + L.tab[fam][a][k]);
      d.cx = cx; d.cy = cy; d.cz = cz;
      const int cc[3] = {cx, cy, cz};
      for (int a = 0; a < 3; ++a) {
        d.own_lo[a] = cc[a] > 0 ? G.ghost : 0;
        d.own_hi[a] = d.own_lo[a] + G.gn[a] / G.nd[a];
      }
      if (c->fp64) {                                  // same geometry, double state
        DomainViewT<double>& w = d.v64;
        w.nx = v.nx; w.ny = v.ny; w.nz = v.nz; w.pitch = v.pitch; w.plane = v.plane; w.ox = v.ox; w.oy = v.oy; w.oz = v.oz;
        w.periodic = v.periodic; w.kc = nullptr; w.kc0 = v.kc0; w.b0 = v.b0;
        for (int a = 0; a < 3; ++a) {
          w.gn[a] = v.gn[a]; w.bq[a] = nullptr;
          for (int s = 0; s < 2; ++s) {
            w.ls[a][s] = v.ls[a][s]; w.ln[a][s] = v.ln[a][s];
            for (int fam = 0; fam < 2; ++fam) w.psi[fam][a][s] = (double*)(c->ws + ld.psi[fam][a][s]);
          }
          for (int fam = 0; fam < 2; ++fam)
            for (int k = 0; k < 3; ++k) w.tab[fam][a][k] = v.tab[fam][a][k];
        }
        for (int f = 0; f < 4; ++f) w.f[f] = (double*)(c->ws + ld.f[f]);
      }
      d.src_offset = (long long*)(c->ws + ld.src_off);
      d.counters = (unsigned int*)(c->ws + ld.counters);
      if (!c->use_ref) {
        float* kcbase = L.has_kc ? (float*)(c->ws + ld.kc) : (float*)(c->ws + ld.f[0]);   // no Kc slot: the map is never used
        auto make_maps = [&](TMaps& tm, float* const f[4], float* const psi[2][3][2]) -> int {
          float* tile_base[5] = {f[0], f[1], f[2], f[3], kcbase};
          int bad = make_tmap(enc, &tm.p_halo, f[0], v, HW, VH) || make_tmap(enc, &tm.vx_halo, f[1], v, HW, TY) ||
                    make_tmap(enc, &tm.vy_halo, f[2], v, TX, PH) || make_tmap(enc, &tm.p_box, f[0], v, BW, BH);
          for (int t = 0; t < 5 && !bad; ++t) bad = make_tmap(enc, &tm.tile[t], tile_base[t], v, TX, TY);
          if (!bad && P->density == FDTD_DENSITY_ARRAY)
            bad = make_tmap(enc, &tm.bq_halo[0], (float*)(c->ws + ld.bq[0]), v, HW, TY) ||
                  make_tmap(enc, &tm.bq_halo[1], (float*)(c->ws + ld.bq[1]), v, TX, PH) ||
                  make_tmap(enc, &tm.bq_tile, (float*)(c->ws + ld.bq[2]), v, TX, TY);
          if (c->fused && psi)
            for (int fam = 0; fam < 2 && !bad; ++fam)
              for (int s = 0; s < 2 && !bad; ++s) {
                if (v.ln[0][s] > 0) bad = make_tmap_psi(enc, &tm.psi_x[fam][s], psi[fam][0][s], v.ln[0][s], v.ny, v.nz, v.ln[0][s], PXW);
                if (v.ln[1][s] > 0 && !bad) bad = make_tmap_psi(enc, &tm.psi_y[fam][s], psi[fam][1][s], v.nx, v.ln[1][s], v.nz, v.pitch, TX);
              }
          return bad;
        };
        int bad = make_maps(d.tm, v.f, v.psi);
        if (c->fused && !bad) {
          for (int f = 0; f < 4; ++f) d.alt.f[f] = (float*)(c->ws + ld.f2[f]);
          for (int fam = 0; fam < 2; ++fam)
            for (int a = 0; a < 3; ++a)
              for (int s = 0; s < 2; ++s) d.alt.psi[fam][a][s] = (float*)(c->ws + ld.psi2[fam][a][s]);
          bad = make_maps(d.tm_alt, d.alt.f, d.alt.psi);
          for (int x = 0; x < (P->time_block > 2 ? 2 : (P->time_block > 1 ? 1 : 0)) && !bad; ++x) {
            for (int f = 0; f < 4; ++f) d.xs[x].f[f] = (float*)(c->ws + ld.fx[x][f]);
            for (int fam = 0; fam < 2; ++fam)
              for (int a = 0; a < 3; ++a)
                for (int s = 0; s < 2; ++s) d.xs[x].psi[fam][a][s] = (float*)(c->ws + ld.psix[x][fam][a][s]);
            bad = make_maps(d.tm_xs[x], d.xs[x].f, d.xs[x].psi);
          }
        }
        if (bad) { delete c; return nullptr; }
      }
      c->doms.push_back(d);
    }

  if (!c->use_ref) {
    if ((e = cudaFuncSetAttribute(update_v_tiled<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, V_SMEM_BYTES)) != cudaSuccess ||
        (e = cudaFuncSetAttribute(update_v_tiled<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, V_SMEM_BYTES)) != cudaSuccess)
      return fail(c, e, "cudaFuncSetAttribute(update_v_tiled)");
    if ((e = cudaFuncSetAttribute(update_p_tiled, cudaFuncAttributeMaxDynamicSharedMemorySize, P_SMEM_BYTES)) != cudaSuccess)
      return fail(c, e, "cudaFuncSetAttribute(update_p_tiled)");
    if (plan_launch(c, P->density == FDTD_DENSITY_ARRAY ? (const void*)update_v_tiled<true> : (const void*)update_v_tiled<false>,
                    V_SMEM_BYTES, &c->grid_v) ||
        plan_launch(c, (const void*)update_p_tiled, P_SMEM_BYTES, &c->grid_p)) { delete c; return nullptr; }
    for (auto& d : c->doms) plan_items(d, std::min(c->grid_v, c->grid_p));
    if (c->fused) {
      if ((e = cudaFuncSetAttribute(step_fused<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, f_smem_bytes<0>())) != cudaSuccess ||
          (e = cudaFuncSetAttribute(step_fused<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, f_smem_bytes<1>())) != cudaSuccess ||
          (e = cudaFuncSetAttribute(step_fused<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, f_smem_bytes<2>())) != cudaSuccess)
        return fail(c, e, "cudaFuncSetAttribute(step_fused)");
      const bool hb = P->density == FDTD_DENSITY_ARRAY;
      if (plan_launch(c, hb ? (const void*)step_fused<1> : (const void*)step_fused<2>, hb ? f_smem_bytes<1>() : f_smem_bytes<2>(),
                      &c->grid_f, FNT)) { delete c; return nullptr; }
      for (size_t k = 0; k < c->doms.size(); ++k) {
        Domain& d = c->doms[k];
        std::vector<int4> table;
        plan_items_fused(d, c->grid_f, table);
        if (table.size() > L.doms[k].items_cap) { set_err("item table larger than its workspace slot"); delete c; return nullptr; }
        if ((e = cudaMemcpyAsync(c->ws + L.doms[k].items, table.data(), table.size() * sizeof(int4), cudaMemcpyHostToDevice, c->stream)) != cudaSuccess ||
            (e = cudaStreamSynchronize(c->stream)) != cudaSuccess)
          return fail(c, e, "cudaMemcpyAsync(item table)");
        d.sched_f.table = (const int4*)(c->ws + L.doms[k].items);
      }
      c->time_block = std::max(1, (int)P->time_block);
      if (c->time_block > 1) {
        Domain& d = c->doms[0];
        const Layout::Dom& ld = L.doms[0];
        const int k = c->time_block, nz = d.v.nz, zs = ld.tb_planes;
        std::vector<int4> all;
        std::vector<size_t> first;
        for (int a = 0; a < nz; a += zs) {
          const int b = std::min(nz, a + zs);
          for (int j = 1; j <= k; ++j) {
            const int ext = 8 * (k - j);
            Domain::TbLaunch T{};
            T.zlo = std::max(0, a - ext); T.zhi = std::min(nz, b + ext);
            T.in_state = j == 1 ? 0 : 2 + (j - 2) % 2;
            T.out_state = j == k ? 1 : 2 + (j - 1) % 2;
            T.step = j - 1;
            std::vector<int4> t;
            plan_items_range(d, T.zlo, T.zhi, t);
            T.nitems = (int)t.size();
            first.push_back(all.size());
            all.insert(all.end(), t.begin(), t.end());
            d.tb.push_back(T);
          }
        }
        if (all.size() > ld.tb_items_cap) { set_err("time-block item tables larger than their workspace slot"); delete c; return nullptr; }
        if ((e = cudaMemcpyAsync(c->ws + ld.tb_items, all.data(), all.size() * sizeof(int4), cudaMemcpyHostToDevice, c->stream)) != cudaSuccess ||
            (e = cudaStreamSynchronize(c->stream)) != cudaSuccess)
          return fail(c, e, "cudaMemcpyAsync(time-block item tables)");
        for (size_t t = 0; t < d.tb.size(); ++t) d.tb[t].table = (const int4*)(c->ws + ld.tb_items) + first[t];
      }
    }
  }
  return c;
}

int fdtd_dims(const fdtd_ctx* c, int32_t out[3]) {
  if (!c || !out) return FDTD_EINVAL;
  for (int a = 0; a < 3; ++a) out[a] = c->G.gn[a];
  return FDTD_OK;
}

int64_t fdtd_launch_count(const fdtd_ctx* c) { return c ? c->launches : -1; }

// Heterogeneous density ("coefficients are absorbed"; reading R6): K dt/dx = rho c^2 dt/dx at the nodes and
// dt/(rho_bar dx) at the half nodes of vx, vy, vz with rho_bar the mean of the two adjacent nodes (the last node of an
// axis repeats itself; that half node is pinned anyway, R3).  Formed on the host in double from the fp32 inputs, rounded
// once, then scattered to the domains (ghost cells included, so subdomains see the global neighbour).
// the fp64 view shares the medium (fp32 coefficients) with the fp32 view
static void sync_v64(fdtd_ctx* c) {
  for (auto& d : c->doms) {
    d.v64.kc = d.v.kc; d.v64.kc0 = d.v.kc0; d.v64.b0 = d.v.b0;
    for (int a = 0; a < 3; ++a) d.v64.bq[a] = d.v.bq[a];
  }
}

static int set_model_density_array(fdtd_ctx* c, const float* c_host, const float* rho_host) {
  if (c->P.density != FDTD_DENSITY_ARRAY) {
    set_err("a heterogeneous rho needs params.density = FDTD_DENSITY_ARRAY (the workspace must hold the three dt/(rho_bar dx) arrays)");
    return FDTD_EUNSUPPORTED;
  }
  const long long nx = c->G.gn[0], ny = c->G.gn[1], nz = c->G.gn[2];
  const size_t n = (size_t)nx * ny * nz;
  const double dt = c->P.dt, dx = c->P.dx;
  std::vector<float> kc(n), bq[3];
  for (int a = 0; a < 3; ++a) bq[a].resize(n);
  for (size_t q = 0; q < n; ++q) {
    const double cc = c_host ? (double)c_host[q] : 1.0, rr = (double)rho_host[q];
    if (!(rr > 0.0) || rr > 1e30 || !(cc > 0.0) || cc > 1e30) { set_err("c and rho must be positive and finite"); return FDTD_EINVAL; }
    kc[q] = (float)(rr * cc * cc * dt / dx);
  }
  for (long long k = 0; k < nz; ++k)
    for (long long j = 0; j < ny; ++j)
      for (long long i = 0; i < nx; ++i) {
        const size_t q = (size_t)((k * ny + j) * nx + i);
        const double r0 = rho_host[q];
        const double rx = rho_host[i + 1 < nx ? q + 1 : q], ry = rho_host[j + 1 < ny ? q + (size_t)nx : q],
                     rz = rho_host[k + 1 < nz ? q + (size_t)(nx * ny) : q];
        bq[0][q] = (float)(dt / (0.5 * (r0 + rx) * dx));
        bq[1][q] = (float)(dt / (0.5 * (r0 + ry) * dx));
        bq[2][q] = (float)(dt / (0.5 * (r0 + rz) * dx));
      }
  std::vector<float*> bases;
  for (size_t k = 0; k < c->doms.size(); ++k) bases.push_back((float*)(c->ws + c->L.doms[k].kc));
  int r = copy_field(c, bases.data(), kc.data(), false, false);
  for (int a = 0; a < 3 && !r; ++a) {
    std::vector<float*> bb;
    for (size_t k = 0; k < c->doms.size(); ++k) bb.push_back((float*)(c->ws + c->L.doms[k].bq[a]));
    r = copy_field(c, bb.data(), bq[a].data(), false, false);
  }
  if (r) return r;
  for (size_t k = 0; k < c->doms.size(); ++k) {
    DomainView& v = c->doms[k].v;
    v.kc = bases[k];
    for (int a = 0; a < 3; ++a) v.bq[a] = (const float*)(c->ws + c->L.doms[k].bq[a]);
  }
  sync_v64(c);
  return FDTD_OK;
}

int fdtd_set_model(fdtd_ctx* c, const float* c_host, const float* rho_host) {
  if (!c) return FDTD_EINVAL;
  const size_t n = (size_t)c->G.gn[0] * c->G.gn[1] * c->G.gn[2];
  double rho = 1.0;
  if (rho_host) {
    rho = rho_host[0];
    bool uniform = true;
    for (size_t q = 1; q < n && uniform; ++q) uniform = rho_host[q] == rho_host[0];
    if (!uniform) return set_model_density_array(c, c_host, rho_host);
    if (!(rho > 0.0) || rho > 1e30) { set_err("rho must be positive and finite"); return FDTD_EINVAL; }
  }
  // validate before anything is touched, so that an error leaves the context as it was
  if (c_host && !c->L.has_kc) {
    set_err("a wave-speed array needs params.medium = FDTD_MEDIUM_ARRAY (this workspace was sized without the K dt/dx array)");
    return FDTD_EUNSUPPORTED;
  }
  if (c_host && !all_positive_finite(c_host, n)) { set_err("c must be positive and finite"); return FDTD_EINVAL; }
  for (auto& d : c->doms)
    for (int a = 0; a < 3; ++a) d.v.bq[a] = nullptr;
  const float b0 = (float)(c->P.dt / (rho * c->P.dx));
  if (!c_host) {
    for (auto& d : c->doms) { d.v.kc = nullptr; d.v.kc0 = (float)(rho * 1.0 * 1.0 * c->P.dt / c->P.dx); d.v.b0 = b0; }
    sync_v64(c);
    return FDTD_OK;
  }
  // c goes up as fp32; K dt/dx = rho c^2 dt/dx (R6) is formed on the device in double and rounded once
  std::vector<float*> bases;
  for (size_t k = 0; k < c->doms.size(); ++k) bases.push_back((float*)(c->ws + c->L.doms[k].kc));
  int r = copy_field(c, bases.data(), const_cast<float*>(c_host), false, false);
  if (r) return r;
  for (size_t k = 0; k < c->doms.size(); ++k) {
    const DomainView& v = c->doms[k].v;
    speed_to_kc_kernel<<<148 * 8, 256, 0, c->stream>>>(bases[k], (long long)v.plane * v.nz, v.pitch, v.nx, rho, c->P.dt, c->P.dx);
    c->launches++;
  }
  CK(cudaGetLastError());
  CK(cudaStreamSynchronize(c->stream));
  for (size_t k = 0; k < c->doms.size(); ++k) { c->doms[k].v.kc = bases[k]; c->doms[k].v.b0 = b0; }
  sync_v64(c);
  return FDTD_OK;
}

int fdtd_set_sources(fdtd_ctx* c, int32_t n, const int32_t* ijk, const float* wav, int32_t len) {
  if (!c || n < 0 || n > MAX_SRC) { set_err("bad source count"); return FDTD_EINVAL; }
  if (n == 0) { c->nsrc = 0; c->wlen = 0; return FDTD_OK; }
  if (!ijk || !wav || len <= 0 || (long long)n * len > MAX_WAV_FLOATS) { set_err("bad source table"); return FDTD_EINVAL; }
  for (int s = 0; s < n; ++s)
    for (int a = 0; a < 3; ++a)
      if (ijk[3 * s + a] < 0 || ijk[3 * s + a] >= c->G.gn[a]) { set_err("source outside the grid"); return FDTD_EINVAL; }
  for (auto& d : c->doms) {
    std::vector<long long> off(n, -1);
    for (int s = 0; s < n; ++s) {
      const int li = ijk[3 * s] - d.v.ox, lj = ijk[3 * s + 1] - d.v.oy, lk = ijk[3 * s + 2] - d.v.oz;
      if (li >= 0 && li < d.v.nx && lj >= 0 && lj < d.v.ny && lk >= 0 && lk < d.v.nz)
        off[s] = (long long)lk * d.v.plane + (long long)lj * d.v.pitch + li;
    }
    CK(cudaMemcpyAsync(d.src_offset, off.data(), n * sizeof(long long), cudaMemcpyHostToDevice, c->stream));
    CK(cudaStreamSynchronize(c->stream));
  }
  CK(cudaMemcpyAsync(c->d_wav, wav, (size_t)n * len * 4, cudaMemcpyHostToDevice, c->stream));
  CK(cudaStreamSynchronize(c->stream));
  c->nsrc = n; c->wlen = len;
  return FDTD_OK;
}

int fdtd_step(fdtd_ctx* c, int32_t n) {
  if (!c || n < 0) return FDTD_EINVAL;
  for (int s = 0; s < n; ++s) {
    int r;
    if (c->time_block > 1 && n - s >= c->time_block) {      // k steps per pass over the z slabs, sources included
      if ((r = do_time_block(c))) return r;
      s += c->time_block - 1;
      continue;
    }
    if (c->fused) {
      if ((r = do_fused_step(c))) return r;   // both sub-updates in one pass (a7)
    } else {
      if ((r = do_substep(c, 0))) return r;   // velocity sub-update
      if ((r = do_substep(c, 1))) return r;   // pressure sub-update
    }
    if ((r = launch_inject(c))) return r;     // source (R14)
  }
  return FDTD_OK;
}

int fdtd_step_profiled(fdtd_ctx* c, int32_t n, double out_ms[4]) {
  if (!c || n < 0 || !out_ms) return FDTD_EINVAL;
  // One CUDA event on the launching stream after every launch group; the interval that ends at a mark is
  // charged to the mark's category (0 = update_v / step_fused, 1 = update_p, 2 = inject, 3 = exchange).  The events are
  // created up front and destroyed on every way out.
  std::vector<cudaEvent_t> ev((size_t)n * 5 + 2, nullptr);
  std::vector<int> cat(ev.size(), -1);
  size_t used = 0;
  int r = FDTD_OK;
  cudaError_t ce = cudaSuccess;
  for (auto& e : ev)
    if (ce == cudaSuccess) ce = cudaEventCreate(&e);
  auto mark = [&](int category) {
    if (ce == cudaSuccess) ce = cudaEventRecord(ev[used], c->stream);
    cat[used++] = category;
  };
  if (ce == cudaSuccess) mark(-1);
  for (int s = 0; s < n && !r && ce == cudaSuccess; ++s) {
    if (c->time_block > 1 && n - s >= c->time_block) {
      r = do_time_block(c);
      mark(0);
      s += c->time_block - 1;
      continue;
    }
    if (c->fused) {
      if (c->doms.size() > 1 && c->substeps_done % c->G.msub == 0) {
        r = exchange_halos(c);
        mark(3);
      }
      for (auto& d : c->doms) if (!r) r = launch_fused(c, d);
      c->substeps_done += 2;
      mark(0);
    }
    for (int which = 0; which < 2 && !r && !c->fused; ++which) {
      if (c->doms.size() > 1 && c->substeps_done % c->G.msub == 0) {
        r = exchange_halos(c);
        mark(3);
      }
      for (auto& d : c->doms) if (!r) r = launch_substep(c, d, which);
      c->substeps_done++;
      mark(which);
    }
    if (!r) { const int64_t l0 = c->launches; r = launch_inject(c); if (c->launches > l0) mark(2); }
  }
  if (ce == cudaSuccess) ce = cudaStreamSynchronize(c->stream);
  out_ms[0] = out_ms[1] = out_ms[2] = out_ms[3] = 0.0;
  if (!r && ce == cudaSuccess)
    for (size_t k = 1; k < used; ++k) {
      float ms = 0.f;
      cudaEventElapsedTime(&ms, ev[k - 1], ev[k]);
      out_ms[cat[k]] += ms;
    }
  for (auto& e : ev)
    if (e) cudaEventDestroy(e);
  CK(ce);
  return r;
}

int fdtd_time_block_stats(const fdtd_ctx* c, int64_t out[2]) {
  if (!c || !out) return FDTD_EINVAL;
  out[0] = c->plane_steps_computed; out[1] = c->plane_steps_owned;
  return FDTD_OK;
}

int fdtd_kernel_in_use(const fdtd_ctx* c) {
  if (!c) return FDTD_EINVAL;
  return c->fused ? FDTD_KERNEL_FUSED : (c->use_ref ? FDTD_KERNEL_REF : FDTD_KERNEL_AUTO);
}

static int field_bases(fdtd_ctx* c, int which, std::vector<float*>& bases, bool want_f64) {
  if (which < 0 || which > 3) { set_err("bad field selector"); return FDTD_EINVAL; }
  if (want_f64 != c->fp64) {
    set_err(c->fp64 ? "this context holds fp64 fields: use the _f64 entry points" : "this context holds fp32 fields: use the fp32 entry points");
    return FDTD_EUNSUPPORTED;
  }
  for (auto& d : c->doms) bases.push_back(c->fp64 ? (float*)d.v64.f[which] : d.v.f[which]);
  return FDTD_OK;
}

int fdtd_get_field(fdtd_ctx* c, int32_t which, float* dst) {
  if (!c || !dst) return FDTD_EINVAL;
  std::vector<float*> b;
  int r = field_bases(c, which, b, false);
  return r ? r : copy_field(c, b.data(), dst, true, true);
}

int fdtd_set_field(fdtd_ctx* c, int32_t which, const float* src) {
  if (!c || !src) return FDTD_EINVAL;
  std::vector<float*> b;
  int r = field_bases(c, which, b, false);
  if (r) return r;
  c->substeps_done = 0;                       // ghosts are written consistently: restart the exchange cadence
  return copy_field(c, b.data(), const_cast<float*>(src), false, false);
}

int fdtd_get_field_f64(fdtd_ctx* c, int32_t which, double* dst) {
  if (!c || !dst) return FDTD_EINVAL;
  std::vector<float*> b;
  int r = field_bases(c, which, b, true);
  return r ? r : copy_field(c, b.data(), (float*)dst, true, true, 8);
}

int fdtd_set_field_f64(fdtd_ctx* c, int32_t which, const double* src) {
  if (!c || !src) return FDTD_EINVAL;
  std::vector<float*> b;
  int r = field_bases(c, which, b, true);
  return r ? r : copy_field(c, b.data(), (float*)const_cast<double*>(src), false, false, 8);
}

int fdtd_get_field_box(fdtd_ctx* c, int32_t which, const int32_t lo[3], const int32_t size[3], float* dst) {
  if (!c || !lo || !size || !dst || which < 0 || which > 3) return FDTD_EINVAL;
  if (c->fp64) { set_err("fdtd_get_field_box reads fp32 fields: use fdtd_get_field_f64 on an fp64 context"); return FDTD_EUNSUPPORTED; }
  for (int a = 0; a < 3; ++a)
    if (lo[a] < 0 || size[a] <= 0 || lo[a] + size[a] > c->G.gn[a]) { set_err("box outside the grid"); return FDTD_EINVAL; }
  for (auto& d : c->doms) {
    const DomainView& v = d.v;
    // intersection of the box with this domain's owned cells, in global coordinates
    int g0[3], g1[3];
    const int o[3] = {v.ox, v.oy, v.oz};
    bool empty = false;
    for (int a = 0; a < 3; ++a) {
      g0[a] = std::max(lo[a], o[a] + d.own_lo[a]);
      g1[a] = std::min(lo[a] + size[a], o[a] + d.own_hi[a]);
      if (g1[a] <= g0[a]) empty = true;
    }
    if (empty) continue;
    for (int gk = g0[2]; gk < g1[2]; ++gk) {
      const float* dev = v.f[which] + (long long)(gk - v.oz) * v.plane + (long long)(g0[1] - v.oy) * v.pitch + (g0[0] - v.ox);
      float* h = dst + ((long long)(gk - lo[2]) * size[1] + (g0[1] - lo[1])) * size[0] + (g0[0] - lo[0]);
      CK(cudaMemcpy2DAsync(h, (size_t)size[0] * 4, dev, (size_t)v.pitch * 4, (size_t)(g1[0] - g0[0]) * 4, g1[1] - g0[1],
                           cudaMemcpyDeviceToHost, c->stream));
    }
  }
  CK(cudaStreamSynchronize(c->stream));
  return FDTD_OK;
}

int fdtd_fill_hash(fdtd_ctx* c, int32_t which, uint64_t seed, double scale) {
  if (!c || which < 0 || which > 3) return FDTD_EINVAL;
  for (auto& d : c->doms) {
    if (c->fp64) fill_hash_kernel<<<148 * 8, 256, 0, c->stream>>>(d.v64, which, seed, (float)scale);
    else fill_hash_kernel<<<148 * 8, 256, 0, c->stream>>>(d.v, which, seed, (float)scale);
    c->launches++;
  }
  c->substeps_done = 0;
  CK(cudaGetLastError());
  return FDTD_OK;
}

int fdtd_field_absmax(fdtd_ctx* c, int32_t which, const int32_t lo[3], const int32_t size[3], float* out) {
  if (!c || !lo || !size || !out || which < 0 || which > 3) return FDTD_EINVAL;
  for (int a = 0; a < 3; ++a)
    if (lo[a] < 0 || size[a] <= 0 || lo[a] + size[a] > c->G.gn[a]) { set_err("box outside the grid"); return FDTD_EINVAL; }
  unsigned int* acc = (unsigned int*)(c->ws + c->L.absmax);
  CK(cudaMemsetAsync(acc, 0, 4, c->stream));
  for (auto& d : c->doms) {
    const DomainView& v = d.v;
    const int o[3] = {v.ox, v.oy, v.oz};
    int g0[3], g1[3];
    bool empty = false;
    for (int a = 0; a < 3; ++a) {
      g0[a] = std::max(lo[a], o[a] + d.own_lo[a]);
      g1[a] = std::min(lo[a] + size[a], o[a] + d.own_hi[a]);
      if (g1[a] <= g0[a]) empty = true;
    }
    if (empty) continue;
    if (c->fp64)
      absmax_kernel<<<148 * 4, 256, 0, c->stream>>>(d.v64, which, g0[0] - o[0], g0[1] - o[1], g0[2] - o[2], g1[0] - g0[0], g1[1] - g0[1],
                                                    g1[2] - g0[2], acc);
    else
      absmax_kernel<<<148 * 4, 256, 0, c->stream>>>(v, which, g0[0] - o[0], g0[1] - o[1], g0[2] - o[2], g1[0] - g0[0], g1[1] - g0[1],
                                                    g1[2] - g0[2], acc);
    c->launches++;
  }
  CK(cudaGetLastError());
  unsigned int bits = 0;
  CK(cudaMemcpyAsync(&bits, acc, 4, cudaMemcpyDeviceToHost, c->stream));
  CK(cudaStreamSynchronize(c->stream));
  memcpy(out, &bits, 4);
  return FDTD_OK;
}

int fdtd_get_psi(fdtd_ctx* c, int32_t which, float* dst) {
  if (!c || !dst || which < 0 || which > 5) return FDTD_EINVAL;
  if (c->fp64) { set_err("this context holds fp64 memory variables: use fdtd_get_psi_f64"); return FDTD_EUNSUPPORTED; }
  for (auto& d : c->doms) {
    int r = get_psi_impl(c, d, d.v, which / 3, which % 3, dst);
    if (r) return r;
  }
  return FDTD_OK;
}

int fdtd_get_psi_f64(fdtd_ctx* c, int32_t which, double* dst) {
  if (!c || !dst || which < 0 || which > 5) return FDTD_EINVAL;
  if (!c->fp64) { set_err("this context holds fp32 memory variables: use fdtd_get_psi"); return FDTD_EUNSUPPORTED; }
  for (auto& d : c->doms) {
    int r = get_psi_impl(c, d, d.v64, which / 3, which % 3, dst);
    if (r) return r;
  }
  return FDTD_OK;
}

int fdtd_cpml_table(fdtd_ctx* c, int32_t axis, int32_t half, float* a, float* b, float* ik) {
  if (!c || axis < 0 || axis > 2 || !a || !b || !ik) return FDTD_EINVAL;
  const AxisTable& t = c->tabs[half ? 0 : 1][axis];
  const size_t n = (size_t)c->G.gn[axis];
  memcpy(a, t.a.data(), n * 4); memcpy(b, t.b.data(), n * 4); memcpy(ik, t.ik.data(), n * 4);
  return FDTD_OK;
}

}  // extern "C"

// ---- fdtd_absmax_noalloc: max |f| of a caller-owned device array with no allocation at all ---------------------------------
// The variant of absmax_kernel for callers that cannot allocate (CUDA graph capture, serving loops): absmax_kernel reduces
// into a scratch word of the context's workspace with atomicMax; this one keeps its scratch — one ticket counter and one
// partial maximum per thread block — in a file-scope device array of fixed size that every GPU loading the library holds
// until exit (FDTD_NOALLOC_SCRATCH_BYTES, 64.25 KB).  Block b reduces the fixed chunk [b, b+1) x NOALLOC_CHUNK of the
// input into partial[b]; the last block to finish (ticket) reduces the partials, writes the result and re-arms the ticket.
namespace {
constexpr int NOALLOC_MAX_BLOCKS = 16384;                 // partial maxima held by the static scratch
constexpr int NOALLOC_CHUNK = 65536;                      // floats per block: 256 threads x 64 float4
constexpr int NOALLOC_HEAD = 64;                          // words before the partials: word 0 is the ticket counter
static_assert((uint64_t)NOALLOC_MAX_BLOCKS * NOALLOC_CHUNK == FDTD_NOALLOC_MAX_ELEMS, "header and kernel disagree on the limit");
static_assert((NOALLOC_HEAD + NOALLOC_MAX_BLOCKS) * 4 == FDTD_NOALLOC_SCRATCH_BYTES, "header and kernel disagree on the scratch size");
// In host code this name is a host-side stand-in, not a device address: the host gets the address from cudaGetSymbolAddress.
static __device__ __align__(256) unsigned int g_noalloc_scratch[NOALLOC_HEAD + NOALLOC_MAX_BLOCKS];

__global__ void __launch_bounds__(256) absmax_noalloc_kernel(const float* __restrict__ in, unsigned long long n, unsigned int* scratch,
                                                             float* __restrict__ out) {
  __shared__ float s_m[8];
  __shared__ bool s_last;
  const unsigned long long lo = (unsigned long long)blockIdx.x * NOALLOC_CHUNK;
  const unsigned long long hi = lo + NOALLOC_CHUNK < n ? lo + NOALLOC_CHUNK : n;
  float m = 0.f;
  if ((reinterpret_cast<uintptr_t>(in) & 15) == 0) {       // lo is a multiple of 4 floats: whole float4s, then a scalar tail
    const unsigned long long v0 = lo >> 2, v1 = hi >> 2;
    for (unsigned long long t = v0 + threadIdx.x; t < v1; t += 256) {
      const float4 f = __ldg(reinterpret_cast<const float4*>(in) + t);
      m = fmaxf(m, fmaxf(fmaxf(fabsf(f.x), fabsf(f.y)), fmaxf(fabsf(f.z), fabsf(f.w))));
    }
    for (unsigned long long t = (v1 << 2) + threadIdx.x; t < hi; t += 256) m = fmaxf(m, fabsf(__ldg(in + t)));
  } else {
    for (unsigned long long t = lo + threadIdx.x; t < hi; t += 256) m = fmaxf(m, fabsf(__ldg(in + t)));
  }
  for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
  if ((threadIdx.x & 31) == 0) s_m[threadIdx.x >> 5] = m;
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < 8; ++w) m = fmaxf(m, s_m[w]);
    scratch[NOALLOC_HEAD + blockIdx.x] = __float_as_uint(m);
    __threadfence();                                       // the partial is visible before the ticket is taken
    s_last = atomicAdd(&scratch[0], 1u) == gridDim.x - 1;
  }
  __syncthreads();
  if (!s_last) return;
  __threadfence();
  float r = 0.f;
  for (unsigned int b = threadIdx.x; b < gridDim.x; b += 256) r = fmaxf(r, __uint_as_float(((volatile unsigned int*)scratch)[NOALLOC_HEAD + b]));
  for (int o = 16; o > 0; o >>= 1) r = fmaxf(r, __shfl_xor_sync(0xffffffffu, r, o));
  if ((threadIdx.x & 31) == 0) s_m[threadIdx.x >> 5] = r;
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < 8; ++w) r = fmaxf(r, s_m[w]);
    *out = r;
    scratch[0] = 0u;                                       // re-armed for the next call on this device
  }
}

constexpr int NOALLOC_MAX_DEVICES = 64;
unsigned int* g_noalloc_ptr[NOALLOC_MAX_DEVICES] = {nullptr};   // device address of g_noalloc_scratch, per device ordinal
std::mutex g_noalloc_mutex;
}  // namespace

extern "C" {

int fdtd_absmax_noalloc(const float* in_dev, uint64_t n, float* out_dev, void* stream) {
  if (!out_dev || (!in_dev && n > 0)) { set_err("fdtd_absmax_noalloc: null pointer"); return FDTD_EINVAL; }
  if (n > (uint64_t)FDTD_NOALLOC_MAX_ELEMS) {
    set_err("fdtd_absmax_noalloc: " + std::to_string((unsigned long long)n) + " elements exceed the maximum of " +
            std::to_string((unsigned long long)FDTD_NOALLOC_MAX_ELEMS) + " that the static scratch array supports");
    return FDTD_EINVAL;
  }
  int dev = -1;
  CK(cudaGetDevice(&dev));
  if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) { set_err("fdtd_absmax_noalloc: device ordinal out of range"); return FDTD_EINVAL; }
  unsigned int* scratch = nullptr;
  {
    std::lock_guard<std::mutex> lock(g_noalloc_mutex);
    if (!g_noalloc_ptr[dev]) {                            // set-up, once per device, with that device current
      void* ptr = nullptr;
      CK(cudaGetSymbolAddress(&ptr, g_noalloc_scratch));
      g_noalloc_ptr[dev] = (unsigned int*)ptr;
    }
    scratch = g_noalloc_ptr[dev];
  }
  cudaStream_t st = (cudaStream_t)stream;
  // The ticket must start at zero.  The kernel re-arms it, but a call that died half-way would leave it armed wrongly, so it
  // is cleared here as well (a memset node on the stream: no allocation).  The partials are overwritten before they are read.
  CK(cudaMemsetAsync(scratch, 0, NOALLOC_HEAD * 4, st));
  const unsigned int blocks = n == 0 ? 1u : (unsigned int)((n + NOALLOC_CHUNK - 1) / NOALLOC_CHUNK);
  absmax_noalloc_kernel<<<blocks, 256, 0, st>>>(in_dev, (unsigned long long)n, scratch, out_dev);
  CK(cudaGetLastError());
  return FDTD_OK;
}

int fdtd_destroy(fdtd_ctx* c) {
  if (!c) return FDTD_EINVAL;
  cudaError_t e = cudaStreamSynchronize(c->stream);
  delete c;
  if (e != cudaSuccess) { set_err(std::string("cudaStreamSynchronize: ") + cudaGetErrorString(e)); return FDTD_ECUDA; }
  return FDTD_OK;
}

}  // extern "C"
