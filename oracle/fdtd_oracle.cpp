// ORACLE — TEST INFRASTRUCTURE ONLY.
//
// Plain, slow, obviously-correct CPU implementation of one time step of the
// staggered-grid 8th-order 3-D acoustic pressure-velocity FDTD update with
// CPML layers (Table 2).  It exists to check the
// CUDA path; only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
// --impl reference legs may build, load or call it.  It shares no code,
// header, table or constant generator with paper_2606_06910_b200/csrc.
//
// Written as the recurrence itself: a triple loop, one point at a time, sums
// in the order stated, no tiling, no fusion, no intrinsics.  `#pragma omp
// parallel for` over z planes is the only concession (every point of one
// sub-update is independent, so results are bit-identical to one thread).
// Compile with -O2 -ffp-contract=off (no FMA contraction, reading R25).
//
// Pins (tests/test_oracle_pins.py): coefficient bit patterns and Taylor
// conditions, discrete dispersion relation, one-step impulse response,
// spatial order 8, reflection / permutation symmetries, CPML -> interior
// reduction, leapfrog energy conservation / decay, stability edge, temporal
// order 2, worked CPML tables.
// PARITY UNPINNED (no printed values in the paper to check against; fixed by
// DESIGN.md readings): R8 exact rho offsets of the staggered CPML profiles,
// R10 psi update-then-use ordering, R14 source time shift / amplitude.

#include <cmath>
#include <cstdint>
#include <cstring>
#include <cstdlib>
#include <vector>
#include <xmmintrin.h>
#ifdef _OPENMP
#include <omp.h>
#endif

extern "C" {
// Plain-data parameter block (mirrors the paper's Table 2).
struct orc_params {
  int32_t n_interior[3];   // interior cells x,y,z
  int32_t cpml[6];         // CPML thickness per face x-,x+,y-,y+,z-,z+ (0 = plain wall)
  double dx, dt;           // cubic cell size, time step
  int32_t cpml_order;      // q (3; BASELINE configs: 2)
  int32_t boundary;        // 0 = WALL (reads outside return 0), 1 = PERIODIC
  double cpml_R0;          // target reflection R
  double cpml_kappa_max;
  double cpml_alpha_max;
  double cpml_c_ref;       // wave speed absorbed in sigma_max (reading R7)
};
}

namespace {

// Staggered 8th-order weights (BASELINE.json config 1; the a_l of P:38 in the
// staggered reading R1), stored as fp32 and used as such in both precisions.
const float kCoef[4] = {1225.0f / 1024.0f, -245.0f / 3072.0f, 49.0f / 5120.0f, -5.0f / 7168.0f};

// CPML profile at normalised depth rho.  Doubles in, fp32 out.
struct Tab { std::vector<float> a, b, ik; std::vector<uint8_t> in; };

void profile_point(double rho, double sigma_max, const orc_params& P, float& a, float& b, float& ik, uint8_t& in) {
  if (!(rho > 0.0)) { a = 0.0f; b = 1.0f; ik = 1.0f; in = 0; return; }   // outside the layer
  double rq = std::pow(rho, (double)P.cpml_order);
  double sigma = sigma_max * rq;                                   // sigma(rho) = sigma_max rho^q
  double kappa = 1.0 + (P.cpml_kappa_max - 1.0) * rq;              // kappa(rho)
  double alpha = P.cpml_alpha_max * std::fmax(0.0, 1.0 - rho);     // alpha(rho) = alpha_max (1 - rho)
  double bb = std::exp(-(sigma / kappa + alpha) * P.dt);           // b = exp[-(sigma/kappa + alpha) dt]
  double den = kappa * (sigma + kappa * alpha);
  double aa = (den == 0.0) ? 0.0 : sigma * (bb - 1.0) / den;       // a = sigma (b-1) / [kappa (sigma + kappa alpha)]  (R9)
  a = (float)aa; b = (float)bb; ik = (float)(1.0 / kappa); in = 1;
}

// Tables of one axis for one staggering (half = 1: nodes at i+1/2, the v family;
// half = 0: integer nodes, the p family).  Reading R8: the layer interface sits
// on the first interior node.
Tab make_table(int N, int L0, int L1, int half, const orc_params& P) {
  Tab t; t.a.resize(N); t.b.resize(N); t.ik.resize(N); t.in.resize(N);
  for (int i = 0; i < N; ++i) {
    double pos = i + (half ? 0.5 : 0.0);
    double rho = 0.0, smax = 0.0;
    if (L0 > 0 && (double)L0 - pos > 0.0) {
      rho = ((double)L0 - pos) / L0;
      smax = -(P.cpml_order + 1.0) * P.cpml_c_ref * std::log(P.cpml_R0) / (2.0 * L0 * P.dx);   // R7
    } else if (L1 > 0 && pos - (double)(N - 1 - L1) > 0.0) {
      rho = (pos - (double)(N - 1 - L1)) / L1;
      smax = -(P.cpml_order + 1.0) * P.cpml_c_ref * std::log(P.cpml_R0) / (2.0 * L1 * P.dx);
    }
    profile_point(rho, smax, P, t.a[i], t.b[i], t.ik[i], t.in[i]);
  }
  return t;
}

// Counter-based generator for synthetic initial states at any grid size:
// splitmix64 of (seed + global linear index), top 24 bits -> [-1, 1).
inline uint64_t splitmix64(uint64_t x) {
  x += 0x9E3779B97F4A7C15ull;
  x = (x ^ (x >> 30)) * 0xBF58476D1CE4E5B9ull;
  x = (x ^ (x >> 27)) * 0x94D049BB133111EBull;
  return x ^ (x >> 31);
}
inline float hash_unit(uint64_t seed, uint64_t idx) {
  uint64_t h = splitmix64(seed + idx);
  return (float)(int32_t)((uint32_t)(h >> 40)) * (1.0f / 8388608.0f) - 1.0f;
}

template <class T>
struct Sim {
  orc_params P;
  int nx, ny, nz;
  bool periodic;
  size_t n;
  std::vector<T> f[4];       // p, vx, vy, vz
  std::vector<T> psi[6];     // psi_vx, psi_vy, psi_vz, psi_px, psi_py, psi_pz (full volume: simplicity over memory)
  std::vector<T> p_prev;     // p^n kept for the leapfrog energy
  std::vector<float> Kc;     // rho c^2 dt/dx per node (R6), rounded once to fp32
  std::vector<float> Bx, By, Bz;  // dt/(rho_bar dx) per half node; empty = scalar B0
  float B0;
  bool have_rho;
  std::vector<float> rho_node, c_node;
  Tab th[3], tf[3];          // half-node (v family) and integer-node (p family) tables per axis
  int nsrc = 0, wlen = 0;
  std::vector<int32_t> src;  // 3*nsrc total-grid indices
  std::vector<float> wav;    // nsrc*wlen
  long step_count = 0;
  int ftz = 0;
  int track_energy = 0;

  explicit Sim(const orc_params& p) : P(p) {
    nx = p.n_interior[0] + p.cpml[0] + p.cpml[1];
    ny = p.n_interior[1] + p.cpml[2] + p.cpml[3];
    nz = p.n_interior[2] + p.cpml[4] + p.cpml[5];
    periodic = p.boundary == 1;
    n = (size_t)nx * ny * nz;
    for (auto& a : f) a.assign(n, T(0));
    for (auto& a : psi) a.assign(n, T(0));
    int N[3] = {nx, ny, nz};
    for (int a = 0; a < 3; ++a) {
      th[a] = make_table(N[a], p.cpml[2 * a], p.cpml[2 * a + 1], 1, p);
      tf[a] = make_table(N[a], p.cpml[2 * a], p.cpml[2 * a + 1], 0, p);
    }
    set_model(nullptr, nullptr);
  }

  size_t idx(long i, long j, long k) const { return (size_t)i + (size_t)nx * ((size_t)j + (size_t)ny * (size_t)k); }

  // Field read with the outer boundary rule (R4): WALL returns 0 outside, PERIODIC wraps.
  T rd(const std::vector<T>& a, long i, long j, long k) const {
    if (periodic) {
      i = ((i % nx) + nx) % nx; j = ((j % ny) + ny) % ny; k = ((k % nz) + nz) % nz;
    } else if (i < 0 || i >= nx || j < 0 || j >= ny || k < 0 || k >= nz) {
      return T(0);
    }
    return a[idx(i, j, k)];
  }

  // Medium (R6): B = dt/(rho_bar dx) at half nodes, Kc = rho c^2 dt/dx at nodes;
  // double arithmetic on the fp32 inputs, rounded once to fp32.
  void set_model(const float* c, const float* rho) {
    Kc.resize(n);
    c_node.assign(n, 1.0f); rho_node.assign(n, 1.0f);
    if (c) std::memcpy(c_node.data(), c, n * sizeof(float));
    if (rho) std::memcpy(rho_node.data(), rho, n * sizeof(float));
    have_rho = rho != nullptr;
    for (size_t q = 0; q < n; ++q) {
      double cc = c_node[q], rr = rho_node[q];
      Kc[q] = (float)(rr * cc * cc * P.dt / P.dx);
    }
    B0 = (float)(P.dt / (1.0 * P.dx));
    Bx.clear(); By.clear(); Bz.clear();
    if (have_rho) {
      Bx.resize(n); By.resize(n); Bz.resize(n);
      for (long k = 0; k < nz; ++k) for (long j = 0; j < ny; ++j) for (long i = 0; i < nx; ++i) {
        auto R = [&](long ii, long jj, long kk) -> double {
          if (periodic) { ii = (ii + nx) % nx; jj = (jj + ny) % ny; kk = (kk + nz) % nz; }
          else { if (ii >= nx) ii = nx - 1; if (jj >= ny) jj = ny - 1; if (kk >= nz) kk = nz - 1; }
          return rho_node[idx(ii, jj, kk)];
        };
        double r0 = R(i, j, k);
        Bx[idx(i, j, k)] = (float)(P.dt / (0.5 * (r0 + R(i + 1, j, k)) * P.dx));
        By[idx(i, j, k)] = (float)(P.dt / (0.5 * (r0 + R(i, j + 1, k)) * P.dx));
        Bz[idx(i, j, k)] = (float)(P.dt / (0.5 * (r0 + R(i, j, k + 1)) * P.dx));
      }
    }
  }

  void enter_parallel() const { if (ftz) _mm_setcsr(_mm_getcsr() | 0x8040); }

  // Velocity sub-update: v_a <- v_a - (dt/rho) [ (1/kappa_a) D+_a p + psi_va ].
  void substep_v() {
    const T c1 = kCoef[0], c2 = kCoef[1], c3 = kCoef[2], c4 = kCoef[3];
    const std::vector<T>& p = f[0];
#pragma omp parallel
    {
      enter_parallel();
#pragma omp for schedule(static)
      for (long k = 0; k < nz; ++k)
        for (long j = 0; j < ny; ++j)
          for (long i = 0; i < nx; ++i) {
            const size_t q = idx(i, j, k);
            // x: D+ p at half node i+1/2 = sum_l c_l (p[i+l] - p[i-l+1])   (R1)
            if (periodic || i < nx - 1) {           // last half node is pinned (R3)
              T d = c1 * (rd(p, i + 1, j, k) - rd(p, i, j, k));
              d += c2 * (rd(p, i + 2, j, k) - rd(p, i - 1, j, k));
              d += c3 * (rd(p, i + 3, j, k) - rd(p, i - 2, j, k));
              d += c4 * (rd(p, i + 4, j, k) - rd(p, i - 3, j, k));
              if (th[0].in[i]) {                     // CPML: psi <- b psi + a d ; d <- d/kappa + psi   (R10)
                psi[0][q] = T(th[0].b[i]) * psi[0][q] + T(th[0].a[i]) * d;
                d = d * T(th[0].ik[i]) + psi[0][q];
              }
              const T B = have_rho ? T(Bx[q]) : T(B0);
              f[1][q] -= B * d;
            }
            if (periodic || j < ny - 1) {
              T d = c1 * (rd(p, i, j + 1, k) - rd(p, i, j, k));
              d += c2 * (rd(p, i, j + 2, k) - rd(p, i, j - 1, k));
              d += c3 * (rd(p, i, j + 3, k) - rd(p, i, j - 2, k));
              d += c4 * (rd(p, i, j + 4, k) - rd(p, i, j - 3, k));
              if (th[1].in[j]) {
                psi[1][q] = T(th[1].b[j]) * psi[1][q] + T(th[1].a[j]) * d;
                d = d * T(th[1].ik[j]) + psi[1][q];
              }
              const T B = have_rho ? T(By[q]) : T(B0);
              f[2][q] -= B * d;
            }
            if (periodic || k < nz - 1) {
              T d = c1 * (rd(p, i, j, k + 1) - rd(p, i, j, k));
              d += c2 * (rd(p, i, j, k + 2) - rd(p, i, j, k - 1));
              d += c3 * (rd(p, i, j, k + 3) - rd(p, i, j, k - 2));
              d += c4 * (rd(p, i, j, k + 4) - rd(p, i, j, k - 3));
              if (th[2].in[k]) {
                psi[2][q] = T(th[2].b[k]) * psi[2][q] + T(th[2].a[k]) * d;
                d = d * T(th[2].ik[k]) + psi[2][q];
              }
              const T B = have_rho ? T(Bz[q]) : T(B0);
              f[3][q] -= B * d;
            }
          }
    }
  }

  // Pressure sub-update (P:40 with the z term restored per P:56, R2):
  // p <- p - K dt [ sum_a (1/kappa_a) D-_a v_a + psi_pa ].
  void substep_p() {
    const T c1 = kCoef[0], c2 = kCoef[1], c3 = kCoef[2], c4 = kCoef[3];
    if (track_energy) p_prev = f[0];
    const std::vector<T>&vx = f[1], &vy = f[2], &vz = f[3];
#pragma omp parallel
    {
      enter_parallel();
#pragma omp for schedule(static)
      for (long k = 0; k < nz; ++k)
        for (long j = 0; j < ny; ++j)
          for (long i = 0; i < nx; ++i) {
            const size_t q = idx(i, j, k);
            // D- v at node i = sum_l c_l (v[i+l-1] - v[i-l])   (R1)
            T dxv = c1 * (rd(vx, i, j, k) - rd(vx, i - 1, j, k));
            dxv += c2 * (rd(vx, i + 1, j, k) - rd(vx, i - 2, j, k));
            dxv += c3 * (rd(vx, i + 2, j, k) - rd(vx, i - 3, j, k));
            dxv += c4 * (rd(vx, i + 3, j, k) - rd(vx, i - 4, j, k));
            if (tf[0].in[i]) {
              psi[3][q] = T(tf[0].b[i]) * psi[3][q] + T(tf[0].a[i]) * dxv;
              dxv = dxv * T(tf[0].ik[i]) + psi[3][q];
            }
            T dyv = c1 * (rd(vy, i, j, k) - rd(vy, i, j - 1, k));
            dyv += c2 * (rd(vy, i, j + 1, k) - rd(vy, i, j - 2, k));
            dyv += c3 * (rd(vy, i, j + 2, k) - rd(vy, i, j - 3, k));
            dyv += c4 * (rd(vy, i, j + 3, k) - rd(vy, i, j - 4, k));
            if (tf[1].in[j]) {
              psi[4][q] = T(tf[1].b[j]) * psi[4][q] + T(tf[1].a[j]) * dyv;
              dyv = dyv * T(tf[1].ik[j]) + psi[4][q];
            }
            T dzv = c1 * (rd(vz, i, j, k) - rd(vz, i, j, k - 1));
            dzv += c2 * (rd(vz, i, j, k + 1) - rd(vz, i, j, k - 2));
            dzv += c3 * (rd(vz, i, j, k + 2) - rd(vz, i, j, k - 3));
            dzv += c4 * (rd(vz, i, j, k + 3) - rd(vz, i, j, k - 4));
            if (tf[2].in[k]) {
              psi[5][q] = T(tf[2].b[k]) * psi[5][q] + T(tf[2].a[k]) * dzv;
              dzv = dzv * T(tf[2].ik[k]) + psi[5][q];
            }
            f[0][q] -= T(Kc[q]) * ((dxv + dyv) + dzv);
          }
    }
  }

  // Additive pressure source (R14): p[src] += w[n] after the pressure sub-update of step n.
  void inject() {
    for (int s = 0; s < nsrc; ++s) {
      if (step_count < wlen) {
        f[0][idx(src[3 * s], src[3 * s + 1], src[3 * s + 2])] += T(wav[(size_t)s * wlen + step_count]);
      }
    }
  }

  void step(int nsteps) {
    for (int s = 0; s < nsteps; ++s) { substep_v(); substep_p(); inject(); ++step_count; }
  }

  // Leapfrog-conserved energy at time n+1/2 (R19), over the interior cells:
  // E = 1/2 sum_a sum rho_bar v_a^2 + 1/2 sum p^n p^{n+1} / (rho c^2), in units of dx^3.
  // Valid after at least one step() with track_energy set.
  double energy() const {
    if (p_prev.size() != n) return -1.0;
    int lo[3] = {P.cpml[0], P.cpml[2], P.cpml[4]};
    int hi[3] = {nx - P.cpml[1], ny - P.cpml[3], nz - P.cpml[5]};
    double e = 0.0;
    for (long k = lo[2]; k < hi[2]; ++k) for (long j = lo[1]; j < hi[1]; ++j) for (long i = lo[0]; i < hi[0]; ++i) {
      size_t q = idx(i, j, k);
      double rr = rho_node[q], cc = c_node[q];
      double rbx = 1.0, rby = 1.0, rbz = 1.0;
      if (have_rho) { rbx = P.dt / ((double)Bx[q] * P.dx); rby = P.dt / ((double)By[q] * P.dx); rbz = P.dt / ((double)Bz[q] * P.dx); }
      double vx = f[1][q], vy = f[2][q], vz = f[3][q];
      e += 0.5 * (rbx * vx * vx + rby * vy * vy + rbz * vz * vz);
      e += 0.5 * (double)p_prev[q] * (double)f[0][q] / (rr * cc * cc);
    }
    return e;
  }
};

struct Handle { int is64; Sim<float>* s32; Sim<double>* s64; };

}  // namespace

#define DISPATCH(h, expr) do { Handle* H = (Handle*)(h); if (H->is64) { auto& S = *H->s64; expr; } else { auto& S = *H->s32; expr; } } while (0)

extern "C" {

void orc_coeffs(float out[4]) { for (int i = 0; i < 4; ++i) out[i] = kCoef[i]; }

void* orc_create(const orc_params* p, int use_fp64) {
  Handle* H = new Handle{use_fp64, nullptr, nullptr};
  if (use_fp64) H->s64 = new Sim<double>(*p); else H->s32 = new Sim<float>(*p);
  return H;
}
void orc_destroy(void* h) { Handle* H = (Handle*)h; delete H->s32; delete H->s64; delete H; }

void orc_dims(void* h, int32_t out[3]) { DISPATCH(h, out[0] = S.nx; out[1] = S.ny; out[2] = S.nz); }
void orc_set_threads(int n) {
#ifdef _OPENMP
  omp_set_num_threads(n);
#else
  (void)n;
#endif
}
int orc_max_threads() {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}
void orc_set_ftz(void* h, int on) { DISPATCH(h, S.ftz = on); }
void orc_track_energy(void* h, int on) { DISPATCH(h, S.track_energy = on); }
void orc_set_model(void* h, const float* c, const float* rho) { DISPATCH(h, S.set_model(c, rho)); }
void orc_set_sources(void* h, int n, const int32_t* ijk, const float* wavelets, int len) {
  DISPATCH(h, S.nsrc = n; S.wlen = len; S.src.assign(ijk, ijk + 3 * n); S.wav.assign(wavelets, wavelets + (size_t)n * len));
}
void orc_step(void* h, int n) { DISPATCH(h, S.step(n)); }
void orc_substep_v(void* h) { DISPATCH(h, S.substep_v()); }
void orc_substep_p(void* h) { DISPATCH(h, S.substep_p()); }
double orc_energy(void* h) { double e = 0; DISPATCH(h, e = S.energy()); return e; }

// which: 0..3 = p,vx,vy,vz ; 4..9 = psi_vx,psi_vy,psi_vz,psi_px,psi_py,psi_pz.  Always exchanged as double.
void orc_get_field(void* h, int which, double* dst) {
  DISPATCH(h, { auto& a = which < 4 ? S.f[which] : S.psi[which - 4]; for (size_t q = 0; q < S.n; ++q) dst[q] = (double)a[q]; });
}
void orc_set_field(void* h, int which, const double* src) {
  DISPATCH(h, { auto& a = which < 4 ? S.f[which] : S.psi[which - 4]; for (size_t q = 0; q < S.n; ++q) a[q] = (decltype(a[0] + 0))src[q]; });
}

// Fill field `which` (0..3) with the counter-based generator evaluated at GLOBAL
// coordinates: this grid is the window [off, off + n) of a gdim grid.
void orc_fill_hash(void* h, int which, uint64_t seed, const int64_t gdim[3], const int64_t off[3], double scale) {
  DISPATCH(h, {
    auto& a = S.f[which];
    for (long k = 0; k < S.nz; ++k) for (long j = 0; j < S.ny; ++j) for (long i = 0; i < S.nx; ++i) {
      uint64_t g = (uint64_t)(i + off[0]) + (uint64_t)gdim[0] * ((uint64_t)(j + off[1]) + (uint64_t)gdim[1] * (uint64_t)(k + off[2]));
      a[S.idx(i, j, k)] = (decltype(a[0] + 0))((float)scale * hash_unit(seed + ((uint64_t)which << 56), g));
    }
  });
}

// CPML tables of one axis (0..2), one staggering (half = 1: v family), as fp32: a, b, 1/kappa, in-layer flag.
void orc_cpml_table(void* h, int axis, int half, float* a, float* b, float* ik, uint8_t* in) {
  DISPATCH(h, {
    const Tab& t = half ? S.th[axis] : S.tf[axis];
    for (size_t i = 0; i < t.a.size(); ++i) { a[i] = t.a[i]; b[i] = t.b[i]; ik[i] = t.ik[i]; in[i] = t.in[i]; }
  });
}

}  // extern "C"
