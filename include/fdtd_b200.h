/* fdtd_b200.h — C ABI of the B200-native 3-D acoustic FDTD + CPML time step.
 *
 * The operation is one time step of the staggered-grid, radius-4 (8th-order) pressure-velocity update of
 * PAPER.md section 3.1 with the CPML memory-variable recursion of section 3.2 in the
 * outer absorbing layer, parameters of Table 2.  P:NN = line NN of the paper text; Rn = a
 * reading listed in DESIGN.md where the paper is silent or ambiguous.
 *
 * Conventions
 *   - Total grid N_a = n_interior[a] + cpml[2a] + cpml[2a+1]; x fastest: idx = i + Nx (j + Ny k).
 *   - p lives on nodes (i,j,k); vx on (i+1/2,j,k); vy on (i,j+1/2,k); vz on (i,j,k+1/2) (R1, R3).
 *   - All fields are fp32.  Every pointer argument says HOST or DEVICE.
 *   - Every entry point except fdtd_create / fdtd_workspace_bytes / fdtd_last_error returns 0 on success
 *     and a negative FDTD_E* code on error; on error the context is left unchanged.  CUDA errors are
 *     captured and returned (FDTD_ECUDA), never abort().  No exception crosses this boundary.
 *   - Nothing here has a CPU fallback: without a CUDA device every compute call fails with FDTD_ECUDA.
 *   - Work is enqueued on params.stream; calls are asynchronous unless the comment says "synchronises".
 */
#ifndef FDTD_B200_H
#define FDTD_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct fdtd_ctx fdtd_ctx; /* opaque */

enum {
  FDTD_OK = 0,
  FDTD_EINVAL = -1,     /* bad size / parameter (dt <= 0, grid smaller than the layers, source out of range ...) */
  FDTD_EWORKSPACE = -2, /* workspace NULL, misaligned (256 B) or smaller than fdtd_workspace_bytes() */
  FDTD_ECUDA = -3,      /* a CUDA runtime / driver call failed; fdtd_last_error() has the text */
  FDTD_EUNSUPPORTED = -4 /* valid per the paper but not built in this configuration (e.g. a density array without */
                         /* params.density = FDTD_DENSITY_ARRAY, or FDTD_PRECISION_FP64 with FDTD_KERNEL_FUSED)   */
};

enum { FDTD_P = 0, FDTD_VX = 1, FDTD_VY = 2, FDTD_VZ = 3 };                 /* field selectors */
enum { FDTD_PSI_VX = 0, FDTD_PSI_VY = 1, FDTD_PSI_VZ = 2, FDTD_PSI_PX = 3, FDTD_PSI_PY = 4, FDTD_PSI_PZ = 5 };
enum { FDTD_WALL = 0, FDTD_PERIODIC = 1 };
enum {
  FDTD_DENSITY_UNIFORM = 0, /* rho is one number: dt/(rho dx) is a scalar                                     */
  FDTD_DENSITY_ARRAY = 1    /* the workspace also holds dt/(rho_bar dx) at the half nodes of vx, vy, vz (+12 B */
                            /* per point), so fdtd_set_model accepts a heterogeneous rho (R6)     */
};
enum {
  FDTD_MEDIUM_ARRAY = 0,  /* the workspace holds a per-node K dt/dx array (+4 B per point), so fdtd_set_model accepts a   */
                          /* wave-speed array c(x) (BASELINE config 3)                                                   */
  FDTD_MEDIUM_UNIFORM = 1 /* c is one number: no per-node array is reserved (saves one field: 16.4 GB at 1600^3);        */
                          /* fdtd_set_model with a c array then returns FDTD_EUNSUPPORTED                                */
};
enum {
  FDTD_PRECISION_FP32 = 0, /* single precision state and arithmetic: the product path                     */
  FDTD_PRECISION_FP64 = 1  /* "verification precision": fields, memory variables and arithmetic in double; every */
                           /* coefficient stays the fp32 number of the fp32 path.  One-thread-per-point kernels only,    */
                           /* monolithic only; fields move through the *_f64 entry points                                */
};
enum {
  FDTD_KERNEL_AUTO = 0, /* TMA-staged, z-streaming tile kernels (the product path)                        */
  FDTD_KERNEL_REF = 1,  /* one thread per point, global loads only; also the only path for FDTD_PERIODIC   */
  FDTD_KERNEL_FUSED = 2 /* one launch per time step: both sub-updates in a single pass over the fields (32 B  */
                        /* per point instead of 48), the single-GPU form of the enlarged ghost of P:42 (a     */
                        /* ghost of 2r = 8 cells per step, recomputed in x and y, streamed in z).  Out of      */
                        /* place: the workspace holds two copies of the fields and psi.  Same bits as AUTO.   */
                        /* Needs FDTD_WALL; in subdomain mode also a total Nx % 4 == 0 and an even            */
                        /* substeps_per_exchange.                                                              */
};

/* Problem statement and Table 2 as one plain-data block. */
typedef struct {
  int32_t n_interior[3];  /* interior cells x, y, z                                                        */
  int32_t cpml[6];        /* CPML thickness per global face x-,x+,y-,y+,z-,z+ in cells; 0 = plain wall (R13) */
  double dx, dt;          /* cubic cell size; time step chosen by the caller (Courant * dx / c_max, R15)    */
  int32_t cpml_order;     /* q: grading order (P:50 uses 3; BASELINE configs use 2)                         */
  int32_t boundary;       /* FDTD_WALL: reads outside the grid return 0 (R4); FDTD_PERIODIC: wrap (tests)   */
  double cpml_R0;         /* target reflection R of sigma_max                                 */
  double cpml_kappa_max;  /* kappa_max                                                        */
  double cpml_alpha_max;  /* alpha_max                                                        */
  double cpml_c_ref;      /* wave speed absorbed into sigma_max = -(q+1) c_ref ln(R0) / (2 L dx) (R7)        */
  int32_t decomp[3];      /* in-HBM subdomain grid Px, Py, Pz; {1,1,1} (or zeros) = monolithic.  1 x Py x Pz is */
                          /* the paper's pencil-yz (x stays local and contiguous), 1 x 1 x Pz slab-z,     */
                          /* Px x Py x 1 block-xy; an x cut needs widths and ghost that are multiples of 4      */
  int32_t ghost;          /* ghost depth g in cells on every internal interface                 */
  int32_t substeps_per_exchange; /* m sub-updates (v or p) between halo exchanges; needs g >= 4 m (R20)      */
  int32_t kernel;         /* FDTD_KERNEL_AUTO / FDTD_KERNEL_REF / FDTD_KERNEL_FUSED                          */
  int32_t density;        /* FDTD_DENSITY_UNIFORM / FDTD_DENSITY_ARRAY                                       */
  int32_t medium;         /* FDTD_MEDIUM_ARRAY (default) / FDTD_MEDIUM_UNIFORM                               */
  int32_t precision;      /* FDTD_PRECISION_FP32 (default) / FDTD_PRECISION_FP64                             */
  int32_t time_block;     /* k = 0 / 1: one time step per pass over the grid.  k >= 2 (FDTD_KERNEL_FUSED,    */
                          /* monolithic): k steps per pass over z slabs, each slab recomputing a ghost of    */
                          /* 2r = 8 planes per remaining step on both sides (the enlarged ghost of P:42,     */
                          /* P:82 inside one GPU); two more copies of the state; same bits as k = 1          */
  int32_t time_block_planes; /* slab thickness for time_block >= 2; 0 = sized to keep a slab's planes in L2  */
  int32_t device;         /* CUDA device ordinal                                                             */
  void* stream;           /* cudaStream_t the work is enqueued on (0 = legacy default stream)                */
  void* workspace;        /* DEVICE memory, 256-byte aligned, owned by the caller, must outlive the context  */
  uint64_t workspace_bytes;
} fdtd_params;

/* Bytes of device workspace fdtd_create needs for these parameters (fields p, vx, vy, vz, the per-node
 * K dt/dx array unless params.medium = FDTD_MEDIUM_UNIFORM, slab-local psi arrays, CPML tables, source tables;
 * FDTD_KERNEL_FUSED: a second copy of the fields and psi).  0 on invalid parameters.
 * Reads only the size fields; no CUDA call. */
uint64_t fdtd_workspace_bytes(const fdtd_params* params);

/* Builds a context: lays the arrays out in params->workspace, zero-fills fields and psi (BASELINE config 1:
 * "fields initialised to zero"), computes the CPML tables b = exp[-(sigma/kappa + alpha) dt],
 * a = sigma (b-1) / [kappa (sigma + kappa alpha)] in double on the host and uploads them as fp32,
 * sets the homogeneous medium c = rho = 1, step counter 0.  Returns NULL on error (see fdtd_last_error). */
fdtd_ctx* fdtd_create(const fdtd_params* params);

/* Medium (R6): c and rho are HOST arrays of the total grid (Nz*Ny*Nx fp32, x fastest) or NULL for 1.0
 * everywhere.  The library forms K dt/dx = rho c^2 dt/dx per node and dt/(rho_bar dx) per half node, rho_bar = mean
 * of the two adjacent nodes (the last node repeats itself), in double arithmetic rounded once to fp32, and copies
 * them to the device before returning (synchronises the stream).  A non-uniform rho needs
 * params.density = FDTD_DENSITY_ARRAY, else FDTD_EUNSUPPORTED. */
int fdtd_set_model(fdtd_ctx* ctx, const float* c_host, const float* rho_host);

/* Point sources injected into p (P:193 gives the Ricker shape; R14): after the pressure sub-update of step n,
 * p[ijk_s] += wavelets[s*len + n]; steps n >= len inject nothing.  ijk: HOST, 3*n total-grid indices;
 * wavelets: HOST, n*len fp32.  Copied before return (synchronises the stream).  n = 0 clears the sources.  n counts
 * every step since fdtd_create, also those taken before this call; sources that share a node are all added, in order. */
int fdtd_set_sources(fdtd_ctx* ctx, int32_t n, const int32_t* ijk_host, const float* wavelets_host, int32_t len);

/* Advances n time steps: for each step the velocity sub-update v_a -= (dt/rho)[(1/kappa_a) D+_a p + psi_va],
 * psi_va <- b psi_va + a D+_a p, then the pressure sub-update
 * p -= K dt sum_a [(1/kappa_a) D-_a v_a + psi_pa] (the z term per R2), then the source.  In subdomain
 * mode a halo exchange (pack / copy / unpack) runs every substeps_per_exchange sub-updates.
 * Asynchronous on params.stream; no host synchronisation. */
int fdtd_step(fdtd_ctx* ctx, int32_t n);

/* fdtd_step with CUDA events recorded on params.stream around every launch group: out_ms_host[0] = total time of
 * the velocity sub-update kernels, [1] = pressure sub-update kernels, [2] = source injection, [3] = halo exchange,
 * in milliseconds over the n steps (FDTD_KERNEL_FUSED: [0] = the fused step kernel, [1] = 0).  Same arithmetic and
 * launches as fdtd_step.  Synchronises. */
int fdtd_step_profiled(fdtd_ctx* ctx, int32_t n, double out_ms_host[4]);

/* Copies one field (FDTD_P..FDTD_VZ) of the total grid, unpadded, to dst_host (Nz*Ny*Nx fp32).  In subdomain
 * mode the owned cells of every subdomain are gathered.  Synchronises the stream. */
int fdtd_get_field(fdtd_ctx* ctx, int32_t which, float* dst_host);

/* The same two calls for a context created with FDTD_PRECISION_FP64 (Nz*Ny*Nx doubles).  The fp32 calls refuse an fp64
 * context and the other way round (FDTD_EUNSUPPORTED). */
int fdtd_get_field_f64(fdtd_ctx* ctx, int32_t which, double* dst_host);
int fdtd_set_field_f64(fdtd_ctx* ctx, int32_t which, const double* src_host);

/* Sub-box [lo, lo+size) of one field to dst_host (size[2]*size[1]*size[0] fp32, x fastest).  Synchronises. */
int fdtd_get_field_box(fdtd_ctx* ctx, int32_t which, const int32_t lo[3], const int32_t size[3], float* dst_host);

/* Overwrites one field from a HOST array of the total grid (initial conditions for tests).  In subdomain mode
 * ghost cells are filled consistently.  Synchronises. */
int fdtd_set_field(fdtd_ctx* ctx, int32_t which, const float* src_host);

/* Fills one field on the device with the counter-based generator scale * u(seed + (which << 56), global linear
 * index), u = top 24 bits of splitmix64 mapped to [-1, 1) — synthetic initial states at any grid size
 * (DESIGN.md "Input recipe").  Asynchronous. */
int fdtd_fill_hash(fdtd_ctx* ctx, int32_t which, uint64_t seed, double scale);

/* One CPML memory variable (FDTD_PSI_*) expanded from its slab-local storage to the full total grid (zeros
 * outside the slabs) into dst_host — debugging / parity of the recursion.  Synchronises. */
int fdtd_get_psi(fdtd_ctx* ctx, int32_t which, float* dst_host);

int fdtd_get_psi_f64(fdtd_ctx* ctx, int32_t which, double* dst_host);   /* the same for an fp64 context */

/* max |f| over the box [lo, lo+size) of one field, reduced on the device; result to *out_host.  Synchronises. */
int fdtd_field_absmax(fdtd_ctx* ctx, int32_t which, const int32_t lo[3], const int32_t size[3], float* out_host);

/* The CPML tables of one axis (0..2) and one staggering (half = 1: v family at i+1/2; 0: p family at nodes), as
 * uploaded: a, b, 1/kappa, each N_axis fp32 into HOST arrays (R8).  Outside the layer a = 0, b = 1,
 * 1/kappa = 1. */
int fdtd_cpml_table(fdtd_ctx* ctx, int32_t axis, int32_t half, float* a_host, float* b_host, float* ik_host);

/* The four staggered difference weights c_1..c_4 as the kernels use them (fp32; BASELINE: bit-exact). */
int fdtd_coeffs(float out_host[4]);

/* The kernel family this context runs: FDTD_KERNEL_AUTO (the TMA-tiled kernels), FDTD_KERNEL_REF or FDTD_KERNEL_FUSED.
 * A context created with FDTD_KERNEL_AUTO runs the much slower one-thread-per-point FDTD_KERNEL_REF kernels when the
 * tiled ones do not apply (FDTD_PERIODIC, FDTD_PRECISION_FP64, or subdomain mode with a total Nx that is not a multiple
 * of 4: the halo copies move whole float4s); this call is how a caller finds out.  A monolithic grid of any Nx runs the
 * tiled kernels. */
int fdtd_kernel_in_use(const fdtd_ctx* ctx);

/* time_block >= 2: plane-steps computed (ghost planes included) and plane-steps owned since fdtd_create, into
 * out_host[0], out_host[1]; their ratio is the redundant compute of the temporal blocking (P:315 reports the same trade
 * across GPUs).  Zeros for a context without time blocking. */
int fdtd_time_block_stats(const fdtd_ctx* ctx, int64_t out_host[2]);

/* Number of kernel launches (the library's own kernels) enqueued since the context was created. */
int64_t fdtd_launch_count(const fdtd_ctx* ctx);

/* Total grid extents. */
int fdtd_dims(const fdtd_ctx* ctx, int32_t out[3]);

/* max |f| over a contiguous DEVICE array of n fp32 values, written to *out_dev (DEVICE), for callers that cannot allocate:
 * code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  Needs no context and no workspace,
 * and calls no cudaMalloc / cudaFree or allocating library routine: the reduction's scratch (one partial maximum per thread
 * block and a ticket counter) lives in a static device array of FDTD_NOALLOC_SCRATCH_BYTES that every GPU loading the library
 * holds until exit.  One block reduces 65,536 values, so n is limited to FDTD_NOALLOC_MAX_ELEMS (2^30 values = 4 GiB; a
 * 1024^3 field); a larger n returns FDTD_EINVAL with the limit in fdtd_last_error() and launches nothing.  Same value as
 * fdtd_field_absmax over the same data (NaNs are ignored by both); n = 0 gives 0.  Runs on the CURRENT device, asynchronous
 * on `stream` (a cudaStream_t; the result is in *out_dev once the stream has reached it).  All calls on one device share
 * the scratch array, which keeps the last call's contents: the ticket is cleared by every call, the partials are rewritten
 * before they are read.  Calls that overlap on the GPU (different streams, or graphs replayed concurrently) race on it:
 * serialise them. */
#define FDTD_NOALLOC_MAX_ELEMS (1ull << 30)
#define FDTD_NOALLOC_SCRATCH_BYTES 65792
int fdtd_absmax_noalloc(const float* in_dev, uint64_t n, float* out_dev, void* stream);

/* Releases the context (not the workspace).  Synchronises the stream first. */
int fdtd_destroy(fdtd_ctx* ctx);

/* Text of the last error on the calling thread ("" if none). */
const char* fdtd_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* FDTD_B200_H */
