/*
 * sph.h -- C ABI of libsph_b200.so: the neighbour-search + particle-interaction + system-update
 * hot path of weakly compressible SPH (arxiv 2104.00537, DualSPHysics v5.0 paper) on one B200.
 *
 * Reference for every call: /root/reference/PAPER.md (cited as PAPER.md:<line>) and the readings
 * A1..A29 / canonical definitions C1..C3 listed in DESIGN.md.
 *
 * General conventions
 *   - Every function returns SPH_OK (0) or a negative SPH_E_* code; nothing throws or exits.
 *     sph_last_error() gives a human-readable message for the last failure on that context.
 *   - "host" pointers are plain CPU memory owned by the caller; the library copies and never
 *     retains them.  All device state is owned by the library and released by sph_destroy().
 *   - Device memory is obtained through params.dev_alloc / dev_free when given (PyTorch's caching
 *     allocator in the Python binding), else cudaMalloc/cudaFree.  All work is enqueued on
 *     params.cuda_stream (a cudaStream_t; NULL = legacy default stream).
 *   - Calls are asynchronous on that stream except sph_load_particles (synchronous H2D from
 *     pageable memory), sph_read_state, sph_get_info and sph_get_timings, which synchronise it.
 *   - Asynchronous device-side faults (a non-finite acceleration or density rate in an interaction
 *     pass, a non-finite state in an update) set device flag bit 0, which the next sph_get_info
 *     reports as SPH_E_NAN.  SPH_E_OVERFLOW is a host-side result only (grid too large for 32-bit
 *     keys at sph_create, destination buffer too small at sph_read_state); flag bit 1 is reserved.
 *   - One context per host thread at a time.  There is no CPU fallback: without a CUDA device
 *     sph_create fails with SPH_E_CUDA.
 */
#ifndef SPH_B200_H
#define SPH_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SPH_OK 0
#define SPH_E_BADARG (-1)   /* invalid parameter or NULL pointer                     */
#define SPH_E_NOMEM (-2)    /* device allocation failed                              */
#define SPH_E_CUDA (-3)     /* CUDA runtime error (message in sph_last_error)        */
#define SPH_E_STATE (-4)    /* call out of order (e.g. step before load)             */
#define SPH_E_OVERFLOW (-5) /* grid too large for 32-bit keys / buffer too small     */
#define SPH_E_NAN (-6)      /* non-finite acceleration or density detected on device */

typedef struct sph_ctx sph_ctx; /* opaque, owned by the library */

typedef void* (*sph_alloc_fn)(size_t bytes, void* user); /* returns a device pointer or NULL */
typedef void (*sph_free_fn)(void* dev_ptr, void* user);

/* Parameters of the problem as the paper states it (dp, h: PAPER.md:60,78; rho0, c0, gamma:
 * 214-218, Eq. 28; alpha: 176-178, Eq. 21; delta: 153, Eq. 17; g: 129; CFL: 285-288, Eq. 35). */
typedef struct sph_params {
  int32_t dim;               /* 2 or 3.  The 2-D plane is (x, z); y is ignored (A19).                */
  double dp;                 /* initial particle spacing; particle mass m = rho0 * dp^dim (A9)       */
  double h;                  /* smoothing length; support radius 2h (Eq. 4, 11)                      */
  double rho0, c0, gamma;    /* Tait EOS, Eq. 28: P = c0^2 rho0/gamma ((rho/rho0)^gamma - 1)         */
  double alpha;              /* artificial viscosity coefficient, Eq. 21                             */
  double delta;              /* density diffusion coefficient, Eq. 17-18 (Molteni-Colagrossi)        */
  double g[3];               /* external acceleration f of Eq. 22                                    */
  double cfl;                /* C_CFL of Eq. 35                                                      */
  double domain_min[3];      /* cell-grid extent; particles outside on a non-periodic axis are       */
  double domain_max[3];      /*   flagged "out", excluded and counted (A16)                          */
  int32_t periodic[3];       /* periodic axes; length must be a multiple of cell size */
  double eta2_coef;          /* eta^2 = eta2_coef * h^2, paper value 0.001 (A6)                      */
  int32_t ddt_over_boundary; /* 0: D_a sums fluid neighbours only (A4); 1: all neighbours            */
  int32_t rho_bound_floor;   /* 1: clamp boundary density at rho0 (A10); default 0                   */
  int32_t cell_div;          /* k in {1,2,3}: cubic cells of size 2h/k, (2k+1)^dim-cell stencil.     */
                             /*   k=1: "cells of size 2h"; k=2: "size h" (635)        */
  double cell_size;          /* 0 -> 2h/k; else >= 2h/k, one value for all axes (C1)                 */
  int32_t pi_kernel;         /* interaction kernel: 0 auto, 1 gather (thread/particle), 2 tiled smem, */
                             /*   3 quad (3-D, cell_div 1: conflict-free smem + packed FP32x2)       */
  int32_t count_neighbours;  /* 1: keep per-particle neighbour counts (SPH_NBCOUNT); costs a store   */
  int32_t integrator;        /* 0: symplectic predictor-corrector, Eq. 33-34 (two passes per step);  */
                             /*   1: Verlet, Eq. 30-31 (one pass per step)         */
  int32_t verlet_steps;      /* N_S of Eq. 31: step k is corrective when k mod N_S == 0 (the first   */
                             /*   step included); 0 -> 40 ("N_S ~ 40 is recommended")  */
  int32_t visco_model;       /* 0: artificial viscosity, Eq. 21-22 (alpha); 1: laminar viscosity, Eq. 23  */
                             /*   (nu0 replaces the artificial term of Eq. 22)      */
  int32_t ddt_model;         /* density diffusion term: 0 Molteni-Colagrossi, Eq. 18; 1 Fourtakas et al.,   */
                             /*   Eq. 19-20 (only the dynamic part of the density difference diffuses, A23) */
  double nu0;                /* kinematic viscosity of Eq. 23                                        */
  int32_t boundary_model;    /* 0: DBC, Eq. 36 (boundary density from the continuity equation);      */
                             /*   1: mDBC, Eq. 38-39: before every interaction pass the */
                             /*   density of each boundary particle is extrapolated from its ghost node    */
                             /*   (corrected SPH gradient over the fluid particles, sph_set_boundary_normals) */
                             /*   and is not integrated in time (A24-A25)                                   */
  int32_t mdbc_slip;         /* mDBC velocity of a boundary particle: 0 its imposed wall velocity (0 if     */
                             /*   fixed); 1 no-slip, v_B = 2 v_wall - v_G with v_G the Shepard sum of Eq. 39 (A26) */
  double mdbc_det_min;       /* the corrected-gradient system is solved when |det| >= this (0 -> 1e-3),     */
                             /*   else the Shepard density is used without gradient (A25)                   */
  int32_t shift_model;       /* 0: none; 1: Fickian particle shifting, Eq. 40-41 with grad C of Eq. 53 and  */
                             /*   the free-surface form Eq. 54 (A27-A29): an     */
                             /*   extra pair of passes after the last interaction pass of a step            */
  double shift_coef;         /* A_s of Eq. 41 ("range [1 - 6], with a value of 2 recommended"); 0 -> 2      */
  double shift_fs_conc;      /* a fluid particle with concentration C_a below this is a free-surface        */
                             /*   particle and follows Eq. 54 (A29); 0 disables the free-surface form       */
  double shift_alpha_n;      /* a_n of Eq. 54 ("0 for violent flows, 0.1 for long slow flows")              */
  double shift_beta_n;       /* beta_n of Eq. 54 (initial concentration gradient)                           */
  int32_t compensated_sums;  /* 1: the momentum sums of Eq. 22 are accumulated with a running compensation  */
                             /*   (Kahan).  Under deep hydrostatic pressure the pair terms add up to ~100    */
                             /*   times the net acceleration and plain fp32 sums leave a few 1e-5 m/s^2; with */
                             /*   this option the full-size config 4 meets rel 1e-4 / floor 1e-6 max|a| for   */
                             /*   every particle, at +15 % time per interaction pass.  Default 0.  The quad   */
                             /*   and gather kernels have it; where the tiled kernel would run (pi_kernel 2,  */
                             /*   2-D, cell_div > 1) the gather kernel runs instead (sph_info.pi_kernel = 1). */
  sph_alloc_fn dev_alloc;    /* may be NULL (cudaMalloc)                                             */
  sph_free_fn dev_free;      /* may be NULL (cudaFree)                                               */
  void* user;                /* passed back to dev_alloc / dev_free                                  */
  void* cuda_stream;         /* cudaStream_t                                                         */
} sph_params;

/* Derived quantities and counters, filled by sph_get_info (synchronises the stream). */
typedef struct sph_info {
  int64_t n;               /* particles loaded                                                       */
  int64_t n_out;           /* particles currently flagged out of the grid (A16)                      */
  int64_t n_bound;         /* boundary particles in the grid (sorted first, C3)                      */
  int32_t ncell[3];        /* cells per axis                                                         */
  int64_t ncells;          /* ncell[0]*ncell[1]*ncell[2]; keys run 0 .. 2*ncells (C3)                */
  double cell_size;        /* cs                                                                     */
  float r2u;               /* (2h/cs)^2 as float: squared support in cell units (C2)                 */
  uint64_t n_interactions; /* ordered neighbour pairs found by the last interaction pass             */
  uint64_t n_interactions_total; /* accumulated over all passes since load                           */
  int64_t steps_done;
  double t, dt;            /* simulated time and last step's dt                                      */
  int32_t pi_kernel;       /* kernel actually used                                                   */
  int32_t device_flags;    /* bit 0: non-finite value seen; bit 1: reserved                          */
} sph_info;

/* Accumulated device time per phase, measured with CUDA events on the context's stream while
 * profiling is on (sph_set_profiling).  Phases follow SURVEY.md 8(a): a1 key, a2 sort,
 * a3 cell-range table, a4 reorder (+a7 EOS), a5/a6 interaction, a8 dt, a9 update. */
typedef struct sph_timings {
  double ms_key, ms_sort, ms_cellstart, ms_reorder, ms_interaction, ms_dt, ms_update;
  int64_t n_nl_builds, n_interaction_passes, n_kernel_launches;
  double ms_mdbc, ms_shift;   /* NEXT-3 ghost-node pass, NEXT-4 concentration + shifting passes */
} sph_timings;

/* What sph_read_state copies out.  Per-particle fields come back in the caller's ORIGINAL particle
 * order; SPH_KEY / SPH_PERM / SPH_CELLSTART describe the sorted order of the last neighbour-list
 * build (C3). */
enum sph_field {
  SPH_POS = 1,        /* double[n*3]  x = domain_min + (cell + u) * cs  (inverse of C1)             */
  SPH_VEL = 2,        /* float[n*3]                                                                 */
  SPH_RHO = 3,        /* float[n]                                                                   */
  SPH_ACC = 4,        /* float[n*3]   dv/dt of the last pass incl. g (Eq. 22); 0 for boundary       */
  SPH_DRHODT = 5,     /* float[n]     d rho/dt of the last pass (Eq. 15 / 36)                       */
  SPH_KEY = 6,        /* uint32[n]    sorted keys                                                   */
  SPH_PERM = 7,       /* uint32[n]    original index of the j-th sorted particle                    */
  SPH_CELLSTART = 8,  /* uint32[2*ncells+2]  cellstart[k] = #{keys < k}                             */
  SPH_NBCOUNT = 9,    /* uint32[n]    neighbours per particle (needs count_neighbours = 1)          */
  SPH_CELL = 10,      /* int32[n*3]   canonical cell coordinates (C1)                               */
  SPH_OFFSET = 11,    /* float[n*3]   canonical in-cell offsets u in [0,1) on the 2^-22 grid (C1)   */
  SPH_PRESS = 12,     /* float[n]     P of the last reorder (Eq. 28)                                */
  SPH_CONC = 13,      /* float[n]     particle concentration C_a of the last pass (Eq. 53; shift_model = 1);    */
                      /*              0 for particles out of the grid (A16)                                     */
  SPH_SHIFT = 14      /* float[n*3]   shifting velocity delta r_a / dt of the last pass (Eq. 40-41, 54); 0 for  */
                      /*              boundary particles and for particles out of the grid                      */
};

/* Create a context.  Validates params, derives constants (m, B, alpha_D, eta^2, cell grid).
 * Fails with SPH_E_BADARG on bad parameters, SPH_E_OVERFLOW if 2*ncells+2 does not fit 32 bits,
 * SPH_E_CUDA if no CUDA device is usable. */
int sph_create(const sph_params* params, sph_ctx** out);

/* Release all device memory of the context.  NULL is allowed. */
void sph_destroy(sph_ctx* ctx);

/* Load n particles from host arrays (copied).  pos: double[n*3]; vel: float[n*3]; rho: float[n];
 * type: uint8[n], 0 fluid, 1 fixed boundary, >= 2 moving-boundary group id (Eq. 37).
 * Positions are converted on the device, in IEEE double, to the canonical state (C1):
 * s = (x-min)/cs, c = floor(s), u = rint((s-c) 2^22) 2^-22 ("relative position of the
 * particle within its cell (using single precision)").  Resets t, step count and counters.
 * This is the one host->device crossing of the run.
 * Memory: the raw inputs pass through a device staging buffer of 41 bytes per particle.  When that is at most
 * 512 MiB (about 13 M particles) the buffer stays allocated for the next load on this context; a larger one is
 * released before the call returns. */
int sph_load_particles(sph_ctx* ctx, int64_t n, const double* pos, const float* vel,
                       const float* rho, const uint8_t* type);

/* Imposed motion of boundary group `group` (>= 2) along `axis` (Eq. 37):
 * x(t) = x(0) + (stroke/2) (sin(2 pi t/period + phase) - sin(phase)), v = dx/dt. */
int sph_set_motion(sph_ctx* ctx, int32_t group, int32_t axis, double stroke, double period,
                   double phase);

/* mDBC input (boundary_model = 1): for every particle, the vector n (metres, double[n*3], original particle
 * order; read for boundary particles only) from the particle to the boundary interface.  The ghost node of a
 * boundary particle is r_G = r_B + 2 n ("a ghost node is projected into the fluid across a boundary interface",
 * PAPER.md:308; the paper does not say how the interface is described, A24).  The vectors move with the particle
 * (imposed motions are translations).  Call after sph_load_particles; without it every n = 0 (ghost node on the
 * particle).  Copied; synchronises the stream. */
int sph_set_boundary_normals(sph_ctx* ctx, const double* normals);

/* One neighbour-list build (cell key, radix sort, cell-range table, reorder) plus one
 * particle-interaction pass (Eq. 15, 17-18 or 19-20, 21-22 or 23, 28, 36) on the current state.
 * With boundary_model = 1 the ghost-node pass (Eq. 38-39) runs between the two; with shift_model = 1 the
 * concentration and shifting passes (Eq. 53, 40-41, 54) follow.
 * Results: SPH_ACC, SPH_DRHODT, SPH_NBCOUNT (+ SPH_CONC, SPH_SHIFT) and the dt candidates of Eq. 35. */
int sph_compute_interactions(sph_ctx* ctx);

/* nsteps time steps with the variable dt of Eq. 35 taken from the pass at state n (A8), all on the device,
 * no host synchronisation.
 *   integrator 0: symplectic predictor-corrector (Eq. 33-34); each step = 2 x (neighbour-list
 *                 build + interaction pass) + dt reduction + predictor + corrector.
 *   integrator 1: Verlet (Eq. 30-31; A21); each step = neighbour-list build + interaction
 *                 pass + dt reduction + update; step k since the last sph_load_particles uses Eq. 31 when
 *                 k mod verlet_steps == 0, else Eq. 30.
 * shift_model = 1: r^{n+1} += dt * (shifting velocity of the state the step's last pass saw) (A28). */
int sph_step(sph_ctx* ctx, int32_t nsteps);

/* Copy one field to host memory `dst` of `dst_bytes` bytes (must be at least the field's size, else
 * SPH_E_OVERFLOW).  Synchronises the stream.  The other device->host crossing. */
int sph_read_state(sph_ctx* ctx, int32_t field, void* dst, size_t dst_bytes);

/* Several fields in one call ("what" names a set of fields): fields[k] goes to host memory
 * dsts[k] of dst_bytes[k] bytes.  All arguments are checked before any work is enqueued (same error codes as
 * sph_read_state); the gathers back to the caller's particle order and the device->host copies are enqueued
 * together and the stream is synchronised once.  nfields = 0 is a no-op. */
int sph_read_fields(sph_ctx* ctx, int32_t nfields, const int32_t* fields, void* const* dsts, const size_t* dst_bytes);

/* Fill *info (synchronises the stream). */
int sph_get_info(sph_ctx* ctx, sph_info* info);

/* Per-phase CUDA-event timing.  on = 1 starts (and clears) accumulation; on = 0 stops it.
 * While on, every phase is bracketed by events on the context's stream. */
int sph_set_profiling(sph_ctx* ctx, int32_t on);
int sph_get_timings(sph_ctx* ctx, sph_timings* out);

/* The neighbour-list sort ("the particles ... are sorted according to the cell to which they belong";
 * order convention C3) on its own, for callers that are not allowed to allocate device memory.
 *
 * Who that is: a host code that took all of the GPU's memory into its own pool at start-up, so that a cudaMalloc made
 * behind its back fails or eats into what it thinks it has (a coupled solver with a fixed memory budget, a plug-in that
 * gets no allocator callback to put into sph_params.dev_alloc); and a caller inside a time loop that must not stall,
 * because cudaMalloc and cudaFree make every stream of the device wait.  The context calls above take their sort work
 * space from dev_alloc / cudaMalloc in sph_load_particles.  This call does not: it never calls cudaMalloc, cudaFree or
 * any routine that allocates.  Its work space (ping-pong buffers, digit histograms) is a fixed array compiled into the
 * library, about 8.3 MiB, which each GPU that loads the library keeps until the process ends.  The price is a size
 * limit: n <= SPH_SORT_STATIC_MAX_N.
 *
 *   key         device, uint32[n]: one key per particle, e.g. the C3 cell key; only read.
 *   n           number of keys; 0 is a no-op; n > SPH_SORT_STATIC_MAX_N returns SPH_E_OVERFLOW and does nothing.
 *   key_bits    the keys are ordered by their low key_bits bits (1..32; 8 bits per pass), so any higher bit should be 0.
 *   key_sorted  device, uint32[n], written: the keys in ascending order.
 *   perm        device, uint32[n], written: perm[j] = position in `key` of the j-th sorted key.  Equal keys keep their
 *               input order (stable), so the result is unique and equals SPH_KEY / SPH_PERM of the context path.
 *   cuda_stream cudaStream_t (NULL = legacy default stream) of the CURRENT device; the three arrays live on that device,
 *               are owned by the caller and must not overlap.  The work is only enqueued; the call does not wait for it.
 *   errmsg      NULL, or host memory of errmsg_bytes bytes that receives a message when the result is not SPH_OK.
 *
 * Returns SPH_OK, SPH_E_BADARG (negative n, key_bits out of range, NULL or aliased arrays), SPH_E_OVERFLOW (n above
 * the limit) or SPH_E_CUDA.
 *
 * First call on a device: the library looks up where its work space lives on that device (cudaGetSymbolAddress) and
 * remembers it; the device must be current on the calling thread.  Make this first call during set-up, before any
 * stream capture is begun.
 * Sharing: all calls on one device use the same work space, and it keeps whatever the previous call left (the call
 * clears the part that has to start at zero itself).  Two calls whose GPU work can overlap in time -- different streams
 * without an ordering between them, or two host threads -- race on it and give wrong results; put them on one stream or
 * order them with events. */
#define SPH_SORT_STATIC_MAX_N 1048576
int sph_sort_keys_static(const uint32_t* key, int64_t n, int32_t key_bits, uint32_t* key_sorted, uint32_t* perm,
                         void* cuda_stream, char* errmsg, size_t errmsg_bytes);

/* Message of the last error on this context ("" if none).  Valid until the next call.
 * With ctx = NULL: the reason of the last failed sph_create on the calling thread. */
const char* sph_last_error(const sph_ctx* ctx);

/* Library version string, e.g. "sph_b200 0.1 (sm_100a)". */
const char* sph_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SPH_B200_H */
