// C ABI of libsph_b200.so (include/sph.h): host-side logic only -- parameter validation, derived
// constants, device memory, the order of kernel launches for the NL -> PI -> SU loop of the paper
// (Fig. 7), and the two host<->device crossings.
#include <math.h>
#include <stdio.h>
#include <string.h>

#include <new>
#include <string>
#include <vector>

#include "sph_internal.cuh"

#define SPH_EXPORT extern "C" __attribute__((visibility("default")))

enum Phase { PH_KEY = 0, PH_SORT, PH_CELLSTART, PH_REORDER, PH_PI, PH_DT, PH_UPDATE, PH_MDBC, PH_SHIFT, PH_COUNT };

struct EventPair {
  int phase;
  cudaEvent_t a, b;
};

struct sph_ctx {
  sph_params prm;
  DevConsts C;
  cudaStream_t stream;
  std::string err;
  std::vector<void*> allocs;

  int64_t n = 0, cap = 0;
  bool loaded = false, nl_valid = false;
  bool has_build = false, has_pass = false;   // since the last load: a neighbour-list build / an interaction pass
  ParticleSet set[2];
  int cur = 0;
  float4* acc = nullptr;
  uint32_t* nbcount = nullptr;
  uint32_t *key[2] = {nullptr, nullptr}, *idx[2] = {nullptr, nullptr};
  int sorted_buf = 0;
  uint32_t *block_hist = nullptr, *digit_total = nullptr, *cellstart = nullptr, *tile_ws = nullptr;
  uint32_t nkeys = 0;
  int key_bits = 0;
  DevScalars* sc = nullptr;
  double* pos0 = nullptr;
  void* stage = nullptr;        // raw inputs of sph_load_particles (kept across loads)
  size_t stage_bytes = 0;
  double* normals = nullptr;    // mDBC: vector to the boundary interface, original particle order (sph_set_boundary_normals)
  double* conc = nullptr;       // shifting: concentration C_a of the last pass, sorted order
  float4* shiftv = nullptr;     // shifting velocity of the last pass, sorted order
  bool has_shift = false;
  bool has_moving = false;
  std::vector<Motion> motions;
  Motion* d_motions = nullptr;
  int pi_kernel = 1;
  int n_sm = 0;               // multiprocessors of the device this context was created on
  int integrator = 0, verlet_steps = 40;
  int64_t kstep = 0;          // Verlet step counter since the last load (Eq. 31 every verlet_steps)

  bool profiling = false;
  std::vector<EventPair> events;
  std::vector<cudaEvent_t> pool;
  double ms[PH_COUNT] = {0};
  int64_t n_nl = 0, n_pi = 0, n_launch = 0;
};

namespace {

int fail(sph_ctx* c, int code, const char* fmt, const char* detail = "") {
  if (c) {
    char buf[512];
    snprintf(buf, sizeof(buf), fmt, detail);
    c->err = buf;
  }
  return code;
}

// sph_create has no context to hang a message on: the reason of its last failure on this thread is kept here and
// returned by sph_last_error(NULL).
thread_local std::string g_create_err;
int create_fail(int code, const std::string& why) {
  g_create_err = why;
  return code;
}

int cuda_fail(sph_ctx* c, cudaError_t e, const char* where) {
  if (c) c->err = std::string(where) + ": " + cudaGetErrorString(e);
  return e == cudaErrorMemoryAllocation ? SPH_E_NOMEM : SPH_E_CUDA;
}

#define CK(call)                                                   \
  do {                                                             \
    cudaError_t e__ = (call);                                      \
    if (e__ != cudaSuccess) return cuda_fail(ctx, e__, #call);     \
  } while (0)

void* dalloc(sph_ctx* c, size_t bytes) {
  if (bytes == 0) bytes = 16;
  void* p = nullptr;
  if (c->prm.dev_alloc) {
    p = c->prm.dev_alloc(bytes, c->prm.user);
  } else if (cudaMalloc(&p, bytes) != cudaSuccess) {
    cudaGetLastError();
    p = nullptr;
  }
  if (p) c->allocs.push_back(p);
  return p;
}

void dfree(sph_ctx* c, void* p) {
  if (!p) return;
  for (size_t i = 0; i < c->allocs.size(); i++)
    if (c->allocs[i] == p) {
      c->allocs.erase(c->allocs.begin() + i);
      break;
    }
  if (c->prm.dev_free) c->prm.dev_free(p, c->prm.user);
  else cudaFree(p);
}

void free_all(sph_ctx* c) {
  while (!c->allocs.empty()) dfree(c, c->allocs.back());
}

// ---- profiling: one event pair per phase instance, folded into ms[] at synchronisation points ----
cudaEvent_t get_event(sph_ctx* c) {
  if (!c->pool.empty()) {
    cudaEvent_t e = c->pool.back();
    c->pool.pop_back();
    return e;
  }
  cudaEvent_t e;
  cudaEventCreate(&e);
  return e;
}

void fold_events(sph_ctx* c) {
  if (c->events.empty()) return;
  cudaStreamSynchronize(c->stream);
  for (auto& ev : c->events) {
    float t = 0.f;
    if (cudaEventElapsedTime(&t, ev.a, ev.b) == cudaSuccess) c->ms[ev.phase] += t;
    c->pool.push_back(ev.a);
    c->pool.push_back(ev.b);
  }
  c->events.clear();
}

struct PhaseTimer {
  sph_ctx* c;
  EventPair ev;
  bool on;
  PhaseTimer(sph_ctx* ctx, int phase) : c(ctx), on(ctx->profiling) {
    if (!on) return;
    ev.phase = phase;
    ev.a = get_event(c);
    ev.b = get_event(c);
    cudaEventRecord(ev.a, c->stream);
  }
  ~PhaseTimer() {
    if (!on) return;
    cudaEventRecord(ev.b, c->stream);
    c->events.push_back(ev);
    if (c->events.size() >= 8192) fold_events(c);
  }
};

int validate(const sph_params* p, std::string& why) {
  auto bad = [&](const char* s) { why = s; return SPH_E_BADARG; };
  if (p->dim != 2 && p->dim != 3) return bad("dim must be 2 or 3");
  if (!(p->dp > 0) || !(p->h > 0)) return bad("dp and h must be positive");
  if (!(p->rho0 > 0) || !(p->c0 > 0) || !(p->gamma > 0)) return bad("rho0, c0, gamma must be positive");
  if (!(p->cfl > 0)) return bad("cfl must be positive");
  if (p->alpha < 0 || p->delta < 0 || p->eta2_coef < 0) return bad("alpha, delta, eta2_coef must be >= 0");
  if (p->cell_div < 1 || p->cell_div > 3) return bad("cell_div must be 1, 2 or 3");
  if (p->pi_kernel < 0 || p->pi_kernel > 3) return bad("pi_kernel must be 0, 1, 2 or 3");
  if (p->integrator < 0 || p->integrator > 1) return bad("integrator must be 0 (symplectic) or 1 (Verlet)");
  if (p->verlet_steps < 0) return bad("verlet_steps must be >= 0");
  if (p->visco_model < 0 || p->visco_model > 1) return bad("visco_model must be 0 (artificial) or 1 (laminar)");
  if (p->nu0 < 0) return bad("nu0 must be >= 0");
  if (p->ddt_model < 0 || p->ddt_model > 1) return bad("ddt_model must be 0 (Molteni) or 1 (Fourtakas)");
  if (p->boundary_model < 0 || p->boundary_model > 1) return bad("boundary_model must be 0 (DBC) or 1 (mDBC)");
  if (p->mdbc_slip < 0 || p->mdbc_slip > 1) return bad("mdbc_slip must be 0 (wall velocity) or 1 (no-slip)");
  if (p->mdbc_det_min < 0) return bad("mdbc_det_min must be >= 0");
  if (p->shift_model < 0 || p->shift_model > 1) return bad("shift_model must be 0 (none) or 1 (Fickian shifting)");
  if (p->shift_coef < 0 || p->shift_fs_conc < 0) return bad("shift_coef and shift_fs_conc must be >= 0");
  if (p->compensated_sums < 0 || p->compensated_sums > 1) return bad("compensated_sums must be 0 or 1");
  const double cs_min = 2.0 * p->h / p->cell_div;
  if (p->cell_size != 0.0 && p->cell_size < cs_min * (1.0 - 1e-12)) return bad("cell_size smaller than 2h/cell_div");
  for (int k = 0; k < 3; k++) {
    if (p->dim == 2 && k == 1) continue;
    if (!(p->domain_max[k] > p->domain_min[k])) return bad("domain_max must exceed domain_min");
  }
  if ((p->dev_alloc == nullptr) != (p->dev_free == nullptr)) return bad("dev_alloc and dev_free must be given together");
  return SPH_OK;
}

// Derived constants: m = rho0 dp^d (A9), B = c0^2 rho0/gamma (Eq. 28),
// alpha_D (Eq. 11), eta^2 = eta2_coef h^2 (A6), grid n_k = ceil((max-min)/cs) (C3).
int derive(const sph_params* p, DevConsts& C, std::string& why) {
  const double pi = 3.14159265358979323846;
  memset(&C, 0, sizeof(C));
  C.dim = p->dim;
  C.k = p->cell_div;
  const double cs = p->cell_size > 0.0 ? p->cell_size : 2.0 * p->h / (double)p->cell_div;
  C.cs = cs;
  double ncells = 1.0;
  for (int k = 0; k < 3; k++) {
    C.per[k] = p->periodic[k] ? 1 : 0;
    C.dmin[k] = p->domain_min[k];
    if (p->dim == 2 && k == 1) { C.nc[k] = 1; C.per[k] = 0; continue; }
    double ext = (p->domain_max[k] - p->domain_min[k]) / cs;
    double nk = ceil(ext - 1e-9);
    if (nk < 1) nk = 1;
    if (nk > 2.0e9) { why = "grid too large"; return SPH_E_OVERFLOW; }
    C.nc[k] = (int)nk;
    ncells *= nk;
    if (C.per[k] && fabs(ext - rint(ext)) > 1e-9 * ext) {
      why = "periodic length must be an integer multiple of the cell size (pass cell_size = L / floor(L / (2h/cell_div)))";
      return SPH_E_BADARG;
    }
    if (C.per[k] && C.nc[k] < 2 * C.k + 1) { why = "periodic axis needs at least 2*cell_div+1 cells"; return SPH_E_BADARG; }
  }
  if (2.0 * ncells + 2.0 >= 4294967295.0 || ncells >= 2147483647.0) { why = "2*ncells+2 does not fit 32-bit keys"; return SPH_E_OVERFLOW; }
  C.ncells = (uint32_t)ncells;
  const double s = 2.0 * p->h / cs;
  C.R2u = (float)(s * s);
  C.qscale = (float)(cs / (2.0 * p->h));
  const double eta2 = p->eta2_coef * p->h * p->h;
  C.eta2u = (float)(eta2 / (cs * cs));
  C.rho0 = (float)p->rho0;
  C.inv_rho0 = (float)(1.0 / p->rho0);
  C.Beos = (float)(p->c0 * p->c0 * p->rho0 / p->gamma);
  C.gamma = (float)p->gamma;
  C.gamma_is7 = p->gamma == 7.0;
  for (int k = 0; k < 3; k++) C.g[k] = (float)p->g[k];
  const double m = p->rho0 * pow(p->dp, p->dim);
  const double aD = p->dim == 2 ? 7.0 / (4.0 * pi * p->h * p->h) : 21.0 / (16.0 * pi * p->h * p->h * p->h);
  const double Cf = -5.0 * aD / (p->h * p->h);     // grad_a W_ab = Cf (1 - q/2)^3 r_ab
  C.c_cont = (float)(m * cs * Cf);
  C.c_ddt = (float)(2.0 * p->delta * p->h * p->c0 * m * Cf);
  C.c_mom = (float)(-m * Cf * cs);
  C.c_pi = (float)(-2.0 * p->alpha * p->c0 * (p->h / cs));
  C.c_mu = (float)(p->h / cs);
  C.ddt_over_boundary = p->ddt_over_boundary;
  C.rho_bound_floor = p->rho_bound_floor;
  C.comp_sums = p->compensated_sums;
  C.ddt_model = p->ddt_model;
  {
    // Fourtakas DDT (Eq. 19-20, A23): rho^H_ab = rho0 [(1 + e)^(1/gamma) - 1], e = rho0 g.r_ab / B, |r_ab| < 2h
    const double B = p->c0 * p->c0 * p->rho0 / p->gamma, a = 1.0 / p->gamma;
    double gn = 0.0;
    for (int k = 0; k < 3; k++) { C.c_hyd[k] = (float)(p->rho0 * cs * p->g[k] / B); gn += p->g[k] * p->g[k]; }
    C.hyd_series_ok = p->rho0 * sqrt(gn) * 2.0 * p->h / B <= 0.02;
    C.hyd_k[0] = (float)(p->rho0 * a);
    C.hyd_k[1] = (float)(p->rho0 * a * (a - 1.0) / 2.0);
    C.hyd_k[2] = (float)(p->rho0 * a * (a - 1.0) * (a - 2.0) / 6.0);
    C.hyd_k[3] = (float)(p->rho0 * a * (a - 1.0) * (a - 2.0) * (a - 3.0) / 24.0);
    C.inv_gamma = (float)a;
  }
  C.visco_model = p->visco_model;
  C.c_lam = (float)(4.0 * m * p->nu0 * Cf);
  if (p->visco_model == 1) C.c_pi = 0.f;          // Eq. 23 replaces the artificial term of Eq. 22
  C.h = p->h;
  C.c0 = p->c0;
  C.cfl = p->cfl;
  C.inv_cs = (float)(1.0 / cs);
  C.boundary_model = p->boundary_model;
  C.mdbc_slip = p->mdbc_slip;
  C.mdbc_det_min = p->mdbc_det_min > 0.0 ? p->mdbc_det_min : 1e-3;
  C.shift_model = p->shift_model;
  C.mass = m;
  C.aD = aD;
  C.c_w = (float)(m * aD);
  C.c_gw = (float)(m * Cf * cs);
  C.shift_ds = (float)((p->shift_coef > 0.0 ? p->shift_coef : 2.0) * p->h);
  C.shift_fs_conc = p->shift_fs_conc;
  C.shift_alpha_n = (float)p->shift_alpha_n;
  C.shift_beta_n = (float)p->shift_beta_n;
  return SPH_OK;
}

int alloc_set(sph_ctx* c, ParticleSet& P, int64_t n) {
  P.posu = (float4*)dalloc(c, sizeof(float4) * n);
  P.velp = (float4*)dalloc(c, sizeof(float4) * n);
  P.cell = (int*)dalloc(c, sizeof(int) * n);
  P.id = (uint32_t*)dalloc(c, sizeof(uint32_t) * n);
  P.type = (uint8_t*)dalloc(c, n);
  P.posu_n = (float4*)dalloc(c, sizeof(float4) * n);
  P.vel_n = (float4*)dalloc(c, sizeof(float4) * n);
  P.cell_n = (int*)dalloc(c, sizeof(int) * n);
  return (P.posu && P.velp && P.cell && P.id && P.type && P.posu_n && P.vel_n && P.cell_n) ? 0 : -1;
}

// sph_load_particles copies the caller's arrays into a device staging buffer (41 B per particle).  Up to this size the
// buffer stays allocated so that a reload (a checkpoint restore, the end-to-end bench) does not allocate again; a
// larger one (config 4: 1.4 GB) is released as soon as the load is done, so it does not lower the largest N that fits.
constexpr size_t STAGE_KEEP_MAX_BYTES = (size_t)512 << 20;

// NL task: a1 key -> a2 sort -> a3 cell ranges -> a4 reorder (+a7 EOS)
int build_nl(sph_ctx* ctx, bool with_n_state) {
  const int64_t n = ctx->n;
  cudaStream_t s = ctx->stream;
  {
    PhaseTimer t(ctx, PH_KEY);
    nl_compute_keys(ctx->C, ctx->set[ctx->cur], n, ctx->key[0], ctx->idx[0], s);
    ctx->n_launch += 1;
  }
  {
    PhaseTimer t(ctx, PH_SORT);
    int nl = 0;
    ctx->sorted_buf = nl_radix_sort(ctx->key[0], ctx->idx[0], ctx->key[1], ctx->idx[1], n, ctx->key_bits,
                                    ctx->block_hist, ctx->digit_total, &nl, s);
    ctx->n_launch += nl;
  }
  {
    PhaseTimer t(ctx, PH_CELLSTART);
    nl_cellstart(ctx->key[ctx->sorted_buf], n, ctx->nkeys, ctx->cellstart, s);
    ctx->n_launch += 1;
  }
  {
    PhaseTimer t(ctx, PH_REORDER);
    nl_reorder(ctx->C, ctx->set[ctx->cur], ctx->set[1 - ctx->cur], ctx->idx[ctx->sorted_buf], n, with_n_state, s);
    ctx->cur = 1 - ctx->cur;
    ctx->n_launch += 1;
  }
  ctx->n_nl += 1;
  ctx->nl_valid = true;
  ctx->has_build = true;
  CK(cudaGetLastError());
  return SPH_OK;
}

// PI task: a5/a6 (+ dt candidates for a8)
int run_pi(sph_ctx* ctx) {
  cudaStream_t s = ctx->stream;
  PhaseTimer t(ctx, PH_PI);
  pi_reset_scalars(ctx->sc, s);
  PiArgs A;
  const ParticleSet& P = ctx->set[ctx->cur];
  A.posu = P.posu;
  A.velp = P.velp;
  A.cell = P.cell;
  A.cellstart = ctx->cellstart;
  A.acc = ctx->acc;
  A.nbcount = ctx->prm.count_neighbours ? ctx->nbcount : nullptr;
  A.sc = ctx->sc;
  A.n = ctx->n;
  A.tile_ws = ctx->tile_ws;
  A.n_sm = ctx->n_sm;
  bool done = false;
  if (ctx->pi_kernel == 3) {
    done = pi_quad(ctx->C, A, s) == 0;
    if (!done) ctx->pi_kernel = 2;                 // configuration not supported by the quad kernel
  }
  if (!done && ctx->pi_kernel == 2) done = pi_tiled(ctx->C, A, s) == 0;
  if (!done) {
    pi_gather(ctx->C, A, s);
    if (ctx->pi_kernel == 2) ctx->pi_kernel = 1;   // configuration not supported by the tiled kernel
  }
  ctx->n_launch += ctx->pi_kernel == 3 ? 4 : 2;   // reset + PI kernel (+ the quad kernel's active-tile list and |F|max pass)
  ctx->n_pi += 1;
  ctx->has_pass = true;
  CK(cudaGetLastError());
  return SPH_OK;
}

// NEXT-3: ghost-node pass on the freshly sorted state, before the interaction pass.  tfrac: the state's time is
// t + tfrac * dt (1/2 for the second pass of a symplectic step).
int run_mdbc(sph_ctx* ctx, double tfrac) {
  if (ctx->C.boundary_model != 1) return SPH_OK;
  PhaseTimer t(ctx, PH_MDBC);
  const int nm = ctx->has_moving ? (int)ctx->motions.size() : 0;
  bx_mdbc(ctx->C, ctx->set[ctx->cur], ctx->cellstart, ctx->n, ctx->normals, ctx->d_motions, nm, ctx->sc, tfrac,
          ctx->stream);
  ctx->n_launch += 1;
  CK(cudaGetLastError());
  return SPH_OK;
}

// NEXT-4: concentration + shifting velocity of the state the interaction pass just saw.
int run_shift(sph_ctx* ctx) {
  if (ctx->C.shift_model != 1) return SPH_OK;
  PhaseTimer t(ctx, PH_SHIFT);
  bx_shift(ctx->C, ctx->set[ctx->cur], ctx->cellstart, ctx->n, ctx->conc, ctx->shiftv, ctx->stream);
  ctx->n_launch += 2;
  ctx->has_shift = true;
  CK(cudaGetLastError());
  return SPH_OK;
}

int check_flags(sph_ctx* ctx, const DevScalars& h) {
  if (h.flags & 1u) return fail(ctx, SPH_E_NAN, "non-finite acceleration or density rate detected on the device");
  if (h.flags & 2u) return fail(ctx, SPH_E_OVERFLOW, "device-side overflow");
  return SPH_OK;
}

}  // namespace

SPH_EXPORT const char* sph_version(void) { return "sph_b200 0.1 (sm_100a)"; }

SPH_EXPORT const char* sph_last_error(const sph_ctx* ctx) { return ctx ? ctx->err.c_str() : g_create_err.c_str(); }

SPH_EXPORT int sph_create(const sph_params* params, sph_ctx** out) {
  if (!params || !out) return create_fail(SPH_E_BADARG, "null params or out pointer");
  *out = nullptr;
  g_create_err.clear();
  std::string why;
  int rc = validate(params, why);
  if (rc != SPH_OK) return create_fail(rc, why);
  sph_ctx* ctx = new (std::nothrow) sph_ctx();
  if (!ctx) return create_fail(SPH_E_NOMEM, "out of host memory");
  ctx->prm = *params;
  rc = derive(params, ctx->C, why);
  if (rc != SPH_OK) { delete ctx; return create_fail(rc, why); }
  int ndev = 0;
  cudaError_t e = cudaGetDeviceCount(&ndev);
  if (e != cudaSuccess || ndev == 0) {       // no CPU fallback: fail loudly
    cudaGetLastError();
    delete ctx;
    return create_fail(SPH_E_CUDA, "no usable CUDA device (there is no CPU fallback)");
  }
  {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&ctx->n_sm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || ctx->n_sm <= 0) {
      cudaGetLastError();
      delete ctx;
      return create_fail(SPH_E_CUDA, "cannot query the CUDA device");
    }
  }
  ctx->stream = (cudaStream_t)params->cuda_stream;
  ctx->nkeys = 2u * ctx->C.ncells + 1u;      // keys 0 .. 2*ncells (C3)
  ctx->key_bits = 0;
  for (uint32_t v = 2u * ctx->C.ncells; v; v >>= 1) ctx->key_bits++;
  if (ctx->key_bits == 0) ctx->key_bits = 1;
  ctx->integrator = params->integrator;
  ctx->verlet_steps = params->verlet_steps > 0 ? params->verlet_steps : 40;
  ctx->pi_kernel = params->pi_kernel == 0 ? 3 : params->pi_kernel;   // auto: quad -> tiled -> gather, falling back per call
  ctx->cellstart = (uint32_t*)dalloc(ctx, sizeof(uint32_t) * ((size_t)ctx->nkeys + 1));
  ctx->sc = (DevScalars*)dalloc(ctx, sizeof(DevScalars));
  ctx->digit_total = (uint32_t*)dalloc(ctx, sizeof(uint32_t) * 256 * 4);
  ctx->tile_ws = (uint32_t*)dalloc(ctx, sizeof(uint32_t) * pi_quad_workspace_words(ctx->C));
  if (!ctx->cellstart || !ctx->sc || !ctx->digit_total || !ctx->tile_ws) {
    free_all(ctx);
    delete ctx;
    return create_fail(SPH_E_NOMEM, "device allocation failed (cell table)");
  }
  if (cudaMemsetAsync(ctx->sc, 0, sizeof(DevScalars), ctx->stream) != cudaSuccess) {
    free_all(ctx);
    delete ctx;
    return create_fail(SPH_E_CUDA, "cudaMemsetAsync failed");
  }
  *out = ctx;
  return SPH_OK;
}

SPH_EXPORT void sph_destroy(sph_ctx* ctx) {
  if (!ctx) return;
  cudaStreamSynchronize(ctx->stream);
  for (auto& ev : ctx->events) { cudaEventDestroy(ev.a); cudaEventDestroy(ev.b); }
  for (auto e : ctx->pool) cudaEventDestroy(e);
  free_all(ctx);
  delete ctx;
}

SPH_EXPORT int sph_load_particles(sph_ctx* ctx, int64_t n, const double* pos, const float* vel, const float* rho,
                                  const uint8_t* type) {
  if (!ctx) return SPH_E_BADARG;
  if (n < 0 || n > 0x7fffffff - 8192) return fail(ctx, SPH_E_BADARG, "n out of range");
  if (n > 0 && (!pos || !vel || !rho || !type)) return fail(ctx, SPH_E_BADARG, "null input array");
  cudaStream_t s = ctx->stream;
  // a failed (re)load leaves the context unloaded, never half-valid
  ctx->loaded = false;
  ctx->has_build = ctx->has_pass = ctx->has_shift = false;
  ctx->nl_valid = false;
  if (ctx->normals) {                         // normals belong to one particle set
    cudaStreamSynchronize(s);
    dfree(ctx, ctx->normals);
    ctx->normals = nullptr;
  }
  if (n > ctx->cap || !ctx->acc) {            // (re)allocate particle storage
    cudaStreamSynchronize(s);
    ctx->n = 0;
    ctx->acc = nullptr;
    ctx->nbcount = nullptr;
    ctx->block_hist = nullptr;
    for (int i = 0; i < 2; i++) { ctx->key[i] = ctx->idx[i] = nullptr; ctx->set[i] = ParticleSet(); }
    void* keep[] = {ctx->cellstart, ctx->sc, ctx->digit_total, ctx->tile_ws, ctx->d_motions, ctx->stage};
    std::vector<void*> old = ctx->allocs;
    for (void* p : old) {
      bool k = false;
      for (void* q : keep) k = k || (p == q);
      if (!k) dfree(ctx, p);
    }
    ctx->cap = 0;
    const int64_t cap = n;
    bool ok = alloc_set(ctx, ctx->set[0], cap) == 0 && alloc_set(ctx, ctx->set[1], cap) == 0;
    ctx->acc = (float4*)dalloc(ctx, sizeof(float4) * cap);
    ctx->nbcount = (uint32_t*)dalloc(ctx, sizeof(uint32_t) * cap);
    for (int i = 0; i < 2; i++) {
      ctx->key[i] = (uint32_t*)dalloc(ctx, sizeof(uint32_t) * cap);
      ctx->idx[i] = (uint32_t*)dalloc(ctx, sizeof(uint32_t) * cap);
    }
    ctx->block_hist = (uint32_t*)dalloc(ctx, sizeof(uint32_t) * nl_radix_hist_entries(cap));
    ctx->pos0 = nullptr;
    ctx->conc = nullptr;
    ctx->shiftv = nullptr;
    if (ctx->C.shift_model == 1) {
      ctx->conc = (double*)dalloc(ctx, sizeof(double) * cap);
      ctx->shiftv = (float4*)dalloc(ctx, sizeof(float4) * cap);
      ok = ok && ctx->conc && ctx->shiftv;
      if (ok) cudaMemsetAsync(ctx->shiftv, 0, sizeof(float4) * cap, s);
    }
    ok = ok && ctx->acc && ctx->nbcount && ctx->key[0] && ctx->key[1] && ctx->idx[0] && ctx->idx[1] && ctx->block_hist;
    if (!ok) return fail(ctx, SPH_E_NOMEM, "device allocation failed for %s particles", std::to_string(n).c_str());
    ctx->cap = cap;
  }
  // any moving-boundary group (type >= 2)?  Eight type bytes per test (sph_set_motion may follow the load, so
  // the start positions of such particles are kept whether or not a motion law is known yet)
  ctx->has_moving = false;
  {
    int64_t i = 0;
    for (; i + 8 <= n && !ctx->has_moving; i += 8) {
      uint64_t w;
      memcpy(&w, type + i, 8);
      ctx->has_moving = (w & 0xfefefefefefefefeull) != 0;
    }
    for (; i < n && !ctx->has_moving; i++) ctx->has_moving = type[i] >= 2;
  }
  if (ctx->has_moving && !ctx->pos0) {
    ctx->pos0 = (double*)dalloc(ctx, sizeof(double) * 3 * ctx->cap);
    if (!ctx->pos0) return fail(ctx, SPH_E_NOMEM, "device allocation failed (pos0)");
  }
  // staging buffer for the raw inputs, kept for the next load: [pos | vel | rho | type], each 256-byte aligned
  auto up = [](size_t b) { return (b + 255) & ~(size_t)255; };
  const size_t o_vel = up(sizeof(double) * 3 * n), o_rho = o_vel + up(sizeof(float) * 3 * n),
               o_type = o_rho + up(sizeof(float) * n), stage_need = o_type + up((size_t)n);
  if (stage_need > ctx->stage_bytes) {
    if (ctx->stage) { cudaStreamSynchronize(s); dfree(ctx, ctx->stage); }
    ctx->stage_bytes = 0;
    ctx->stage = dalloc(ctx, stage_need);
    if (!ctx->stage) return fail(ctx, SPH_E_NOMEM, "device allocation failed (staging)");
    ctx->stage_bytes = stage_need;
  }
  double* d_pos = (double*)ctx->stage;
  float* d_vel = (float*)((char*)ctx->stage + o_vel);
  float* d_rho = (float*)((char*)ctx->stage + o_rho);
  uint8_t* d_type = (uint8_t*)ctx->stage + o_type;
  CK(cudaMemsetAsync(ctx->sc, 0, sizeof(DevScalars), s));
  if (n > 0) {
    CK(cudaMemcpyAsync(d_pos, pos, sizeof(double) * 3 * n, cudaMemcpyHostToDevice, s));
    CK(cudaMemcpyAsync(d_vel, vel, sizeof(float) * 3 * n, cudaMemcpyHostToDevice, s));
    CK(cudaMemcpyAsync(d_rho, rho, sizeof(float) * n, cudaMemcpyHostToDevice, s));
    CK(cudaMemcpyAsync(d_type, type, n, cudaMemcpyHostToDevice, s));
  }
  ctx->cur = 0;
  su_canonicalize(ctx->C, d_pos, d_vel, d_rho, d_type, n, ctx->set[0], ctx->has_moving ? ctx->pos0 : nullptr,
                  ctx->sc, s);
  ctx->n_launch += 1;
  CK(cudaGetLastError());
  CK(cudaStreamSynchronize(s));      // the caller's buffers are free again on return
  if (ctx->stage_bytes > STAGE_KEEP_MAX_BYTES) {   // a large staging copy is not worth holding for a reload that may never come
    dfree(ctx, ctx->stage);
    ctx->stage = nullptr;
    ctx->stage_bytes = 0;
  }
  ctx->n = n;
  ctx->loaded = true;
  ctx->kstep = 0;
  ctx->nl_valid = false;
  return SPH_OK;
}

SPH_EXPORT int sph_set_motion(sph_ctx* ctx, int32_t group, int32_t axis, double stroke, double period, double phase) {
  if (!ctx) return SPH_E_BADARG;
  if (group < 2 || group > 255) return fail(ctx, SPH_E_BADARG, "motion group must be in 2..255");
  if (axis < 0 || axis > 2 || !(period > 0)) return fail(ctx, SPH_E_BADARG, "bad axis or period");
  Motion m = {group, axis, stroke, period, phase};
  bool found = false;
  for (auto& q : ctx->motions)
    if (q.group == group && q.axis == axis) { q = m; found = true; }
  if (!found) ctx->motions.push_back(m);
  if (ctx->d_motions) { cudaStreamSynchronize(ctx->stream); dfree(ctx, ctx->d_motions); }
  ctx->d_motions = (Motion*)dalloc(ctx, sizeof(Motion) * ctx->motions.size());
  if (!ctx->d_motions) return fail(ctx, SPH_E_NOMEM, "device allocation failed (motions)");
  CK(cudaMemcpyAsync(ctx->d_motions, ctx->motions.data(), sizeof(Motion) * ctx->motions.size(),
                     cudaMemcpyHostToDevice, ctx->stream));
  CK(cudaStreamSynchronize(ctx->stream));
  return SPH_OK;
}

SPH_EXPORT int sph_set_boundary_normals(sph_ctx* ctx, const double* normals) {
  if (!ctx) return SPH_E_BADARG;
  if (!ctx->loaded) return fail(ctx, SPH_E_STATE, "sph_set_boundary_normals before sph_load_particles");
  if (!normals && ctx->n > 0) return fail(ctx, SPH_E_BADARG, "null normals array");
  cudaStream_t s = ctx->stream;
  if (!ctx->normals) {
    ctx->normals = (double*)dalloc(ctx, sizeof(double) * 3 * (size_t)ctx->n);
    if (!ctx->normals) return fail(ctx, SPH_E_NOMEM, "device allocation failed (normals)");
  }
  if (ctx->n > 0) CK(cudaMemcpyAsync(ctx->normals, normals, sizeof(double) * 3 * (size_t)ctx->n, cudaMemcpyHostToDevice, s));
  CK(cudaStreamSynchronize(s));
  return SPH_OK;
}

SPH_EXPORT int sph_compute_interactions(sph_ctx* ctx) {
  if (!ctx) return SPH_E_BADARG;
  if (!ctx->loaded) return fail(ctx, SPH_E_STATE, "sph_compute_interactions before sph_load_particles");
  int rc = build_nl(ctx, ctx->integrator == 1);   // Verlet: the state n-1 travels with every reorder
  if (rc != SPH_OK) return rc;
  if ((rc = run_mdbc(ctx, 0.0)) != SPH_OK) return rc;
  rc = run_pi(ctx);
  if (rc != SPH_OK) return rc;
  if ((rc = run_shift(ctx)) != SPH_OK) return rc;
  {
    PhaseTimer t(ctx, PH_DT);
    su_compute_dt(ctx->C, ctx->sc, ctx->stream);
    ctx->n_launch += 1;
  }
  return SPH_OK;
}

SPH_EXPORT int sph_step(sph_ctx* ctx, int32_t nsteps) {
  if (!ctx) return SPH_E_BADARG;
  if (!ctx->loaded) return fail(ctx, SPH_E_STATE, "sph_step before sph_load_particles");
  if (nsteps < 0) return fail(ctx, SPH_E_BADARG, "nsteps < 0");
  cudaStream_t s = ctx->stream;
  const int nm = ctx->has_moving ? (int)ctx->motions.size() : 0;
  for (int it = 0; it < nsteps && ctx->integrator == 1; it++) {   // Verlet, Eq. 30-31: one pass per step
    int rc;
    if ((rc = build_nl(ctx, true)) != SPH_OK) return rc;         // NL at state n; carries (v, rho)^{n-1}
    if ((rc = run_mdbc(ctx, 0.0)) != SPH_OK) return rc;          // mDBC: boundary rho, v from the ghost nodes
    if ((rc = run_pi(ctx)) != SPH_OK) return rc;                 // F^n, R^n
    if ((rc = run_shift(ctx)) != SPH_OK) return rc;              // shifting velocity of state n
    {
      PhaseTimer t(ctx, PH_DT);
      su_compute_dt(ctx->C, ctx->sc, s);                         // dt^n (Eq. 35)
      ctx->n_launch += 1;
    }
    {
      PhaseTimer t(ctx, PH_UPDATE);
      su_verlet(ctx->C, ctx->set[ctx->cur], ctx->acc, ctx->n, ctx->sc, ctx->d_motions, nm, ctx->pos0,
                ctx->kstep % ctx->verlet_steps == 0, ctx->C.shift_model == 1 ? ctx->shiftv : nullptr, s);
      ctx->n_launch += 2;
    }
    ctx->kstep++;
    ctx->nl_valid = false;
    CK(cudaGetLastError());
  }
  for (int it = 0; it < nsteps && ctx->integrator == 0; it++) {
    int rc;
    if ((rc = build_nl(ctx, false)) != SPH_OK) return rc;        // NL at state n
    if ((rc = run_mdbc(ctx, 0.0)) != SPH_OK) return rc;          // mDBC: boundary rho, v from the ghost nodes
    if ((rc = run_pi(ctx)) != SPH_OK) return rc;                 // F^n, R^n
    {
      PhaseTimer t(ctx, PH_DT);
      su_compute_dt(ctx->C, ctx->sc, s);                         // dt^n (Eq. 35, A8)
      ctx->n_launch += 1;
    }
    {
      PhaseTimer t(ctx, PH_UPDATE);
      su_predictor(ctx->C, ctx->set[ctx->cur], ctx->acc, ctx->n, ctx->sc, ctx->d_motions, nm, ctx->pos0, s);
      ctx->n_launch += 1;
    }
    if ((rc = build_nl(ctx, true)) != SPH_OK) return rc;         // NL at state n+1/2
    if ((rc = run_mdbc(ctx, 0.5)) != SPH_OK) return rc;
    if ((rc = run_pi(ctx)) != SPH_OK) return rc;                 // F^{n+1/2}, R^{n+1/2}
    if ((rc = run_shift(ctx)) != SPH_OK) return rc;              // shifting velocity of state n+1/2
    {
      PhaseTimer t(ctx, PH_UPDATE);
      su_corrector(ctx->C, ctx->set[ctx->cur], ctx->acc, ctx->n, ctx->sc, ctx->d_motions, nm, ctx->pos0,
                   ctx->C.shift_model == 1 ? ctx->shiftv : nullptr, s);
      ctx->n_launch += 2;
    }
    ctx->nl_valid = false;   // positions moved after the last build
    CK(cudaGetLastError());
  }
  return SPH_OK;
}

// bytes of one field (0 for an unknown field)
static size_t field_bytes(const sph_ctx* ctx, int32_t field) {
  const size_t n = (size_t)ctx->n;
  switch (field) {
    case SPH_POS: return sizeof(double) * 3 * n;
    case SPH_VEL: case SPH_ACC: case SPH_OFFSET: case SPH_SHIFT: return sizeof(float) * 3 * n;
    case SPH_RHO: case SPH_DRHODT: case SPH_PRESS: case SPH_CONC: return sizeof(float) * n;
    case SPH_KEY: case SPH_PERM: case SPH_NBCOUNT: return sizeof(uint32_t) * n;
    case SPH_CELL: return sizeof(int32_t) * 3 * n;
    case SPH_CELLSTART: return sizeof(uint32_t) * ((size_t)ctx->nkeys + 1);
    default: return (size_t)-1;
  }
}

SPH_EXPORT int sph_read_fields(sph_ctx* ctx, int32_t nfields, const int32_t* fields, void* const* dsts,
                               const size_t* dst_bytes) {
  if (!ctx || nfields < 0 || (nfields > 0 && (!fields || !dsts || !dst_bytes))) return SPH_E_BADARG;
  if (!ctx->loaded) return fail(ctx, SPH_E_STATE, "sph_read_state / sph_read_fields before sph_load_particles");
  const int64_t n = ctx->n;
  cudaStream_t s = ctx->stream;
  const ParticleSet& P = ctx->set[ctx->cur];
  // every argument is checked before anything is launched
  size_t tmp_bytes = 0;
  for (int32_t k = 0; k < nfields; k++) {
    const int32_t field = fields[k];
    if (!dsts[k]) return fail(ctx, SPH_E_BADARG, "null destination");
    const size_t need = field_bytes(ctx, field);
    if (need == (size_t)-1) return fail(ctx, SPH_E_BADARG, "unknown field");
    if (dst_bytes[k] < need) return fail(ctx, SPH_E_OVERFLOW, "destination buffer too small");
    if ((field == SPH_KEY || field == SPH_CELLSTART) && !ctx->has_build)
      return fail(ctx, SPH_E_STATE, "field needs a neighbour-list build since the last load");
    if ((field == SPH_ACC || field == SPH_DRHODT || field == SPH_NBCOUNT) && !ctx->has_pass)
      return fail(ctx, SPH_E_STATE, "field needs an interaction pass since the last load");
    if ((field == SPH_CONC || field == SPH_SHIFT) && !ctx->has_shift)
      return fail(ctx, SPH_E_STATE, "field needs shift_model = 1 and an interaction pass since the last load");
    if (field == SPH_NBCOUNT && !ctx->prm.count_neighbours)
      return fail(ctx, SPH_E_STATE, "SPH_NBCOUNT needs params.count_neighbours = 1");
    if (field != SPH_KEY && field != SPH_PERM && field != SPH_CELLSTART) tmp_bytes += (need + 255) & ~(size_t)255;
  }
  // all gathers back to the caller's particle order first, then the copies, then one synchronisation
  char* tmp = nullptr;
  if (tmp_bytes) {
    tmp = (char*)dalloc(ctx, tmp_bytes);
    if (!tmp) return fail(ctx, SPH_E_NOMEM, "device allocation failed (read buffer)");
  }
  std::vector<void*> src((size_t)nfields, nullptr);
  size_t off = 0;
  for (int32_t k = 0; k < nfields; k++) {
    const int32_t field = fields[k];
    const size_t need = field_bytes(ctx, field);
    if (need == 0) continue;
    if (field == SPH_KEY) { src[k] = ctx->key[ctx->sorted_buf]; continue; }
    if (field == SPH_PERM) { src[k] = P.id; continue; }
    if (field == SPH_CELLSTART) { src[k] = ctx->cellstart; continue; }
    void* t = tmp + off;
    off += (need + 255) & ~(size_t)255;
    src[k] = t;
    switch (field) {
      case SPH_POS: su_unsort_pos(ctx->C, P, n, (double*)t, nullptr, nullptr, s); break;
      case SPH_CELL: su_unsort_pos(ctx->C, P, n, nullptr, (int*)t, nullptr, s); break;
      case SPH_OFFSET: su_unsort_pos(ctx->C, P, n, nullptr, nullptr, (float*)t, s); break;
      case SPH_VEL: su_unsort_f4(P.velp, P.id, n, 3, 0, (float*)t, s); break;
      case SPH_PRESS: su_unsort_f4(P.velp, P.id, n, 1, 3, (float*)t, s); break;
      case SPH_RHO: su_unsort_f4(P.posu, P.id, n, 1, 3, (float*)t, s); break;
      case SPH_ACC: su_unsort_f4(ctx->acc, P.id, n, 3, 0, (float*)t, s); break;
      case SPH_DRHODT: su_unsort_f4(ctx->acc, P.id, n, 1, 3, (float*)t, s); break;
      case SPH_NBCOUNT: su_unsort_u32(ctx->nbcount, P.id, n, (uint32_t*)t, s); break;
      case SPH_SHIFT: su_unsort_f4(ctx->shiftv, P.id, n, 3, 0, (float*)t, s); break;
      case SPH_CONC: su_unsort_f64(ctx->conc, P.id, n, (float*)t, s); break;
    }
    ctx->n_launch += 1;
  }
  cudaError_t e = cudaGetLastError();
  for (int32_t k = 0; k < nfields && e == cudaSuccess; k++)
    if (src[k]) e = cudaMemcpyAsync(dsts[k], src[k], field_bytes(ctx, fields[k]), cudaMemcpyDeviceToHost, s);
  const cudaError_t e2 = cudaStreamSynchronize(s);
  if (e == cudaSuccess) e = e2;
  if (tmp) dfree(ctx, tmp);
  if (e != cudaSuccess) return cuda_fail(ctx, e, "sph_read_state / sph_read_fields");
  return SPH_OK;
}

SPH_EXPORT int sph_read_state(sph_ctx* ctx, int32_t field, void* dst, size_t dst_bytes) {
  if (!ctx || !dst) return SPH_E_BADARG;
  return sph_read_fields(ctx, 1, &field, &dst, &dst_bytes);
}

SPH_EXPORT int sph_get_info(sph_ctx* ctx, sph_info* info) {
  if (!ctx || !info) return SPH_E_BADARG;
  DevScalars h;
  CK(cudaMemcpyAsync(&h, ctx->sc, sizeof(h), cudaMemcpyDeviceToHost, ctx->stream));
  uint32_t nb = 0;
  if (ctx->has_build) CK(cudaMemcpyAsync(&nb, ctx->cellstart + ctx->C.ncells, sizeof(nb), cudaMemcpyDeviceToHost, ctx->stream));
  CK(cudaStreamSynchronize(ctx->stream));
  memset(info, 0, sizeof(*info));
  info->n = ctx->n;
  info->n_out = h.n_out;
  info->n_bound = nb;
  for (int k = 0; k < 3; k++) info->ncell[k] = ctx->C.nc[k];
  info->ncells = ctx->C.ncells;
  info->cell_size = ctx->C.cs;
  info->r2u = ctx->C.R2u;
  info->n_interactions = h.n_inter;
  info->n_interactions_total = h.n_inter_total + h.n_inter;
  info->steps_done = (int64_t)h.steps;
  info->t = h.t;
  info->dt = h.dt;
  info->pi_kernel = ctx->pi_kernel;
  info->device_flags = (int32_t)h.flags;
  return check_flags(ctx, h);
}

SPH_EXPORT int sph_set_profiling(sph_ctx* ctx, int32_t on) {
  if (!ctx) return SPH_E_BADARG;
  fold_events(ctx);
  if (on) {
    for (int i = 0; i < PH_COUNT; i++) ctx->ms[i] = 0.0;   // timings restart; the counters keep running
  }
  ctx->profiling = on != 0;
  return SPH_OK;
}

SPH_EXPORT int sph_get_timings(sph_ctx* ctx, sph_timings* out) {
  if (!ctx || !out) return SPH_E_BADARG;
  fold_events(ctx);
  CK(cudaStreamSynchronize(ctx->stream));
  out->ms_key = ctx->ms[PH_KEY];
  out->ms_sort = ctx->ms[PH_SORT];
  out->ms_cellstart = ctx->ms[PH_CELLSTART];
  out->ms_reorder = ctx->ms[PH_REORDER];
  out->ms_interaction = ctx->ms[PH_PI];
  out->ms_dt = ctx->ms[PH_DT];
  out->ms_update = ctx->ms[PH_UPDATE];
  out->n_nl_builds = ctx->n_nl;
  out->n_interaction_passes = ctx->n_pi;
  out->n_kernel_launches = ctx->n_launch;
  out->ms_mdbc = ctx->ms[PH_MDBC];
  out->ms_shift = ctx->ms[PH_SHIFT];
  return SPH_OK;
}
