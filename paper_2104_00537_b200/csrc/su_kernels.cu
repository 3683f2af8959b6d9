// System update (SU) task: variable time step (Eq. 35) and the symplectic position-Verlet
// predictor-corrector (Eq. 33-34), plus the canonical position conversions (C1)
// used at load / read time.  "the duration of the simulation step is calculated, together with the
// new values of the properties of SPH particles".
//
// Positions live as (linear cell index, offset u in [0,1) in cell units on a 2^-22 grid).  The paper
// performs SU in double precision to protect small position increments in large
// domains; the (cell, offset) form gives the same protection in fp32 because the increment is added to
// a number of magnitude < 1 whatever the domain size.
#include "sph_internal.cuh"

namespace {

constexpr float TWO22 = 4194304.0f;
constexpr float INV_TWO22 = 1.0f / 4194304.0f;

__device__ __forceinline__ void decode_cell(const DevConsts& C, int lin, int c[3]) {
  c[0] = lin % C.nc[0];
  int r = lin / C.nc[0];
  c[1] = r % C.nc[1];
  c[2] = r / C.nc[1];
}

// C1 in IEEE double, every operation individually rounded: s = (x - min)/cs; c = floor(s);
// u = rint((s - c) 2^22) 2^-22; u == 1 -> c += 1, u = 0.  Returns linear cell or -1 (out, A16).
__device__ __forceinline__ int canon_double(const DevConsts& C, const double x[3], float u[3]) {
  int c[3];
  bool out = false;
#pragma unroll
  for (int k = 0; k < 3; k++) {
    if (C.dim == 2 && k == 1) { c[k] = 0; u[k] = 0.f; continue; }
    double s = __ddiv_rn(__dsub_rn(x[k], C.dmin[k]), C.cs);
    double fl = floor(s);
    double uu = __dmul_rn(rint(__dmul_rn(__dsub_rn(s, fl), 4194304.0)), 1.0 / 4194304.0);
    if (uu >= 1.0) { fl += 1.0; uu = 0.0; }
    long long ci = (long long)fl;
    if (C.per[k]) {
      ci %= C.nc[k];
      if (ci < 0) ci += C.nc[k];
    } else if (ci < 0 || ci >= C.nc[k] || !(s == s)) {
      out = true; ci = 0; uu = 0.0;
    }
    c[k] = (int)ci;
    u[k] = (float)uu;
  }
  if (out) { u[0] = u[1] = u[2] = 0.f; return -1; }
  return c[0] + C.nc[0] * (c[1] + C.nc[1] * c[2]);
}

// fp32 position advance in cell units with carry into the cell and re-quantisation to the 2^-22 grid.
__device__ __forceinline__ int advance_cell(const DevConsts& C, int lin, float u[3], const float du[3]) {
  int c[3];
  decode_cell(C, lin, c);
  bool out = false;
#pragma unroll
  for (int k = 0; k < 3; k++) {
    if (C.dim == 2 && k == 1) continue;
    float un = u[k] + du[k];
    float fl = floorf(un);
    float r = rintf((un - fl) * TWO22) * INV_TWO22;
    if (r >= 1.0f) { fl += 1.0f; r = 0.0f; }
    int ci = c[k] + (int)fl;
    if (C.per[k]) {
      ci %= C.nc[k];
      if (ci < 0) ci += C.nc[k];
    } else if (ci < 0 || ci >= C.nc[k] || !(un == un)) {
      out = true;
    }
    c[k] = ci;
    u[k] = r;
  }
  if (out) return -1;
  return c[0] + C.nc[0] * (c[1] + C.nc[1] * c[2]);
}

__global__ void k_canonicalize(DevConsts C, const double* __restrict__ pos, const float* __restrict__ vel,
                               const float* __restrict__ rho, const uint8_t* __restrict__ type, int64_t n,
                               ParticleSet P, double* __restrict__ pos0, DevScalars* sc) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  double x[3] = {pos[3 * i], pos[3 * i + 1], pos[3 * i + 2]};
  float u[3];
  int lin = canon_double(C, x, u);
  if (lin < 0) atomicAdd(&sc->n_out, 1u);
  P.posu[i] = make_float4(u[0], u[1], u[2], rho[i]);
  P.velp[i] = make_float4(vel[3 * i], vel[3 * i + 1], vel[3 * i + 2], 0.f);
  P.cell[i] = lin;
  P.id[i] = (uint32_t)i;
  P.type[i] = type[i];
  if (pos0) { pos0[3 * i] = x[0]; pos0[3 * i + 1] = x[1]; pos0[3 * i + 2] = x[2]; }
}

// a8: dt = CFL min( sqrt(h / max_a |F_a|), h / (c0 + max |mu_ab|) )   (Eq. 35, A12, A13)
__global__ void k_compute_dt(DevConsts C, DevScalars* sc) {
  double f2 = (double)__uint_as_float(sc->fmax2_bits);
  double visc = (double)__uint_as_float(sc->visc_bits);
  double fa = sqrt(f2);
  double dtf = fa > 0.0 ? sqrt(C.h / fa) : 1e300;
  double dtcv = C.h / (C.c0 + visc);
  sc->dt = C.cfl * (dtf < dtcv ? dtf : dtcv);
}

// Boundary particle with imposed motion (Eq. 37): position and velocity from the motion law at time t.
__device__ __forceinline__ int moved_boundary(const DevConsts& C, const Motion* motions, int nmotions, int group,
                                              const double* pos0, uint32_t id, double t, float u[3], float v[3]) {
  double x[3] = {pos0[3 * (size_t)id], pos0[3 * (size_t)id + 1], pos0[3 * (size_t)id + 2]};
  v[0] = v[1] = v[2] = 0.f;
  for (int j = 0; j < nmotions; j++)
    if (motions[j].group == group) {
      double d, vv;
      motion_eval(motions[j], t, &d, &vv);
      x[motions[j].axis] += d;
      v[motions[j].axis] = (float)vv;
    }
  return canon_double(C, x, u);
}

// a9, predictor:  r^{n+1/2} = r^n + dt/2 v^n;  v^{n+1/2} = v^n + dt/2 F^n;  rho^{n+1/2} = rho^n + dt/2 R^n
// (Eq. 33-34 first halves).  Saves state n.  Boundary: rho only (A11), + imposed motion.
__global__ void k_predictor(DevConsts C, ParticleSet P, const float4* __restrict__ acc, int64_t n, DevScalars* sc,
                            const Motion* __restrict__ motions, int nmotions, const double* __restrict__ pos0) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  int lin = P.cell[i];
  if (lin < 0) return;
  const double dtd = sc->dt;
  const float hdt = 0.5f * (float)dtd;
  float4 p = P.posu[i];
  float4 v = P.velp[i];
  float4 a = acc[i];
  uint8_t ty = P.type[i];
  P.posu_n[i] = p;
  P.vel_n[i] = v;
  P.cell_n[i] = lin;
  if (!(isfinite(a.x) && isfinite(a.y) && isfinite(a.z) && isfinite(a.w))) atomicOr(&sc->flags, 1u);
  float u[3] = {p.x, p.y, p.z};
  if (ty == 0) {
    float s = hdt * C.inv_cs;
    float du[3] = {s * v.x, s * v.y, s * v.z};
    lin = advance_cell(C, lin, u, du);
    v.x = fmaf(hdt, a.x, v.x);
    v.y = fmaf(hdt, a.y, v.y);
    v.z = fmaf(hdt, a.z, v.z);
  } else if (ty >= 2 && nmotions > 0) {
    float vv[3];
    lin = moved_boundary(C, motions, nmotions, ty, pos0, P.id[i], sc->t + 0.5 * dtd, u, vv);
    v.x = vv[0]; v.y = vv[1]; v.z = vv[2];
  }
  float rho = fmaf(hdt, a.w, p.w);
  if (ty != 0 && C.rho_bound_floor) rho = fmaxf(rho, C.rho0);
  if (ty != 0 && C.boundary_model == 1) rho = p.w;   // mDBC: set by the ghost-node pass, not integrated (A24)
  if (lin < 0) atomicAdd(&sc->n_out, 1u);
  P.posu[i] = make_float4(u[0], u[1], u[2], rho);
  P.velp[i] = v;
  P.cell[i] = lin;
}

// NEXT-1, Verlet scheme, Eq. 30-31, one interaction pass per step:
//   regular:    v^{n+1} = v^{n-1} + 2 dt F^n;  rho^{n+1} = rho^{n-1} + 2 dt R^n     (Eq. 30)
//   corrective: v^{n+1} = v^n + dt F^n;        rho^{n+1} = rho^n + dt R^n           (Eq. 31, every N_S steps)
//   both:       r^{n+1} = r^n + dt v^n + dt^2/2 F^n
// P.vel_n holds (v^{n-1}, rho^{n-1}) on entry and (v^n, rho^n) on exit.  Boundary: rho only, + imposed motion.
__global__ void k_verlet(DevConsts C, ParticleSet P, const float4* __restrict__ acc, int64_t n, DevScalars* sc,
                         const Motion* __restrict__ motions, int nmotions, const double* __restrict__ pos0,
                         int corrective, const float4* __restrict__ shiftv) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  int lin = P.cell[i];
  if (lin < 0) return;
  const double dtd = sc->dt;
  const float dt = (float)dtd;
  const float4 p = P.posu[i];      // r^n (offsets), rho^n
  float4 v = P.velp[i];            // v^n
  const float4 m1 = P.vel_n[i];    // v^{n-1}, rho^{n-1}
  const float4 a = acc[i];         // F^n, R^n
  const uint8_t ty = P.type[i];
  if (!(isfinite(a.x) && isfinite(a.y) && isfinite(a.z) && isfinite(a.w))) atomicOr(&sc->flags, 1u);
  P.vel_n[i] = make_float4(v.x, v.y, v.z, p.w);
  float u[3] = {p.x, p.y, p.z};
  if (ty == 0) {
    const float s = dt * C.inv_cs, hs = 0.5f * dt * s;
    float du[3] = {fmaf(hs, a.x, s * v.x), fmaf(hs, a.y, s * v.y), fmaf(hs, a.z, s * v.z)};
    if (shiftv) {   // delta r_a = -D_s grad C_a, Eq. 40-41 (A28)
      const float4 sh = shiftv[i];
      du[0] = fmaf(s, sh.x, du[0]); du[1] = fmaf(s, sh.y, du[1]); du[2] = fmaf(s, sh.z, du[2]);
    }
    lin = advance_cell(C, lin, u, du);
    if (corrective) {
      v.x = fmaf(dt, a.x, v.x);
      v.y = fmaf(dt, a.y, v.y);
      v.z = fmaf(dt, a.z, v.z);
    } else {
      v.x = fmaf(2.0f * dt, a.x, m1.x);
      v.y = fmaf(2.0f * dt, a.y, m1.y);
      v.z = fmaf(2.0f * dt, a.z, m1.z);
    }
  } else if (ty >= 2 && nmotions > 0) {
    float vv[3];
    lin = moved_boundary(C, motions, nmotions, ty, pos0, P.id[i], sc->t + dtd, u, vv);
    v.x = vv[0]; v.y = vv[1]; v.z = vv[2];
  }
  float rho = corrective ? fmaf(dt, a.w, p.w) : fmaf(2.0f * dt, a.w, m1.w);
  if (ty != 0 && C.rho_bound_floor) rho = fmaxf(rho, C.rho0);
  if (ty != 0 && C.boundary_model == 1) rho = p.w;   // mDBC (A24)
  if (lin < 0) atomicAdd(&sc->n_out, 1u);
  P.posu[i] = make_float4(u[0], u[1], u[2], rho);
  P.velp[i] = v;
  P.cell[i] = lin;
}

// a9, corrector:  v^{n+1} = v^n + dt F^{n+1/2};  r^{n+1} = r^n + dt (v^{n+1} + v^n)/2;
// eps = -(R^{n+1/2}/rho^{n+1/2}) dt;  rho^{n+1} = rho^n (2 - eps)/(2 + eps)       (Eq. 33-34)
__global__ void k_corrector(DevConsts C, ParticleSet P, const float4* __restrict__ acc, int64_t n, DevScalars* sc,
                            const Motion* __restrict__ motions, int nmotions, const double* __restrict__ pos0,
                            const float4* __restrict__ shiftv) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  int lin = P.cell[i];
  if (lin < 0) return;
  const double dtd = sc->dt;
  const float dt = (float)dtd;
  float4 ph = P.posu[i];      // state n+1/2
  float4 pn = P.posu_n[i];    // state n
  float4 vn = P.vel_n[i];
  float4 a = acc[i];          // F^{n+1/2}, R^{n+1/2}
  uint8_t ty = P.type[i];
  if (!(isfinite(a.x) && isfinite(a.y) && isfinite(a.z) && isfinite(a.w))) atomicOr(&sc->flags, 1u);
  float u[3] = {ph.x, ph.y, ph.z};
  float4 v = P.velp[i];
  if (ty == 0) {
    v.x = fmaf(dt, a.x, vn.x);
    v.y = fmaf(dt, a.y, vn.y);
    v.z = fmaf(dt, a.z, vn.z);
    float s = 0.5f * dt * C.inv_cs;
    float du[3] = {s * (v.x + vn.x), s * (v.y + vn.y), s * (v.z + vn.z)};
    if (shiftv) {   // delta r_a = -D_s grad C_a, Eq. 40-41 (A28)
      const float4 sh = shiftv[i];
      const float sd = dt * C.inv_cs;
      du[0] = fmaf(sd, sh.x, du[0]); du[1] = fmaf(sd, sh.y, du[1]); du[2] = fmaf(sd, sh.z, du[2]);
    }
    u[0] = pn.x; u[1] = pn.y; u[2] = pn.z;
    lin = advance_cell(C, P.cell_n[i], u, du);
  } else if (ty >= 2 && nmotions > 0) {
    float vv[3];
    lin = moved_boundary(C, motions, nmotions, ty, pos0, P.id[i], sc->t + dtd, u, vv);
    v.x = vv[0]; v.y = vv[1]; v.z = vv[2];
  }
  float eps = -(a.w / ph.w) * dt;
  float rho = pn.w * (2.0f - eps) / (2.0f + eps);
  if (ty != 0 && C.rho_bound_floor) rho = fmaxf(rho, C.rho0);
  if (ty != 0 && C.boundary_model == 1) rho = ph.w;  // mDBC: the value of the last ghost-node pass (A24)
  if (lin < 0) atomicAdd(&sc->n_out, 1u);
  P.posu[i] = make_float4(u[0], u[1], u[2], rho);
  P.velp[i] = v;
  P.cell[i] = lin;
}

__global__ void k_advance_time(DevScalars* sc) {
  sc->t += sc->dt;
  sc->steps += 1;
}

__global__ void k_unsort_pos(DevConsts C, ParticleSet P, int64_t n, double* __restrict__ pos_out,
                             int* __restrict__ cell_out, float* __restrict__ off_out) {
  int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= n) return;
  size_t i = P.id[j];
  int lin = P.cell[j];
  float4 p = P.posu[j];
  float u[3] = {p.x, p.y, p.z};
  int c[3] = {-1, -1, -1};
  if (lin >= 0) decode_cell(C, lin, c);
#pragma unroll
  for (int k = 0; k < 3; k++) {
    if (pos_out) {
      double x;
      if (lin < 0) x = __longlong_as_double(0x7ff8000000000000LL);
      else if (C.dim == 2 && k == 1) x = 0.0;
      else x = __dadd_rn(C.dmin[k], __dmul_rn(__dadd_rn((double)c[k], (double)u[k]), C.cs));  // inverse of C1
      pos_out[3 * i + k] = x;
    }
    if (cell_out) cell_out[3 * i + k] = c[k];
    if (off_out) off_out[3 * i + k] = u[k];
  }
}

__global__ void k_unsort_f4(const float4* __restrict__ src, const uint32_t* __restrict__ id, int64_t n, int ncomp,
                            int comp0, float* __restrict__ out) {
  int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= n) return;
  float4 v = src[j];
  float a[4] = {v.x, v.y, v.z, v.w};
  size_t i = id[j];
  for (int k = 0; k < ncomp; k++) out[(size_t)ncomp * i + k] = a[comp0 + k];
}

__global__ void k_unsort_f64(const double* __restrict__ src, const uint32_t* __restrict__ id, int64_t n,
                             float* __restrict__ out) {
  int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= n) return;
  out[id[j]] = (float)src[j];
}

__global__ void k_unsort_u32(const uint32_t* __restrict__ src, const uint32_t* __restrict__ id, int64_t n,
                             uint32_t* __restrict__ out) {
  int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= n) return;
  out[id[j]] = src[j];
}

}  // namespace

static inline unsigned grid_for(int64_t n, int threads) { return (unsigned)((n + threads - 1) / threads); }

void su_canonicalize(const DevConsts& C, const double* pos, const float* vel, const float* rho,
                     const uint8_t* type, int64_t n, const ParticleSet& P, double* pos0, DevScalars* sc,
                     cudaStream_t s) {
  if (n == 0) return;
  k_canonicalize<<<grid_for(n, 256), 256, 0, s>>>(C, pos, vel, rho, type, n, P, pos0, sc);
}

void su_compute_dt(const DevConsts& C, DevScalars* sc, cudaStream_t s) { k_compute_dt<<<1, 1, 0, s>>>(C, sc); }

void su_predictor(const DevConsts& C, const ParticleSet& P, const float4* acc, int64_t n, DevScalars* sc,
                  const Motion* motions, int nmotions, const double* pos0, cudaStream_t s) {
  if (n == 0) return;
  k_predictor<<<grid_for(n, 256), 256, 0, s>>>(C, P, acc, n, sc, motions, nmotions, pos0);
}

void su_corrector(const DevConsts& C, const ParticleSet& P, const float4* acc, int64_t n, DevScalars* sc,
                  const Motion* motions, int nmotions, const double* pos0, const float4* shiftv, cudaStream_t s) {
  if (n > 0) k_corrector<<<grid_for(n, 256), 256, 0, s>>>(C, P, acc, n, sc, motions, nmotions, pos0, shiftv);
  k_advance_time<<<1, 1, 0, s>>>(sc);
}

void su_verlet(const DevConsts& C, const ParticleSet& P, const float4* acc, int64_t n, DevScalars* sc,
               const Motion* motions, int nmotions, const double* pos0, int corrective, const float4* shiftv,
               cudaStream_t s) {
  if (n > 0) k_verlet<<<grid_for(n, 256), 256, 0, s>>>(C, P, acc, n, sc, motions, nmotions, pos0, corrective, shiftv);
  k_advance_time<<<1, 1, 0, s>>>(sc);
}

void su_unsort_pos(const DevConsts& C, const ParticleSet& P, int64_t n, double* pos_out, int* cell_out,
                   float* off_out, cudaStream_t s) {
  if (n == 0) return;
  k_unsort_pos<<<grid_for(n, 256), 256, 0, s>>>(C, P, n, pos_out, cell_out, off_out);
}

void su_unsort_f4(const float4* src, const uint32_t* id, int64_t n, int ncomp, int comp0, float* out,
                  cudaStream_t s) {
  if (n == 0) return;
  k_unsort_f4<<<grid_for(n, 256), 256, 0, s>>>(src, id, n, ncomp, comp0, out);
}

void su_unsort_u32(const uint32_t* src, const uint32_t* id, int64_t n, uint32_t* out, cudaStream_t s) {
  if (n == 0) return;
  k_unsort_u32<<<grid_for(n, 256), 256, 0, s>>>(src, id, n, out);
}

void su_unsort_f64(const double* src, const uint32_t* id, int64_t n, float* out, cudaStream_t s) {
  if (n == 0) return;
  k_unsort_f64<<<grid_for(n, 256), 256, 0, s>>>(src, id, n, out);
}
