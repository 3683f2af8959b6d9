// Internal declarations shared by the translation units of libsph_b200.so.
// Not part of the ABI (include/sph.h is).  sm_100a only.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/sph.h"

// Constants of one problem, derived on the host in double (sph_api.cu) and passed by value.
struct DevConsts {
  int dim, k;              // k = cell_div; stencil radius in cells
  int nc[3];               // cells per axis
  int per[3];              // periodic flags
  uint32_t ncells;         // nc[0]*nc[1]*nc[2]
  float R2u;               // (2h/cs)^2, canonical predicate threshold (C2)
  float qscale;            // cs/(2h): q/2 = sqrt(r2u) * qscale
  float eta2u;             // eta^2 / cs^2
  float rho0, inv_rho0, Beos, gamma;
  int gamma_is7;
  float g[3];
  // accumulated raw sums are scaled once per particle:
  float c_cont;            // m * cs * Cf            : R_cont = rho_a * c_cont * sum (1/rho_b) w^3 (dv.du)
  float c_ddt;             // 2 delta h c0 m Cf      : D_a    = c_ddt * sum_F (1/rho_b) w^3 (rho_a - rho_b)
  float c_mom;             // -m * Cf * cs           : F_a    = c_mom * sum w^3 [(Pa+Pb)/(rho_a rho_b) + Pi] du
  float c_pi;              // -alpha c0 * 2 * (h/cs) : Pi_ab  = c_pi * min(dv.du,0) / ((r2u+eta2u)(rho_a+rho_b))
  float c_mu;              // h/cs                   : mu_ab  = c_mu * (dv.du) / (r2u + eta2u)
  int ddt_over_boundary, rho_bound_floor;
  int comp_sums;           // sph_params.compensated_sums: Kahan accumulation of the momentum sums of Eq. 22
  int visco_model;         // 0 artificial (Eq. 21-22), 1 laminar (Eq. 23)
  int ddt_model;           // 0 Molteni (Eq. 18), 1 Fourtakas (Eq. 19-20)
  int hyd_series_ok;       // |e| <= 0.02 for every pair: the binomial series below is exact to fp32 rounding
  float c_hyd[3];          // e = P^H_ab / B = sum_k c_hyd[k] du_k,  c_hyd[k] = rho0 cs g_k / B   (Eq. 20)
  float hyd_k[4];          // rho^H_ab = e (k0 + e (k1 + e (k2 + e k3))) = rho0 [(1 + e)^(1/gamma) - 1]
  float inv_gamma;
  float c_lam;             // 4 m nu0 Cf             : F_lam = c_lam * sum w^3 r2u / ((r2u+eta2u)(rho_a+rho_b)) dv
  double cs, dmin[3];
  double h, c0, cfl;
  float inv_cs;            // 1/cs (update kernel: du = dt * v / cs)
  // NEXT-3 mDBC (Eq. 38-39) and NEXT-4 shifting (Eq. 40-41, 53-54)
  int boundary_model, mdbc_slip, shift_model;
  double mdbc_det_min;
  double mass, aD;         // m = rho0 dp^d (A9), alpha_D of Eq. 11
  float c_w;               // m alpha_D          : V_b W_ab = c_w (1/rho_b) w^4 (2q + 1)
  float c_gw;              // m Cf cs            : V_b grad_a W_ab = c_gw (1/rho_b) w^3 du
  float shift_ds;          // A_s h              : D_s / dt = shift_ds |v_a|   (Eq. 41)
  float shift_alpha_n, shift_beta_n;
  double shift_fs_conc;    // free-surface switch of Eq. 54: compared with the double C_a, as the oracle does
};

// Tait EOS, Eq. 28, evaluated without the cancellation of (rho/rho0)^gamma - 1:
// with e = (rho - rho0)/rho0,  (1+e)^7 - 1 = e (7 + 21 e + 35 e^2 + 35 e^3 + 21 e^4 + 7 e^5 + e^6).
__device__ __forceinline__ float eos_pressure(const DevConsts& C, float rho) {
  float e = (rho - C.rho0) * C.inv_rho0;
  float x;
  if (C.gamma_is7) {
    float p = e + 7.f;
    p = fmaf(p, e, 21.f);
    p = fmaf(p, e, 35.f);
    p = fmaf(p, e, 35.f);
    p = fmaf(p, e, 21.f);
    p = fmaf(p, e, 7.f);
    x = p * e;
  } else {
    x = expm1f(C.gamma * log1pf(e));
  }
  return C.Beos * x;
}

// Device-resident scalars (one small struct in global memory).
struct DevScalars {
  unsigned int fmax2_bits;   // max_a |F_a|^2 over fluid a (float bits; non-negative floats order as uints)
  unsigned int visc_bits;    // max |mu_ab| over evaluated pairs
  unsigned int flags;        // bit0 non-finite, bit1 overflow
  unsigned int n_out;        // particles flagged out
  unsigned long long n_inter;        // neighbour pairs of the last pass
  unsigned long long n_inter_total;  // accumulated
  double dt;                 // current step's dt (Eq. 35)
  double t;                  // simulated time
  unsigned long long steps;
};

struct Motion {
  int group, axis;
  double stroke, period, phase;
};

// Imposed motion of a boundary group (Eq. 37): displacement since t = 0 and velocity along the group's axis.
__device__ __forceinline__ void motion_eval(const Motion& m, double t, double* disp, double* velc) {
  const double w = 6.283185307179586476925286766559 / m.period;
  *disp = 0.5 * m.stroke * (sin(w * t + m.phase) - sin(m.phase));
  *velc = 0.5 * m.stroke * w * cos(w * t + m.phase);
}

// Particle arrays in the current (sorted) order.  Two sets; a reorder gathers set `cur` into `1-cur`.
struct ParticleSet {
  float4* posu;     // (ux, uy, uz, rho): in-cell offsets on the 2^-22 grid + density
  float4* velp;     // (vx, vy, vz, P)
  int* cell;        // linear cell index cx + nx (cy + ny cz); -1 if out of the grid
  uint32_t* id;     // original particle index
  uint8_t* type;
  // state at step n, carried through the half-step reorder (Eq. 33-34 need r^n, v^n, rho^n)
  float4* posu_n;
  float4* vel_n;    // (vx, vy, vz, unused)
  int* cell_n;
};

// ---- neighbour list (nl_kernels.cu) ----
void nl_compute_keys(const DevConsts& C, const ParticleSet& P, int64_t n, uint32_t* key, uint32_t* idx,
                     cudaStream_t s);
// Stable LSD radix sort of (key, idx) pairs over `key_bits` bits; result ends in (key_out, idx_out).
// key/idx are ping-pong buffers a/b; returns which buffer holds the result (0 = a, 1 = b).
int nl_radix_sort(uint32_t* key_a, uint32_t* idx_a, uint32_t* key_b, uint32_t* idx_b, int64_t n, int key_bits,
                  uint32_t* block_hist, uint32_t* digit_total, int* n_launch, cudaStream_t s);
size_t nl_radix_hist_entries(int64_t n);
void nl_cellstart(const uint32_t* sorted_key, int64_t n, uint32_t nkeys, uint32_t* cellstart, cudaStream_t s);
void nl_reorder(const DevConsts& C, const ParticleSet& src, const ParticleSet& dst, const uint32_t* idx,
                int64_t n, bool with_n_state, cudaStream_t s);

// ---- particle interaction (pi_kernels.cu) ----
struct PiArgs {
  const float4* posu;
  const float4* velp;
  const int* cell;
  const uint32_t* cellstart;   // 2*ncells + 2 entries
  float4* acc;                 // (ax, ay, az, drho/dt)
  uint32_t* nbcount;           // may be NULL
  DevScalars* sc;
  int64_t n;
  uint32_t* tile_ws;           // quad kernel work space: [0] number of active tiles, [1] next tile, [4..] tile list
  int n_sm;                    // multiprocessors of the context's device (persistent kernels: one CTA per SM)
};
size_t pi_quad_workspace_words(const DevConsts& C);   // size of tile_ws in 32-bit words
void pi_gather(const DevConsts& C, const PiArgs& A, cudaStream_t s);
int pi_tiled(const DevConsts& C, const PiArgs& A, cudaStream_t s);   // returns 0, or -1 if unsupported config
int pi_quad(const DevConsts& C, const PiArgs& A, cudaStream_t s);    // 3-D, cell_div 1 only; 0 or -1 likewise
void pi_reset_scalars(DevScalars* sc, cudaStream_t s);

// ---- NEXT-3 mDBC and NEXT-4 shifting (bx_kernels.cu) ----
// Ghost-node pass: density (Eq. 38), velocity (Eq. 39) and pressure (Eq. 28) of every boundary particle of the sorted
// set P.  normals: double[n*3] in original order or NULL; wall velocities from the motion laws at sc->t + tfrac * sc->dt.
void bx_mdbc(const DevConsts& C, const ParticleSet& P, const uint32_t* cellstart, int64_t n, const double* normals,
             const Motion* motions, int nmotions, DevScalars* sc, double tfrac, cudaStream_t s);
// Concentration C_a (Eq. 53) of every particle, then the shifting velocity (Eq. 40-41, 54) of every fluid particle.
void bx_shift(const DevConsts& C, const ParticleSet& P, const uint32_t* cellstart, int64_t n, double* conc,
              float4* shiftv, cudaStream_t s);

// ---- system update (su_kernels.cu) ----
void su_canonicalize(const DevConsts& C, const double* pos, const float* vel, const float* rho,
                     const uint8_t* type, int64_t n, const ParticleSet& P, double* pos0, DevScalars* sc,
                     cudaStream_t s);
void su_compute_dt(const DevConsts& C, DevScalars* sc, cudaStream_t s);
void su_predictor(const DevConsts& C, const ParticleSet& P, const float4* acc, int64_t n, DevScalars* sc,
                  const Motion* motions, int nmotions, const double* pos0, cudaStream_t s);
// shiftv: shifting velocity of the last pass (NEXT-4) or NULL
void su_corrector(const DevConsts& C, const ParticleSet& P, const float4* acc, int64_t n, DevScalars* sc,
                  const Motion* motions, int nmotions, const double* pos0, const float4* shiftv, cudaStream_t s);
// Verlet step, Eq. 30-31: corrective != 0 selects Eq. 31.  State n-1 lives in P.vel_n = (v^{n-1}, rho^{n-1}).
void su_verlet(const DevConsts& C, const ParticleSet& P, const float4* acc, int64_t n, DevScalars* sc,
               const Motion* motions, int nmotions, const double* pos0, int corrective, const float4* shiftv,
               cudaStream_t s);
// scatter sorted-order fields back to original order for sph_read_state
void su_unsort_pos(const DevConsts& C, const ParticleSet& P, int64_t n, double* pos_out, int* cell_out,
                   float* off_out, cudaStream_t s);
void su_unsort_f4(const float4* src, const uint32_t* id, int64_t n, int ncomp, int comp0, float* out,
                  cudaStream_t s);
void su_unsort_u32(const uint32_t* src, const uint32_t* id, int64_t n, uint32_t* out, cudaStream_t s);
void su_unsort_f64(const double* src, const uint32_t* id, int64_t n, float* out, cudaStream_t s);
