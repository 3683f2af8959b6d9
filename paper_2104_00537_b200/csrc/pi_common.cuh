// Per-pair arithmetic of the particle interaction (PI) task, shared by the PI kernels of this library.
// Everything is evaluated in "cell units": du = (r_a - r_b)/cs with r_a, r_b taken from the canonical
// (cell, offset) state (C1), so distances use the particle's single-precision position relative to its
// cell.  The scale factors that turn the raw sums into physical rates are applied once
// per particle (DevConsts::c_*).
#pragma once
#include "sph_internal.cuh"

__device__ __forceinline__ float fast_sqrt(float x) {
  float r;
  asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}
__device__ __forceinline__ float fast_rcp(float x) {
  float r;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}

// C2, the canonical pair predicate: r2u = fma(duz,duz, fma(duy,duy, dux*dux)) in fp32 with individually
// rounded operations (the 2-D form has no y term); pair <=> r2u < R2u.  du_k are exact (2^-22 grid).
template <int DIM>
__device__ __forceinline__ float pair_r2u(float dux, float duy, float duz) {
  float r2 = __fmul_rn(dux, dux);
  if (DIM == 3) r2 = __fmaf_rn(duy, duy, r2);
  return __fmaf_rn(duz, duz, r2);
}

// Raw sums accumulated for one particle a.
struct PairAcc {
  float sx, sy, sz;   // sum w^3 [(Pa+Pb)/(rho_a rho_b) + Pi_ab] du          -> momentum, Eq. 22
  float sc;           // sum (1/rho_b) w^3 (dv.du)                            -> continuity, Eq. 15 / 36
  float sd;           // sum_F (1/rho_b) w^3 (rho_a - rho_b)                  -> density diffusion, Eq. 17-18 (A3)
  float visc;         // max |mu_ab| / c_mu
};

// One accepted ordered pair, fluid a.  DDT: include the diffusion term for this b (fluid b, or any b
// when ddt_over_boundary; A4).
template <bool DDT>
__device__ __forceinline__ void pair_fluid(const DevConsts& C, float dux, float duy, float duz, float r2u,
                                           float rho_a, float inv_rho_a, float P_a, float vax, float vay,
                                           float vaz, float4 pb, float4 vb, PairAcc& A) {
  float s = fast_sqrt(r2u);
  float w = fmaf(-s, C.qscale, 1.0f);            // 1 - q/2   (Eq. 11)
  float w3 = w * w * w;                          // grad_a W_ab = Cf w^3 cs du
  float inv_rho_b = fast_rcp(pb.w);
  float dvx = vax - vb.x, dvy = vay - vb.y, dvz = vaz - vb.z;
  float dot = fmaf(dvz, duz, fmaf(dvy, duy, dvx * dux));       // v_ab . r_ab / cs
  float gb = w3 * inv_rho_b;
  A.sc = fmaf(gb, dot, A.sc);
  if (DDT) A.sd = fmaf(gb, rho_a - pb.w, A.sd);
  float rs = rho_a + pb.w;
  float x = fast_rcp((r2u + C.eta2u) * rs);
  float mu = fabsf(dot) * x * rs;                // |mu_ab| / c_mu   (Eq. 21, A12)
  A.visc = fmaxf(A.visc, mu);
  float pi = C.c_pi * fminf(dot, 0.0f) * x;      // Pi_ab, non-zero only for approaching pairs (Eq. 21)
  float coef = w3 * fmaf(P_a + vb.w, inv_rho_a * inv_rho_b, pi);
  A.sx = fmaf(coef, dux, A.sx);
  A.sy = fmaf(coef, duy, A.sy);
  A.sz = fmaf(coef, duz, A.sz);
}

// One accepted ordered pair, boundary a <- fluid b (Eq. 36): continuity only.
__device__ __forceinline__ void pair_bound(const DevConsts& C, float dux, float duy, float duz, float r2u,
                                           float vax, float vay, float vaz, float4 pb, float4 vb, PairAcc& A) {
  float s = fast_sqrt(r2u);
  float w = fmaf(-s, C.qscale, 1.0f);
  float w3 = w * w * w;
  float inv_rho_b = fast_rcp(pb.w);
  float dvx = vax - vb.x, dvy = vay - vb.y, dvz = vaz - vb.z;
  float dot = fmaf(dvz, duz, fmaf(dvy, duy, dvx * dux));
  A.sc = fmaf(w3 * inv_rho_b, dot, A.sc);
}

// Scale the raw sums: returns (ax, ay, az, drho/dt).
__device__ __forceinline__ float4 finish_particle(const DevConsts& C, bool fluid, float rho_a, const PairAcc& A) {
  float4 r;
  if (fluid) {
    r.x = fmaf(C.c_mom, A.sx, C.g[0]);
    r.y = fmaf(C.c_mom, A.sy, C.g[1]);
    r.z = fmaf(C.c_mom, A.sz, C.g[2]);
    r.w = fmaf(rho_a * C.c_cont, A.sc, C.c_ddt * A.sd);
  } else {
    r.x = r.y = r.z = 0.f;
    r.w = rho_a * C.c_cont * A.sc;
  }
  return r;
}

// Block-level reduction of the dt candidates and the interaction count into DevScalars.
__device__ __forceinline__ void reduce_scalars(DevScalars* sc, float f2, float visc, unsigned int nb) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    f2 = fmaxf(f2, __shfl_xor_sync(0xffffffffu, f2, o));
    visc = fmaxf(visc, __shfl_xor_sync(0xffffffffu, visc, o));
    nb += __shfl_xor_sync(0xffffffffu, nb, o);
  }
  if ((threadIdx.x & 31) == 0) {
    if (f2 > 0.f) atomicMax(&sc->fmax2_bits, __float_as_uint(f2));
    if (visc > 0.f) atomicMax(&sc->visc_bits, __float_as_uint(visc));
    if (nb) atomicAdd(&sc->n_inter, (unsigned long long)nb);
  }
}
