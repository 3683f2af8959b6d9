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

// Fourtakas DDT, Eq. 19-20 (A23): hydrostatic density difference rho^H_ab = rho0 [(1 + e)^(1/gamma) - 1] with
// e = P^H_ab / B = rho0 g.r_ab / B.  For |e| <= 0.02 the binomial series to e^4 is exact to fp32 rounding
// (and avoids the cancellation of forming 1 + e); otherwise expm1(log1p(e) / gamma).
__device__ __forceinline__ float hydrostatic_drho(const DevConsts& C, float dux, float duy, float duz) {
  const float e = fmaf(C.c_hyd[2], duz, fmaf(C.c_hyd[1], duy, C.c_hyd[0] * dux));
  if (C.hyd_series_ok) return e * fmaf(e, fmaf(e, fmaf(e, C.hyd_k[3], C.hyd_k[2]), C.hyd_k[1]), C.hyd_k[0]);
  return C.rho0 * expm1f(log1pf(e) * C.inv_gamma);
}

// Development builds that split the fp32 error of the momentum sum of Eq. 22 into its parts (never in a release build;
// gather kernel, pi_kernel = 1, only; reading T3, profiles/r3_momentum_error_split.md):
//   SPH_NVCC_EXTRA=-DPI_ACC_F64   the fp32 pair terms are summed in double            -> removes the summation error
//   SPH_NVCC_EXTRA=-DPI_TERM_F64  ... and the pair coefficient itself (r^2, 1 - q/2, (Pa + Pb) / (rho_a rho_b)) is
//                                 evaluated in double from the stored fp32 state      -> removes the per-pair rounding;
//                                 what is left comes from the fp32 state itself (P of the fp32 EOS, the constants)
#if defined(PI_TERM_F64) && !defined(PI_ACC_F64)
#define PI_ACC_F64
#endif

// Raw sums accumulated for one particle a.
struct PairAcc {
  float sx, sy, sz;   // sum w^3 [(Pa+Pb)/(rho_a rho_b) + Pi_ab] du          -> momentum, Eq. 22
  float sc;           // sum (1/rho_b) w^3 (dv.du)                            -> continuity, Eq. 15 / 36
  float sd;           // sum_F (1/rho_b) w^3 (rho_a - rho_b)                  -> density diffusion, Eq. 17-18 (A3)
  float visc;         // max |mu_ab| / c_mu
  float lx, ly, lz;   // sum w^3 r2u / ((r2u + eta2u)(rho_a + rho_b)) dv        -> laminar viscosity, Eq. 23
  float kx, ky, kz;   // running compensation of sx, sy, sz (sph_params.compensated_sums; 0 otherwise)
#ifdef PI_ACC_F64
  double dx = 0.0, dy = 0.0, dz = 0.0;   // the momentum sums of pair_fluid, in double (added to sx, sy, sz at the end)
#endif
};

// s += p with the Kahan compensation c (what the rounded sum has in excess of the exact one); no fast-math, so the
// compiler keeps (t - s) - y as written.
__device__ __forceinline__ void kahan_add(float p, float& s, float& c) {
  const float y = p - c;
  const float t = s + y;
  c = (t - s) - y;
  s = t;
}

// Momentum sums of Eq. 22: A.s += coef * du.  Plain FMA, or compensated when sph_params.compensated_sums = 1 (under deep
// hydrostatic pressure the pair terms are ~100 times the net acceleration; profiles/r3_momentum_error_split.md).
__device__ __forceinline__ void momentum_add(const DevConsts& C, float coef, float dux, float duy, float duz, PairAcc& A) {
  if (C.comp_sums) {                             // uniform branch
    kahan_add(coef * dux, A.sx, A.kx);
    kahan_add(coef * duy, A.sy, A.ky);
    kahan_add(coef * duz, A.sz, A.kz);
  } else {
    A.sx = fmaf(coef, dux, A.sx);
    A.sy = fmaf(coef, duy, A.sy);
    A.sz = fmaf(coef, duz, A.sz);
  }
}

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
  if (DDT) {
    float drho = rho_a - pb.w;
    if (C.ddt_model == 1) drho -= hydrostatic_drho(C, dux, duy, duz);   // Eq. 19-20
    A.sd = fmaf(gb, drho, A.sd);
  }
  float rs = rho_a + pb.w;
  float x = fast_rcp((r2u + C.eta2u) * rs);
  float mu = fabsf(dot) * x * rs;                // |mu_ab| / c_mu   (Eq. 21, A12)
  A.visc = fmaxf(A.visc, mu);
  float pi = C.c_pi * fminf(dot, 0.0f) * x;      // Pi_ab, non-zero only for approaching pairs (Eq. 21)
  float coef = w3 * fmaf(P_a + vb.w, inv_rho_a * inv_rho_b, pi);
#ifdef PI_ACC_F64
  double coefd = (double)coef;
#ifdef PI_TERM_F64
  {
    const double r2d = (double)dux * dux + (double)duy * duy + (double)duz * duz;      // du are exact (C1)
    const double wd = fmax(1.0 - sqrt(r2d) * (C.cs / (2.0 * C.h)), 0.0);
    coefd = wd * wd * wd * (((double)P_a + (double)vb.w) / ((double)rho_a * (double)pb.w) + (double)pi);
  }
#endif
  A.dx += coefd * (double)dux;
  A.dy += coefd * (double)duy;
  A.dz += coefd * (double)duz;
#else
  momentum_add(C, coef, dux, duy, duz, A);
#endif
  if (C.visco_model == 1) {                      // Eq. 23 (c_pi = 0 in this model)
    float lam = w3 * r2u * x;
    A.lx = fmaf(lam, dvx, A.lx);
    A.ly = fmaf(lam, dvy, A.ly);
    A.lz = fmaf(lam, dvz, A.lz);
  }
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
#ifdef PI_ACC_F64
    const double cm = -C.mass * (-5.0 * C.aD / (C.h * C.h)) * C.cs;      // c_mom before its rounding to float
    r.x = (float)(cm * (A.dx + (double)A.sx) + (double)C.g[0]);
    r.y = (float)(cm * (A.dy + (double)A.sy) + (double)C.g[1]);
    r.z = (float)(cm * (A.dz + (double)A.sz) + (double)C.g[2]);
#else
    r.x = fmaf(C.c_mom, A.sx - A.kx, C.g[0]);    // k = 0 without compensated sums
    r.y = fmaf(C.c_mom, A.sy - A.ky, C.g[1]);
    r.z = fmaf(C.c_mom, A.sz - A.kz, C.g[2]);
#endif
    if (C.visco_model == 1) {
      r.x = fmaf(C.c_lam, A.lx, r.x);
      r.y = fmaf(C.c_lam, A.ly, r.y);
      r.z = fmaf(C.c_lam, A.lz, r.z);
    }
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

// One particle a against the particles of its adjacent cells, read straight from global memory
// (sorted arrays + cell-range table).  Used by the baseline kernel and as the overflow path of the tiled one.
template <int DIM>
__device__ __forceinline__ void gather_one(const DevConsts& C, const PiArgs& A, uint32_t a, bool a_fluid, float& f2,
                                        float& visc, unsigned int& nb_out) {
  const float4 pa = A.posu[a];
  const float4 va = A.velp[a];
  const int lin = A.cell[a];
  int ca[3];
  ca[0] = lin % C.nc[0];
  int r = lin / C.nc[0];
  ca[1] = r % C.nc[1];
  ca[2] = r / C.nc[1];
  const float inv_rho_a = fast_rcp(pa.w);
  PairAcc S = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
  unsigned int nb = 0;
  const int K = C.k;
  const int ky = DIM == 3 ? K : 0;
  for (int dz = -K; dz <= K; dz++) {
    int cz = ca[2] + dz;
    if (C.per[2]) cz = (cz + C.nc[2]) % C.nc[2];
    else if (cz < 0 || cz >= C.nc[2]) continue;
    for (int dy = -ky; dy <= ky; dy++) {
      int cy = ca[1] + dy;
      if (C.per[1]) cy = (cy + C.nc[1]) % C.nc[1];
      else if (cy < 0 || cy >= C.nc[1]) continue;
      for (int dx = -K; dx <= K; dx++) {
        int cx = ca[0] + dx;
        if (C.per[0]) cx = (cx + C.nc[0]) % C.nc[0];
        else if (cx < 0 || cx >= C.nc[0]) continue;
        const uint32_t lin2 = (uint32_t)cx + (uint32_t)C.nc[0] * ((uint32_t)cy + (uint32_t)C.nc[1] * (uint32_t)cz);
        // offsets of a relative to the neighbour cell's origin: du = ua - (ub + dc)  (exact, C1)
        const float ox = pa.x - (float)dx, oy = pa.y - (float)dy, oz = pa.z - (float)dz;
        // boundary neighbours (block 0): fluid a only (B<-B pairs are never evaluated, Eq. 36)
        if (a_fluid) {
          const uint32_t b0 = A.cellstart[lin2], b1 = A.cellstart[lin2 + 1];
          for (uint32_t b = b0; b < b1; b++) {
            const float4 pb = A.posu[b];
            const float dux = ox - pb.x, duy = DIM == 3 ? oy - pb.y : 0.f, duz = oz - pb.z;
            const float r2u = pair_r2u<DIM>(dux, duy, duz);
            if (r2u < C.R2u) {
              nb++;
              const float4 vb = A.velp[b];
              if (C.ddt_over_boundary)
                pair_fluid<true>(C, dux, duy, duz, r2u, pa.w, inv_rho_a, va.w, va.x, va.y, va.z, pb, vb, S);
              else
                pair_fluid<false>(C, dux, duy, duz, r2u, pa.w, inv_rho_a, va.w, va.x, va.y, va.z, pb, vb, S);
            }
          }
        }
        // fluid neighbours (block 1)
        {
          const uint32_t b0 = A.cellstart[C.ncells + lin2], b1 = A.cellstart[C.ncells + lin2 + 1];
          for (uint32_t b = b0; b < b1; b++) {
            const float4 pb = A.posu[b];
            const float dux = ox - pb.x, duy = DIM == 3 ? oy - pb.y : 0.f, duz = oz - pb.z;
            const float r2u = pair_r2u<DIM>(dux, duy, duz);
            if (r2u < C.R2u && b != a) {          // self excluded by index (A17)
              nb++;
              const float4 vb = A.velp[b];
              if (a_fluid)
                pair_fluid<true>(C, dux, duy, duz, r2u, pa.w, inv_rho_a, va.w, va.x, va.y, va.z, pb, vb, S);
              else
                pair_bound(C, dux, duy, duz, r2u, va.x, va.y, va.z, pb, vb, S);
            }
          }
        }
      }
    }
  }
  const float4 out = finish_particle(C, a_fluid, pa.w, S);
  if (!isfinite(out.x + out.y + out.z + out.w)) atomicOr(&A.sc->flags, 1u);   // reported as SPH_E_NAN
  A.acc[a] = out;
  if (A.nbcount) A.nbcount[a] = nb;
  if (a_fluid) f2 = fmaxf(f2, fmaf(out.x, out.x, fmaf(out.y, out.y, out.z * out.z)));
  visc = fmaxf(visc, S.visc * C.c_mu);
  nb_out += nb;
}
