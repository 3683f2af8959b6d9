// NEXT-3 and NEXT-4 of SURVEY.md 8(f): passes that reuse the neighbour list of the interaction pass.
//
//   k_mdbc  : modified dynamic boundary conditions, Eq. 38-39.  One thread per boundary particle:
//             ghost node r_G = r_B + 2 n_B (n_B from sph_set_boundary_normals, A24), corrected SPH approximation of
//             Liu & Liu over the FLUID particles within 2h of r_G, rho_B = rho_G + (r_B - r_G) . grad rho_G (Eq. 38),
//             v_G = Shepard sum (Eq. 39).  The ghost node is not a particle, so this pass works in double on the
//             exact (cell, offset) positions; it touches N_B << N particles.
//   k_conc  : particle concentration C_a = sum_b V_b W_ab over all particles, self included (Eq. 53, A27).
//   k_shift : grad C_a = sum_b V_b (C_b - C_a) grad_a W_ab (Eq. 53) and the shifting velocity
//             s_a = -A_s h |v_a| grad C_a (Eq. 40-41), with the free-surface form of Eq. 54 (A29).
// k_conc / k_shift use the canonical pair predicate C2, i.e. exactly the neighbour set of the interaction pass.
#include "pi_common.cuh"

namespace {

__device__ __forceinline__ void decode3(const DevConsts& C, int lin, int c[3]) {
  c[0] = lin % C.nc[0];
  int r = lin / C.nc[0];
  c[1] = r % C.nc[1];
  c[2] = r / C.nc[1];
}

// Gaussian elimination with partial pivoting on an M x M system held in registers (every index is static after
// unrolling).  Returns det A (0 if a pivot vanishes; x is then not set).
template <int M>
__device__ __forceinline__ double solve_small(double (&A)[M][M], double (&b)[M], double (&x)[M]) {
  double det = 1.0;
#pragma unroll
  for (int c = 0; c < M; c++) {
    int piv = c;
    double best = fabs(A[c][c]);
#pragma unroll
    for (int r = c + 1; r < M; r++) {
      const double v = fabs(A[r][c]);
      if (v > best) { best = v; piv = r; }
    }
    if (best == 0.0) return 0.0;
#pragma unroll
    for (int r = c + 1; r < M; r++)
      if (piv == r) {
#pragma unroll
        for (int k = 0; k < M; k++) { const double t = A[c][k]; A[c][k] = A[r][k]; A[r][k] = t; }
        const double t = b[c]; b[c] = b[r]; b[r] = t;
        det = -det;
      }
    det *= A[c][c];
#pragma unroll
    for (int r = c + 1; r < M; r++) {
      const double f = A[r][c] / A[c][c];
#pragma unroll
      for (int k = c; k < M; k++) A[r][k] -= f * A[c][k];
      b[r] -= f * b[c];
    }
  }
#pragma unroll
  for (int r = M - 1; r >= 0; r--) {
    double s = b[r];
#pragma unroll
    for (int k = r + 1; k < M; k++) s -= A[r][k] * x[k];
    x[r] = s / A[r][r];
  }
  return det;
}

template <int DIM>
__global__ void __launch_bounds__(128) k_mdbc(DevConsts C, ParticleSet P, const uint32_t* __restrict__ cellstart,
                                              const double* __restrict__ normals, const Motion* __restrict__ motions,
                                              int nmotions, const DevScalars* __restrict__ sc, double tfrac) {
  const uint32_t n_bound = cellstart[C.ncells];          // boundary block sorted first (C3)
  const uint32_t a = blockIdx.x * blockDim.x + threadIdx.x;
  if (a >= n_bound) return;
  constexpr int M = DIM + 1;
  const int ax[3] = {0, DIM == 3 ? 1 : 2, 2};            // active axes: (x, y, z) or (x, z)
  const float4 pa = P.posu[a];
  const uint8_t ty = P.type[a];
  const size_t id = P.id[a];
  int ca[3];
  decode3(C, P.cell[a], ca);
  double nrm[3] = {0.0, 0.0, 0.0};
  if (normals) { nrm[0] = normals[3 * id]; nrm[1] = DIM == 3 ? normals[3 * id + 1] : 0.0; nrm[2] = normals[3 * id + 2]; }
  // imposed wall velocity at the time of this state (0 for a fixed particle)
  double vw[3] = {0.0, 0.0, 0.0};
  if (ty >= 2 && nmotions > 0) {
    const double t = sc->t + tfrac * sc->dt;
    for (int j = 0; j < nmotions; j++)
      if (motions[j].group == (int)ty) {
        double d, vv;
        motion_eval(motions[j], t, &d, &vv);
        vw[motions[j].axis] = vv;
      }
  }
  // ghost node in cell units: integer cell + offset in [0, 1)
  const double ua[3] = {(double)pa.x, (double)pa.y, (double)pa.z};
  int cg[3];
  double ug[3];
  bool reach = true;
#pragma unroll
  for (int k = 0; k < 3; k++) {
    if (DIM == 2 && k == 1) { cg[k] = 0; ug[k] = 0.0; continue; }
    const double g = (double)ca[k] + ua[k] + 2.0 * nrm[k] / C.cs;
    const double fl = floor(g);
    ug[k] = g - fl;
    long long ci = (long long)fl;
    if (C.per[k]) { ci %= C.nc[k]; if (ci < 0) ci += C.nc[k]; }
    else if (ci < -(long long)C.k || ci >= (long long)C.nc[k] + C.k) reach = false;   // beyond the stencil of every cell
    cg[k] = (int)ci;
  }

  double A[M][M], rhs[M], sv[3] = {0.0, 0.0, 0.0};
#pragma unroll
  for (int i = 0; i < M; i++) {
    rhs[i] = 0.0;
#pragma unroll
    for (int j = 0; j < M; j++) A[i][j] = 0.0;
  }
  unsigned nb = 0;
  const double R2 = 4.0 * C.h * C.h, inv_h = 1.0 / C.h;
  const int K = C.k, ky = DIM == 3 ? K : 0;
  if (reach)
    for (int dz = -K; dz <= K; dz++) {
      int cz = cg[2] + dz;
      if (C.per[2]) cz = ((cz % C.nc[2]) + C.nc[2]) % C.nc[2];
      else if (cz < 0 || cz >= C.nc[2]) continue;
      for (int dy = -ky; dy <= ky; dy++) {
        int cy = cg[1] + dy;
        if (C.per[1]) cy = ((cy % C.nc[1]) + C.nc[1]) % C.nc[1];
        else if (cy < 0 || cy >= C.nc[1]) continue;
        for (int dx = -K; dx <= K; dx++) {
          int cx = cg[0] + dx;
          if (C.per[0]) cx = ((cx % C.nc[0]) + C.nc[0]) % C.nc[0];
          else if (cx < 0 || cx >= C.nc[0]) continue;
          const uint32_t lin2 = (uint32_t)cx + (uint32_t)C.nc[0] * ((uint32_t)cy + (uint32_t)C.nc[1] * (uint32_t)cz);
          const uint32_t b0 = cellstart[C.ncells + lin2], b1 = cellstart[C.ncells + lin2 + 1];   // fluid block
          for (uint32_t b = b0; b < b1; b++) {
            const float4 pb = P.posu[b];
            // d = r_b - r_G in metres (exact differences of the canonical state, then one scaling)
            double d[3];
            d[0] = (((double)pb.x + (double)dx) - ug[0]) * C.cs;
            d[1] = DIM == 3 ? (((double)pb.y + (double)dy) - ug[1]) * C.cs : 0.0;
            d[2] = (((double)pb.z + (double)dz) - ug[2]) * C.cs;
            const double r2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
            if (!(r2 < R2)) continue;
            const float4 vb = P.velp[b];
            const double q = sqrt(r2) * inv_h, w = 1.0 - 0.5 * q, w3 = w * w * w;
            const double Wb = C.aD * w3 * w * (2.0 * q + 1.0);              // Eq. 11
            const double f = -5.0 * C.aD * w3 * inv_h * inv_h;              // grad W = f * (r_G - r_b) w.r.t. r_G
            const double Vb = C.mass / (double)pb.w;
            nb++;
            A[0][0] += Vb * Wb;
            rhs[0] += C.mass * Wb;
#pragma unroll
            for (int j = 0; j < DIM; j++) A[0][1 + j] += Vb * Wb * d[ax[j]];
#pragma unroll
            for (int i = 0; i < DIM; i++) {
              const double gw = -f * d[ax[i]];
              A[1 + i][0] += Vb * gw;
              rhs[1 + i] += C.mass * gw;
#pragma unroll
              for (int j = 0; j < DIM; j++) A[1 + i][1 + j] += Vb * gw * d[ax[j]];
            }
            sv[0] += Vb * (double)vb.x * Wb;
            sv[1] += Vb * (double)vb.y * Wb;
            sv[2] += Vb * (double)vb.z * Wb;
          }
        }
      }
    }

  double rho_b, vout[3] = {vw[0], vw[1], vw[2]};
  if (nb == 0 || !(A[0][0] > 0.0)) {
    rho_b = (double)C.rho0;                                // no fluid in reach of the ghost node (A25)
  } else {
    const double sumVW = A[0][0], shep = rhs[0] / A[0][0];
    double x[M];
    const double det = solve_small<M>(A, rhs, x);
    if (fabs(det) >= C.mdbc_det_min) {
      rho_b = x[0];
#pragma unroll
      for (int j = 0; j < DIM; j++) rho_b += -2.0 * nrm[ax[j]] * x[1 + j];   // Eq. 38: (r_B - r_G) . grad rho_G
    } else {
      rho_b = shep;                                        // Shepard value, no gradient (A25)
    }
    if (C.mdbc_slip == 1) {                                // Eq. 39, no-slip about the wall velocity (A26)
      vout[0] = 2.0 * vw[0] - sv[0] / sumVW;
      if (DIM == 3) vout[1] = 2.0 * vw[1] - sv[1] / sumVW;
      vout[2] = 2.0 * vw[2] - sv[2] / sumVW;
    }
  }
  const float rho_f = (float)rho_b;
  P.posu[a] = make_float4(pa.x, pa.y, pa.z, rho_f);
  P.velp[a] = make_float4((float)vout[0], (float)vout[1], (float)vout[2], eos_pressure(C, rho_f));
}

// Walks the neighbours of particle a (any type, both blocks) by the canonical predicate C2 and calls
// f(b, dux, duy, duz, r2u) for each, b != a.
template <int DIM, class F>
__device__ __forceinline__ void for_each_neighbour(const DevConsts& C, const float4* __restrict__ posu,
                                                   const uint32_t* __restrict__ cellstart, uint32_t a, const float4 pa,
                                                   int lin, F f) {
  int ca[3];
  decode3(C, lin, ca);
  const int K = C.k, ky = DIM == 3 ? K : 0;
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
        const float ox = pa.x - (float)dx, oy = pa.y - (float)dy, oz = pa.z - (float)dz;   // exact (C1)
#pragma unroll
        for (int blk = 0; blk < 2; blk++) {
          const uint32_t key = (uint32_t)blk * C.ncells + lin2;
          const uint32_t b0 = cellstart[key], b1 = cellstart[key + 1];
          for (uint32_t b = b0; b < b1; b++) {
            const float4 pb = posu[b];
            const float dux = ox - pb.x, duy = DIM == 3 ? oy - pb.y : 0.f, duz = oz - pb.z;
            const float r2u = pair_r2u<DIM>(dux, duy, duz);
            if (r2u < C.R2u && b != a) f(b, pb, dux, duy, duz, r2u);
          }
        }
      }
    }
  }
}

// C_a = V_a W(0) + sum_b V_b W_ab   (Eq. 53, A27); W = alpha_D (1 - q/2)^4 (2q + 1) (Eq. 11)
template <int DIM>
__global__ void __launch_bounds__(128) k_conc(DevConsts C, const float4* __restrict__ posu, const int* __restrict__ cell,
                                              const uint32_t* __restrict__ cellstart, double* __restrict__ conc,
                                              uint32_t n) {
  const uint32_t n_active = cellstart[2u * C.ncells];
  const uint32_t a = blockIdx.x * blockDim.x + threadIdx.x;
  if (a >= n_active) {                        // particles out of the grid (sorted last, C3) take no part: C_a = 0
    if (a < n) conc[a] = 0.0;
    return;
  }
  const float4 pa = posu[a];
  double sum = (double)(fast_rcp(pa.w));      // self term: w = 1, q = 0
  for_each_neighbour<DIM>(C, posu, cellstart, a, pa, cell[a],
                          [&](uint32_t, const float4 pb, float, float, float, float r2u) {
                            const float hq = fast_sqrt(r2u) * C.qscale;      // q / 2
                            const float w = 1.0f - hq, w2 = w * w;
                            sum += (double)(w2 * w2 * fmaf(4.0f, hq, 1.0f) * fast_rcp(pb.w));
                          });
  conc[a] = sum * (double)C.c_w;
}

template <int DIM>
__global__ void __launch_bounds__(128) k_shift(DevConsts C, const float4* __restrict__ posu,
                                               const float4* __restrict__ velp, const int* __restrict__ cell,
                                               const uint32_t* __restrict__ cellstart, const double* __restrict__ conc,
                                               float4* __restrict__ shiftv, uint32_t n) {
  const uint32_t n_bound = cellstart[C.ncells], n_active = cellstart[2u * C.ncells];
  const uint32_t a = blockIdx.x * blockDim.x + threadIdx.x;
  if (a >= n) return;
  // boundary particles and particles out of the grid are not shifted; the slot of an out-of-grid particle would
  // otherwise keep the vector some other particle left there on an earlier pass
  if (a < n_bound || a >= n_active) { shiftv[a] = make_float4(0.f, 0.f, 0.f, 0.f); return; }
  const float4 pa = posu[a];
  const double Ca = conc[a];
  float gx = 0.f, gy = 0.f, gz = 0.f;
  for_each_neighbour<DIM>(C, posu, cellstart, a, pa, cell[a],
                          [&](uint32_t b, const float4 pb, float dux, float duy, float duz, float r2u) {
                            const float w = fmaf(-fast_sqrt(r2u), C.qscale, 1.0f);
                            const float dC = (float)(conc[b] - Ca);
                            const float t = w * w * w * fast_rcp(pb.w) * dC;
                            gx = fmaf(t, dux, gx);
                            gy = fmaf(t, duy, gy);
                            gz = fmaf(t, duz, gz);
                          });
  gx *= C.c_gw; gy *= C.c_gw; gz *= C.c_gw;        // grad C_a  (Eq. 53)
  const float4 va = velp[a];
  const float ds = C.shift_ds * sqrtf(fmaf(va.z, va.z, fmaf(va.y, va.y, va.x * va.x)));   // D_s / dt (Eq. 41)
  float4 out;
  if (Ca < C.shift_fs_conc) {                     // Eq. 54 with n = -grad C / |grad C| (A29); a discontinuous switch, so in double
    const float gn = sqrtf(fmaf(gz, gz, fmaf(gy, gy, gx * gx)));
    const float fac = gn > 0.f ? -ds * C.shift_alpha_n * (-gn - C.shift_beta_n) / gn : 0.f;
    out = make_float4(-fac * gx, -fac * gy, -fac * gz, 0.f);
  } else {
    out = make_float4(-ds * gx, -ds * gy, -ds * gz, 0.f);     // Eq. 40
  }
  shiftv[a] = out;
}

}  // namespace

void bx_mdbc(const DevConsts& C, const ParticleSet& P, const uint32_t* cellstart, int64_t n, const double* normals,
             const Motion* motions, int nmotions, DevScalars* sc, double tfrac, cudaStream_t s) {
  if (n == 0) return;
  const unsigned grid = (unsigned)((n + 127) / 128);     // n_bound is only known on the device; surplus threads exit
  if (C.dim == 3) k_mdbc<3><<<grid, 128, 0, s>>>(C, P, cellstart, normals, motions, nmotions, sc, tfrac);
  else k_mdbc<2><<<grid, 128, 0, s>>>(C, P, cellstart, normals, motions, nmotions, sc, tfrac);
}

void bx_shift(const DevConsts& C, const ParticleSet& P, const uint32_t* cellstart, int64_t n, double* conc,
              float4* shiftv, cudaStream_t s) {
  if (n == 0) return;
  const unsigned grid = (unsigned)((n + 127) / 128);
  if (C.dim == 3) {
    k_conc<3><<<grid, 128, 0, s>>>(C, P.posu, P.cell, cellstart, conc, (uint32_t)n);
    k_shift<3><<<grid, 128, 0, s>>>(C, P.posu, P.velp, P.cell, cellstart, conc, shiftv, (uint32_t)n);
  } else {
    k_conc<2><<<grid, 128, 0, s>>>(C, P.posu, P.cell, cellstart, conc, (uint32_t)n);
    k_shift<2><<<grid, 128, 0, s>>>(C, P.posu, P.velp, P.cell, cellstart, conc, shiftv, (uint32_t)n);
  }
}
