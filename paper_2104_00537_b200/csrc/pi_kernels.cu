// Particle interaction (PI) task, baseline kernel: one CUDA thread per particle walks the particles of
// the adjacent cells straight from global memory (L1/L2), as the paper describes its own GPU kernel
// ("a CUDA thread is created to compute the interactions of each particle"; "only the
// neighbouring particles in the adjacent cells will contribute").  This kernel supports
// every configuration (2-D/3-D, periodic axes, any cell_div) and is the fallback for the tiled kernel.
#include "pi_common.cuh"

namespace {

template <int DIM>
__global__ void __launch_bounds__(128) k_pi_gather(DevConsts C, PiArgs A) {
  const uint32_t n_bound = A.cellstart[C.ncells];        // boundary block sorted first (C3)
  const uint32_t n_active = A.cellstart[2u * C.ncells];  // in-grid particles
  const uint32_t a = blockIdx.x * blockDim.x + threadIdx.x;
  float f2 = 0.f, visc = 0.f;
  unsigned int nb = 0;
  if (a < n_active) {
    const bool a_fluid = a >= n_bound;
    const float4 pa = A.posu[a];
    const float4 va = A.velp[a];
    const int lin = A.cell[a];
    int ca[3];
    ca[0] = lin % C.nc[0];
    int r = lin / C.nc[0];
    ca[1] = r % C.nc[1];
    ca[2] = r / C.nc[1];
    const float inv_rho_a = fast_rcp(pa.w);
    PairAcc S = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
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
    A.acc[a] = out;
    if (A.nbcount) A.nbcount[a] = nb;
    if (a_fluid) f2 = fmaf(out.x, out.x, fmaf(out.y, out.y, out.z * out.z));
    visc = S.visc * C.c_mu;
  }
  reduce_scalars(A.sc, f2, visc, nb);
}

__global__ void k_reset_scalars(DevScalars* sc) {
  sc->n_inter_total += sc->n_inter;
  sc->n_inter = 0;
  sc->fmax2_bits = 0;
  sc->visc_bits = 0;
}

}  // namespace

void pi_reset_scalars(DevScalars* sc, cudaStream_t s) { k_reset_scalars<<<1, 1, 0, s>>>(sc); }

void pi_gather(const DevConsts& C, const PiArgs& A, cudaStream_t s) {
  if (A.n == 0) return;
  const int threads = 128;
  const unsigned grid = (unsigned)((A.n + threads - 1) / threads);
  if (C.dim == 3) k_pi_gather<3><<<grid, threads, 0, s>>>(C, A);
  else k_pi_gather<2><<<grid, threads, 0, s>>>(C, A);
}

int pi_tiled(const DevConsts&, const PiArgs&, cudaStream_t) { return -1; }
