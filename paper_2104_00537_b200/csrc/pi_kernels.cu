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
  if (a < n_active) gather_one<DIM>(C, A, a, a >= n_bound, f2, visc, nb);
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

