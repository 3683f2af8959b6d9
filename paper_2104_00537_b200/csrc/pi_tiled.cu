// Particle interaction (PI) task, tiled kernel for sm_100a (cells of size 2h, cell_div = 1).
//
// One CTA owns a tile of TX x TY x TZ cells.  It stages the particles of the tile and of the one-cell halo
// around it -- (TX+2)(TY+2)(TZ+2) cells, both type blocks -- in shared memory, with positions rewritten as
// exact tile-relative coordinates (offset u + integer cell offset; all values on the 2^-22 grid with
// magnitude < 4, so every difference is exact in fp32 and the canonical predicate C2 is reproduced
// bit for bit).  Each warp then takes chunks of 32 particles a of the tile's centre cells (one a per lane):
//   test phase : every candidate b of the adjacent cells is read once per warp as a shared-memory
//                broadcast (LDS.128) and tested by all 32 lanes; accepted b indices go to a per-lane queue;
//   pair phase : when (almost) all lanes hold queued work, each lane pops one b and evaluates the pair
//                (Eq. 15, 17-18, 21-22, 36), so the ~45-instruction pair body runs with (almost) full lanes
//                instead of the ~15 % that a test-and-branch loop gets (sphere / 27 cells = 15.5 %).
// What is kept from the paper's design: cell-linked list, particles sorted by cell, positions relative to the
// cell in fp32.  What differs: the paper's thread-per-particle loop with a branch per
// candidate is replaced by staging + per-lane compaction.
#include "pi_common.cuh"

namespace {

template <int DIM>
struct TileCfg {
  static constexpr int TX = DIM == 3 ? 2 : 6, TY = DIM == 3 ? 2 : 1, TZ = DIM == 3 ? 2 : 6;   // 2-D: 6x6 cells per tile (swept on config 1)
  static constexpr int SX = TX + 2, SY = DIM == 3 ? TY + 2 : 1, SZ = TZ + 2;
  static constexpr int NCELL = SX * SY * SZ;   // staged cells per type block
  static constexpr int NR = 2 * NCELL;         // staged ranges: block 0 = boundary, block 1 = fluid
  static constexpr int NSEG = 2 * TY * TZ;     // a-segments: (block, cz, cy) rows of TX centre cells
};

constexpr int PT_RQ = 8;          // ring entries (group base, 32-bit accept mask) per lane
constexpr float PT_MARGIN = 6.0e-5f;  // prefilter slack, > worst rounding error of the expanded form

template <int DIM>
__device__ __forceinline__ int range_index(int blk, int ix, int iy, int iz) {   // ix,iy,iz are staged indices (0-based)
  using T = TileCfg<DIM>;
  return ((blk * T::SZ + iz) * T::SY + iy) * T::SX + ix;
}

struct TileSmem {
  float4* tpos;       // (x, y, z, |b|^2): tile-centred exact coordinates + squared norm for the prefilter
  float4* vrho;       // (vx, vy, vz, rho)
  float* press;       // P
  uint2* ring;        // per-lane ring of (group base index, accept mask)
  uint32_t* soff;     // NR + 1
  uint32_t* gstart;   // NR
  uint32_t* misc;     // [0] chunk counter, [1..NSEG+1] chunk prefix
};

// Per-lane state of one particle a.
struct LaneA {
  float x, y, z;          // exact tile-centred coordinates
  float nx, ny, nz, thr;  // -2x, -2y, -2z, (R2u + margin) - |a|^2 : prefilter  |b|^2 - 2 a.b < thr
  float vx, vy, vz, rho, inv_rho, P;
};

struct LaneQ {
  unsigned cur_mask, cur_base;   // entry being consumed
  unsigned rd, wr;               // ring positions
};

// A popped pair whose b data is already on its way from shared memory (software pipelining: the loads
// of pair i+1 are issued before the arithmetic of pair i).
struct Pending {
  float4 pb, vb;
  float Pb;
  unsigned valid;
};

// Pop the next queued candidate of this lane (or the lane's own particle as a harmless dummy: r = 0
// contributes exactly 0, A17) and issue its loads.
template <int NT>
__device__ __forceinline__ void fetch_next(const TileSmem& S, LaneQ& Q, unsigned ja, Pending& N) {
  if (Q.cur_mask == 0u && Q.rd != Q.wr) {
    const uint2 e = S.ring[(Q.rd & (PT_RQ - 1)) * NT + threadIdx.x];
    Q.cur_base = e.x;
    Q.cur_mask = e.y;
    Q.rd++;
  }
  const bool v = Q.cur_mask != 0u;
  const unsigned j = v ? Q.cur_base + (__ffs(Q.cur_mask) - 1) : ja;
  Q.cur_mask &= Q.cur_mask - 1u;
  N.pb = S.tpos[j];
  N.vb = S.vrho[j];
  N.Pb = S.press[j];
  N.valid = v ? 1u : 0u;
}

// Pair arithmetic, branch free.  The canonical predicate C2 is evaluated here on the exact offsets; a
// prefilter false positive (~1e-4 of the pairs) or a dummy gets weight 0.
template <int DIM, bool A_FLUID, bool DDT>
__device__ __forceinline__ void pair_eval(const DevConsts& C, const LaneA& a, const Pending& P, PairAcc& A,
                                          unsigned int& nb) {
  const float dux = a.x - P.pb.x, duy = DIM == 3 ? a.y - P.pb.y : 0.f, duz = a.z - P.pb.z;   // exact (C1)
  const float r2u = pair_r2u<DIM>(dux, duy, duz);
  const bool ok = r2u < C.R2u;
  nb += (ok ? P.valid : 0u);
  const float rho_b = P.vb.w;
  const float s = fast_sqrt(r2u);
  const float w = fmaf(-s, C.qscale, 1.0f);            // 1 - q/2   (Eq. 11)
  const float w3 = ok ? w * w * w : 0.f;               // grad_a W_ab = Cf w^3 cs du
  const float inv_rho_b = fast_rcp(rho_b);
  const float dvx = a.vx - P.vb.x, dvy = a.vy - P.vb.y, dvz = a.vz - P.vb.z;
  float dot = fmaf(dvz, duz, fmaf(dvy, duy, dvx * dux));     // v_ab . r_ab / cs
  dot = ok ? dot : 0.f;
  const float gb = w3 * inv_rho_b;
  A.sc = fmaf(gb, dot, A.sc);
  if (A_FLUID) {
    if (DDT) {
      float drho = a.rho - rho_b;
      if (C.ddt_model == 1) drho -= hydrostatic_drho(C, dux, duy, duz);   // Eq. 19-20 (A23); uniform branch
      A.sd = fmaf(gb, drho, A.sd);
    }
    const float rs = a.rho + rho_b;
    const float x = fast_rcp((r2u + C.eta2u) * rs);
    A.visc = fmaxf(A.visc, fabsf(dot) * x * rs);       // |mu_ab| / c_mu   (Eq. 21, A12)
    const float t = fminf(dot, 0.0f) * x;              // Pi_ab = c_pi * t, approaching pairs only (Eq. 21)
    const float coef = w3 * fmaf(a.P + P.Pb, a.inv_rho * inv_rho_b, C.c_pi * t);
    A.sx = fmaf(coef, dux, A.sx);                      // plain sums only: pi_tiled() declines compensated_sums
    A.sy = fmaf(coef, duy, A.sy);
    A.sz = fmaf(coef, duz, A.sz);
    if (C.visco_model == 1) {                          // Eq. 23 (A22; c_pi = 0 in this model); uniform branch
      const float lam = w3 * r2u * x;
      A.lx = fmaf(lam, dvx, A.lx);
      A.ly = fmaf(lam, dvy, A.ly);
      A.lz = fmaf(lam, dvz, A.lz);
    }
  }
}

template <int DIM, bool A_FLUID>
__device__ __forceinline__ void pair_eval_ddt(const DevConsts& C, bool ddt, const LaneA& a, const Pending& P,
                                              PairAcc& A, unsigned int& nb) {
  if (ddt) pair_eval<DIM, A_FLUID, true>(C, a, P, A, nb);
  else pair_eval<DIM, A_FLUID, false>(C, a, P, A, nb);
}

__device__ __forceinline__ bool lane_has_work(const LaneQ& Q, const Pending& P) {
  return P.valid != 0u || Q.cur_mask != 0u || Q.rd != Q.wr;
}

// Run the pair body in lock step while at least thr_lanes lanes have work, or while some lane's ring is
// nearly full (that lane must make progress even if others are idle).  Two half steps per loop iteration so
// the pending-pair registers ping-pong without moves.
template <int DIM, int NT, bool A_FLUID>
__device__ __forceinline__ void drain(const DevConsts& C, const TileSmem& S, bool ddt, int thr_lanes, unsigned ja,
                                      LaneQ& Q, Pending& P, const LaneA& a, PairAcc& acc, unsigned int& nb) {
  while (true) {
    if (__popc(__ballot_sync(0xffffffffu, lane_has_work(Q, P))) < thr_lanes &&
        !__any_sync(0xffffffffu, Q.wr - Q.rd >= PT_RQ - 1)) break;
    Pending N;
    fetch_next<NT>(S, Q, ja, N);
    pair_eval_ddt<DIM, A_FLUID>(C, ddt, a, P, acc, nb);
    if (__popc(__ballot_sync(0xffffffffu, lane_has_work(Q, N))) < thr_lanes &&
        !__any_sync(0xffffffffu, Q.wr - Q.rd >= PT_RQ - 1)) { P = N; break; }
    fetch_next<NT>(S, Q, ja, P);
    pair_eval_ddt<DIM, A_FLUID>(C, ddt, a, N, acc, nb);
  }
}

template <int DIM>
__device__ __forceinline__ bool prefilter(const LaneA& a, const float4& pb) {
  float s = fmaf(a.nx, pb.x, pb.w);
  if (DIM == 3) s = fmaf(a.ny, pb.y, s);
  s = fmaf(a.nz, pb.z, s);
  return s < a.thr;
}

// Test candidates [j0, j1) for all lanes in groups of 32 (one accept bit per candidate), queue non-empty masks,
// and run the pair body while (almost) all lanes have queued work.
template <int DIM, int NT, bool A_FLUID>
__device__ __forceinline__ void sweep_range(const DevConsts& C, const TileSmem& S, unsigned j0, unsigned j1, bool ddt,
                                            int thr_lanes, unsigned ja, LaneQ& Q, Pending& P, const LaneA& a,
                                            PairAcc& acc, unsigned int& nb) {
  for (unsigned j = j0; j < j1; j += 32) {
    unsigned m = 0;
    if (j + 32 <= j1) {
#pragma unroll
      for (int u = 0; u < 32; u++)
        if (prefilter<DIM>(a, S.tpos[j + u])) m |= 1u << u;
    } else {
      for (unsigned u = 0; j + u < j1; u++)
        if (prefilter<DIM>(a, S.tpos[j + u])) m |= 1u << u;
    }
    if (m != 0u) {
      S.ring[(Q.wr & (PT_RQ - 1)) * NT + threadIdx.x] = make_uint2(j, m);
      Q.wr++;
    }
    drain<DIM, NT, A_FLUID>(C, S, ddt, thr_lanes, ja, Q, P, a, acc, nb);
  }
}

// One chunk of up to 32 particles a (one per lane) of a-segment (blk_a, cy, cz).
template <int DIM, int NT, bool A_FLUID>
__device__ __forceinline__ void process_chunk(const DevConsts& C, const PiArgs& A, const TileSmem& S, int cy, int cz,
                                              int vx, unsigned seg_start, unsigned seg_len, unsigned chunk,
                                              float& f2max, float& viscmax, unsigned int& nbsum) {
  using T = TileCfg<DIM>;
  const int lane = threadIdx.x & 31;
  const int blk_a = A_FLUID ? 1 : 0;
  const unsigned t = chunk * 32 + lane;
  const bool active = t < seg_len;
  const unsigned ja = seg_start + (active ? t : 0);
  const float4 pa = S.tpos[ja];
  const float4 va = S.vrho[ja];
  LaneA a;
  a.x = pa.x; a.y = pa.y; a.z = pa.z;
  a.nx = -2.f * pa.x; a.ny = -2.f * pa.y; a.nz = -2.f * pa.z;
  a.thr = active ? (C.R2u + PT_MARGIN) - pa.w : -1.0e30f;       // inactive lanes never accept
  a.vx = va.x; a.vy = va.y; a.vz = va.z; a.rho = va.w;
  a.inv_rho = fast_rcp(va.w);
  a.P = S.press[ja];
  // cell (x) of this lane's a, and of the chunk's first / last a (uniform)
  int cxa = 0;
  for (int x = 1; x < vx; x++) cxa += ja >= S.soff[range_index<DIM>(blk_a, 1 + x, DIM == 3 ? 1 + cy : 0, 1 + cz)];
  const unsigned t_lo = chunk * 32, t_hi = min(chunk * 32 + 31, seg_len - 1);
  int cx_lo = 0, cx_hi = 0;
  for (int x = 1; x < vx; x++) {
    const unsigned b = S.soff[range_index<DIM>(blk_a, 1 + x, DIM == 3 ? 1 + cy : 0, 1 + cz)];
    cx_lo += seg_start + t_lo >= b;
    cx_hi += seg_start + t_hi >= b;
  }
  const int n_act = min(32u, seg_len - t_lo);
  const int thr_lanes = max(1, n_act - max(2, n_act / 8));

  PairAcc acc = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
  unsigned int nb = 0;
  LaneQ Q = {0u, 0u, 0u, 0u};
  Pending P;
  P.pb = pa; P.vb = va; P.Pb = a.P; P.valid = 0u;             // empty pipeline: a dummy (the particle itself)
  const int dy0 = DIM == 3 ? -1 : 0, dy1 = DIM == 3 ? 1 : 0;
  if (A_FLUID) {   // boundary neighbours of fluid a (no diffusion term unless ddt_over_boundary, A4)
    const bool ddt = C.ddt_over_boundary != 0;
    for (int dz = -1; dz <= 1; dz++)
      for (int dy = dy0; dy <= dy1; dy++) {
        const int iy = DIM == 3 ? 1 + cy + dy : 0, iz = 1 + cz + dz;
        const unsigned j0 = S.soff[range_index<DIM>(0, cx_lo, iy, iz)];
        const unsigned j1 = S.soff[range_index<DIM>(0, cx_hi + 2, iy, iz) + 1];
        sweep_range<DIM, NT, A_FLUID>(C, S, j0, j1, ddt, thr_lanes, ja, Q, P, a, acc, nb);
      }
    drain<DIM, NT, A_FLUID>(C, S, ddt, 1, ja, Q, P, a, acc, nb);
  }
  for (int dz = -1; dz <= 1; dz++)   // fluid neighbours
    for (int dy = dy0; dy <= dy1; dy++) {
      const int iy = DIM == 3 ? 1 + cy + dy : 0, iz = 1 + cz + dz;
      const unsigned j0 = S.soff[range_index<DIM>(1, cx_lo, iy, iz)];
      const unsigned j1 = S.soff[range_index<DIM>(1, cx_hi + 2, iy, iz) + 1];
      sweep_range<DIM, NT, A_FLUID>(C, S, j0, j1, true, thr_lanes, ja, Q, P, a, acc, nb);
    }
  drain<DIM, NT, A_FLUID>(C, S, true, 1, ja, Q, P, a, acc, nb);

  if (active) {
    if (A_FLUID) nb -= 1;   // the particle itself passed the test at r = 0 and contributed exactly 0 (A17)
    const int r_a = range_index<DIM>(blk_a, 1 + cxa, DIM == 3 ? 1 + cy : 0, 1 + cz);
    const unsigned ga = S.gstart[r_a] + (ja - S.soff[r_a]);
    const float4 out = finish_particle(C, A_FLUID, a.rho, acc);
    if (!isfinite(out.x + out.y + out.z + out.w)) atomicOr(&A.sc->flags, 1u);   // reported as SPH_E_NAN
    A.acc[ga] = out;
    if (A.nbcount) A.nbcount[ga] = nb;
    if (A_FLUID) f2max = fmaxf(f2max, fmaf(out.x, out.x, fmaf(out.y, out.y, out.z * out.z)));
    viscmax = fmaxf(viscmax, acc.visc * C.c_mu);
    nbsum += nb;
  }
}

template <int DIM>
__device__ __forceinline__ void overflow_one(const DevConsts& C, const PiArgs& A, uint32_t a, bool a_fluid, float& f2,
                                          float& visc, unsigned int& nb) {
  gather_one<DIM>(C, A, a, a_fluid, f2, visc, nb);
}

template <int DIM, int NT, int NMAX>
__global__ void __launch_bounds__(NT, 1) k_pi_tiled(DevConsts C, PiArgs A, int ntx, int nty) {
  using T = TileCfg<DIM>;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  TileSmem S;
  S.tpos = reinterpret_cast<float4*>(smem_raw);
  S.vrho = S.tpos + NMAX;
  S.ring = reinterpret_cast<uint2*>(S.vrho + NMAX);
  S.press = reinterpret_cast<float*>(S.ring + PT_RQ * NT);
  S.soff = reinterpret_cast<uint32_t*>(S.press + NMAX);
  S.gstart = S.soff + (T::NR + 1);
  S.misc = S.gstart + T::NR;
  __shared__ uint32_t s_cnt[T::NR];

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int tx = blockIdx.x % ntx, ty = (blockIdx.x / ntx) % nty, tz = blockIdx.x / (ntx * nty);
  const int ox = tx * T::TX, oy = ty * T::TY, oz = tz * T::TZ;

  // 1. global ranges of the staged cells
  for (int r = tid; r < T::NR; r += NT) {
    const int blk = r / T::NCELL, c = r % T::NCELL;
    const int ix = c % T::SX, iy = (c / T::SX) % T::SY, iz = c / (T::SX * T::SY);
    int g[3] = {ox + ix - 1, DIM == 3 ? oy + iy - 1 : 0, oz + iz - 1};
    bool valid = true;
#pragma unroll
    for (int k = 0; k < 3; k++) {
      if (DIM == 2 && k == 1) continue;
      if (C.per[k]) g[k] = (g[k] + C.nc[k]) % C.nc[k];
      else if (g[k] < 0 || g[k] >= C.nc[k]) valid = false;
    }
    uint32_t g0 = 0, n = 0;
    if (valid) {
      const uint32_t key = (uint32_t)blk * C.ncells + (uint32_t)g[0] + (uint32_t)C.nc[0] * ((uint32_t)g[1] + (uint32_t)C.nc[1] * (uint32_t)g[2]);
      g0 = A.cellstart[key];
      n = A.cellstart[key + 1] - g0;
    }
    s_cnt[r] = n;
    S.gstart[r] = g0;
  }
  __syncthreads();
  if (warp == 0) {   // exclusive scan of the NR counts
    constexpr int PER = (T::NR + 31) / 32;
    uint32_t v[PER], sum = 0;
#pragma unroll
    for (int i = 0; i < PER; i++) {
      const int r = lane * PER + i;
      v[i] = r < T::NR ? s_cnt[r] : 0u;
      sum += v[i];
    }
    uint32_t inc = sum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t up = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= o) inc += up;
    }
    uint32_t run = inc - sum;
#pragma unroll
    for (int i = 0; i < PER; i++) {
      const int r = lane * PER + i;
      if (r < T::NR) S.soff[r] = run;
      run += v[i];
    }
    if (lane == 31) S.soff[T::NR] = inc;
  }
  __syncthreads();

  // a-segments: rows (block, cz, cy) of the valid centre cells; chunk prefix for dynamic scheduling
  const int vx = min(T::TX, C.nc[0] - ox);
  const int vy = DIM == 3 ? min(T::TY, C.nc[1] - oy) : 1;
  const int vz = min(T::TZ, C.nc[2] - oz);
  if (tid == 0) {
    uint32_t run = 0;
    for (int s = 0; s < T::NSEG; s++) {
      const int blk = s / (T::TY * T::TZ), cz = (s / T::TY) % T::TZ, cy = s % T::TY;
      uint32_t len = 0;
      if (cy < vy && cz < vz) {
        const int iy = DIM == 3 ? 1 + cy : 0;
        len = S.soff[range_index<DIM>(blk, vx, iy, 1 + cz) + 1] - S.soff[range_index<DIM>(blk, 1, iy, 1 + cz)];
      }
      S.misc[1 + s] = run;
      run += (len + 31) / 32;
    }
    S.misc[1 + T::NSEG] = run;
    S.misc[0] = 0;
  }
  __syncthreads();
  const uint32_t nchunks = S.misc[1 + T::NSEG];
  if (nchunks == 0) return;                       // nothing to compute in this tile (air)
  const uint32_t total = S.soff[T::NR];

  float f2max = 0.f, viscmax = 0.f;
  unsigned int nbsum = 0;

  if (total > (uint32_t)NMAX) {
    // staged set does not fit in shared memory (very crowded cells): per-particle global gather
    for (int s = 0; s < T::NSEG; s++) {
      const int blk = s / (T::TY * T::TZ), cz = (s / T::TY) % T::TZ, cy = s % T::TY;
      if (cy >= vy || cz >= vz) continue;
      const int iy = DIM == 3 ? 1 + cy : 0;
      const int r0 = range_index<DIM>(blk, 1, iy, 1 + cz), r1 = range_index<DIM>(blk, vx, iy, 1 + cz);
      const uint32_t g0 = S.gstart[r0], len = S.soff[r1 + 1] - S.soff[r0];
      for (uint32_t i = tid; i < len; i += NT) overflow_one<DIM>(C, A, g0 + i, blk == 1, f2max, viscmax, nbsum);
    }
    reduce_scalars(A.sc, f2max, viscmax, nbsum);
    return;
  }

  // 2. stage particles with tile-centred coordinates: u + integer cell offset - T/2.  Exact: every value is a
  //    multiple of 2^-22 with magnitude <= 2, so all differences are exact in fp32 (C1/C2).
  //    One staged particle per thread and trip: its range is found by bisection of the offsets (NR is a power
  //    of two), so that every lane is busy whatever the cell populations (about 11 particles per cell in 2-D).
  static_assert((T::NR & (T::NR - 1)) == 0, "bisection below assumes a power of two");
  for (uint32_t j = tid; j < total; j += NT) {
    int r = 0;
#pragma unroll
    for (int step = T::NR / 2; step > 0; step >>= 1)
      if (S.soff[r + step] <= j) r += step;         // largest r with soff[r] <= j (empty ranges are skipped over)
    const int c = r % T::NCELL;
    const float fx = (float)(c % T::SX - 1) - 0.5f * T::TX,
                fy = DIM == 3 ? (float)((c / T::SX) % T::SY - 1) - 0.5f * T::TY : 0.f,
                fz = (float)(c / (T::SX * T::SY) - 1) - 0.5f * T::TZ;
    const uint32_t g = S.gstart[r] + (j - S.soff[r]);
    const float4 p = A.posu[g];
    const float4 v = A.velp[g];
    const float x = p.x + fx, y = DIM == 3 ? p.y + fy : 0.f, z = p.z + fz;
    S.tpos[j] = make_float4(x, y, z, fmaf(z, z, fmaf(y, y, x * x)));
    S.vrho[j] = make_float4(v.x, v.y, v.z, p.w);
    S.press[j] = v.w;
  }
  __syncthreads();

  // 3. chunks of 32 a's, taken dynamically by the warps
  while (true) {
    uint32_t ch = 0;
    if (lane == 0) ch = atomicAdd(&S.misc[0], 1u);
    ch = __shfl_sync(0xffffffffu, ch, 0);
    if (ch >= nchunks) break;
    int s = 0;
    while (s + 1 < T::NSEG && ch >= S.misc[1 + s + 1]) s++;
    const int blk = s / (T::TY * T::TZ), cz = (s / T::TY) % T::TZ, cy = s % T::TY;
    const int iy = DIM == 3 ? 1 + cy : 0;
    const unsigned seg_start = S.soff[range_index<DIM>(blk, 1, iy, 1 + cz)];
    const unsigned seg_len = S.soff[range_index<DIM>(blk, vx, iy, 1 + cz) + 1] - seg_start;
    const unsigned chunk = ch - S.misc[1 + s];
    if (blk == 1) process_chunk<DIM, NT, true>(C, A, S, cy, cz, vx, seg_start, seg_len, chunk, f2max, viscmax, nbsum);
    else process_chunk<DIM, NT, false>(C, A, S, cy, cz, vx, seg_start, seg_len, chunk, f2max, viscmax, nbsum);
  }
  reduce_scalars(A.sc, f2max, viscmax, nbsum);
}

template <int DIM, int NT, int NMAX>
int launch_tiled(const DevConsts& C, const PiArgs& A, cudaStream_t s) {
  using T = TileCfg<DIM>;
  const int ntx = (C.nc[0] + T::TX - 1) / T::TX;
  const int nty = DIM == 3 ? (C.nc[1] + T::TY - 1) / T::TY : 1;
  const int ntz = (C.nc[2] + T::TZ - 1) / T::TZ;
  const size_t smem = sizeof(float4) * 2 * NMAX + sizeof(uint2) * PT_RQ * NT + sizeof(float) * NMAX +
                      sizeof(uint32_t) * (T::NR + 1 + T::NR + 2 + T::NSEG);
  // per device, so set on every launch (a cheap host call): a process may hold contexts on several devices
  if (cudaFuncSetAttribute(k_pi_tiled<DIM, NT, NMAX>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) !=
      cudaSuccess) {
    cudaGetLastError();
    return -1;
  }
  const long long ntiles = (long long)ntx * nty * ntz;
  if (ntiles > 0x7fffffffLL) return -1;
  k_pi_tiled<DIM, NT, NMAX><<<(unsigned)ntiles, NT, smem, s>>>(C, A, ntx, nty);
  return 0;
}

}  // namespace

// Returns 0 if the tiled kernel was launched, -1 if this configuration is not supported (caller falls back
// to the gather kernel): cells must have size 2h/1 (27- or 9-cell stencil).
int pi_tiled(const DevConsts& C, const PiArgs& A, cudaStream_t s) {
  if (A.n == 0) return 0;
  if (C.k != 1) return -1;
  if (C.comp_sums) return -1;        // no compensated variant of this kernel: the caller runs the gather kernel (sph.h)
  if (!(C.eta2u > 0.f)) return -1;   // the self pair (r = 0) must evaluate to exactly 0, which needs eta^2 > 0
  if (C.dim == 3) return launch_tiled<3, 512, 4992>(C, A, s);
  return launch_tiled<2, 128, 1024>(C, A, s);
}
