// Neighbour list (NL) task: cell key per particle, stable LSD radix sort of (key, index),
// cell-range table, reorder of the particle arrays.
// PAPER.md:558 "the simulation domain is split up in cubic cells of size 2h ... The particles with
// their data are sorted according to the cell to which they belong and an index array with the first
// and last particle of each cell is created."  Canonical key / order / range conventions: C3.
// All of this is integer work and must be bit-exact against the oracle.
#include <stdarg.h>
#include <stdio.h>

#include <mutex>

#include "sph_internal.cuh"

namespace {

constexpr int RS_THREADS = 256;
constexpr int RS_WARPS = RS_THREADS / 32;
constexpr int RS_ITEMS = 16;                       // keys per thread
constexpr int RS_TILE = RS_THREADS * RS_ITEMS;     // 4096 keys per block
constexpr int RS_RADIX = 256;

// a1: key = block * ncells + cell, block 0 = boundary, 1 = fluid; out-of-grid -> 2 * ncells (C3)
__global__ void k_keys(const int* __restrict__ cell, const uint8_t* __restrict__ type, int64_t n,
                       uint32_t ncells, uint32_t* __restrict__ key, uint32_t* __restrict__ idx) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  int c = cell[i];
  uint32_t k = c < 0 ? 2u * ncells : (type[i] == 0 ? ncells : 0u) + (uint32_t)c;
  key[i] = k;
  idx[i] = (uint32_t)i;
}

// a2, pass part 1: per-block digit histogram + global digit totals
__global__ void __launch_bounds__(RS_THREADS) k_rs_hist(const uint32_t* __restrict__ key, int64_t n, int shift,
                                                       uint32_t nblocks, uint32_t* __restrict__ block_hist,
                                                       uint32_t* __restrict__ digit_total) {
  __shared__ uint32_t h[RS_RADIX];
  h[threadIdx.x] = 0;
  __syncthreads();
  int64_t base = (int64_t)blockIdx.x * RS_TILE;
#pragma unroll
  for (int k = 0; k < RS_ITEMS; k++) {
    int64_t e = base + k * RS_THREADS + threadIdx.x;
    if (e < n) atomicAdd(&h[(key[e] >> shift) & 0xFF], 1u);
  }
  __syncthreads();
  uint32_t c = h[threadIdx.x];
  block_hist[(size_t)threadIdx.x * nblocks + blockIdx.x] = c;
  if (c) atomicAdd(&digit_total[threadIdx.x], c);
}

__device__ __forceinline__ uint32_t warp_incl_scan(uint32_t v) {
  int lane = threadIdx.x & 31;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    uint32_t t = __shfl_up_sync(0xffffffffu, v, o);
    if (lane >= o) v += t;
  }
  return v;
}

// a2, pass part 2: block d turns row d of block_hist into global offsets:
// offset[d][b] = sum_{d' < d} total[d'] + sum_{b' < b} count[d][b']
__global__ void __launch_bounds__(RS_THREADS) k_rs_scan(uint32_t* __restrict__ block_hist, uint32_t nblocks,
                                                       const uint32_t* __restrict__ digit_total) {
  __shared__ uint32_t wsum[RS_WARPS];
  __shared__ uint32_t s_carry;
  const int d = blockIdx.x, t = threadIdx.x, lane = t & 31, w = t >> 5;
  uint32_t v = t < d ? digit_total[t] : 0u;
  uint32_t inc = warp_incl_scan(v);
  if (lane == 31) wsum[w] = inc;
  __syncthreads();
  if (t == 0) {
    uint32_t s = 0;
    for (int i = 0; i < RS_WARPS; i++) s += wsum[i];
    s_carry = s;
  }
  __syncthreads();
  uint32_t* row = block_hist + (size_t)d * nblocks;
  for (uint32_t b0 = 0; b0 < nblocks; b0 += RS_THREADS) {
    uint32_t b = b0 + t;
    uint32_t c = b < nblocks ? row[b] : 0u;
    uint32_t in = warp_incl_scan(c);
    __syncthreads();                 // wsum reuse
    if (lane == 31) wsum[w] = in;
    __syncthreads();
    uint32_t woff = 0;
    for (int i = 0; i < w; i++) woff += wsum[i];
    uint32_t carry = s_carry;
    if (b < nblocks) row[b] = carry + woff + in - c;
    __syncthreads();
    if (t == RS_THREADS - 1) s_carry = carry + woff + in;
    __syncthreads();
  }
}

// a2, pass part 3: stable scatter.  Tile order is (warp, round, lane); ranks are assigned in that order,
// so equal digits keep their relative order (LSD radix sort needs every pass to be stable).
__global__ void __launch_bounds__(RS_THREADS) k_rs_scatter(const uint32_t* __restrict__ key_in,
                                                          const uint32_t* __restrict__ idx_in, int64_t n, int shift,
                                                          uint32_t nblocks, const uint32_t* __restrict__ block_off,
                                                          uint32_t* __restrict__ key_out,
                                                          uint32_t* __restrict__ idx_out, int first_pass) {
  __shared__ uint32_t whist[RS_WARPS][RS_RADIX];
  const int t = threadIdx.x, lane = t & 31, w = t >> 5;
  for (int i = t; i < RS_WARPS * RS_RADIX; i += RS_THREADS) (&whist[0][0])[i] = 0;
  __syncthreads();
  const int64_t base = (int64_t)blockIdx.x * RS_TILE + (int64_t)w * (RS_ITEMS * 32);
  const uint32_t lt = (1u << lane) - 1u;
  uint32_t keys[RS_ITEMS], rank[RS_ITEMS];
#pragma unroll
  for (int k = 0; k < RS_ITEMS; k++) {
    int64_t e = base + k * 32 + lane;
    keys[k] = e < n ? key_in[e] : 0xFFFFFFFFu;
  }
#pragma unroll
  for (int k = 0; k < RS_ITEMS; k++) {
    uint32_t dgt = (keys[k] >> shift) & 0xFF;
    uint32_t peers = __match_any_sync(0xffffffffu, dgt);
    int leader = __ffs(peers) - 1;
    uint32_t old = 0;
    if (lane == leader) {
      old = whist[w][dgt];
      whist[w][dgt] = old + __popc(peers);
    }
    old = __shfl_sync(0xffffffffu, old, leader);
    rank[k] = old + __popc(peers & lt);
    __syncwarp();
  }
  __syncthreads();
  {  // thread t owns digit t: exclusive scan over warps, seeded with this block's global offset
    uint32_t run = block_off[(size_t)t * nblocks + blockIdx.x];
#pragma unroll
    for (int i = 0; i < RS_WARPS; i++) {
      uint32_t c = whist[i][t];
      whist[i][t] = run;
      run += c;
    }
  }
  __syncthreads();
#pragma unroll
  for (int k = 0; k < RS_ITEMS; k++) {
    int64_t e = base + k * 32 + lane;
    if (e < n) {
      uint32_t dgt = (keys[k] >> shift) & 0xFF;
      uint32_t pos = whist[w][dgt] + rank[k];
      key_out[pos] = keys[k];
      idx_out[pos] = first_pass ? (uint32_t)e : idx_in[e];
    }
  }
}

// a3: cellstart[k] = #{sorted keys < k}, k = 0 .. nkeys (nkeys + 1 entries): one lower-bound search per key,
// so empty cells (most of a dam-break grid is air) cost the same as full ones.
__global__ void k_cellstart(const uint32_t* __restrict__ key, int64_t n, uint32_t nkeys,
                            uint32_t* __restrict__ cellstart) {
  uint32_t k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k > nkeys) return;
  int64_t lo = 0, hi = n;            // first index with key[idx] >= k
  while (lo < hi) {
    int64_t mid = (lo + hi) >> 1;
    if (key[mid] < k) lo = mid + 1; else hi = mid;
  }
  cellstart[k] = (uint32_t)lo;
}

// (the Tait EOS, Eq. 28, lives in sph_internal.cuh: eos_pressure)

// a4 (+ a7): gather every per-particle array by the sorted index; P from rho (EOS) on the way.
__global__ void k_reorder(DevConsts C, ParticleSet src, ParticleSet dst, const uint32_t* __restrict__ idx,
                          int64_t n, int with_n) {
  int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= n) return;
  uint32_t i = idx[j];
  float4 p = src.posu[i];
  float4 v = src.velp[i];
  v.w = eos_pressure(C, p.w);
  dst.posu[j] = p;
  dst.velp[j] = v;
  dst.cell[j] = src.cell[i];
  dst.id[j] = src.id[i];
  dst.type[j] = src.type[i];
  if (with_n) {
    dst.posu_n[j] = src.posu_n[i];
    dst.vel_n[j] = src.vel_n[i];
    dst.cell_n[j] = src.cell_n[i];
  }
}

}  // namespace

static inline unsigned grid_for(int64_t n, int threads) { return (unsigned)((n + threads - 1) / threads); }

void nl_compute_keys(const DevConsts& C, const ParticleSet& P, int64_t n, uint32_t* key, uint32_t* idx,
                     cudaStream_t s) {
  if (n == 0) return;
  k_keys<<<grid_for(n, 256), 256, 0, s>>>(P.cell, P.type, n, C.ncells, key, idx);
}

size_t nl_radix_hist_entries(int64_t n) {
  size_t nblocks = (size_t)((n + RS_TILE - 1) / RS_TILE);
  if (nblocks == 0) nblocks = 1;
  return nblocks * RS_RADIX;
}

int nl_radix_sort(uint32_t* key_a, uint32_t* idx_a, uint32_t* key_b, uint32_t* idx_b, int64_t n, int key_bits,
                  uint32_t* block_hist, uint32_t* digit_total, int* n_launch, cudaStream_t s) {
  if (n == 0) return 0;
  const uint32_t nblocks = (uint32_t)((n + RS_TILE - 1) / RS_TILE);
  int passes = (key_bits + 7) / 8;
  if (passes < 1) passes = 1;
  cudaMemsetAsync(digit_total, 0, sizeof(uint32_t) * RS_RADIX * 4, s);
  uint32_t *kin = key_a, *iin = idx_a, *kout = key_b, *iout = idx_b;
  for (int p = 0; p < passes; p++) {
    int shift = 8 * p;
    k_rs_hist<<<nblocks, RS_THREADS, 0, s>>>(kin, n, shift, nblocks, block_hist, digit_total + p * RS_RADIX);
    k_rs_scan<<<RS_RADIX, RS_THREADS, 0, s>>>(block_hist, nblocks, digit_total + p * RS_RADIX);
    k_rs_scatter<<<nblocks, RS_THREADS, 0, s>>>(kin, iin, n, shift, nblocks, block_hist, kout, iout, p == 0);
    uint32_t* tk = kin; kin = kout; kout = tk;
    uint32_t* ti = iin; iin = iout; iout = ti;
    if (n_launch) *n_launch += 3;
  }
  return (passes & 1) ? 1 : 0;   // after an odd number of passes the result is in buffer b
}

void nl_cellstart(const uint32_t* sorted_key, int64_t n, uint32_t nkeys, uint32_t* cellstart, cudaStream_t s) {
  k_cellstart<<<grid_for((int64_t)nkeys + 1, 256), 256, 0, s>>>(sorted_key, n, nkeys, cellstart);
}

void nl_reorder(const DevConsts& C, const ParticleSet& src, const ParticleSet& dst, const uint32_t* idx,
                int64_t n, bool with_n_state, cudaStream_t s) {
  if (n == 0) return;
  k_reorder<<<grid_for(n, 256), 256, 0, s>>>(C, src, dst, idx, n, with_n_state ? 1 : 0);
}

// =====================================================================================================================
// sph_sort_keys_static (include/sph.h): the a2 radix sort above for callers that must not allocate.
//
// The context path (build_nl in sph_api.cu) gets its sort work space -- the ping-pong (key, index) buffers, the
// per-block digit histograms and the digit totals -- from sph_params.dev_alloc or cudaMalloc at sph_load_particles.
// A host program that has already handed every byte of HBM to its own pool, or that calls the sort from inside a
// solver loop it cannot afford to stall (cudaMalloc and cudaFree synchronise the whole device), has neither option.
// For those callers the same three kernels run here on a work space that is part of the library image: one
// file-scope __device__ array, sized for SPH_SORT_STATIC_MAX_N pairs, which every GPU that loads the library holds
// until the process exits (about 8.3 MiB).
//
// Note for whoever edits this: in HOST code the name g_sort_scratch is only a handle of the symbol.  It is not a device
// address and must never be given to a kernel or to cudaMemsetAsync; the address on the current device comes from
// cudaGetSymbolAddress, once per device (sort_scratch_on_current_device).
// =====================================================================================================================
namespace {

constexpr int64_t ST_MAX_N = SPH_SORT_STATIC_MAX_N;
constexpr size_t ST_MAX_BLOCKS = (size_t)((ST_MAX_N + RS_TILE - 1) / RS_TILE);
// layout, in 32-bit words (every part starts on a 256-byte boundary):
constexpr size_t ST_OFF_KEY = 0;                                        // ping-pong keys            [ST_MAX_N]
constexpr size_t ST_OFF_IDX = ST_OFF_KEY + (size_t)ST_MAX_N;            // ping-pong indices         [ST_MAX_N]
constexpr size_t ST_OFF_HIST = ST_OFF_IDX + (size_t)ST_MAX_N;           // per-block digit histogram [256][nblocks]
constexpr size_t ST_OFF_TOTAL = ST_OFF_HIST + ST_MAX_BLOCKS * RS_RADIX; // digit totals, 4 passes    [4][256]
constexpr size_t ST_WORDS = ST_OFF_TOTAL + 4 * RS_RADIX;
static_assert(ST_MAX_N % 64 == 0 && (ST_MAX_BLOCKS * RS_RADIX) % 64 == 0, "parts of the work space are 256-byte aligned");

static __device__ __align__(256) uint32_t g_sort_scratch[ST_WORDS];

constexpr int ST_MAX_DEVICES = 64;
uint32_t* g_scratch_addr[ST_MAX_DEVICES];   // device address of g_sort_scratch, per device ordinal; 0 = not looked up yet
std::mutex g_scratch_mu;

// Address of the work space on the device that is current on the calling thread.  The first call on a device asks the
// runtime for it (this also makes the runtime load the module there); later calls read the cached pointer.
cudaError_t sort_scratch_on_current_device(uint32_t** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= ST_MAX_DEVICES) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(g_scratch_mu);
  if (!g_scratch_addr[dev]) {
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, g_sort_scratch);
    if (e != cudaSuccess) return e;
    if (!p) return cudaErrorInvalidSymbol;
    g_scratch_addr[dev] = (uint32_t*)p;
  }
  *out = g_scratch_addr[dev];
  return cudaSuccess;
}

int static_sort_fail(int code, char* errmsg, size_t errmsg_bytes, const char* fmt, ...) {
  if (errmsg && errmsg_bytes) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(errmsg, errmsg_bytes, fmt, ap);
    va_end(ap);
  }
  return code;
}

}  // namespace

extern "C" __attribute__((visibility("default"))) int sph_sort_keys_static(const uint32_t* key, int64_t n,
                                                                           int32_t key_bits, uint32_t* key_sorted,
                                                                           uint32_t* perm, void* cuda_stream,
                                                                           char* errmsg, size_t errmsg_bytes) {
  if (errmsg && errmsg_bytes) errmsg[0] = 0;
  if (n < 0) return static_sort_fail(SPH_E_BADARG, errmsg, errmsg_bytes, "sph_sort_keys_static: n = %lld is negative", (long long)n);
  if (key_bits < 1 || key_bits > 32)
    return static_sort_fail(SPH_E_BADARG, errmsg, errmsg_bytes, "sph_sort_keys_static: key_bits = %d, must be 1..32", (int)key_bits);
  if (n > ST_MAX_N)
    return static_sort_fail(SPH_E_OVERFLOW, errmsg, errmsg_bytes,
                            "sph_sort_keys_static: n = %lld exceeds SPH_SORT_STATIC_MAX_N = %lld, the size the built-in work "
                            "space was compiled for; larger sorts need a context (sph_create), which allocates",
                            (long long)n, (long long)ST_MAX_N);
  if (n == 0) return SPH_OK;
  if (!key || !key_sorted || !perm)
    return static_sort_fail(SPH_E_BADARG, errmsg, errmsg_bytes, "sph_sort_keys_static: null key, key_sorted or perm pointer");
  if (key == key_sorted || key == perm || key_sorted == perm)
    return static_sort_fail(SPH_E_BADARG, errmsg, errmsg_bytes, "sph_sort_keys_static: key, key_sorted and perm must be three different arrays");

  uint32_t* ws = nullptr;
  cudaError_t e = sort_scratch_on_current_device(&ws);
  if (e != cudaSuccess) {
    cudaGetLastError();
    return static_sort_fail(SPH_E_CUDA, errmsg, errmsg_bytes, "sph_sort_keys_static: cudaGetSymbolAddress(work space): %s",
                            cudaGetErrorString(e));
  }
  cudaStream_t s = (cudaStream_t)cuda_stream;
  uint32_t* tmp_key = ws + ST_OFF_KEY;
  uint32_t* tmp_idx = ws + ST_OFF_IDX;
  uint32_t* block_hist = ws + ST_OFF_HIST;
  uint32_t* digit_total = ws + ST_OFF_TOTAL;

  const uint32_t nblocks = (uint32_t)((n + RS_TILE - 1) / RS_TILE);
  const int passes = (key_bits + 7) / 8;
  // The work space still holds what the previous call left.  Only the digit totals are accumulated into (atomicAdd in
  // k_rs_hist) and have to start at zero; the histograms and the ping-pong buffers are fully written before being read.
  e = cudaMemsetAsync(digit_total, 0, sizeof(uint32_t) * RS_RADIX * 4, s);
  // Pass p writes to the caller's arrays when an even number of passes follow it, else to the work space, so the last
  // pass always lands in (key_sorted, perm) and the caller's input is only ever read.
  const uint32_t *kin = key, *iin = nullptr;
  for (int p = 0; p < passes && e == cudaSuccess; p++) {
    const bool to_caller = ((passes - 1 - p) & 1) == 0;
    uint32_t* kout = to_caller ? key_sorted : tmp_key;
    uint32_t* iout = to_caller ? perm : tmp_idx;
    const int shift = 8 * p;
    k_rs_hist<<<nblocks, RS_THREADS, 0, s>>>(kin, n, shift, nblocks, block_hist, digit_total + p * RS_RADIX);
    k_rs_scan<<<RS_RADIX, RS_THREADS, 0, s>>>(block_hist, nblocks, digit_total + p * RS_RADIX);
    k_rs_scatter<<<nblocks, RS_THREADS, 0, s>>>(kin, iin, n, shift, nblocks, block_hist, kout, iout, p == 0);
    kin = kout;
    iin = iout;
    e = cudaGetLastError();
  }
  if (e != cudaSuccess)
    return static_sort_fail(SPH_E_CUDA, errmsg, errmsg_bytes, "sph_sort_keys_static: %s", cudaGetErrorString(e));
  return SPH_OK;
}
