// Particle interaction (PI) task, "quad" kernel for sm_100a: 3-D, cells of size 2h (cell_div = 1).
//
// A persistent CTA (one per SM) takes 2x2x2-cell tiles from a device-built list of non-empty tiles and stages each
// tile plus a one-cell halo in shared memory with exact tile-centred coordinates (C1/C2 hold bit for bit).  The
// work of a warp is organised so that every shared-memory access of the hot loops is bank-conflict free and the
// pair arithmetic runs on packed FP32x2 instructions (FFMA2/FADD2/FMUL2, new on sm_100):
//
//   a-group : 8 particles a of one cell = 4 quarter-warps x 2.  Quarter-warp q owns the pair (a_2q, a_2q+1);
//             its 8 lanes r = 0..7 own the candidates b whose staged index is congruent to r modulo 8.
//   T phase : (test) lane (q, r) walks the candidate rows 16 candidates per step: one LDS.128 brings the
//             half-precision test records of candidates 16g+r and 16g+r+8 (packed as half2), three HFMA2 and
//             one HSET2 per a evaluate the expanded-form prefilter |b|^2 - 2 a.b < R^2 + margin - |a|^2 for
//             both candidates at once.  The prefilter is conservative (margin > its rounding error, DESIGN.md
//             5.2); the bits of both a are OR-ed into one 32-bit word per 16 steps; non-empty words go to a pool
//             per quarter-warp in shared memory.
//   P phase : (pair) the lanes of a quarter-warp claim the pool words dynamically, in (word, residue) order, so
//             the 8 records loaded by a quarter-warp in one step lie in 8 different bank groups (two conflict-free
//             LDS.128 per popped b) while the work stays balanced.  Every popped b is evaluated against BOTH a of
//             the lane with packed FP32x2 arithmetic, b entering as a broadcast scalar operand.  The exact
//             canonical predicate C2 (fp32, individually rounded) decides membership; a b that is a neighbour
//             of only one of the two a contributes exactly 0 to the other (the kernel weight is clamped at 0).
//   reduce  : the partial sums of the 8 lanes of a quarter-warp are combined with 3 butterfly shuffles
//             (fixed order, deterministic) and lane r = 0 writes the two results.
//
// What is kept from the paper: cell-linked list, particles sorted by cell, fp32 cell-relative positions
// (PAPER.md:558, 572).  What differs: the thread-per-particle loop with a branch per candidate.
#include <cuda_fp16.h>

#include "pi_common.cuh"

namespace {

constexpr int QT = 2;                     // tile: QT^3 centre cells
constexpr int QS = QT + 2;                // staged cells per axis
constexpr int QNCELL = QS * QS * QS;      // 64 staged cells per type block
constexpr int QNR = 2 * QNCELL;           // staged ranges: block 0 = boundary, block 1 = fluid
constexpr int QNSEG = 2 * QT * QT * QT;   // a-segments: (block, centre cell)
constexpr int QCAP = 64;                  // pool entries (non-empty words) per quarter-warp per round
constexpr int QB = 4;                     // T-phase steps whose loads are issued together
constexpr float Q_MARGIN = 0.03f;         // prefilter slack in r2u, > worst-case half-precision error
constexpr float Q_FAR = 100.0f;           // coordinate of the dummy record (never within the support)

// offset of the staged range of row k = (dz + 1) * 3 + (dy + 1) relative to the row dy = dz = 0
__constant__ int c_rowoff[9] = {-QS * QS - QS, -QS * QS, -QS * QS + QS, -QS, 0, QS, QS * QS - QS, QS * QS, QS * QS + QS};

__device__ __forceinline__ int qrange(int blk, int ix, int iy, int iz) {   // staged indices, 0-based
  return ((blk * QS + iz) * QS + iy) * QS + ix;
}

struct QSmem {
  float4* rpos;       // (x, y, z, rho): exact tile-centred coordinates + density
  float4* rvel;       // (vx, vy, vz, P / rho)
  uint4* tst;         // half2-packed test records: entry g*8 + r = candidates 16g+r (low halves) and 16g+r+8
  uint2* bm;          // [warp][4][QCAP] pools: (bitmap word, byte address of the record of its bit 0)
  uint32_t* soff;     // QNR + 1
  uint32_t* gstart;   // QNR
  uint32_t* seg;      // [0] group counter, [1..QNSEG+1] a-group prefix
};

__device__ __forceinline__ uint32_t h2_as_u32(__half2 h) { return *reinterpret_cast<uint32_t*>(&h); }
__device__ __forceinline__ __half2 u32_as_h2(uint32_t u) { return *reinterpret_cast<__half2*>(&u); }

// Packed FP32x2 values live in 64-bit registers (an aligned register pair), so that ptxas keeps the two halves
// together and needs no moves around FADD2 / FMUL2 / FFMA2.  A scalar operand is written as the pair {s, s};
// ptxas folds it into the instruction's scalar-broadcast operand form.
typedef unsigned long long f2;
__device__ __forceinline__ f2 f2_pack(float lo, float hi) {
  f2 r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
  return r;
}
__device__ __forceinline__ f2 f2_bc(float s) { return f2_pack(s, s); }
// Pack two scalars through a packed add of +0 (exact up to the sign of zero), so that the result is born in an aligned register pair
// and stays there (a plain mov.b64 is re-materialised by ptxas with two moves at every use).
__device__ __forceinline__ f2 f2_pack_pinned(float lo, float hi) {
  f2 r;
  asm volatile("{.reg .b64 t, o; mov.b64 t, {%1, %2}; mov.b64 o, {%3, %3}; add.rn.f32x2 %0, t, o;}"
               : "=l"(r) : "f"(lo), "f"(hi), "f"(0.0f));
  return r;
}
__device__ __forceinline__ float f2_lo(f2 v) {
  float lo, hi;
  asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
  return lo;
}
__device__ __forceinline__ float f2_hi(f2 v) {
  float lo, hi;
  asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
  return hi;
}
__device__ __forceinline__ float f_lt(float a, float b) {   // 1.0f if a < b else 0.0f
  float r;
  asm("set.lt.f32.f32 %0, %1, %2;" : "=f"(r) : "f"(a), "f"(b));
  return r;
}
__device__ __forceinline__ f2 f2_add(f2 a, f2 b) {
  f2 r;
  asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
  return r;
}
__device__ __forceinline__ f2 f2_mul(f2 a, f2 b) {
  f2 r;
  asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
  return r;
}
__device__ __forceinline__ f2 f2_fma(f2 a, f2 b, f2 c) {
  f2 r;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
  return r;
}
// acc += a * b, in place (input and output tied to one register pair: no moves around loop-carried sums)
__device__ __forceinline__ void f2_fma_acc(f2 a, f2 b, f2& acc) {
  asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(acc) : "l"(a), "l"(b));
}
__device__ __forceinline__ void f2_add_acc(f2 a, f2& acc) {
  asm("add.rn.f32x2 %0, %0, %1;" : "+l"(acc) : "l"(a));
}

// Packed state of the two particles a of a lane.
struct PairA {
  f2 x, y, z, vx, vy, vz, rho, inv_rho, kap;   // kap = P / rho
};
struct PairAcc2 {
  f2 sx, sy, sz, sc, sd;
  float visc0, visc1;
  f2 nb;              // neighbour counts, kept as floats (exact integers)
  f2 lx, ly, lz;      // laminar viscosity sums, Eq. 23 (LAM instantiations only)
};

// One popped candidate b against both a of the lane (Eq. 15, 17-18, 21-22, 36), branch free.  A b outside the
// support of a_h (prefilter false positive, neighbour of the other a only, or the dummy record) gets weight 0:
// w = max(1 - q/2, 0).  nb counts the exact canonical predicate C2.  pb = (x, y, z, rho_b), vb = (v_b, P_b/rho_b).
// DDT: this b enters the density diffusion term (A4).
template <bool A_FLUID, bool DDT, bool LAM, bool FOURT>
__device__ __forceinline__ void pair2(const DevConsts& C, const PairA& a, const float4 pb, const float4 vb,
                                      PairAcc2& A) {
  const f2 dux = f2_add(a.x, f2_bc(-pb.x));   // exact (C1)
  const f2 duy = f2_add(a.y, f2_bc(-pb.y));
  const f2 duz = f2_add(a.z, f2_bc(-pb.z));
  f2 r2 = f2_mul(dux, dux);                   // C2: individually rounded
  r2 = f2_fma(duy, duy, r2);
  r2 = f2_fma(duz, duz, r2);
  const float r2a = f2_lo(r2), r2b = f2_hi(r2);
  f2_add_acc(f2_pack(f_lt(r2a, C.R2u), f_lt(r2b, C.R2u)), A.nb);   // exact: counts stay far below 2^24
  f2 w = f2_fma(f2_pack(fast_sqrt(r2a), fast_sqrt(r2b)), f2_bc(-C.qscale), f2_bc(1.0f));   // 1 - q/2   (Eq. 11)
  w = f2_pack(fmaxf(f2_lo(w), 0.f), fmaxf(f2_hi(w), 0.f));
  const f2 w3 = f2_mul(f2_mul(w, w), w);      // grad_a W_ab = Cf w^3 cs du
  const float inv_rho_b = fast_rcp(pb.w);
  const f2 dvx = f2_add(a.vx, f2_bc(-vb.x));
  const f2 dvy = f2_add(a.vy, f2_bc(-vb.y));
  const f2 dvz = f2_add(a.vz, f2_bc(-vb.z));
  f2 dot = f2_mul(dvx, dux);                  // v_ab . r_ab / cs
  dot = f2_fma(dvy, duy, dot);
  dot = f2_fma(dvz, duz, dot);
  const f2 gb = f2_mul(w3, f2_bc(inv_rho_b));
  f2_fma_acc(gb, dot, A.sc);
  if (A_FLUID) {
    if (DDT) {
      f2 drho = f2_add(a.rho, f2_bc(-pb.w));
      if (FOURT) {   // Eq. 19-20 (A23): minus rho^H_ab = e (k0 + e (k1 + e (k2 + e k3))), e = c_hyd . du
        f2 e = f2_mul(dux, f2_bc(C.c_hyd[0]));
        e = f2_fma(duy, f2_bc(C.c_hyd[1]), e);
        e = f2_fma(duz, f2_bc(C.c_hyd[2]), e);
        f2 h = f2_fma(e, f2_bc(C.hyd_k[3]), f2_bc(C.hyd_k[2]));
        h = f2_fma(e, h, f2_bc(C.hyd_k[1]));
        h = f2_fma(e, h, f2_bc(C.hyd_k[0]));
        drho = f2_fma(f2_mul(e, f2_bc(-1.0f)), h, drho);
      }
      f2_fma_acc(gb, drho, A.sd);
    }
    const f2 rs = f2_add(a.rho, f2_bc(pb.w));
    const f2 den = f2_mul(f2_add(r2, f2_bc(C.eta2u)), rs);
    const f2 xinv = f2_pack(fast_rcp(f2_lo(den)), fast_rcp(f2_hi(den)));
    const f2 y = f2_mul(dot, xinv);                       // dot / ((r2 + eta2) rs)
    if (LAM) {                                            // Eq. 23: sum w^3 r2u / ((r2u + eta2u) rs) dv
      const f2 lam = f2_mul(f2_mul(w3, r2), xinv);
      f2_fma_acc(lam, dvx, A.lx);
      f2_fma_acc(lam, dvy, A.ly);
      f2_fma_acc(lam, dvz, A.lz);
    }
    const f2 mu = f2_mul(y, rs);                          // mu_ab / c_mu   (Eq. 21, A12)
    A.visc0 = fmaxf(A.visc0, fabsf(f2_lo(mu)));
    A.visc1 = fmaxf(A.visc1, fabsf(f2_hi(mu)));
    const f2 t = f2_pack(fminf(f2_lo(y), 0.f), fminf(f2_hi(y), 0.f));   // approaching pairs only (Eq. 21)
    // (Pa + Pb) / (rho_a rho_b) = kap_a / rho_b + kap_b / rho_a
    const f2 pp = f2_fma(a.kap, f2_bc(inv_rho_b), f2_mul(a.inv_rho, f2_bc(vb.w)));
    const f2 coef = f2_mul(w3, f2_fma(f2_bc(C.c_pi), t, pp));
    f2_fma_acc(coef, dux, A.sx);
    f2_fma_acc(coef, duy, A.sy);
    f2_fma_acc(coef, duz, A.sz);
  }
}

// Predicated 64-bit shared-memory load into an existing register pair (nothing happens if !p).
__device__ __forceinline__ void lds64_if(bool p, unsigned saddr, unsigned& x, unsigned& y) {
  asm volatile("{.reg .pred q; setp.ne.u32 q, %2, 0; @q ld.shared.v2.u32 {%0, %1}, [%3];}"
               : "+r"(x), "+r"(y) : "r"((unsigned)p), "r"(saddr));
}

// Sum over the 8 lanes of a quarter-warp (butterfly, fixed order).
__device__ __forceinline__ float qsum(float v) {
  v += __shfl_xor_sync(0xffffffffu, v, 1);
  v += __shfl_xor_sync(0xffffffffu, v, 2);
  v += __shfl_xor_sync(0xffffffffu, v, 4);
  return v;
}
__device__ __forceinline__ float qmax(float v) {
  v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, 1));
  v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, 2));
  v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, 4));
  return v;
}
__device__ __forceinline__ unsigned qsumu(unsigned v) {
  v += __shfl_xor_sync(0xffffffffu, v, 1);
  v += __shfl_xor_sync(0xffffffffu, v, 2);
  v += __shfl_xor_sync(0xffffffffu, v, 4);
  return v;
}

// One a-group: up to 8 particles a of the centre cell (cx, cy, cz) (tile-local, 0..QT-1), type block
// A_FLUID ? 1 : 0, staged at [cell_start + 8*grp, ...).  bmw is this warp's pool area ([4][QCAP] uint2).
template <bool A_FLUID, bool LAM, bool FOURT>
__device__ __forceinline__ void process_group(const DevConsts& C, const PiArgs& A, const QSmem& S, uint2* bmw, int cx,
                                              int cy, int cz, unsigned cell_start, unsigned n_a, unsigned grp,
                                              unsigned total, float& f2max, float& viscmax, unsigned int& nbsum) {
  const int lane = threadIdx.x & 31, q = lane >> 3, r = lane & 7;
  const unsigned t0 = grp * 8 + 2 * q, t1 = t0 + 1;
  const bool act0 = t0 < n_a, act1 = t1 < n_a;
  const unsigned ja0 = cell_start + (act0 ? t0 : 0), ja1 = cell_start + (act1 ? t1 : 0);

  // ---- state of the two a of this lane (inactive: far away, never accepted) ----
  PairA a;
  __half2 nx0, ny0, nz0, th0, nx1, ny1, nz1, th1;
  float rho_a0, rho_a1;
  {
    float4 p0 = S.rpos[ja0], v0 = S.rvel[ja0], p1 = S.rpos[ja1], v1 = S.rvel[ja1];
    if (!act0) { p0 = make_float4(-Q_FAR, -Q_FAR, -Q_FAR, 1.f); v0 = make_float4(0.f, 0.f, 0.f, 0.f); }
    if (!act1) { p1 = make_float4(-Q_FAR, -Q_FAR, -Q_FAR, 1.f); v1 = make_float4(0.f, 0.f, 0.f, 0.f); }
    a.x = f2_pack_pinned(p0.x, p1.x); a.y = f2_pack_pinned(p0.y, p1.y); a.z = f2_pack_pinned(p0.z, p1.z);
    a.rho = f2_pack_pinned(p0.w, p1.w);
    rho_a0 = p0.w; rho_a1 = p1.w;
    a.inv_rho = f2_pack_pinned(fast_rcp(p0.w), fast_rcp(p1.w));
    a.vx = f2_pack_pinned(v0.x, v1.x); a.vy = f2_pack_pinned(v0.y, v1.y); a.vz = f2_pack_pinned(v0.z, v1.z);
    a.kap = f2_pack_pinned(v0.w, v1.w);
    // prefilter operands (half precision): s = |b|^2 - 2 a.b  <  thr = R2u + margin - |a|^2
    const float thr0 = act0 ? (C.R2u + Q_MARGIN) - fmaf(p0.z, p0.z, fmaf(p0.y, p0.y, p0.x * p0.x)) : -60000.f;
    const float thr1 = act1 ? (C.R2u + Q_MARGIN) - fmaf(p1.z, p1.z, fmaf(p1.y, p1.y, p1.x * p1.x)) : -60000.f;
    nx0 = __float2half2_rn(act0 ? -2.f * p0.x : 0.f); ny0 = __float2half2_rn(act0 ? -2.f * p0.y : 0.f);
    nz0 = __float2half2_rn(act0 ? -2.f * p0.z : 0.f); th0 = __half2half2(__float2half_ru(thr0));
    nx1 = __float2half2_rn(act1 ? -2.f * p1.x : 0.f); ny1 = __float2half2_rn(act1 ? -2.f * p1.y : 0.f);
    nz1 = __float2half2_rn(act1 ? -2.f * p1.z : 0.f); th1 = __half2half2(__float2half_ru(thr1));
  }
  PairAcc2 acc;
  acc.sx = acc.sy = acc.sz = acc.sc = acc.sd = acc.nb = acc.lx = acc.ly = acc.lz = f2_pack(0.f, 0.f);
  acc.visc0 = acc.visc1 = 0.f;

  // Rounds are homogeneous in the type block of b: fluid a sweeps the 9 boundary-block rows first (diffusion
  // term only if ddt_over_boundary, A4), then the 9 fluid rows; boundary a sweeps the fluid rows only (Eq. 36).
  const int nruns = A_FLUID ? 18 : 9;
  int ri = (A_FLUID && S.soff[QNCELL] == 0u) ? 9 : 0;   // no boundary particle staged: skip their 9 rows
  int gw = -1, g_first = 0, g_last = -1;
  unsigned j0 = 0, j1 = 0;
  const unsigned dummy_addr = total * 16u;
  const int row0 = qrange(1, cx, 1 + cy, 1 + cz);        // fluid-block range of the cell left of the centre cell
  uint2* bmq = bmw + q * QCAP;                       // pool of this quarter-warp
  const unsigned bmq_s = (unsigned)__cvta_generic_to_shared(bmq);
  const unsigned qsel = 0x4440u | (unsigned)q;           // byte_perm selector: byte q of a ballot
  const unsigned lt_mask = (1u << r) - 1u;               // lanes of the quarter-warp below this one

  while (ri < nruns) {
    // ================= T phase: fill the pools (until one of them would overflow) =================
    const int ri_end = (A_FLUID && ri < 9) ? 9 : nruns;
    const bool ddt_round = !(A_FLUID && ri < 9 && !C.ddt_over_boundary);
    int nw = 0;
    unsigned npool = 0;
    while (ri < ri_end) {
      if (gw < 0) {   // open run ri
        // row ri of the stencil: cells (cx-1 .. cx+1, cy+dy, cz+dz) of one type block are one contiguous range
        const int row = ((A_FLUID && ri < 9) ? row0 - QNCELL : row0) + c_rowoff[(A_FLUID && ri >= 9) ? ri - 9 : ri];
        j0 = S.soff[row];
        j1 = S.soff[row + 3];
        if (j1 <= j0) { ri++; continue; }
        g_first = (int)(j0 >> 4);
        g_last = (int)((j1 - 1) >> 4);
        gw = g_first;
      }
      const int nstep = min(16, g_last - gw + 1);
      const uint4* tp = S.tst + gw * 8 + r;
      unsigned u = 0;
      // 16 steps in batches of QB: the loads of a batch are issued together, so that they overlap the
      // arithmetic of the previous batch.  Steps beyond nstep read whatever follows (the test records are
      // followed by the pools in shared memory, so the addresses stay valid); their bits are masked below.
#pragma unroll
      for (int b0 = 0; b0 < 16; b0 += QB) {
        if (b0 < nstep) {
          uint4 t[QB];
#pragma unroll
          for (int i = 0; i < QB; i++) t[i] = tp[(b0 + i) * 8];   // may run past the run (never past the pools)
#pragma unroll
          for (int i = 0; i < QB; i++) {
            const __half2 bx = u32_as_h2(t[i].x), by = u32_as_h2(t[i].y), bz = u32_as_h2(t[i].z), bw = u32_as_h2(t[i].w);
            const __half2 s0 = __hfma2(nz0, bz, __hfma2(ny0, by, __hfma2(nx0, bx, bw)));
            const __half2 s1 = __hfma2(nz1, bz, __hfma2(ny1, by, __hfma2(nx1, bx, bw)));
            const unsigned m = __hlt2_mask(s0, th0) | __hlt2_mask(s1, th1);
            u |= m & (0x00010001u << (b0 + i));
          }
        }
      }
      // keep the candidates that lie inside the run [j0, j1): bit i (low half) is candidate c + 16 i, bit
      // 16 + i is candidate c + 8 + 16 i with c = 16 gw + r.  Branch free; this also drops the steps >= nstep.
      {
        const int c = gw * 16 + r;
        const int lo0 = max(((int)j0 - c + 15) >> 4, 0), lo1 = min(max(((int)j1 - c + 15) >> 4, 0), 16);
        const int hi0 = max(((int)j0 - c + 7) >> 4, 0), hi1 = min(max(((int)j1 - c + 7) >> 4, 0), 16);
        const unsigned mlo = (0xffffu >> (16 - lo1)) & (0xffffu << lo0);
        const unsigned mhi = (0xffffu >> (16 - hi1)) & (0xffffu << hi0);
        u &= (mlo & 0xffffu) | (mhi << 16);
      }
      // non-empty words go to the pool of this quarter-warp, compacted in (word, residue) order, together
      // with the byte address of the record of bit 0 (bit p -> + 256 (p & 15) + 128 (p >> 4))
      {
        const unsigned nzq = __byte_perm(__ballot_sync(0xffffffffu, u != 0u), 0u, qsel);
        // a pool would overflow: run the P phase first; this word is recomputed in the next round (rare)
        if (__any_sync(0xffffffffu, npool + (unsigned)__popc(nzq) > (unsigned)QCAP)) break;
        if (u != 0u)
          bmq[npool + (unsigned)__popc(nzq & lt_mask)] = make_uint2(u, ((unsigned)gw * 16u + (unsigned)r) * 16u);
        npool += (unsigned)__popc(nzq);
      }
      nw++;
      gw += 16;
      if (gw > g_last) { ri++; gw = -1; }
    }
    if (nw == 0) continue;
    __syncwarp();

    // ================= P phase: the 8 lanes of a quarter-warp claim words from their pool =================
    // Words are claimed in pool order, so the 8 words in flight are (nearly always) 8 consecutive pool entries
    // = 8 different residues: the record loads stay bank-conflict free while the work is balanced dynamically.
    const unsigned char* rp = reinterpret_cast<const unsigned char*>(S.rpos);
    const unsigned char* rv = reinterpret_cast<const unsigned char*>(S.rvel);
    unsigned cur = 0, base = 0, next = 8;
    if ((unsigned)r < npool) {
      const uint2 e = bmq[r];
      cur = e.x;
      base = e.y;
    }
    // one step: claim (lanes whose word is used up take the next pool entries in lane order), pop the highest
    // set bit and issue the loads of its record; then evaluate the record fetched by the previous step
    // (software pipeline, two steps per loop trip so that records and accumulators ping-pong without moves).
    // Pool words are non-empty, so "no word" means "pool used up"; a lane without work loads the dummy record.
#define Q_FETCH(PB, VB)                                                                                \
  {                                                                                                    \
    const bool need = cur == 0u;                                                                       \
    const unsigned nq = __byte_perm(__ballot_sync(0xffffffffu, need), 0u, qsel);                       \
    const unsigned ei = next + (unsigned)__popc(nq & lt_mask);                                         \
    next += (unsigned)__popc(nq);                                                                      \
    lds64_if(need && ei < npool, bmq_s + ei * 8u, cur, base);                                          \
    more = __any_sync(0xffffffffu, cur != 0u);                                                         \
    const unsigned p = 31u - (unsigned)__clz((int)cur); /* cur == 0 -> p = 0xffffffff (unused) */      \
    const unsigned addr = cur != 0u ? base + ((p & 15u) << 8) + ((p >> 4) << 7) : dummy_addr;          \
    cur &= ~(1u << (p & 31u));                                                                         \
    PB = *reinterpret_cast<const float4*>(rp + addr);                                                  \
    VB = *reinterpret_cast<const float4*>(rv + addr);                                                  \
  }
#define Q_LOOP(DDT)                                                                                    \
  {                                                                                                    \
    float4 pbA, vbA, pbB, vbB;                                                                         \
    bool more;                                                                                         \
    Q_FETCH(pbA, vbA)                                                                                  \
    while (more) { /* single exit: at most one surplus evaluation of dummy records per round */        \
      Q_FETCH(pbB, vbB)                                                                                \
      pair2<A_FLUID, DDT, LAM, FOURT>(C, a, pbA, vbA, acc);                                                        \
      Q_FETCH(pbA, vbA)                                                                                \
      pair2<A_FLUID, DDT, LAM, FOURT>(C, a, pbB, vbB, acc);                                                        \
    }                                                                                                  \
  }
    if (ddt_round) Q_LOOP(true) else Q_LOOP(false)
#undef Q_LOOP
#undef Q_FETCH
    __syncwarp();
  }

  // ---- combine the 8 lanes of each quarter-warp; lane r = 0 writes both particles ----
  PairAcc r0 = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f}, r1 = r0;
  r0.sc = qsum(f2_lo(acc.sc)); r1.sc = qsum(f2_hi(acc.sc));
  const unsigned nb0 = (unsigned)qsum(f2_lo(acc.nb)), nb1 = (unsigned)qsum(f2_hi(acc.nb));
  if (A_FLUID) {
    r0.sx = qsum(f2_lo(acc.sx)); r1.sx = qsum(f2_hi(acc.sx));
    r0.sy = qsum(f2_lo(acc.sy)); r1.sy = qsum(f2_hi(acc.sy));
    r0.sz = qsum(f2_lo(acc.sz)); r1.sz = qsum(f2_hi(acc.sz));
    r0.sd = qsum(f2_lo(acc.sd)); r1.sd = qsum(f2_hi(acc.sd));
    r0.visc = qmax(acc.visc0); r1.visc = qmax(acc.visc1);
    if (LAM) {
      r0.lx = qsum(f2_lo(acc.lx)); r1.lx = qsum(f2_hi(acc.lx));
      r0.ly = qsum(f2_lo(acc.ly)); r1.ly = qsum(f2_hi(acc.ly));
      r0.lz = qsum(f2_lo(acc.lz)); r1.lz = qsum(f2_hi(acc.lz));
    }
  }
  if (r == 0) {
    const int ra = qrange(A_FLUID ? 1 : 0, 1 + cx, 1 + cy, 1 + cz);
    const unsigned gbase = S.gstart[ra] - S.soff[ra];
#pragma unroll
    for (int h = 0; h < 2; h++) {
      if (h == 0 ? act0 : act1) {
        const PairAcc& pa1 = h ? r1 : r0;
        unsigned nb = h ? nb1 : nb0;
        if (A_FLUID) nb -= 1u;   // the particle itself passed the test at r = 0 and contributed exactly 0 (A17)
        const unsigned ga = gbase + (h ? ja1 : ja0);
        const float4 out = finish_particle(C, A_FLUID, h ? rho_a1 : rho_a0, pa1);
        A.acc[ga] = out;
        if (A.nbcount) A.nbcount[ga] = nb;
        if (A_FLUID) f2max = fmaxf(f2max, fmaf(out.x, out.x, fmaf(out.y, out.y, out.z * out.z)));
        viscmax = fmaxf(viscmax, pa1.visc * C.c_mu);
        nbsum += nb;
      }
    }
  }
}

// Active-tile list: most tiles of a dam break are air.  A tile is active if its centre cells hold a particle;
// x-adjacent cells are adjacent keys, so one (block, cy, cz) row of centre cells is one cellstart difference.
// ws[0] = number of active tiles, ws[1] = next tile to take (both zeroed before the launch), ws[4..] = tile ids.
__global__ void __launch_bounds__(256) k_quad_tiles(DevConsts C, const uint32_t* __restrict__ cellstart, int ntx, int nty,
                                                    int ntiles, uint32_t* ws) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= ntiles) return;
  const int ox = (t % ntx) * QT, oy = ((t / ntx) % nty) * QT, oz = (t / (ntx * nty)) * QT;
  const uint32_t w = (uint32_t)min(QT, C.nc[0] - ox);
  bool any = false;
  for (int blk = 0; blk < 2; blk++)
    for (int cz = oz; cz < min(oz + QT, C.nc[2]); cz++)
      for (int cy = oy; cy < min(oy + QT, C.nc[1]); cy++) {
        const uint32_t key = (uint32_t)blk * C.ncells + (uint32_t)ox +
                             (uint32_t)C.nc[0] * ((uint32_t)cy + (uint32_t)C.nc[1] * (uint32_t)cz);
        any = any || cellstart[key + w] != cellstart[key];
      }
  if (any) ws[4 + atomicAdd(&ws[0], 1u)] = (uint32_t)t;
}

// Persistent kernel: one CTA per SM takes active tiles from the list until it is used up.
template <int NT, int NMAX, bool LAM, bool FOURT>
__global__ void __launch_bounds__(NT, 1) k_pi_quad(DevConsts C, PiArgs A, int ntx, int nty) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  constexpr int NWARP = NT / 32;
  QSmem S;
  S.rpos = reinterpret_cast<float4*>(smem_raw);
  S.rvel = S.rpos + NMAX;
  S.tst = reinterpret_cast<uint4*>(S.rvel + NMAX);
  S.bm = reinterpret_cast<uint2*>(S.tst + (NMAX / 16) * 8);
  S.soff = reinterpret_cast<uint32_t*>(S.bm + NWARP * 4 * QCAP);
  S.gstart = S.soff + (QNR + 1);
  S.seg = S.gstart + QNR;
  __shared__ uint32_t s_cnt[QNR];
  __shared__ uint32_t s_tile;

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const uint32_t n_active = A.tile_ws[0];
  float f2max = 0.f, viscmax = 0.f;
  unsigned int nbsum = 0;

 for (;;) {
  __syncthreads();                                  // every warp is done with the previous tile's shared memory
  if (tid == 0) s_tile = atomicAdd(&A.tile_ws[1], 1u);
  __syncthreads();
  if (s_tile >= n_active) break;
  const int tile = (int)A.tile_ws[4 + s_tile];
  const int tx = tile % ntx, ty = (tile / ntx) % nty, tz = tile / (ntx * nty);
  const int ox = tx * QT, oy = ty * QT, oz = tz * QT;

  // A tile whose staged set does not fit in shared memory (compressed or crowded regions) is processed as two
  // half tiles in z: part 1 = centre cells cz = 0 with the staged layers iz = 0..2, part 2 = cz = 1 with
  // iz = 1..3 (the other layer counts as empty).  Only a half that still does not fit takes the global-gather path.
  for (int part = 0; part < 3; part++) {
  const int zlo = part == 2 ? 1 : 0, zhi = part == 1 ? 2 : 3;        // staged layers in use
  const int czlo = part == 2 ? 1 : 0, czhi = part == 1 ? 0 : 1;      // centre layers computed
  if (part) __syncthreads();

  // 1. global ranges of the staged cells (both type blocks)
  for (int rr = tid; rr < QNR; rr += NT) {
    const int blk = rr / QNCELL, c = rr % QNCELL;
    const int ix = c % QS, iy = (c / QS) % QS, iz = c / (QS * QS);
    int g[3] = {ox + ix - 1, oy + iy - 1, oz + iz - 1};
    bool valid = iz >= zlo && iz <= zhi;
#pragma unroll
    for (int k = 0; k < 3; k++) {
      if (C.per[k]) g[k] = (g[k] + C.nc[k]) % C.nc[k];
      else if (g[k] < 0 || g[k] >= C.nc[k]) valid = false;
    }
    uint32_t g0 = 0, n = 0;
    if (valid) {
      const uint32_t key = (uint32_t)blk * C.ncells + (uint32_t)g[0] +
                           (uint32_t)C.nc[0] * ((uint32_t)g[1] + (uint32_t)C.nc[1] * (uint32_t)g[2]);
      g0 = A.cellstart[key];
      n = A.cellstart[key + 1] - g0;
    }
    s_cnt[rr] = n;
    S.gstart[rr] = g0;
  }
  __syncthreads();
  if (warp == 0) {   // exclusive scan of the QNR counts
    constexpr int PER = (QNR + 31) / 32;
    uint32_t v[PER], sum = 0;
#pragma unroll
    for (int i = 0; i < PER; i++) {
      const int rr = lane * PER + i;
      v[i] = rr < QNR ? s_cnt[rr] : 0u;
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
      const int rr = lane * PER + i;
      if (rr < QNR) S.soff[rr] = run;
      run += v[i];
    }
    if (lane == 31) S.soff[QNR] = inc;
  }
  __syncthreads();

  // a-segments (block, centre cell) and the a-group prefix for dynamic scheduling
  const int vx = min(QT, C.nc[0] - ox), vy = min(QT, C.nc[1] - oy), vz = min(QT, C.nc[2] - oz);
  if (tid == 0) {
    uint32_t run = 0;
    for (int s = 0; s < QNSEG; s++) {
      const int blk = 1 - (s >> 3), cz = (s >> 2) & 1, cy = (s >> 1) & 1, cx = s & 1;
      uint32_t n = 0;
      if (cx < vx && cy < vy && cz < vz && cz >= czlo && cz <= czhi) n = s_cnt[qrange(blk, 1 + cx, 1 + cy, 1 + cz)];
      S.seg[1 + s] = run;
      run += (n + 7) / 8;
    }
    S.seg[1 + QNSEG] = run;
    S.seg[0] = 0;
  }
  __syncthreads();
  const uint32_t ngroups = S.seg[1 + QNSEG];
  if (ngroups == 0) {                             // nothing to compute in this (half) tile
    if (part == 0) break;
    continue;
  }
  const uint32_t total = S.soff[QNR];

  if (total + 1 > (uint32_t)NMAX) {
    if (part == 0) continue;                      // retry as two half tiles
    // even the half tile does not fit (very crowded cells): per-particle global gather
    for (int s = 0; s < QNSEG; s++) {
      const int blk = 1 - (s >> 3), cz = (s >> 2) & 1, cy = (s >> 1) & 1, cx = s & 1;
      if (cx >= vx || cy >= vy || cz >= vz || cz < czlo || cz > czhi) continue;
      const int rr = qrange(blk, 1 + cx, 1 + cy, 1 + cz);
      const uint32_t g0 = S.gstart[rr], len = s_cnt[rr];
      for (uint32_t i = tid; i < len; i += NT) gather_one<3>(C, A, g0 + i, blk == 1, f2max, viscmax, nbsum);
    }
    continue;
  }

  // 2. stage particles with tile-centred coordinates: u + integer cell offset - QT/2.  Exact: every value is a
  //    multiple of 2^-22 with magnitude <= 2, so all differences are exact in fp32 (C1/C2).
  for (int rr = warp; rr < QNR; rr += NWARP) {
    const uint32_t n = s_cnt[rr];
    if (n == 0) continue;
    const int c = rr % QNCELL;
    const float fx = (float)(c % QS - 1) - 0.5f * QT, fy = (float)((c / QS) % QS - 1) - 0.5f * QT,
                fz = (float)(c / (QS * QS) - 1) - 0.5f * QT;
    const uint32_t g0 = S.gstart[rr], d0 = S.soff[rr];
    for (uint32_t i = lane; i < n; i += 32) {
      const float4 p = A.posu[g0 + i];
      const float4 v = A.velp[g0 + i];
      S.rpos[d0 + i] = make_float4(p.x + fx, p.y + fy, p.z + fz, p.w);
      S.rvel[d0 + i] = make_float4(v.x, v.y, v.z, __fdiv_rn(v.w, p.w));   // (v, P / rho)
    }
  }
  if (tid == 0) {   // dummy record: popped by lanes that have run out of work, never within any support
    S.rpos[total] = make_float4(Q_FAR, Q_FAR, Q_FAR, 1.0f);
    S.rvel[total] = make_float4(0.f, 0.f, 0.f, 0.f);
  }
  __syncthreads();
  // 3. half-precision test records, two candidates per half2: entry g*8 + r <- candidates 16g + r, 16g + r + 8
  {
    const uint32_t nent = ((total + 15) / 16) * 8;
    for (uint32_t e = tid; e < nent; e += NT) {
      const uint32_t c0 = (e >> 3) * 16 + (e & 7), c1 = c0 + 8;
      float4 p0 = make_float4(0.f, 0.f, 0.f, 0.f), p1 = p0;
      if (c0 < total) p0 = S.rpos[c0];
      if (c1 < total) p1 = S.rpos[c1];
      const __half2 hx = __floats2half2_rn(p0.x, p1.x), hy = __floats2half2_rn(p0.y, p1.y),
                    hz = __floats2half2_rn(p0.z, p1.z);
      const float2 fx = __half22float2(hx), fy = __half22float2(hy), fz = __half22float2(hz);
      float w0 = fmaf(fz.x, fz.x, fmaf(fy.x, fy.x, fx.x * fx.x));   // |b|^2 of the rounded coordinates
      float w1 = fmaf(fz.y, fz.y, fmaf(fy.y, fy.y, fx.y * fx.y));
      if (c0 >= total) w0 = 60000.f;                                 // padding: never accepted
      if (c1 >= total) w1 = 60000.f;
      const __half2 hw = __floats2half2_rn(w0, w1);
      S.tst[e] = make_uint4(h2_as_u32(hx), h2_as_u32(hy), h2_as_u32(hz), h2_as_u32(hw));
    }
  }
  __syncthreads();

  // 4. a-groups, taken dynamically by the warps
  uint2* bmw = S.bm + warp * 4 * QCAP;
  while (true) {
    uint32_t gi = 0;
    if (lane == 0) gi = atomicAdd(&S.seg[0], 1u);
    gi = __shfl_sync(0xffffffffu, gi, 0);
    if (gi >= ngroups) break;
    int s = 0;
    while (s + 1 < QNSEG && gi >= S.seg[1 + s + 1]) s++;
    const int blk = 1 - (s >> 3), cz = (s >> 2) & 1, cy = (s >> 1) & 1, cx = s & 1;
    const int rr = qrange(blk, 1 + cx, 1 + cy, 1 + cz);
    const unsigned cell_start = S.soff[rr], n_a = s_cnt[rr], grp = gi - S.seg[1 + s];
    if (blk == 1) process_group<true, LAM, FOURT>(C, A, S, bmw, cx, cy, cz, cell_start, n_a, grp, total, f2max, viscmax, nbsum);
    else process_group<false, false, false>(C, A, S, bmw, cx, cy, cz, cell_start, n_a, grp, total, f2max, viscmax, nbsum);
  }
  if (part == 0) break;
  }   // parts
 }   // tiles
  reduce_scalars(A.sc, f2max, viscmax, nbsum);
}

template <int NT, int NMAX, bool LAM, bool FOURT>
int launch_quad(const DevConsts& C, const PiArgs& A, cudaStream_t s) {
  const int ntx = (C.nc[0] + QT - 1) / QT, nty = (C.nc[1] + QT - 1) / QT, ntz = (C.nc[2] + QT - 1) / QT;
  constexpr int NWARP = NT / 32;
  const size_t smem = sizeof(float4) * 2 * NMAX + sizeof(uint4) * (NMAX / 16) * 8 +
                      sizeof(uint2) * NWARP * 4 * QCAP + sizeof(uint32_t) * ((QNR + 1) + QNR + (QNSEG + 2));
  static bool configured = false;
  if (!configured) {
    if (cudaFuncSetAttribute(k_pi_quad<NT, NMAX, LAM, FOURT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) !=
        cudaSuccess) {
      cudaGetLastError();
      return -1;
    }
    configured = true;
  }
  const long long ntiles = (long long)ntx * nty * ntz;
  if (ntiles > 0x7fffffffLL || A.tile_ws == nullptr) return -1;
  static int n_sm = 0;
  if (n_sm == 0) {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n_sm <= 0) {
      cudaGetLastError();
      n_sm = 0;
      return -1;
    }
  }
  if (cudaMemsetAsync(A.tile_ws, 0, 4 * sizeof(uint32_t), s) != cudaSuccess) return -1;
  k_quad_tiles<<<(unsigned)((ntiles + 255) / 256), 256, 0, s>>>(C, A.cellstart, ntx, nty, (int)ntiles, A.tile_ws);
  k_pi_quad<NT, NMAX, LAM, FOURT><<<(unsigned)min((long long)n_sm, ntiles), NT, smem, s>>>(C, A, ntx, nty);
  return 0;
}

}  // namespace

size_t pi_quad_workspace_words(const DevConsts& C) {
  const size_t ntx = (C.nc[0] + QT - 1) / QT, nty = (C.nc[1] + QT - 1) / QT, ntz = (C.nc[2] + QT - 1) / QT;
  return 4 + ntx * nty * ntz;
}

// Returns 0 if the quad kernel was launched, -1 if this configuration is not supported (caller falls back to
// the tiled kernel): 3-D, cells of size 2h (27-cell stencil), eta^2 > 0.
int pi_quad(const DevConsts& C, const PiArgs& A, cudaStream_t s) {
  if (A.n == 0) return 0;
  if (C.dim != 3 || C.k != 1) return -1;
  if (!(C.eta2u > 0.f)) return -1;   // the self pair (r = 0) must evaluate to exactly 0, which needs eta^2 > 0
  // the packed Fourtakas term uses the series form of the inverse EOS (exact to fp32 rounding for |e| <= 0.02)
  if (C.ddt_model == 1 && !C.hyd_series_ok) return -1;
  const bool lam = C.visco_model == 1, fourt = C.ddt_model == 1;   // Eq. 23 / Eq. 19-20 instantiations
  if (lam && fourt) return launch_quad<512, 4928, true, true>(C, A, s);
  if (lam) return launch_quad<512, 4928, true, false>(C, A, s);
  if (fourt) return launch_quad<512, 4928, false, true>(C, A, s);
  return launch_quad<512, 4928, false, false>(C, A, s);
}
