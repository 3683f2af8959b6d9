// Particle interaction (PI) task, "quad" kernel for sm_100a: 3-D, cells of size 2h (cell_div = 1).
//
// A persistent CTA (one per SM) takes 2x2x2-cell tiles from a device-built list of non-empty tiles (tiles with fluid
// first, boundary-only tiles last) and stages each tile plus a one-cell halo in shared memory with TMA bulk copies
// (every cell is one contiguous range of the sorted arrays, C3); an in-place pass rewrites the positions as exact
// tile-centred coordinates (C1/C2 hold bit for bit) and builds a half-precision test record per particle.
//
//   work unit : 16 particles a of one centre cell x half of the 27-cell stencil (part 0 / part 1: disjoint row sets with
//             about equal numbers of neighbours); the two units of a group add their partial sums into the zeroed
//             output with atomics.  Units are handed out dynamically to the 16 warps.
//   lanes   : lane (g, t) = (lane / 4, lane % 4).  The four lanes of g own the pair (a_g, a_g+8) of the group; lane t
//             owns the candidates b whose staged index is congruent to 2t or 2t + 1 modulo 8.
//   T phase : (test) one mma.sync m16n8k8 (f16) per 8 candidates evaluates the expanded-form prefilter
//             D = |a|^2 - 2 a.b + |b|^2 - (R^2 + margin) for the 16 a of the warp (-2a split into two halves for
//             precision); b is a candidate of a iff D < 0.  The prefilter is conservative (margin > its rounding
//             error).  The sign bits of both a of a lane are OR-ed and collected, QB steps at a time,
//             into one 32-bit word per residue stream and 32 steps; non-empty words go to the lane's private word
//             list in shared memory together with the address of the record of bit 0 (no votes, no compaction).
//   P phase : (pair) every lane pops the set bits of its own words (one FLO per pop) and loads the two records of b
//             (LDS.128 each).  The trip count is the warp maximum of the per-lane pop counts (one REDUX per round),
//             so the loop carries no vote; a lane out of bits evaluates a dummy record far away.  Every popped b is
//             evaluated against BOTH a of the lane with packed FP32x2 arithmetic (FFMA2/FADD2/FMUL2, new on sm_100),
//             b entering as a broadcast scalar operand; the sums are packed in-place FFMA2 as well.  The exact
//             canonical predicate C2 (fp32, individually rounded) decides membership; a b that is a neighbour
//             of only one of the two a contributes exactly 0 to the other (the kernel weight is clamped at 0).
//   reduce  : the partial sums of the 4 lanes of a pair are combined with 2 butterfly shuffles (fixed order) and
//             lane t = 0 adds the two results to the output.
//
// What is kept from the paper: cell-linked list, particles sorted by cell, fp32 cell-relative positions
// (PAPER.md:558, 572).  What differs: the thread-per-particle loop with a branch per candidate.
#include <cuda_fp16.h>
#include <stdio.h>

#include "pi_common.cuh"

namespace {

constexpr int QT = 2;                     // tile: QT^3 centre cells
constexpr int QS = QT + 2;                // staged cells per axis
constexpr int QNCELL = QS * QS * QS;      // 64 staged cells per type block
constexpr int QNR = 2 * QNCELL;           // staged ranges: block 0 = boundary, block 1 = fluid
constexpr int QNSEG = 2 * QT * QT * QT;   // a-segments: (block, centre cell)
constexpr int QSLOT = 8;                  // non-empty words (32 candidates of the lane's residue each) per lane per round
constexpr int QB = 8;                     // T-phase steps whose loads are issued together
constexpr float Q_MARGIN = 0.03f;         // prefilter slack in r2u, > worst-case half-precision error
constexpr float Q_FAR = 100.0f;           // coordinate of the dummy record (never within the support)

// offset of the staged range of row k = (dz + 1) * 3 + (dy + 1) relative to the row dy = dz = 0
__constant__ int c_rowoff[9] = {-QS * QS - QS, -QS * QS, -QS * QS + QS, -QS, 0, QS, QS * QS - QS, QS * QS, QS * QS + QS};

// A group of 16 a is processed as two work units (part 0, part 1) that cover disjoint rows of the stencil and add
// their partial sums to the zeroed output with atomics: units of half the size halve the idle tail of a tile and
// let the word lists of a unit fit one round.  part 0 = boundary-block rows + the centre and corner rows of the
// fluid block, part 1 = the four edge rows of the fluid block (roughly equal numbers of neighbours).
__constant__ int c_partrow[2][5] = {{4, 0, 2, 6, 8}, {1, 3, 5, 7, 7}};

__device__ __forceinline__ int qrange(int blk, int ix, int iy, int iz) {   // staged indices, 0-based
  return ((blk * QS + iz) * QS + iy) * QS + ix;
}

struct QSmem {
  float4* rpos;       // (x, y, z, rho): exact tile-centred coordinates + density
  float4* rvel;       // (vx, vy, vz, P / rho)
  uint2* tst;         // half-precision test record of every staged particle: (x, y), (z, |b|^2)
  uint2* bm;          // [warp][QSLOT][32] private word lists: (bitmap word, byte address of the record of its bit 0)
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
  // raw sums of the two a of a lane, packed: one in-place FFMA2 per sum and step.  ptxas copies a loop-carried
  // 64-bit value back with two moves per loop trip, so the pair loop carries the halves as scalars across its
  // back edge and packs them at the top of the body (Q_PACK / Q_UNPACK; the packing itself costs nothing).
  f2 sx, sy, sz, sc, sd;
  float visc;         // max |mu_ab| / c_mu over the accepted pairs of both a (only the maximum over all particles is used, Eq. 35)
  f2 nb;              // neighbour counts, kept as floats (exact integers)
  f2 lx, ly, lz;      // laminar viscosity sums, Eq. 23 (LAM instantiations only)
  f2 cx, cy, cz;      // running compensation of sx, sy, sz (KAHAN instantiations only: sph_params.compensated_sums)
};
// Kahan update s += a * b with the running compensation c (c = what the rounded sum has in excess of the exact one).
__device__ __forceinline__ void f2_kahan_acc(f2 a, f2 b, f2& s, f2& c) {
  const f2 m1 = f2_bc(-1.0f);
  const f2 y = f2_fma(c, m1, f2_mul(a, b));        // a b - c
  const f2 t = f2_add(s, y);
  c = f2_fma(y, m1, f2_fma(s, m1, t));             // (t - s) - y
  s = t;
}
// One popped candidate b against both a of the lane (Eq. 15, 17-18, 21-22, 36), branch free, in two parts so that
// the record registers are free again after the head (the P loop reloads them for the next step before the tail).
// A b outside the support of a_h (prefilter false positive, neighbour of the other a only, or the dummy record)
// gets weight 0: w = max(1 - q/2, 0), and is masked out of the viscous dt candidate (A12) by the exact predicate.
// nb counts the exact canonical predicate C2.  pb = (x, y, z, rho_b), vb = (v_b, P_b/rho_b).
// DDT: this b enters the density diffusion term (A4).
struct PairTmp {
  f2 dux, duy, duz, dvx, dvy, dvz, drho, rs, ppb;
  float inv_rho_b;
};
template <bool A_FLUID, bool DDT>
__device__ __forceinline__ void pair2_head(const PairA& a, const float4 pb, const float4 vb, PairTmp& T) {
  T.dux = f2_add(a.x, f2_bc(-pb.x));   // exact (C1)
  T.duy = f2_add(a.y, f2_bc(-pb.y));
  T.duz = f2_add(a.z, f2_bc(-pb.z));
  T.dvx = f2_add(a.vx, f2_bc(-vb.x));
  T.dvy = f2_add(a.vy, f2_bc(-vb.y));
  T.dvz = f2_add(a.vz, f2_bc(-vb.z));
  T.inv_rho_b = fast_rcp(pb.w);
  if (A_FLUID) {
    if (DDT) T.drho = f2_add(a.rho, f2_bc(-pb.w));
    T.rs = f2_add(a.rho, f2_bc(pb.w));
    T.ppb = f2_mul(a.inv_rho, f2_bc(vb.w));       // kap_b / rho_a
  }
}
template <bool A_FLUID, bool DDT, bool LAM, bool FOURT, bool KAHAN>
__device__ __forceinline__ void pair2_tail(const DevConsts& C, const PairA& a, const PairTmp& T, PairAcc2& A) {
  f2 r2 = f2_mul(T.dux, T.dux);                   // C2: individually rounded
  r2 = f2_fma(T.duy, T.duy, r2);
  r2 = f2_fma(T.duz, T.duz, r2);
  const float r2a = f2_lo(r2), r2b = f2_hi(r2);
  const f2 inside = f2_pack(f_lt(r2a, C.R2u), f_lt(r2b, C.R2u));
  f2_add_acc(inside, A.nb);                       // exact: counts stay far below 2^24
  f2 w = f2_fma(f2_pack(fast_sqrt(r2a), fast_sqrt(r2b)), f2_bc(-C.qscale), f2_bc(1.0f));   // 1 - q/2   (Eq. 11)
  w = f2_pack(fmaxf(f2_lo(w), 0.f), fmaxf(f2_hi(w), 0.f));
  const f2 w3 = f2_mul(f2_mul(w, w), w);          // grad_a W_ab = Cf w^3 cs du
  f2 dot = f2_mul(T.dvx, T.dux);                  // v_ab . r_ab / cs
  dot = f2_fma(T.dvy, T.duy, dot);
  dot = f2_fma(T.dvz, T.duz, dot);
  const f2 gb = f2_mul(w3, f2_bc(T.inv_rho_b));
  f2_fma_acc(gb, dot, A.sc);
  if (A_FLUID) {
    if (DDT) {
      f2 drho = T.drho;
      if (FOURT) {   // Eq. 19-20 (A23): minus rho^H_ab = e (k0 + e (k1 + e (k2 + e k3))), e = c_hyd . du
        f2 e = f2_mul(T.dux, f2_bc(C.c_hyd[0]));
        e = f2_fma(T.duy, f2_bc(C.c_hyd[1]), e);
        e = f2_fma(T.duz, f2_bc(C.c_hyd[2]), e);
        f2 h = f2_fma(e, f2_bc(C.hyd_k[3]), f2_bc(C.hyd_k[2]));
        h = f2_fma(e, h, f2_bc(C.hyd_k[1]));
        h = f2_fma(e, h, f2_bc(C.hyd_k[0]));
        drho = f2_fma(f2_mul(e, f2_bc(-1.0f)), h, drho);
      }
      f2_fma_acc(gb, drho, A.sd);
    }
    const f2 den = f2_mul(f2_add(r2, f2_bc(C.eta2u)), T.rs);
    const f2 xinv = f2_pack(fast_rcp(f2_lo(den)), fast_rcp(f2_hi(den)));
    const f2 y = f2_mul(dot, xinv);                       // dot / ((r2 + eta2) rs)
    if (LAM) {                                            // Eq. 23: sum w^3 r2u / ((r2u + eta2u) rs) dv
      const f2 lam = f2_mul(f2_mul(w3, r2), xinv);
      f2_fma_acc(lam, T.dvx, A.lx);
      f2_fma_acc(lam, T.dvy, A.ly);
      f2_fma_acc(lam, T.dvz, A.lz);
    }
    const f2 mu = f2_mul(f2_mul(y, T.rs), inside);        // mu_ab / c_mu over accepted pairs only (Eq. 21, A12)
    A.visc = fmaxf(fmaxf(A.visc, fabsf(f2_lo(mu))), fabsf(f2_hi(mu)));   // one FMNMX3
    const f2 t = f2_pack(fminf(f2_lo(y), 0.f), fminf(f2_hi(y), 0.f));   // approaching pairs only (Eq. 21)
    // (Pa + Pb) / (rho_a rho_b) = kap_a / rho_b + kap_b / rho_a
    const f2 pp = f2_fma(a.kap, f2_bc(T.inv_rho_b), T.ppb);
    const f2 coef = f2_mul(w3, f2_fma(f2_bc(C.c_pi), t, pp));
    if (KAHAN) {   // compensated momentum sums: the pair terms are ~100x the net under deep hydrostatic pressure
      f2_kahan_acc(coef, T.dux, A.sx, A.cx);
      f2_kahan_acc(coef, T.duy, A.sy, A.cy);
      f2_kahan_acc(coef, T.duz, A.sz, A.cz);
    } else {
      f2_fma_acc(coef, T.dux, A.sx);
      f2_fma_acc(coef, T.duy, A.sy);
      f2_fma_acc(coef, T.duz, A.sz);
    }
  }
}

__device__ __forceinline__ unsigned bfind32(unsigned x) {   // index of the highest set bit; 0xffffffff if x == 0
  unsigned r;
  asm("bfind.u32 %0, %1;" : "=r"(r) : "r"(x));
  return r;
}

// Take the next (word, base) entry of a lane's list if the current word is used up and the list is not:
// one predicate drives the 64-bit shared-memory load and the pointer increment (nothing happens otherwise).
__device__ __forceinline__ void next_word_if_empty(unsigned& cur, unsigned& base, unsigned& wptr, unsigned wend) {
  asm volatile(
      "{.reg .pred q;\n\t"
      "setp.lt.u32 q, %2, %3;\n\t"
      "setp.eq.and.u32 q, %0, 0, q;\n\t"
      "@q ld.shared.v2.u32 {%0, %1}, [%2];\n\t"
      "@q add.u32 %2, %2, 256;}"
      : "+r"(cur), "+r"(base), "+r"(wptr) : "r"(wend));
}

// Sum over the 4 lanes that share a pair of a (butterfly, fixed order).
__device__ __forceinline__ float qsum(float v) {
  v += __shfl_xor_sync(0xffffffffu, v, 1);
  v += __shfl_xor_sync(0xffffffffu, v, 2);
  return v;
}
__device__ __forceinline__ float qmax(float v) {
  v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, 1));
  v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, 2));
  return v;
}

#ifdef Q_STATS
__device__ unsigned long long g_qstats[8];
__global__ void k_qstats_print() {
  printf("QSTATS warp_steps %llu pops %llu rounds %llu slots %llu groups %llu eff %.4f\n", g_qstats[0], g_qstats[1], g_qstats[2],
         g_qstats[3], g_qstats[4], (double)g_qstats[1] / (32.0 * (double)g_qstats[0]));
  for (int i = 0; i < 8; i++) g_qstats[i] = 0;
}
#endif

// ---- TMA bulk copy global -> shared memory, completion counted in bytes on an mbarrier ----
__device__ __forceinline__ void mbar_init(unsigned mbar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(mbar), "r"(count));
}
__device__ __forceinline__ void mbar_arrive_expect_tx(unsigned mbar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(mbar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned mbar, unsigned parity) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "WAIT_%=:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
      "@p bra DONE_%=;\n\t"
      "bra WAIT_%=;\n\t"
      "DONE_%=:\n\t}" ::"r"(mbar), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst_smem, const void* src_gmem, unsigned bytes, unsigned mbar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                   (unsigned)__cvta_generic_to_shared(dst_smem)),
               "l"(src_gmem), "r"(bytes), "r"(mbar)
               : "memory");
}

// m16n8k8 half-precision MMA with half accumulators: D (16 x 8) = A (16 x 8, row) * B (8 x 8, col) + C.
// Lane (g = lane / 4, t = lane % 4) holds A[g][2t, 2t+1] and A[g+8][2t, 2t+1], B[2t, 2t+1][g], and the
// same elements of C / D as of A.
__device__ __forceinline__ void mma_m16n8k8(unsigned& d0, unsigned& d1, unsigned a0, unsigned a1, unsigned b0, unsigned c0,
                                            unsigned c1) {
  asm volatile("mma.sync.aligned.m16n8k8.row.col.f16.f16.f16.f16 {%0, %1}, {%2, %3}, {%4}, {%5, %6};"
               : "=r"(d0), "=r"(d1) : "r"(a0), "r"(a1), "r"(b0), "r"(c0), "r"(c1));
}

// One a-group: up to 16 particles a of the centre cell (cx, cy, cz) (tile-local, 0..QT-1), type block
// A_FLUID ? 1 : 0, staged at [cell_start + 16*grp, ...).  bmw is this warp's word-list area ([QSLOT][32] uint2).
// Lane (g, t) = (lane / 4, lane % 4): the 4 lanes of g own the pair (a_2g, a_2g+1); lane t owns the candidates
// whose staged index is congruent to 2t or 2t+1 modulo 8.
template <bool A_FLUID, bool LAM, bool FOURT, bool KAHAN>
__device__ __forceinline__ void process_group(const DevConsts& C, const PiArgs& A, const QSmem& S, uint2* bmw, int cx,
                                              int cy, int cz, unsigned cell_start, unsigned n_a, unsigned grp, int part,
                                              unsigned total, float& viscmax, unsigned int& nbsum) {
  const int lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
  const unsigned t0 = grp * 16 + 2 * g, t1 = t0 + 1;
  const bool act0 = t0 < n_a, act1 = t1 < n_a;
  const unsigned ja0 = cell_start + (act0 ? t0 : 0), ja1 = cell_start + (act1 ? t1 : 0);

  // ---- state of the two a of this lane (inactive: far away, never accepted) ----
  PairA a;
  unsigned fa0, fa1, fc0, fc1;    // MMA fragments of the prefilter: rows g (a_2g) and g + 8 (a_2g+1)
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
    // Prefilter as a 16 x 8 x 8 product: row of a = (-2a_hi, 1, -2a_lo, 0) with -2a = hi + lo in
    // half precision, column of b = (b, |b|^2, b, |b|^2), C = |a|^2 - R2u - margin, so that
    // D = |b|^2 - 2 a.b + |a|^2 - (R2u + margin) and b is a candidate of a iff D < 0.  An inactive a has a zero
    // row and C = +60000: never accepted.
    float e0[3] = {-2.f * p0.x, -2.f * p0.y, -2.f * p0.z}, e1[3] = {-2.f * p1.x, -2.f * p1.y, -2.f * p1.z};
    float k0a, k0b, k1a, k1b;       // elements (2t, 2t+1) of the two rows
    {
      float h0[3], l0[3], h1[3], l1[3];
#pragma unroll
      for (int k = 0; k < 3; k++) {
        h0[k] = __half2float(__float2half_rn(e0[k])); l0[k] = e0[k] - h0[k];
        h1[k] = __half2float(__float2half_rn(e1[k])); l1[k] = e1[k] - h1[k];
      }
      k0a = t == 0 ? h0[0] : t == 1 ? h0[2] : t == 2 ? l0[0] : l0[2];
      k0b = t == 0 ? h0[1] : t == 1 ? 1.f : t == 2 ? l0[1] : 0.f;
      k1a = t == 0 ? h1[0] : t == 1 ? h1[2] : t == 2 ? l1[0] : l1[2];
      k1b = t == 0 ? h1[1] : t == 1 ? 1.f : t == 2 ? l1[1] : 0.f;
    }
    const float c0f = fmaf(p0.z, p0.z, fmaf(p0.y, p0.y, p0.x * p0.x)) - (C.R2u + Q_MARGIN);
    const float c1f = fmaf(p1.z, p1.z, fmaf(p1.y, p1.y, p1.x * p1.x)) - (C.R2u + Q_MARGIN);
    fa0 = act0 ? h2_as_u32(__floats2half2_rn(k0a, k0b)) : 0u;
    fa1 = act1 ? h2_as_u32(__floats2half2_rn(k1a, k1b)) : 0u;
    fc0 = h2_as_u32(__half2half2(act0 ? __float2half_rd(c0f) : __float2half_rn(60000.f)));   // rounded down: conservative
    fc1 = h2_as_u32(__half2half2(act1 ? __float2half_rd(c1f) : __float2half_rn(60000.f)));
  }
#ifdef Q_STATS
  if (lane == 0) atomicAdd(&g_qstats[4], 1ull);
#endif
  PairAcc2 acc;
  acc.lx = acc.ly = acc.lz = f2_pack(0.f, 0.f);
  acc.sx = acc.sy = acc.sz = acc.sc = acc.sd = acc.nb = f2_pack(0.f, 0.f);
  acc.visc = 0.f;
  acc.cx = acc.cy = acc.cz = f2_pack(0.f, 0.f);

  // Rounds are homogeneous in the type block of b: fluid a sweeps the 9 boundary-block rows first (diffusion
  // term only if ddt_over_boundary, A4), then the 9 fluid rows; boundary a sweeps the fluid rows only (Eq. 36).
  // Runs of this unit: fluid a, part 0: the 9 boundary-block rows, then 5 fluid rows; otherwise fluid rows only.
  const int nbr = (A_FLUID && part == 0) ? 9 : 0;       // boundary-block runs come first
  const int nruns = nbr + (part == 0 ? 5 : 4);
  int ri = (nbr && S.soff[QNCELL] == 0u) ? nbr : 0;     // no boundary particle staged: skip their 9 rows
  int sw = -1, s_last = -1;                             // next block of 8 candidates of the open run, its last block
  int j0 = 0, j1 = 0;
  const unsigned dummy_addr = total * 16u;
  const int row0 = qrange(1, cx, 1 + cy, 1 + cz);        // fluid-block range of the cell left of the centre cell
  uint2* wl = bmw + lane;                                // private word list of this lane: entries wl[32 * k]
  const unsigned wl_s = (unsigned)__cvta_generic_to_shared(wl);
  const uint32_t* tst32 = reinterpret_cast<const uint32_t*>(S.tst) + 2 * g + (t & 1);   // B fragment of block 0

  while (ri < nruns) {
    // ================= T phase: fill the private word lists (at most QSLOT non-empty words per lane and round) =================
    const int ri_end = ri < nbr ? nbr : nruns;
    const bool ddt_round = !(ri < nbr && !C.ddt_over_boundary);
    int nslot = 0;
    unsigned nw = 0, npop = 0;
    while (ri < ri_end) {
      // a slot adds up to two words to a list: if one might not fit, run the P phase first (the round resumes here)
      if (__any_sync(0xffffffffu, nw > (unsigned)(QSLOT - 2))) break;
      if (sw < 0) {   // open run ri
        // row ri of the stencil: cells (cx-1 .. cx+1, cy+dy, cz+dz) of one type block are one contiguous range
        const int row = ri < nbr ? row0 - QNCELL + c_rowoff[ri] : row0 + c_rowoff[c_partrow[part][ri - nbr]];
        j0 = (int)S.soff[row];
        j1 = (int)S.soff[row + 3];
        if (j1 <= j0) { ri++; continue; }
        sw = j0 >> 3;
        s_last = (j1 - 1) >> 3;
      }
      // One slot = up to 32 steps; a step tests the 8 candidates of block sw + i against the 16 a of the warp with
      // one MMA.  d0 | d1 carries the sign of D for (either a of the lane, candidate 8 (sw + i) + 2t) in bit 15 and
      // for candidate + 1 in bit 31; they are appended to the words of the two residue streams QB steps at a
      // time, so that after ne steps bit p of a word belongs to step ne - 1 - p.  The loads of QB steps are issued
      // together.  Steps beyond the run read whatever follows (the test records are followed by the word lists
      // in shared memory, so the addresses stay valid); their bits are masked below.
      const int nstep = min(32, s_last - sw + 1);
      const int ne = (nstep + QB - 1) & ~(QB - 1);       // steps executed
      const uint32_t* tq = tst32 + sw * 16;
      unsigned accL = 0, accH = 0;
#pragma unroll
      for (int b0 = 0; b0 < 32; b0 += QB) {
        if (b0 < nstep) {
          unsigned bb[QB];
#pragma unroll
          for (int i = 0; i < QB; i++) bb[i] = tq[(b0 + i) * 16];   // may run past the run (never past the lists)
#ifdef Q_CHECK   // development build (SPH_NVCC_EXTRA=-DQ_CHECK): every test-record load stays inside the test records + word lists
          if (reinterpret_cast<const unsigned char*>(tq + (b0 + QB - 1) * 16 + 1) > reinterpret_cast<const unsigned char*>(S.soff))
            atomicOr(&A.sc->flags, 1u);
#endif
          // the sign bits of the QB steps of a batch are merged first (top QB bits of the upper half-word: candidate 2t + 1, of the
          // lower half-word: candidate 2t; earlier step = higher bit), so that the batches do not form one long dependency chain
          unsigned y = 0;
#pragma unroll
          for (int i = 0; i < QB; i++) {
            unsigned d0, d1;
            mma_m16n8k8(d0, d1, fa0, fa1, bb[i], fc0, fc1);
            y += ((d0 | d1) & 0x80008000u) >> i;
          }
          accH = __funnelshift_l(y, accH, QB);
          accL = __funnelshift_l(y << 16, accL, QB);
        }
      }
      // keep the candidates that lie inside the run [j0, j1): step i of stream h is candidate c0 + 8 i with
      // c0 = 8 sw + 2t + h, valid for i in [ilo, ihi], i.e. bits ne - 1 - ihi .. ne - 1 - ilo.  Branch free.
      const int cL = 8 * sw + 2 * t;
#pragma unroll
      for (int h = 0; h < 2; h++) {
        const int c0 = cL + h;
        const int ilo = max((j0 - c0 + 7) >> 3, 0), ihi = min((j1 - 1 - c0) >> 3, ne - 1);   // arithmetic shifts
        const unsigned m = ihi >= ilo ? (0xffffffffu >> (31 - (ne - 1 - ilo))) & (0xffffffffu << (ne - 1 - ihi)) : 0u;
        unsigned& w = h ? accH : accL;
        w &= m;
        // a non-empty word goes to this lane's list, together with the byte address of the record of its bit 0
        // (bit p -> record address - 128 p); no other lane reads it
        if (w != 0u) {
          wl[nw * 32u] = make_uint2(w, (unsigned)(c0 + 8 * (ne - 1)) * 16u);
          nw++;
          npop += (unsigned)__popc(w);
        }
      }
      nslot++;
      sw += 32;
      if (sw > s_last) { ri++; sw = -1; }
    }
    if (nslot == 0) continue;

    // ================= P phase: every lane pops the bits of its own words =================
    // Lane t holds candidates of residues 2t and 2t + 1 only.  The trip count is the warp maximum of the pop
    // counts; a lane that has run out of bits evaluates the dummy record (exactly zero contribution).
    const unsigned nmax = __reduce_max_sync(0xffffffffu, npop);
#ifdef Q_STATS
    {
      const unsigned tot = __reduce_add_sync(0xffffffffu, npop);
      if (lane == 0) {
        atomicAdd(&g_qstats[0], (unsigned long long)nmax);      // warp steps
        atomicAdd(&g_qstats[1], (unsigned long long)tot);       // pops
        atomicAdd(&g_qstats[2], 1ull);                          // rounds
        atomicAdd(&g_qstats[3], (unsigned long long)nslot);     // word slots
      }
    }
#endif
    const unsigned char* rp = reinterpret_cast<const unsigned char*>(S.rpos);
    const unsigned char* rv = reinterpret_cast<const unsigned char*>(S.rvel);
    unsigned cur = 0, base = 0;
    unsigned wptr = wl_s;
    const unsigned wend = wl_s + nw * 256u;
    // one pop: take the next word if the current one is used up and turn its highest set bit into a record
    // address.  Software pipeline, two steps per loop trip (records ping-pong without moves): while step k is
    // evaluated, the record of step k + 1 is being loaded and the address of step k + 2 is popped; a lane out of
    // bits gets the dummy record.
#define Q_POP(ADDR)                                                                                    \
  {                                                                                                    \
    next_word_if_empty(cur, base, wptr, wend);                                                         \
    const unsigned p = bfind32(cur); /* cur == 0 -> 0xffffffff (unused) */                              \
    ADDR = cur != 0u ? base - (p << 7) : dummy_addr;                                                   \
    cur &= ~(1u << (p & 31u));                                                                         \
  }
#ifdef Q_CHECK   // development build: every popped record address is a staged record or the dummy record
#define Q_CHECK_ADDR(ADDR) if ((ADDR) > dummy_addr || ((ADDR) & 15u)) atomicOr(&A.sc->flags, 1u);
#else
#define Q_CHECK_ADDR(ADDR)
#endif
#define Q_LOAD(ADDR, PB, VB)                                                                           \
  Q_CHECK_ADDR(ADDR)                                                                                   \
  PB = *reinterpret_cast<const float4*>(rp + ADDR);                                                    \
  VB = *reinterpret_cast<const float4*>(rv + ADDR);
#define Q_UNPACK()                                                                                     \
  q_s[0] = f2_lo(acc.sx); q_s[1] = f2_hi(acc.sx); q_s[2] = f2_lo(acc.sy); q_s[3] = f2_hi(acc.sy);    \
  q_s[4] = f2_lo(acc.sz); q_s[5] = f2_hi(acc.sz); q_s[6] = f2_lo(acc.sc); q_s[7] = f2_hi(acc.sc);    \
  q_s[8] = f2_lo(acc.sd); q_s[9] = f2_hi(acc.sd); q_s[16] = f2_lo(acc.nb); q_s[17] = f2_hi(acc.nb);   \
  if (LAM) {                                                                                           \
    q_s[10] = f2_lo(acc.lx); q_s[11] = f2_hi(acc.lx); q_s[12] = f2_lo(acc.ly); q_s[13] = f2_hi(acc.ly); \
    q_s[14] = f2_lo(acc.lz); q_s[15] = f2_hi(acc.lz);                                                 \
  }                                                                                                    \
  Q_UNPACK_K()
#define Q_UNPACK_K()                                                                                   \
  if (KAHAN) {                                                                                         \
    q_s[18] = f2_lo(acc.cx); q_s[19] = f2_hi(acc.cx); q_s[20] = f2_lo(acc.cy); q_s[21] = f2_hi(acc.cy); \
    q_s[22] = f2_lo(acc.cz); q_s[23] = f2_hi(acc.cz);                                                 \
  }
#define Q_PACK_K()                                                                                     \
  if (KAHAN) { acc.cx = f2_pack(q_s[18], q_s[19]); acc.cy = f2_pack(q_s[20], q_s[21]); acc.cz = f2_pack(q_s[22], q_s[23]); }
#define Q_PACK()                                                                                       \
  acc.sx = f2_pack(q_s[0], q_s[1]); acc.sy = f2_pack(q_s[2], q_s[3]); acc.sz = f2_pack(q_s[4], q_s[5]); \
  acc.sc = f2_pack(q_s[6], q_s[7]); acc.sd = f2_pack(q_s[8], q_s[9]); acc.nb = f2_pack(q_s[16], q_s[17]); \
  if (LAM) { acc.lx = f2_pack(q_s[10], q_s[11]); acc.ly = f2_pack(q_s[12], q_s[13]); acc.lz = f2_pack(q_s[14], q_s[15]); } \
  Q_PACK_K()
#define Q_LOOP(DDT)                                                                                    \
  {                                                                                                    \
    float4 pbA, vbA, pbB, vbB;                                                                         \
    PairTmp T;                                                                                         \
    unsigned addr;                                                                                     \
    float q_s[24];             /* the packed sums, as scalars across the back edge of the loop */      \
    Q_POP(addr)                                                                                        \
    Q_LOAD(addr, pbA, vbA)                                                                             \
    Q_POP(addr)                                                                                        \
    Q_UNPACK()                                                                                         \
    _Pragma("unroll 2") /* two trips = four steps per iteration: 4.675 against 4.722 ms (unroll 3: 4.760, 4: 4.819) */     \
    for (unsigned k = 0; k < nmax; k += 2) { /* at most one surplus evaluation of dummy records */     \
      Q_PACK()                                                                                         \
      Q_LOAD(addr, pbB, vbB)   /* record of step k + 1: its address was popped during step k - 1 */    \
      Q_POP(addr)              /* address of step k + 2 */                                             \
      pair2_head<A_FLUID, DDT>(a, pbA, vbA, T);                                                        \
      pair2_tail<A_FLUID, DDT, LAM, FOURT, KAHAN>(C, a, T, acc);                                              \
      Q_LOAD(addr, pbA, vbA)                                                                           \
      Q_POP(addr)                                                                                      \
      pair2_head<A_FLUID, DDT>(a, pbB, vbB, T);                                                        \
      pair2_tail<A_FLUID, DDT, LAM, FOURT, KAHAN>(C, a, T, acc);                                              \
      Q_UNPACK()                                                                                       \
    }                                                                                                  \
    Q_PACK()                                                                                           \
  }
    if (ddt_round) Q_LOOP(true) else Q_LOOP(false)
#undef Q_LOOP
#undef Q_PACK
#undef Q_UNPACK
#undef Q_PACK_K
#undef Q_UNPACK_K
#undef Q_LOAD
#undef Q_CHECK_ADDR
#undef Q_POP
  }

  // ---- combine the 4 lanes of each pair; lane t = 0 writes both particles ----
  PairAcc r0 = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f}, r1 = r0;
  r0.sc = qsum(f2_lo(acc.sc)); r1.sc = qsum(f2_hi(acc.sc));
  const unsigned nb0 = (unsigned)qsum(f2_lo(acc.nb)), nb1 = (unsigned)qsum(f2_hi(acc.nb));
  if (A_FLUID) {
    if (KAHAN) {
      acc.sx = f2_fma(acc.cx, f2_bc(-1.0f), acc.sx);   // sum - compensation
      acc.sy = f2_fma(acc.cy, f2_bc(-1.0f), acc.sy);
      acc.sz = f2_fma(acc.cz, f2_bc(-1.0f), acc.sz);
    }
    r0.sx = qsum(f2_lo(acc.sx)); r1.sx = qsum(f2_hi(acc.sx));
    r0.sy = qsum(f2_lo(acc.sy)); r1.sy = qsum(f2_hi(acc.sy));
    r0.sz = qsum(f2_lo(acc.sz)); r1.sz = qsum(f2_hi(acc.sz));
    r0.sd = qsum(f2_lo(acc.sd)); r1.sd = qsum(f2_hi(acc.sd));
    r0.visc = r1.visc = qmax(acc.visc);
    if (LAM) {
      r0.lx = qsum(f2_lo(acc.lx)); r1.lx = qsum(f2_hi(acc.lx));
      r0.ly = qsum(f2_lo(acc.ly)); r1.ly = qsum(f2_hi(acc.ly));
      r0.lz = qsum(f2_lo(acc.lz)); r1.lz = qsum(f2_hi(acc.lz));
    }
  }
  if (t == 0) {
    const int ra = qrange(A_FLUID ? 1 : 0, 1 + cx, 1 + cy, 1 + cz);
    const unsigned gbase = S.gstart[ra] - S.soff[ra];
#pragma unroll
    for (int h = 0; h < 2; h++) {
      if (h == 0 ? act0 : act1) {
        const PairAcc& pa1 = h ? r1 : r0;
        unsigned nb = h ? nb1 : nb0;
        if (A_FLUID && part == 0) nb -= 1u;   // the particle itself (centre row) passed the test at r = 0, contributing exactly 0 (A17)
        const unsigned ga = gbase + (h ? ja1 : ja0);
        const float rho_a = h ? rho_a1 : rho_a0;
        // scaled partial sums of this unit (finish_particle of pi_common.cuh, with g entering through part 0 only);
        // the two units of a group add into the zeroed output: x1 + x2 is the same in either order
        float4 out = make_float4(0.f, 0.f, 0.f, 0.f);
        if (A_FLUID) {
          out.x = fmaf(C.c_mom, pa1.sx, part == 0 ? C.g[0] : 0.f);
          out.y = fmaf(C.c_mom, pa1.sy, part == 0 ? C.g[1] : 0.f);
          out.z = fmaf(C.c_mom, pa1.sz, part == 0 ? C.g[2] : 0.f);
          if (LAM) {
            out.x = fmaf(C.c_lam, pa1.lx, out.x);
            out.y = fmaf(C.c_lam, pa1.ly, out.y);
            out.z = fmaf(C.c_lam, pa1.lz, out.z);
          }
          out.w = fmaf(rho_a * C.c_cont, pa1.sc, C.c_ddt * pa1.sd);
        } else {
          out.w = rho_a * C.c_cont * pa1.sc;
        }
        if (!isfinite(out.x + out.y + out.z + out.w)) atomicOr(&A.sc->flags, 1u);   // reported as SPH_E_NAN
        atomicAdd(&A.acc[ga], out);
        if (A.nbcount) atomicAdd(&A.nbcount[ga], nb);
        viscmax = fmaxf(viscmax, pa1.visc * C.c_mu);
        nbsum += nb;
      }
    }
  }
}

// max_a |F_a|^2 over the fluid particles (dt candidate of Eq. 35), from the summed output of the work units.
__global__ void __launch_bounds__(256) k_quad_fmax(DevConsts C, const float4* __restrict__ acc,
                                                   const uint32_t* __restrict__ cellstart, DevScalars* sc) {
  const uint32_t f0 = cellstart[C.ncells], f1 = cellstart[2u * C.ncells];   // the fluid block in sorted order (C3)
  float f2 = 0.f;
  for (uint32_t i = f0 + blockIdx.x * blockDim.x + threadIdx.x; i < f1; i += gridDim.x * blockDim.x) {
    const float4 o = acc[i];
    f2 = fmaxf(f2, fmaf(o.x, o.x, fmaf(o.y, o.y, o.z * o.z)));
  }
  reduce_scalars(sc, f2, 0.f, 0u);
}

// Active-tile list: most tiles of a dam break are air.  A tile is active if its centre cells hold a particle;
// x-adjacent cells are adjacent keys, so one (block, cy, cz) row of centre cells is one cellstart difference.
// ws[0] = number of tiles with fluid, ws[1] = next tile to take, ws[2] = number of boundary-only tiles (all zeroed
// before the launch), ws[4..] = tile ids (fluid tiles from the front, boundary-only tiles from the back).
__global__ void __launch_bounds__(256) k_quad_tiles(DevConsts C, const uint32_t* __restrict__ cellstart, int ntx, int nty,
                                                    int ntiles, uint32_t* ws) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= ntiles) return;
  const int ox = (t % ntx) * QT, oy = ((t / ntx) % nty) * QT, oz = (t / (ntx * nty)) * QT;
  const uint32_t w = (uint32_t)min(QT, C.nc[0] - ox);
  bool any[2] = {false, false};
  for (int blk = 0; blk < 2; blk++)
    for (int cz = oz; cz < min(oz + QT, C.nc[2]); cz++)
      for (int cy = oy; cy < min(oy + QT, C.nc[1]); cy++) {
        const uint32_t key = (uint32_t)blk * C.ncells + (uint32_t)ox +
                             (uint32_t)C.nc[0] * ((uint32_t)cy + (uint32_t)C.nc[1] * (uint32_t)cz);
        any[blk] = any[blk] || cellstart[key + w] != cellstart[key];
      }
  // Tiles with fluid centre particles fill the list from the front, tiles with boundary particles only (short ones:
  // B <- F pairs, no momentum) from the back: the CTAs take the list in order, so the launch ends with short tiles
  // (4.720 against 4.787 ms per pass on config 2).
  if (any[1]) ws[4 + atomicAdd(&ws[0], 1u)] = (uint32_t)t;
  else if (any[0]) ws[4 + (uint32_t)ntiles - 1u - atomicAdd(&ws[2], 1u)] = (uint32_t)t;
}

// Persistent kernel: one CTA per SM takes active tiles from the list until it is used up.
template <int NT, int NMAX, bool LAM, bool FOURT, bool KAHAN>
__global__ void __launch_bounds__(NT, 1) k_pi_quad(DevConsts C, PiArgs A, int ntx, int nty) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  constexpr int NWARP = NT / 32;
  QSmem S;
  S.rpos = reinterpret_cast<float4*>(smem_raw);
  S.rvel = S.rpos + NMAX;
  S.tst = reinterpret_cast<uint2*>(S.rvel + NMAX);
  S.bm = S.tst + NMAX;
  S.soff = reinterpret_cast<uint32_t*>(S.bm + NWARP * QSLOT * 32);
  S.gstart = S.soff + (QNR + 1);
  S.seg = S.gstart + QNR;
  __shared__ uint32_t s_cnt[QNR];
  __shared__ uint32_t s_tile;
  __shared__ __align__(8) unsigned long long s_mbar;
  const unsigned mbar_s = (unsigned)__cvta_generic_to_shared(&s_mbar);
  unsigned mbar_phase = 0;
  if (threadIdx.x == 0) {
    mbar_init(mbar_s, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const uint32_t n_front = A.tile_ws[0], n_active = n_front + A.tile_ws[2];   // fluid tiles from the front, boundary-only ones from the back
  const uint32_t n_tiles_all = (uint32_t)(ntx * nty) * (uint32_t)((C.nc[2] + QT - 1) / QT);
  float f2max = 0.f, viscmax = 0.f;   // f2max: overflow path only (k_quad_fmax covers every fluid particle)
  unsigned int nbsum = 0;

 // One thread claims the next tile while the CTA computes the current one (the atomic is a global round trip that
 // would otherwise stall all 16 warps once per tile); the result is read after the next tile barrier
 // (4.658 against 4.676 ms; reading the tile id ahead as well is slower: 4.677).
 if (tid == 0) s_tile = atomicAdd(&A.tile_ws[1], 1u);
 for (;;) {
  __syncthreads();                                  // every warp is done with the previous tile's shared memory
  const uint32_t cur_tile = s_tile;
  if (cur_tile >= n_active) break;
  bool claimed = false;
  const int tile = (int)A.tile_ws[4 + (cur_tile < n_front ? cur_tile : n_tiles_all - 1u - (cur_tile - n_front))];
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
      run += (n + 15) / 16;
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

  // 2. stage the particles: the sorted arrays hold every cell as one contiguous range (C3), so each non-empty staged
  //    range is two TMA bulk copies (positions + density, velocities + pressure) straight into shared memory,
  //    completing on one mbarrier (no register staging, all copies of the tile in flight at once).
  //    (The generic-proxy accesses of the previous tile were fenced by the threads that made them, before the barrier,
  //    at the end of step 4; this second fence in the issuing threads is kept as well: one instruction per tile.)
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  if (tid == 0) mbar_arrive_expect_tx(mbar_s, total * 32u);
  for (int rr = tid; rr < QNR; rr += NT) {
    const uint32_t n = s_cnt[rr];
    if (n == 0) continue;
    const uint32_t g0 = S.gstart[rr], d0 = S.soff[rr];
    bulk_g2s(S.rpos + d0, A.posu + g0, n * 16u, mbar_s);
    bulk_g2s(S.rvel + d0, A.velp + g0, n * 16u, mbar_s);
  }
  mbar_wait(mbar_s, mbar_phase);
  mbar_phase ^= 1u;
  // 3. in place: tile-centred coordinates u + integer cell offset - QT/2 (exact: every value is a multiple of
  //    2^-22 with magnitude <= 2, so all differences are exact in fp32, C1/C2), P -> P / rho, and the
  //    half-precision test records (x, y, z, |b|^2 of the rounded coordinates): the columns of the prefilter product
  for (int rr = warp; rr < QNR; rr += NWARP) {
    const uint32_t n = s_cnt[rr];
    if (n == 0) continue;
    const int c = rr % QNCELL;
    const float fx = (float)(c % QS - 1) - 0.5f * QT, fy = (float)((c / QS) % QS - 1) - 0.5f * QT,
                fz = (float)(c / (QS * QS) - 1) - 0.5f * QT;
    const uint32_t d0 = S.soff[rr];
    for (uint32_t i = lane; i < n; i += 32) {
      float4 pp = S.rpos[d0 + i];
      pp.x += fx; pp.y += fy; pp.z += fz;
      S.rpos[d0 + i] = pp;
      float* kap = reinterpret_cast<float*>(S.rvel + d0 + i) + 3;
      *kap = __fdiv_rn(*kap, pp.w);                                       // (v, P / rho)
      const __half2 hxy = __floats2half2_rn(pp.x, pp.y);
      const __half hz = __float2half_rn(pp.z);
      const float2 fxy = __half22float2(hxy);
      const float gz = __half2float(hz);
      const float w = fmaf(gz, gz, fmaf(fxy.y, fxy.y, fxy.x * fxy.x));
      S.tst[d0 + i] = make_uint2(h2_as_u32(hxy), h2_as_u32(__halves2half2(hz, __float2half_rn(w))));
    }
  }
  if (tid == 0) {   // dummy record: popped by lanes that have run out of work, never within any support
    S.rpos[total] = make_float4(Q_FAR, Q_FAR, Q_FAR, 1.0f);
    S.rvel[total] = make_float4(0.f, 0.f, 0.f, 0.f);
  }
  __syncthreads();

  if (!claimed) {                                   // every thread has read s_tile (two barriers ago)
    if (tid == NT - 1) s_tile = atomicAdd(&A.tile_ws[1], 1u);
    claimed = true;
  }
  // 4. a-groups, taken dynamically by the warps
  uint2* bmw = S.bm + warp * QSLOT * 32;
  while (true) {
    uint32_t gi = 0;
    if (lane == 0) gi = atomicAdd(&S.seg[0], 1u);
    gi = __shfl_sync(0xffffffffu, gi, 0);
    if (gi >= 2u * ngroups) break;
    const int part = gi & 1u;                       // the two units of a group are handed out one after the other, so
    gi >>= 1;                                       // that neighbouring warps are in different phases (4.791 against 4.806 ms)
    int s = 0;
    while (s + 1 < QNSEG && gi >= S.seg[1 + s + 1]) s++;
    const int blk = 1 - (s >> 3), cz = (s >> 2) & 1, cy = (s >> 1) & 1, cx = s & 1;
    const int rr = qrange(blk, 1 + cx, 1 + cy, 1 + cz);
    const unsigned cell_start = S.soff[rr], n_a = s_cnt[rr], grp = gi - S.seg[1 + s];
    if (blk == 1) process_group<true, LAM, FOURT, KAHAN>(C, A, S, bmw, cx, cy, cz, cell_start, n_a, grp, part, total, viscmax, nbsum);
    else process_group<false, false, false, false>(C, A, S, bmw, cx, cy, cz, cell_start, n_a, grp, part, total, viscmax, nbsum);
  }
  // This thread is done with the staged records: its generic-proxy accesses (the in-place rewrite of step 3, the dummy
  // record, the reads of step 4) are ordered before the next barrier here, in the thread that made them, so that the
  // bulk copies (async proxy) of the next tile or half tile, issued after that barrier, may overwrite the memory.
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  if (part == 0) break;
  }   // parts
  if (!claimed && tid == NT - 1) s_tile = atomicAdd(&A.tile_ws[1], 1u);   // no (half) tile reached the a-groups
 }   // tiles
  reduce_scalars(A.sc, f2max, viscmax, nbsum);
}

template <int NT, int NMAX, bool LAM, bool FOURT, bool KAHAN>
int launch_quad(const DevConsts& C, const PiArgs& A, cudaStream_t s) {
  const int ntx = (C.nc[0] + QT - 1) / QT, nty = (C.nc[1] + QT - 1) / QT, ntz = (C.nc[2] + QT - 1) / QT;
  constexpr int NWARP = NT / 32;
  const size_t smem = sizeof(float4) * 2 * NMAX + sizeof(uint2) * NMAX +
                      sizeof(uint2) * NWARP * QSLOT * 32 + sizeof(uint32_t) * ((QNR + 1) + QNR + (QNSEG + 2));
  // per device, so set on every launch (a cheap host call): a process may hold contexts on several devices
  if (cudaFuncSetAttribute(k_pi_quad<NT, NMAX, LAM, FOURT, KAHAN>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) !=
      cudaSuccess) {
    cudaGetLastError();
    return -1;
  }
  const long long ntiles = (long long)ntx * nty * ntz;
  if (ntiles > 0x7fffffffLL || A.tile_ws == nullptr) return -1;
  const int n_sm = A.n_sm;                            // of the context's device (sph_create)
  if (n_sm <= 0) return -1;
  if (cudaMemsetAsync(A.tile_ws, 0, 4 * sizeof(uint32_t), s) != cudaSuccess) return -1;
  // the work units add their partial sums into the outputs
  if (cudaMemsetAsync(A.acc, 0, sizeof(float4) * (size_t)A.n, s) != cudaSuccess) return -1;
  if (A.nbcount && cudaMemsetAsync(A.nbcount, 0, sizeof(uint32_t) * (size_t)A.n, s) != cudaSuccess) return -1;
  k_quad_tiles<<<(unsigned)((ntiles + 255) / 256), 256, 0, s>>>(C, A.cellstart, ntx, nty, (int)ntiles, A.tile_ws);
  k_pi_quad<NT, NMAX, LAM, FOURT, KAHAN><<<(unsigned)min((long long)n_sm, ntiles), NT, smem, s>>>(C, A, ntx, nty);
#ifdef Q_STATS
  k_qstats_print<<<1, 1, 0, s>>>();
#endif
  k_quad_fmax<<<n_sm * 4, 256, 0, s>>>(C, A.acc, A.cellstart, A.sc);
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
  if (C.comp_sums) {                                               // sph_params.compensated_sums: Kahan momentum sums
    if (lam && fourt) return launch_quad<512, 4928, true, true, true>(C, A, s);
    if (lam) return launch_quad<512, 4928, true, false, true>(C, A, s);
    if (fourt) return launch_quad<512, 4928, false, true, true>(C, A, s);
    return launch_quad<512, 4928, false, false, true>(C, A, s);
  }
  if (lam && fourt) return launch_quad<512, 4928, true, true, false>(C, A, s);
  if (lam) return launch_quad<512, 4928, true, false, false>(C, A, s);
  if (fourt) return launch_quad<512, 4928, false, true, false>(C, A, s);
  return launch_quad<512, 4928, false, false, false>(C, A, s);
}
