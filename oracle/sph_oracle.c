/*
 * sph_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, double-precision CPU oracle for the hot path of the weakly compressible SPH
 * method of arxiv 2104.00537 (DualSPHysics v5.0 paper, /root/reference/PAPER.md):
 * neighbour search + particle interaction + variable dt + symplectic step (+ the Verlet scheme, Eq. 30-31).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may call this.  It shares no code with the CUDA library (paper_2104_00537_b200/csrc):
 * no common headers, helpers, tables or constants.
 *
 * Every function cites the passage of PAPER.md it follows; where the paper is silent,
 * garbled or ambiguous the reading is the one listed in DESIGN.md section "Readings"
 * (labels A1..A20, C1..C3 from SURVEY.md section 8(c)).
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): Wendland normalisation = 1 by quadrature;
 * gradient vs finite difference; EOS P(rho0)=0 and dP/drho=c0^2; brute force == cell list;
 * lattice neighbour counts 304 / 36 / 250; momentum antisymmetry; diffusion conservation
 * and sign/magnitude against the analytic Laplacian; continuity against an independently
 * computed moment matrix; uniform lattice F = g; worked two-particle example
 * (tests/golden/two_particle.txt); dt closed form; integrator closed forms (free fall,
 * Pade density; Verlet free fall and corrective-step rule); hydrostatic column.  The Verlet density leapfrog has no
 * closed form to pin it: "parity unpinned" for that line beyond the free-fall and N_S = 1 (Euler) cases.  Everything else (absolute per-particle values on the
 * configs) is pinned only by these plus oracle-vs-GPU agreement: "parity otherwise unpinned".
 * Imposed motion (Eq. 37): closed form x(t), v(t) and the half-step evaluation time; rho_bound_floor (A10).
 * NEXT-3 mDBC (tests/test_oracle_next34.py): exact reproduction of linear density fields at ghost node and boundary
 * particle on arbitrary clouds, the system against numpy.linalg.solve on a non-linear field, ghost node at twice
 * the normal, Shepard / no-neighbour fallbacks, Shepard velocity and no-slip, brute force == cell list,
 * "set, not integrated" in both steppers.  NEXT-4 shifting: C = 1.00049 and grad C = 0 on the full lattice, grad C
 * against an independent numpy brute force at two free surfaces (direction, magnitude), linearity in A_s and |v|,
 * the Eq. 54 form, and r^{n+1}(shift) - r^{n+1}(no shift) = dt s in both steppers.
 *
 * Build: gcc -O2 -fopenmp -ffp-contract=off -shared -fPIC (see oracle/build.py).
 * -ffp-contract=off matters: the canonical conversions (C1) and the fp32 pair predicate
 * (C2) must be evaluated with individually rounded IEEE operations.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_API __attribute__((visibility("default")))

typedef struct {
  int dim;                /* 2 (plane x,z) or 3 */
  double dp, h, rho0, c0, gamma, alpha, delta;
  double g[3];
  double cfl;
  double domain_min[3], domain_max[3];
  int periodic[3];
  double eta2_coef;       /* eta^2 = eta2_coef * h^2 (A6) */
  int ddt_over_boundary;  /* A4 */
  int rho_bound_floor;    /* A10 */
  int cell_div;           /* k: cells of size 2h/k, stencil (2k+1)^dim */
  double cell_size;       /* 0 -> 2h/k */
  int visco_model;        /* 0: artificial viscosity, Eq. 21-22; 1: laminar viscosity, Eq. 23 (NEXT-2) */
  double nu0;             /* kinematic viscosity of Eq. 23 */
  int ddt_model;          /* 0: Molteni-Colagrossi, Eq. 18; 1: Fourtakas et al., Eq. 19-20 (NEXT-2) */
  int boundary_model;     /* 0: DBC, Eq. 36; 1: mDBC, Eq. 38-39 (NEXT-3) */
  int mdbc_slip;          /* 0: boundary velocity stays the imposed one; 1: no-slip, v_B = 2 v_wall - v_G (Eq. 39, A26) */
  double mdbc_det_min;    /* smallest |det| of the corrected-gradient system that is still solved (A25) */
  int shift_model;        /* 0: none; 1: Fickian shifting, Eq. 40-41, 53-54 (NEXT-4) */
  double shift_coef;      /* A_s of Eq. 41 */
  double shift_fs_conc;   /* a fluid particle with C_a below this value is treated as a free-surface particle (A29) */
  double shift_alpha_n;   /* a_n of Eq. 54 */
  double shift_beta_n;    /* beta_n of Eq. 54 */
} orc_params;

typedef struct {
  int group, axis;
  double stroke, period, phase;
} orc_motion;

/* ------------------------------------------------------------------------------------ */
/* Kernel, gradient, equation of state                                                  */
/* ------------------------------------------------------------------------------------ */

/* alpha_D of the Wendland C2 kernel: 7/(4 pi h^2) in 2-D, 21/(16 pi h^3) in 3-D
 * (below Eq. 11). */
ORC_API double orc_alphaD(int dim, double h) {
  const double pi = 3.14159265358979323846;
  return dim == 2 ? 7.0 / (4.0 * pi * h * h) : 21.0 / (16.0 * pi * h * h * h);
}

/* Wendland C2: W = alpha_D (1 - q/2)^4 (2q + 1), 0 <= q <= 2, q = r/h (Eq. 11). */
ORC_API double orc_W(int dim, double h, double r) {
  double q = r / h;
  if (q >= 2.0) return 0.0;
  double w = 1.0 - 0.5 * q;
  return orc_alphaD(dim, h) * w * w * w * w * (2.0 * q + 1.0);
}

/* grad_a W_ab = f_ab * r_ab with f_ab = -5 alpha_D (1 - q/2)^3 / h^2.
 * Derivation from Eq. 11: dW/dq = alpha_D [ -2 (1-q/2)^3 (2q+1) + 2 (1-q/2)^4 ]
 *                               = -5 alpha_D q (1-q/2)^3;
 * grad W = (dW/dq) (1/h) r_ab / r = -5 alpha_D (1-q/2)^3 / h^2 * r_ab. */
ORC_API double orc_fab(int dim, double h, double r) {
  double q = r / h;
  if (q >= 2.0) return 0.0;
  double w = 1.0 - 0.5 * q;
  return -5.0 * orc_alphaD(dim, h) * w * w * w / (h * h);
}

/* Tait equation of state, Eq. 28: P = (c_s^2 rho0 / gamma) [ (rho/rho0)^gamma - 1 ]. */
ORC_API double orc_eos(const orc_params* p, double rho) {
  double B = p->c0 * p->c0 * p->rho0 / p->gamma;
  return B * (pow(rho / p->rho0, p->gamma) - 1.0);
}

/* ------------------------------------------------------------------------------------ */
/* Cell grid, canonical position state (C1), keys / order / ranges (C3)                 */
/* ------------------------------------------------------------------------------------ */

static double cell_size_of(const orc_params* p) {
  return p->cell_size > 0.0 ? p->cell_size : 2.0 * p->h / (double)p->cell_div;
}

/* Grid: cubic cells of size cs = 2h/k ("cubic cells of size 2h", 635 "size h");
 * n_k = ceil((max_k - min_k)/cs); a 2-D case has one cell layer in y.  R2u = (2h/cs)^2 as float
 * is the squared support in cell units used by the pair predicate C2. */
ORC_API void orc_grid(const orc_params* p, double* cs_out, int ncell[3], float* R2u_out) {
  double cs = cell_size_of(p);
  for (int k = 0; k < 3; k++) {
    if (p->dim == 2 && k == 1) { ncell[k] = 1; continue; }
    double ext = (p->domain_max[k] - p->domain_min[k]) / cs;
    int n = (int)ceil(ext - 1e-9);  /* a periodic length that is an exact multiple must not gain a cell */
    if (n < 1) n = 1;
    ncell[k] = n;
  }
  if (cs_out) *cs_out = cs;
  if (R2u_out) { double s = 2.0 * p->h / cs; *R2u_out = (float)(s * s); }
}

/* C1: canonical position state.  s = (x - min)/cs; c = floor(s); u = rint((s - c) 2^22) 2^-22;
 * u == 1 -> c += 1, u = 0.  IEEE double, each operation rounded on its own (-ffp-contract=off).
 * This is the paper's "relative position of the particle within its cell (using single
 * precision)" made exactly reproducible.  Particles outside the grid on a
 * non-periodic axis are flagged out (A16); on a periodic axis the cell index wraps. */
static void canon1(const orc_params* p, const int ncell[3], double cs, const double x[3],
                   int32_t c[3], float u[3], uint8_t* out) {
  *out = 0;
  for (int k = 0; k < 3; k++) {
    if (p->dim == 2 && k == 1) { c[k] = 0; u[k] = 0.0f; continue; }
    double s = (x[k] - p->domain_min[k]) / cs;
    double fl = floor(s);
    double uu = rint((s - fl) * 4194304.0) * (1.0 / 4194304.0);
    if (uu >= 1.0) { fl += 1.0; uu = 0.0; }
    long ci = (long)fl;
    if (p->periodic[k]) {
      ci %= ncell[k];
      if (ci < 0) ci += ncell[k];
    } else if (ci < 0 || ci >= ncell[k] || !(s == s)) {
      *out = 1;
      ci = 0; uu = 0.0;
    }
    c[k] = (int32_t)ci;
    u[k] = (float)uu;
  }
}

ORC_API void orc_canonicalize(const orc_params* p, int64_t n, const double* pos,
                              int32_t* cell, float* u, uint8_t* out) {
  int ncell[3]; double cs;
  orc_grid(p, &cs, ncell, NULL);
  for (int64_t i = 0; i < n; i++) canon1(p, ncell, cs, pos + 3 * i, cell + 3 * i, u + 3 * i, out + i);
}

/* Inverse of C1: x = min + (c + u) cs in double; this is taken as the true position. */
ORC_API void orc_position(const orc_params* p, int64_t n, const int32_t* cell, const float* u,
                          double* pos) {
  int ncell[3]; double cs;
  orc_grid(p, &cs, ncell, NULL);
  for (int64_t i = 0; i < n; i++)
    for (int k = 0; k < 3; k++) {
      if (p->dim == 2 && k == 1) { pos[3 * i + k] = 0.0; continue; }
      pos[3 * i + k] = p->domain_min[k] + ((double)cell[3 * i + k] + (double)u[3 * i + k]) * cs;
    }
}

/* C3: key = block * ncells + (cx + nx (cy + ny cz)); block 0 = boundary, 1 = fluid;
 * out-of-grid particles get key 2*ncells (sorted last, excluded). */
ORC_API void orc_keys(const orc_params* p, int64_t n, const int32_t* cell, const uint8_t* type,
                      const uint8_t* out, uint32_t* key) {
  int nc[3];
  orc_grid(p, NULL, nc, NULL);
  uint32_t ncells = (uint32_t)nc[0] * (uint32_t)nc[1] * (uint32_t)nc[2];
  for (int64_t i = 0; i < n; i++) {
    if (out[i]) { key[i] = 2u * ncells; continue; }
    uint32_t lin = (uint32_t)cell[3 * i] + (uint32_t)nc[0] * ((uint32_t)cell[3 * i + 1] + (uint32_t)nc[1] * (uint32_t)cell[3 * i + 2]);
    key[i] = (type[i] == 0 ? ncells : 0u) + lin;
  }
}

/* Stable sort by key: a counting sort over the key range, which visits particles in their
 * current order -> the unique stable permutation ("particles with their data are sorted
 * according to the cell").  perm[j] = index (current order) of the j-th sorted
 * particle; cellstart[k] = #{keys < k}, k = 0..nkeys (prefix-count convention: range of key k is
 * [cellstart[k], cellstart[k+1]), empty cells have begin = end) -- the paper's "index array with
 * the first and last particle of each cell". */
ORC_API void orc_sort(int64_t n, const uint32_t* key, uint32_t nkeys, uint32_t* perm,
                      uint32_t* cellstart /* nkeys + 1 */) {
  memset(cellstart, 0, sizeof(uint32_t) * ((size_t)nkeys + 1));
  for (int64_t i = 0; i < n; i++) cellstart[key[i] + 1]++;      /* counts, shifted by one */
  for (uint32_t k = 0; k < nkeys; k++) cellstart[k + 1] += cellstart[k];
  uint32_t* cur = (uint32_t*)malloc(sizeof(uint32_t) * (size_t)nkeys);
  memcpy(cur, cellstart, sizeof(uint32_t) * (size_t)nkeys);
  for (int64_t i = 0; i < n; i++) perm[cur[key[i]]++] = (uint32_t)i;
  free(cur);
}

/* ------------------------------------------------------------------------------------ */
/* Pair evaluation                                                                       */
/* ------------------------------------------------------------------------------------ */

typedef struct {
  int dim, k;
  int nc[3];
  double cs, h, m, B, aD, eta2, c0, alpha, delta, rho0, gamma;
  float R2u;
  double R2exact;   /* (2h)^2 */
} consts_t;

static void make_consts(const orc_params* p, consts_t* C) {
  C->dim = p->dim; C->k = p->cell_div;
  orc_grid(p, &C->cs, C->nc, &C->R2u);
  C->h = p->h;
  C->m = p->rho0 * pow(p->dp, p->dim);             /* A9: m = rho0 dp^d for every particle (V = dr^d) */
  C->B = p->c0 * p->c0 * p->rho0 / p->gamma;       /* Eq. 28 */
  C->aD = orc_alphaD(p->dim, p->h);                /* Eq. 11 */
  C->eta2 = p->eta2_coef * p->h * p->h;            /* A6: eta^2 = 0.001 h^2 */
  C->c0 = p->c0; C->alpha = p->alpha; C->delta = p->delta; C->rho0 = p->rho0; C->gamma = p->gamma;
  C->R2exact = 4.0 * p->h * p->h;
}

typedef struct {
  double F[3];      /* momentum sum (without gravity) */
  double R;         /* continuity sum incl. D_a */
  double visc;      /* max |mu_ab| over this particle's evaluated pairs */
  uint32_t nb;      /* number of neighbours (C2 predicate) */
  uint32_t nb_exact_diff;  /* pairs where the exact double predicate disagrees with C2 */
} accum_t;

/* C2, canonical pair predicate, evaluated in fp32 exactly as stated:
 *   du_k = u_a - (u_b + dc_k)  (exact on the 2^-22 grid, |values| < 4)
 *   r2u  = fmaf(du_z,du_z, fmaf(du_y,du_y, du_x*du_x))   (2-D: no y term)
 *   pair <=> b != a and r2u < R2u.
 * Returns 1 if pair; du_out receives the (exact) offsets in cell units as doubles. */
static inline int pair_predicate(const consts_t* C, const float ua[3], const float ub[3],
                                 const int dc[3], double du_out[3], int* exact_pair) {
  float dux = ua[0] - (ub[0] + (float)dc[0]);
  float duy = C->dim == 3 ? ua[1] - (ub[1] + (float)dc[1]) : 0.0f;
  float duz = ua[2] - (ub[2] + (float)dc[2]);
  float r2u = dux * dux;
  if (C->dim == 3) r2u = fmaf(duy, duy, r2u);
  r2u = fmaf(duz, duz, r2u);
  du_out[0] = dux; du_out[1] = duy; du_out[2] = duz;
  /* exact double predicate |r_ab| < 2h (Eq. 4 with k = 2, A2), for the report only */
  double rx = (double)dux * C->cs, ry = (double)duy * C->cs, rz = (double)duz * C->cs;
  *exact_pair = (rx * rx + ry * ry + rz * rz) < C->R2exact;
  return r2u < C->R2u;
}

/* One ordered pair (a receives from b). Steps 4-6 of SURVEY 8(c), i.e. Eq. 15, 17-18, 21-22, 36.
 * a_fluid / b_fluid select the evaluated pair types: (F<-F), (F<-B), (B<-F); B<-B never. */
static inline void pair_terms(const consts_t* C, const orc_params* p, int a_fluid, int b_fluid,
                              const double du[3], const double va[3], const double vb[3],
                              double rho_a, double rho_b, double P_a, double P_b, accum_t* A) {
  /* r_ab = r_a - r_b, v_ab = v_a - v_b */
  double r[3] = {du[0] * C->cs, du[1] * C->cs, du[2] * C->cs};
  double v[3] = {va[0] - vb[0], va[1] - vb[1], va[2] - vb[2]};
  double r2 = r[0] * r[0] + r[1] * r[1] + r[2] * r[2];
  double rr = sqrt(r2);
  double f = orc_fab(C->dim, C->h, rr);                 /* grad_a W_ab = f r_ab */
  double vr = v[0] * r[0] + v[1] * r[1] + v[2] * r[2];  /* v_ab . r_ab */
  double Vb = C->m / rho_b;                             /* V_b = m_b / rho_b */

  /* continuity, Eq. 15 (fluid a) / Eq. 36 (boundary a, fluid b only): rho_a sum V_b v_ab.grad W */
  A->R += rho_a * Vb * vr * f;

  /* density diffusion, Eq. 17-18, diffusive reading A3: D_a = 2 delta h c0 sum (rho_a - rho_b) f V_b,
   * fluid a only, fluid b only unless ddt_over_boundary (A4); c_a = c0 (A5). */
  if (a_fluid && (b_fluid || p->ddt_over_boundary)) {
    double drho = rho_a - rho_b;
    if (p->ddt_model == 1) {
      /* Fourtakas et al., Eq. 19-20: only the dynamic part of the density difference
       * diffuses.  The hydrostatic part is built locally from P^H_ab = rho0 g z_ab (Eq. 20; written here as
       * rho0 g . r_ab for any direction of g) through the inverse of the Tait EOS (Eq. 28, "barotropic"):
       * rho^H_ab = rho0 [ (1 + P^H_ab / B)^(1/gamma) - 1 ]  (reading A23). */
      double PH = C->rho0 * (p->g[0] * r[0] + p->g[1] * r[1] + p->g[2] * r[2]);
      double rhoH = C->rho0 * (pow(1.0 + PH / C->B, 1.0 / C->gamma) - 1.0);
      drho -= rhoH;
    }
    A->R += 2.0 * C->delta * C->h * C->c0 * drho * f * Vb;
  }

  /* mu_ab = h v_ab.r_ab / (r^2 + eta^2)  (Eq. 21; A12 for the dt) */
  double mu = C->h * vr / (r2 + C->eta2);
  if (fabs(mu) > A->visc) A->visc = fabs(mu);

  if (a_fluid) {
    /* artificial viscosity, Eq. 21: Pi_ab = -alpha cbar mu / rhobar if v_ab.r_ab < 0 else 0;
     * cbar = c0 (A5), rhobar = (rho_a + rho_b)/2 (A7) */
    double Pi = 0.0;
    if (vr < 0.0) Pi = -C->alpha * C->c0 * mu / (0.5 * (rho_a + rho_b));
    /* momentum, Eq. 22: - sum m_b ( (P_a + P_b)/(rho_a rho_b) + Pi_ab ) grad W */
    if (p->visco_model == 1) Pi = 0.0;    /* laminar: Eq. 23 replaces the artificial term of Eq. 22 (A22) */
    double coef = -C->m * ((P_a + P_b) / (rho_a * rho_b) + Pi) * f;
    A->F[0] += coef * r[0]; A->F[1] += coef * r[1]; A->F[2] += coef * r[2];
    if (p->visco_model == 1) {
      /* laminar viscosity, Eq. 23 (Lo & Shao):
       * nu0 lap(v)_a = sum_b m_b 4 nu0 (r_ab . grad_a W_ab) / ((rho_a + rho_b)(r_ab^2 + eta^2)) v_ab,
       * with r_ab . grad_a W_ab = f r^2 */
      double lam = C->m * 4.0 * p->nu0 * (f * r2) / ((rho_a + rho_b) * (r2 + C->eta2));
      A->F[0] += lam * v[0]; A->F[1] += lam * v[1]; A->F[2] += lam * v[2];
    }
  }
}

/* One interaction pass on state {cell,u,v,rho,type}:  acc (n x 3) = F_a incl. gravity for fluid,
 * 0 for boundary;  drho (n) = R_a;  nbcount;  *viscmax = max |mu_ab|;
 * *n_diff = number of ordered pairs where C2 (fp32) and the exact double predicate disagree.
 * mode 0: brute force O(N^2) over all ordered pairs; mode 1: the oracle's own cell list.
 * Out-of-grid particles (A16) are excluded on both sides. */
ORC_API int orc_interactions(const orc_params* p, int64_t n, const int32_t* cell, const float* u,
                             const uint8_t* out, const double* vel, const double* rho,
                             const uint8_t* type, int mode, double* acc, double* drho,
                             uint32_t* nbcount, double* viscmax, uint64_t* n_diff) {
  consts_t C; make_consts(p, &C);
  const int K = C.k;
  double* P = (double*)malloc(sizeof(double) * (size_t)n);
  for (int64_t i = 0; i < n; i++) P[i] = orc_eos(p, rho[i]);   /* step 2: P_a for all a */

  uint32_t *perm = NULL, *cellstart = NULL, *key = NULL;
  uint32_t ncells = (uint32_t)C.nc[0] * (uint32_t)C.nc[1] * (uint32_t)C.nc[2];
  if (mode == 1) {
    /* own cell list, keyed by cell only (types mixed; independent of the C3 layout) */
    key = (uint32_t*)malloc(sizeof(uint32_t) * (size_t)n);
    for (int64_t i = 0; i < n; i++)
      key[i] = out[i] ? ncells
                      : (uint32_t)cell[3 * i] + (uint32_t)C.nc[0] * ((uint32_t)cell[3 * i + 1] + (uint32_t)C.nc[1] * (uint32_t)cell[3 * i + 2]);
    perm = (uint32_t*)malloc(sizeof(uint32_t) * (size_t)n);
    cellstart = (uint32_t*)malloc(sizeof(uint32_t) * ((size_t)ncells + 2));
    orc_sort(n, key, ncells + 1, perm, cellstart);
  }

  double vmax = 0.0;
  uint64_t ndiff = 0;
#pragma omp parallel for schedule(dynamic, 256) reduction(max : vmax) reduction(+ : ndiff)
  for (int64_t a = 0; a < n; a++) {
    accum_t A; memset(&A, 0, sizeof(A));
    acc[3 * a] = acc[3 * a + 1] = acc[3 * a + 2] = 0.0; drho[a] = 0.0; nbcount[a] = 0;
    if (out[a]) continue;
    const int a_fluid = type[a] == 0;
    const float* ua = u + 3 * a;
    const int32_t* ca = cell + 3 * a;

    if (mode == 0) {
      for (int64_t b = 0; b < n; b++) {
        if (b == a || out[b]) continue;                 /* A17: self excluded by index */
        const int b_fluid = type[b] == 0;
        if (!a_fluid && !b_fluid) continue;             /* B<-B never evaluated (Eq. 36) */
        int dc[3]; int far = 0;
        for (int k = 0; k < 3; k++) {
          int d = cell[3 * b + k] - ca[k];
          if (p->periodic[k]) {                         /* minimum image in whole cells (A15) */
            int nk = C.nc[k];
            d %= nk; if (d < 0) d += nk;                /* 0..nk-1 */
            if (d > nk / 2) d -= nk;
            /* for tiny periodic grids (nk <= 2K) several images could be in range; not supported */
          }
          dc[k] = d;
          if (d > K || d < -K) far = 1;                 /* |du| > K >= sqrt(R2u): cannot be a pair */
        }
        if (far) continue;
        double du[3]; int ex;
        int pr = pair_predicate(&C, ua, u + 3 * b, dc, du, &ex);
        if (pr != ex) A.nb_exact_diff++;
        if (!pr) continue;
        A.nb++;
        pair_terms(&C, p, a_fluid, b_fluid, du, vel + 3 * a, vel + 3 * b, rho[a], rho[b], P[a], P[b], &A);
      }
    } else {
      const int kz0 = -K, kz1 = K;
      const int ky0 = C.dim == 3 ? -K : 0, ky1 = C.dim == 3 ? K : 0;
      for (int dz = kz0; dz <= kz1; dz++)
        for (int dy = ky0; dy <= ky1; dy++)
          for (int dx = -K; dx <= K; dx++) {
            int d3[3] = {dx, dy, dz}; int cc[3]; int skip = 0;
            for (int k = 0; k < 3; k++) {
              int c2 = ca[k] + d3[k];
              if (p->periodic[k]) { c2 %= C.nc[k]; if (c2 < 0) c2 += C.nc[k]; }
              else if (c2 < 0 || c2 >= C.nc[k]) skip = 1;
              cc[k] = c2;
            }
            if (skip) continue;
            uint32_t lin = (uint32_t)cc[0] + (uint32_t)C.nc[0] * ((uint32_t)cc[1] + (uint32_t)C.nc[1] * (uint32_t)cc[2]);
            for (uint32_t j = cellstart[lin]; j < cellstart[lin + 1]; j++) {
              int64_t b = perm[j];
              if (b == a) continue;
              const int b_fluid = type[b] == 0;
              if (!a_fluid && !b_fluid) continue;
              double du[3]; int ex;
              int pr = pair_predicate(&C, ua, u + 3 * b, d3, du, &ex);
              if (pr != ex) A.nb_exact_diff++;
              if (!pr) continue;
              A.nb++;
              pair_terms(&C, p, a_fluid, b_fluid, du, vel + 3 * a, vel + 3 * b, rho[a], rho[b], P[a], P[b], &A);
            }
          }
    }
    if (a_fluid) {   /* + f: external acceleration, gravity (Eq. 22) */
      acc[3 * a] = A.F[0] + p->g[0]; acc[3 * a + 1] = A.F[1] + p->g[1]; acc[3 * a + 2] = A.F[2] + p->g[2];
    }
    drho[a] = A.R;
    nbcount[a] = A.nb;
    if (A.visc > vmax) vmax = A.visc;
    ndiff += A.nb_exact_diff;
  }
  *viscmax = vmax;
  if (n_diff) *n_diff = ndiff;
  free(P); free(perm); free(cellstart); free(key);
  return 0;
}

/* ------------------------------------------------------------------------------------ */
/* Neighbour enumeration for the NEXT-3 / NEXT-4 sums                                   */
/* ------------------------------------------------------------------------------------ */

/* The oracle's own cell list, keyed by cell only (all types mixed), as in orc_interactions mode 1. */
typedef struct {
  uint32_t *perm, *cellstart;
} celllist_t;

static void celllist_build(const consts_t* C, int64_t n, const int32_t* cell, const uint8_t* out, celllist_t* L) {
  uint32_t ncells = (uint32_t)C->nc[0] * (uint32_t)C->nc[1] * (uint32_t)C->nc[2];
  uint32_t* key = (uint32_t*)malloc(sizeof(uint32_t) * (size_t)(n > 0 ? n : 1));
  for (int64_t i = 0; i < n; i++)
    key[i] = out[i] ? ncells
                    : (uint32_t)cell[3 * i] + (uint32_t)C->nc[0] * ((uint32_t)cell[3 * i + 1] + (uint32_t)C->nc[1] * (uint32_t)cell[3 * i + 2]);
  L->perm = (uint32_t*)malloc(sizeof(uint32_t) * (size_t)(n > 0 ? n : 1));
  L->cellstart = (uint32_t*)malloc(sizeof(uint32_t) * ((size_t)ncells + 2));
  orc_sort(n, key, ncells + 1, L->perm, L->cellstart);
  free(key);
}
static void celllist_free(celllist_t* L) { free(L->perm); free(L->cellstart); }

/* Calls cb(user, b, du) for every particle b != a, of any type, that is a neighbour of a by the canonical
 * predicate C2 (the same neighbour set as the interaction pass, plus boundary-boundary pairs).
 * du = (r_a - r_b)/cs.  mode 0: brute force; mode 1: cell list L. */
typedef void (*pair_cb)(void* user, int64_t b, const double du[3]);
static void each_neighbour(const consts_t* C, const orc_params* p, int64_t n, const int32_t* cell, const float* u,
                           const uint8_t* out, int mode, const celllist_t* L, int64_t a, pair_cb cb, void* user) {
  const int K = C->k;
  const float* ua = u + 3 * a;
  const int32_t* ca = cell + 3 * a;
  if (mode == 0) {
    for (int64_t b = 0; b < n; b++) {
      if (b == a || out[b]) continue;
      int dc[3]; int far = 0;
      for (int k = 0; k < 3; k++) {
        int d = cell[3 * b + k] - ca[k];
        if (p->periodic[k]) {
          int nk = C->nc[k];
          d %= nk; if (d < 0) d += nk;
          if (d > nk / 2) d -= nk;
        }
        dc[k] = d;
        if (d > K || d < -K) far = 1;
      }
      if (far) continue;
      double du[3]; int ex;
      if (pair_predicate(C, ua, u + 3 * b, dc, du, &ex)) cb(user, b, du);
    }
    return;
  }
  const int ky = C->dim == 3 ? K : 0;
  for (int dz = -K; dz <= K; dz++)
    for (int dy = -ky; dy <= ky; dy++)
      for (int dx = -K; dx <= K; dx++) {
        int d3[3] = {dx, dy, dz}; int cc[3]; int skip = 0;
        for (int k = 0; k < 3; k++) {
          int c2 = ca[k] + d3[k];
          if (p->periodic[k]) { c2 %= C->nc[k]; if (c2 < 0) c2 += C->nc[k]; }
          else if (c2 < 0 || c2 >= C->nc[k]) skip = 1;
          cc[k] = c2;
        }
        if (skip) continue;
        uint32_t lin = (uint32_t)cc[0] + (uint32_t)C->nc[0] * ((uint32_t)cc[1] + (uint32_t)C->nc[1] * (uint32_t)cc[2]);
        for (uint32_t j = L->cellstart[lin]; j < L->cellstart[lin + 1]; j++) {
          int64_t b = L->perm[j];
          if (b == a) continue;
          double du[3]; int ex;
          if (pair_predicate(C, ua, u + 3 * b, d3, du, &ex)) cb(user, b, du);
        }
      }
}

/* ------------------------------------------------------------------------------------ */
/* NEXT-3: modified dynamic boundary conditions, Eq. 38-39            */
/* ------------------------------------------------------------------------------------ */

/* Solve the m x m system A x = b (m <= 4) by Gaussian elimination with partial pivoting.
 * Returns the determinant of A (0 if a pivot vanishes; x is then not set). */
static double solve_small(int m, double A[4][4], double b[4], double x[4]) {
  double det = 1.0;
  for (int c = 0; c < m; c++) {
    int piv = c;
    for (int r = c + 1; r < m; r++) if (fabs(A[r][c]) > fabs(A[piv][c])) piv = r;
    if (A[piv][c] == 0.0) return 0.0;
    if (piv != c) {
      for (int k = 0; k < m; k++) { double t = A[c][k]; A[c][k] = A[piv][k]; A[piv][k] = t; }
      double t = b[c]; b[c] = b[piv]; b[piv] = t;
      det = -det;
    }
    det *= A[c][c];
    for (int r = c + 1; r < m; r++) {
      double f = A[r][c] / A[c][c];
      for (int k = c; k < m; k++) A[r][k] -= f * A[c][k];
      b[r] -= f * b[c];
    }
  }
  for (int r = m - 1; r >= 0; r--) {
    double s = b[r];
    for (int k = r + 1; k < m; k++) s -= A[r][k] * x[k];
    x[r] = s / A[r][r];
  }
  return det;
}

/* mDBC.  For every boundary particle B (type != 0, in the grid):
 *   ghost node  r_G = r_B + 2 n_B, n_B = the vector from the particle to the boundary interface, supplied by the
 *               caller ("a ghost node is projected into the fluid across a boundary interface", A24);
 *   corrected SPH approximation of Liu & Liu at r_G over the FLUID particles b within 2h of r_G:  with
 *               d = r_b - r_G, W = W(|d|), grad_G W = -f d, V_b = m/rho_b, the unknowns (rho_G, grad rho_G) solve
 *                 [ sum V W          sum V W d_j          ] [ rho_G      ]   [ sum m W          ]
 *                 [ sum V grad_i W   sum V grad_i W d_j   ] [ grad_j rho ] = [ sum m grad_i W   ]
 *               (the Taylor expansion rho_b = rho_G + grad rho_G . d, multiplied by V_b W and by V_b grad_i W and
 *               summed; rho_b V_b = m);
 *   Eq. 38      rho_B = rho_G + (r_B - r_G) . grad rho_G = rho_G - 2 n_B . grad rho_G;
 *   Eq. 39      v_G = sum V v_b W / sum V W;  mdbc_slip = 1: v_B = 2 v_wall - v_G ("this velocity with the
 *               direction reversed", generalised to a moving wall, A26); mdbc_slip = 0: v_B = v_wall.
 * Fallbacks (the paper is silent, A25): |det| < mdbc_det_min -> Shepard value rho_B = sum m W / sum V W, no
 * gradient; no fluid particle within 2h of the ghost node -> rho_B = rho0, v_B = v_wall.
 * The ghost node is not a particle, so distances are evaluated in double from the canonical positions (the
 * exact predicate |d| < 2h), with the minimum image on periodic axes.
 * vel, rho: in/out (fluid entries read, boundary entries written).  vwall: n x 3 or NULL (= 0).
 * status (n, may be NULL): 0 not a boundary particle / out, 1 full solve, 2 Shepard, 3 no neighbour. */
ORC_API int orc_mdbc(const orc_params* p, int64_t n, const int32_t* cell, const float* u, const uint8_t* out,
                     double* vel, double* rho, const uint8_t* type, const double* normals, const double* vwall,
                     int mode, uint8_t* status) {
  consts_t C; make_consts(p, &C);
  const int K = C.k;
  const int dim = C.dim, m1 = dim + 1;
  const int ax[3] = {0, dim == 3 ? 1 : 2, 2};        /* active axes: (x, y, z) or (x, z) */
  double* pos = (double*)malloc(sizeof(double) * 3 * (size_t)(n > 0 ? n : 1));
  orc_position(p, n, cell, u, pos);
  celllist_t L = {NULL, NULL};
  if (mode == 1) celllist_build(&C, n, cell, out, &L);
  double Lk[3];
  for (int k = 0; k < 3; k++) Lk[k] = (double)C.nc[k] * C.cs;
  double* rho_new = (double*)malloc(sizeof(double) * (size_t)(n > 0 ? n : 1));
  double* vel_new = (double*)malloc(sizeof(double) * 3 * (size_t)(n > 0 ? n : 1));

#pragma omp parallel for schedule(dynamic, 64)
  for (int64_t a = 0; a < n; a++) {
    if (status) status[a] = 0;
    rho_new[a] = rho[a];
    for (int k = 0; k < 3; k++) vel_new[3 * a + k] = vel[3 * a + k];
    if (type[a] == 0 || out[a]) continue;
    double nrm[3] = {0.0, 0.0, 0.0}, vw[3] = {0.0, 0.0, 0.0};
    for (int k = 0; k < 3; k++) {
      if (normals) nrm[k] = normals[3 * a + k];
      if (vwall) vw[k] = vwall[3 * a + k];
    }
    if (dim == 2) nrm[1] = 0.0;
    double xg[3];
    for (int k = 0; k < 3; k++) xg[k] = pos[3 * a + k] + 2.0 * nrm[k];

    double A[4][4] = {{0}}, rhs[4] = {0}, sv[3] = {0, 0, 0};
    uint32_t nb = 0;
    /* candidate fluid particles: brute force, or the cells around the ghost node's cell */
    int cg[3]; int cg_valid = 1;
    for (int k = 0; k < 3; k++) {
      if (dim == 2 && k == 1) { cg[k] = 0; continue; }
      double sg = floor((xg[k] - p->domain_min[k]) / C.cs);
      long ci = (long)sg;
      if (p->periodic[k]) { ci %= C.nc[k]; if (ci < 0) ci += C.nc[k]; }
      else if (ci < -K || ci >= C.nc[k] + K) cg_valid = 0;    /* farther than the stencil from every cell */
      cg[k] = (int)ci;
    }
#define MDBC_PAIR(b)                                                                               \
    do {                                                                                           \
      if (type[b] != 0 || out[b]) break;                                                           \
      double d[3], r2 = 0.0;                                                                       \
      for (int k = 0; k < 3; k++) {                                                                \
        d[k] = pos[3 * (b) + k] - xg[k];                                                           \
        if (dim == 2 && k == 1) d[k] = 0.0;                                                        \
        if (p->periodic[k]) d[k] -= Lk[k] * rint(d[k] / Lk[k]);                                    \
        r2 += d[k] * d[k];                                                                         \
      }                                                                                            \
      if (!(r2 < C.R2exact)) break;                                                                \
      double rr = sqrt(r2), Wb = orc_W(dim, C.h, rr), f = orc_fab(dim, C.h, rr);                   \
      double Vb = C.m / rho[b];                                                                    \
      double gW[3] = {-f * d[0], -f * d[1], -f * d[2]};     /* gradient w.r.t. the ghost node */   \
      nb++;                                                                                        \
      A[0][0] += Vb * Wb; rhs[0] += C.m * Wb;                                                      \
      for (int j = 0; j < dim; j++) A[0][1 + j] += Vb * Wb * d[ax[j]];                             \
      for (int i = 0; i < dim; i++) {                                                              \
        A[1 + i][0] += Vb * gW[ax[i]]; rhs[1 + i] += C.m * gW[ax[i]];                              \
        for (int j = 0; j < dim; j++) A[1 + i][1 + j] += Vb * gW[ax[i]] * d[ax[j]];                \
      }                                                                                            \
      for (int k = 0; k < 3; k++) sv[k] += Vb * vel[3 * (b) + k] * Wb;                             \
    } while (0)
    if (mode == 0) {
      for (int64_t b = 0; b < n; b++) MDBC_PAIR(b);
    } else if (cg_valid) {
      const int ky = dim == 3 ? K : 0;
      for (int dz = -K; dz <= K; dz++)
        for (int dy = -ky; dy <= ky; dy++)
          for (int dx = -K; dx <= K; dx++) {
            int d3[3] = {dx, dy, dz}; int cc[3]; int skip = 0;
            for (int k = 0; k < 3; k++) {
              int c2 = cg[k] + d3[k];
              if (p->periodic[k]) { c2 %= C.nc[k]; if (c2 < 0) c2 += C.nc[k]; }
              else if (c2 < 0 || c2 >= C.nc[k]) skip = 1;
              cc[k] = c2;
            }
            if (skip) continue;
            uint32_t lin = (uint32_t)cc[0] + (uint32_t)C.nc[0] * ((uint32_t)cc[1] + (uint32_t)C.nc[1] * (uint32_t)cc[2]);
            for (uint32_t j = L.cellstart[lin]; j < L.cellstart[lin + 1]; j++) { int64_t b = L.perm[j]; MDBC_PAIR(b); }
          }
    }
#undef MDBC_PAIR
    if (nb == 0 || !(A[0][0] > 0.0)) {       /* no fluid in reach of the ghost node (A25) */
      rho_new[a] = p->rho0;
      for (int k = 0; k < 3; k++) vel_new[3 * a + k] = vw[k];
      if (status) status[a] = 3;
      continue;
    }
    const double shep_rho = rhs[0] / A[0][0], sumVW = A[0][0];
    double x[4] = {0, 0, 0, 0};
    double det = solve_small(m1, A, rhs, x);
    if (fabs(det) >= p->mdbc_det_min) {
      double rb = x[0];
      for (int j = 0; j < dim; j++) rb += -2.0 * nrm[ax[j]] * x[1 + j];     /* Eq. 38 */
      rho_new[a] = rb;
      if (status) status[a] = 1;
    } else {
      rho_new[a] = shep_rho;
      if (status) status[a] = 2;
    }
    for (int k = 0; k < 3; k++) {
      double vg = sv[k] / sumVW;                                             /* Eq. 39 */
      vel_new[3 * a + k] = p->mdbc_slip == 1 ? 2.0 * vw[k] - vg : vw[k];
    }
    if (dim == 2) vel_new[3 * a + 1] = vw[1];
  }
  for (int64_t a = 0; a < n; a++) {
    if (type[a] == 0 || out[a]) continue;
    rho[a] = rho_new[a];
    for (int k = 0; k < 3; k++) vel[3 * a + k] = vel_new[3 * a + k];
  }
  free(pos); free(rho_new); free(vel_new);
  if (mode == 1) celllist_free(&L);
  return 0;
}

/* ------------------------------------------------------------------------------------ */
/* NEXT-4: particle shifting, Eq. 40-41 with Eq. 53-54 (434-442)     */
/* ------------------------------------------------------------------------------------ */

typedef struct { const consts_t* C; const double* rho; double sum; } conc_ctx;
static void conc_cb(void* user, int64_t b, const double du[3]) {
  conc_ctx* X = (conc_ctx*)user;
  double r = sqrt(du[0] * du[0] + du[1] * du[1] + du[2] * du[2]) * X->C->cs;
  X->sum += X->C->m / X->rho[b] * orc_W(X->C->dim, X->C->h, r);
}

/* Particle concentration, second half of Eq. 53: C_a = sum_{b in P} (m_b/rho_b) W_ab "computed through the sum
 * of the smoothing kernel", for every particle a of any type, over every particle b of any type within 2h,
 * b = a included (W(0); reading A27).  Neighbours by the canonical predicate C2. */
ORC_API int orc_concentration(const orc_params* p, int64_t n, const int32_t* cell, const float* u,
                              const uint8_t* out, const double* rho, const uint8_t* type, int mode, double* conc) {
  (void)type;
  consts_t C; make_consts(p, &C);
  celllist_t L = {NULL, NULL};
  if (mode == 1) celllist_build(&C, n, cell, out, &L);
#pragma omp parallel for schedule(dynamic, 256)
  for (int64_t a = 0; a < n; a++) {
    conc[a] = 0.0;
    if (out[a]) continue;
    conc_ctx X = {&C, rho, C.m / rho[a] * orc_W(C.dim, C.h, 0.0)};
    each_neighbour(&C, p, n, cell, u, out, mode, &L, a, conc_cb, &X);
    conc[a] = X.sum;
  }
  if (mode == 1) celllist_free(&L);
  return 0;
}

typedef struct { const consts_t* C; const double* rho; const double* conc; double Ca; double g[3]; } gradc_ctx;
static void gradc_cb(void* user, int64_t b, const double du[3]) {
  gradc_ctx* X = (gradc_ctx*)user;
  const consts_t* C = X->C;
  double r[3] = {du[0] * C->cs, du[1] * C->cs, du[2] * C->cs};
  double f = orc_fab(C->dim, C->h, sqrt(r[0] * r[0] + r[1] * r[1] + r[2] * r[2]));
  double w = C->m / X->rho[b] * (X->conc[b] - X->Ca) * f;          /* V_b (C_b - C_a), grad_a W_ab = f r_ab */
  X->g[0] += w * r[0]; X->g[1] += w * r[1]; X->g[2] += w * r[2];
}

/* Shifting velocity s_a = delta r_a / dt of every fluid particle (0 for boundary particles):
 *   Eq. 53   grad C_a = sum_{b in P} (m_b/rho_b) (C_b - C_a) grad_a W_ab  (conc = C of orc_concentration);
 *   Eq. 40-41  delta r_a = -D_s grad C_a,  D_s = A_s h |v_a| dt   =>  s_a = -A_s h |v_a| grad C_a;
 *   Eq. 54   for a free-surface particle (C_a < shift_fs_conc, A29) the shift is restricted to
 *            -D_s [ dC/ds s + dC/db b + a_n (dC/dn - beta_n) n ] with the surface normal taken along the
 *            concentration gradient, n = -grad C_a/|grad C_a| (pointing out of the fluid, A29); the tangential
 *            derivatives then vanish identically and dC/dn = -|grad C_a|, leaving
 *            s_a = -A_s h |v_a| a_n (-|grad C_a| - beta_n) n.
 * gradc (n x 3, may be NULL) receives grad C_a. */
ORC_API int orc_shift_velocity(const orc_params* p, int64_t n, const int32_t* cell, const float* u,
                               const uint8_t* out, const double* vel, const double* rho, const uint8_t* type,
                               const double* conc, int mode, double* shift, double* gradc) {
  consts_t C; make_consts(p, &C);
  celllist_t L = {NULL, NULL};
  if (mode == 1) celllist_build(&C, n, cell, out, &L);
#pragma omp parallel for schedule(dynamic, 256)
  for (int64_t a = 0; a < n; a++) {
    shift[3 * a] = shift[3 * a + 1] = shift[3 * a + 2] = 0.0;
    if (gradc) gradc[3 * a] = gradc[3 * a + 1] = gradc[3 * a + 2] = 0.0;
    if (out[a] || type[a] != 0) continue;
    gradc_ctx X = {&C, rho, conc, conc[a], {0.0, 0.0, 0.0}};
    each_neighbour(&C, p, n, cell, u, out, mode, &L, a, gradc_cb, &X);
    if (gradc) { gradc[3 * a] = X.g[0]; gradc[3 * a + 1] = X.g[1]; gradc[3 * a + 2] = X.g[2]; }
    const double* v = vel + 3 * a;
    double vmag = sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
    double Ds = p->shift_coef * C.h * vmag;                         /* D_s / dt, Eq. 41 */
    if (conc[a] < p->shift_fs_conc) {                               /* Eq. 54 */
      double gn = sqrt(X.g[0] * X.g[0] + X.g[1] * X.g[1] + X.g[2] * X.g[2]);
      if (gn > 0.0) {
        double fac = -Ds * p->shift_alpha_n * (-gn - p->shift_beta_n);
        for (int k = 0; k < 3; k++) shift[3 * a + k] = fac * (-X.g[k] / gn);
      }
    } else {
      for (int k = 0; k < 3; k++) shift[3 * a + k] = -Ds * X.g[k];  /* Eq. 40 */
    }
  }
  if (mode == 1) celllist_free(&L);
  return 0;
}

/* Eq. 35 with A12/A13: dt_f = min_{a in F} sqrt(h/|F_a|) (F_a incl. gravity),
 * dt_cv = h / (c0 + max_pairs |mu_ab|), dt = CFL min(dt_f, dt_cv). */
ORC_API double orc_dt(const orc_params* p, int64_t n, const double* acc, const uint8_t* type,
                      const uint8_t* out, double viscmax) {
  double dtf = INFINITY;
  for (int64_t a = 0; a < n; a++) {
    if (type[a] != 0 || out[a]) continue;
    double fa = sqrt(acc[3 * a] * acc[3 * a] + acc[3 * a + 1] * acc[3 * a + 1] + acc[3 * a + 2] * acc[3 * a + 2]);
    if (fa > 0.0) { double d = sqrt(p->h / fa); if (d < dtf) dtf = d; }
  }
  double dtcv = p->h / (p->c0 + viscmax);
  return p->cfl * (dtf < dtcv ? dtf : dtcv);
}

/* Imposed motion of a boundary group (Eq. 37, config 4): displacement of the group at time t
 * relative to t = 0 along `axis`: (stroke/2) [sin(2 pi t/T + phase) - sin(phase)], and its
 * time derivative as the imposed velocity. */
static void motion_at(const orc_motion* m, double t, double* disp, double* velc) {
  const double pi = 3.14159265358979323846;
  double w = 2.0 * pi / m->period;
  *disp = 0.5 * m->stroke * (sin(w * t + m->phase) - sin(m->phase));
  *velc = 0.5 * m->stroke * w * cos(w * t + m->phase);
}

/* Before an interaction pass on the state at time t_state, with boundary_model = 1: the boundary particles take
 * their density and velocity from the ghost nodes (orc_mdbc); v_wall is the imposed velocity of the particle
 * (the motion law at t_state for a moving group, else 0). */
static void mdbc_before_pass(const orc_params* p, int64_t n, const int32_t* cell, const float* u, const uint8_t* out,
                             double* vel, double* rho, const uint8_t* type, const double* normals,
                             const orc_motion* motions, int nmotions, double t_state, int mode) {
  if (p->boundary_model != 1) return;
  double* vw = (double*)calloc(3 * (size_t)(n > 0 ? n : 1), sizeof(double));
  for (int64_t a = 0; a < n; a++)
    if (type[a] >= 2)
      for (int j = 0; j < nmotions; j++)
        if (motions[j].group == type[a]) {
          double d, vv; motion_at(&motions[j], t_state, &d, &vv);
          vw[3 * a + motions[j].axis] = vv;
        }
  orc_mdbc(p, n, cell, u, out, vel, rho, type, normals, vw, mode, NULL);
  free(vw);
}

/* After the last interaction pass of a step, with shift_model = 1: shifting velocity of that state (Eq. 40-41, 53-54). */
static void shift_after_pass(const orc_params* p, int64_t n, const int32_t* cell, const float* u, const uint8_t* out,
                             const double* vel, const double* rho, const uint8_t* type, int mode, double* shift) {
  double* conc = (double*)malloc(sizeof(double) * (size_t)(n > 0 ? n : 1));
  orc_concentration(p, n, cell, u, out, rho, type, mode, conc);
  orc_shift_velocity(p, n, cell, u, out, vel, rho, type, conc, mode, shift, NULL);
  free(conc);
}

/* nsteps symplectic position-Verlet predictor-corrector steps, Eq. 33-34,
 * variable dt from the pass at state n (A8).  Positions live in the canonical (cell,u) state and are
 * re-quantised (C1) after every position update.  vel, rho are double in/out.
 * pos0 (n x 3 double): positions at t = 0 of moving-boundary particles (only read for type >= 2).
 * Returns 0; *t is advanced; dt_hist (nsteps) receives each step's dt if not NULL. */
ORC_API int orc_step(const orc_params* p, int64_t n, int32_t* cell, float* u, uint8_t* out,
                     double* vel, double* rho, const uint8_t* type, int nsteps,
                     const orc_motion* motions, int nmotions, const double* pos0, const double* normals,
                     double* t, double* dt_hist, int mode) {
  int ncell[3]; double cs;
  orc_grid(p, &cs, ncell, NULL);
  const int mdbc = p->boundary_model == 1;
  double* shift = p->shift_model == 1 ? (double*)calloc(3 * (size_t)(n > 0 ? n : 1), sizeof(double)) : NULL;
  double* pos_n = (double*)malloc(sizeof(double) * 3 * (size_t)n);
  double* vel_n = (double*)malloc(sizeof(double) * 3 * (size_t)n);
  double* rho_n = (double*)malloc(sizeof(double) * (size_t)n);
  double* F = (double*)malloc(sizeof(double) * 3 * (size_t)n);
  double* R = (double*)malloc(sizeof(double) * (size_t)n);
  uint32_t* nb = (uint32_t*)malloc(sizeof(uint32_t) * (size_t)n);
  double x[3];

  for (int s = 0; s < nsteps; s++) {
    double visc;
    /* state n */
    orc_position(p, n, cell, u, pos_n);
    mdbc_before_pass(p, n, cell, u, out, vel, rho, type, normals, motions, nmotions, *t, mode);
    memcpy(vel_n, vel, sizeof(double) * 3 * (size_t)n);
    memcpy(rho_n, rho, sizeof(double) * (size_t)n);
    orc_interactions(p, n, cell, u, out, vel, rho, type, mode, F, R, nb, &visc, NULL);   /* F^n, R^n */
    double dt = orc_dt(p, n, F, type, out, visc);
    if (dt_hist) dt_hist[s] = dt;

    /* predictor: r^{n+1/2} = r^n + dt/2 v^n ; v^{n+1/2} = v^n + dt/2 F^n ; rho^{n+1/2} = rho^n + dt/2 R^n */
    for (int64_t a = 0; a < n; a++) {
      if (out[a]) continue;
      if (type[a] == 0) {
        for (int k = 0; k < 3; k++) {
          x[k] = pos_n[3 * a + k] + 0.5 * dt * vel_n[3 * a + k];
          vel[3 * a + k] = vel_n[3 * a + k] + 0.5 * dt * F[3 * a + k];
        }
        canon1(p, ncell, cs, x, cell + 3 * a, u + 3 * a, out + a);
      } else if (type[a] >= 2) {          /* boundary with imposed motion: law at t + dt/2 */
        for (int k = 0; k < 3; k++) { x[k] = pos0[3 * a + k]; vel[3 * a + k] = 0.0; }
        for (int j = 0; j < nmotions; j++)
          if (motions[j].group == type[a]) {
            double d, vv; motion_at(&motions[j], *t + 0.5 * dt, &d, &vv);
            x[motions[j].axis] += d; vel[3 * a + motions[j].axis] = vv;
          }
        canon1(p, ncell, cs, x, cell + 3 * a, u + 3 * a, out + a);
      }
      if (mdbc && type[a] != 0) continue;            /* mDBC: the boundary density is not integrated (A24) */
      rho[a] = rho_n[a] + 0.5 * dt * R[a];           /* fluid and boundary alike (A11) */
      if (type[a] != 0 && p->rho_bound_floor && rho[a] < p->rho0) rho[a] = p->rho0;   /* A10 */
    }

    /* second pass at (r, v, rho)^{n+1/2}: neighbours rebuilt */
    mdbc_before_pass(p, n, cell, u, out, vel, rho, type, normals, motions, nmotions, *t + 0.5 * dt, mode);
    orc_interactions(p, n, cell, u, out, vel, rho, type, mode, F, R, nb, &visc, NULL);   /* F^{n+1/2}, R^{n+1/2} */
    if (shift) shift_after_pass(p, n, cell, u, out, vel, rho, type, mode, shift);       /* of the state n+1/2 */

    /* corrector: v^{n+1} = v^n + dt F^{n+1/2}; r^{n+1} = r^n + dt (v^{n+1} + v^n)/2;
     * eps = -(R^{n+1/2}/rho^{n+1/2}) dt; rho^{n+1} = rho^n (2 - eps)/(2 + eps)   (Eq. 33-34) */
    for (int64_t a = 0; a < n; a++) {
      if (out[a]) continue;
      double eps = -(R[a] / rho[a]) * dt;
      if (type[a] == 0) {
        for (int k = 0; k < 3; k++) {
          double vn1 = vel_n[3 * a + k] + dt * F[3 * a + k];
          x[k] = pos_n[3 * a + k] + dt * 0.5 * (vn1 + vel_n[3 * a + k]);
          if (shift) x[k] += dt * shift[3 * a + k];      /* delta r_a = -D_s grad C_a, Eq. 40-41 (A28) */
          vel[3 * a + k] = vn1;
        }
        canon1(p, ncell, cs, x, cell + 3 * a, u + 3 * a, out + a);
      } else if (type[a] >= 2) {          /* law at t + dt */
        for (int k = 0; k < 3; k++) { x[k] = pos0[3 * a + k]; vel[3 * a + k] = 0.0; }
        for (int j = 0; j < nmotions; j++)
          if (motions[j].group == type[a]) {
            double d, vv; motion_at(&motions[j], *t + dt, &d, &vv);
            x[motions[j].axis] += d; vel[3 * a + motions[j].axis] = vv;
          }
        canon1(p, ncell, cs, x, cell + 3 * a, u + 3 * a, out + a);
      }
      if (mdbc && type[a] != 0) continue;
      rho[a] = rho_n[a] * (2.0 - eps) / (2.0 + eps);
      if (type[a] != 0 && p->rho_bound_floor && rho[a] < p->rho0) rho[a] = p->rho0;
    }
    *t += dt;
  }
  free(shift);
  free(pos_n); free(vel_n); free(rho_n); free(F); free(R); free(nb);
  return 0;
}

/* nsteps Verlet steps, Eq. 30-31: ONE interaction pass per step.
 *   regular step  (Eq. 30): v^{n+1} = v^{n-1} + 2 dt F^n ; rho^{n+1} = rho^{n-1} + 2 dt R^n
 *   corrective step (Eq. 31): v^{n+1} = v^n + dt F^n     ; rho^{n+1} = rho^n + dt R^n
 *   both                    : r^{n+1} = r^n + dt v^n + dt^2/2 F^n
 * Readings (A21): the step counter k starts at 0 at load; step k is corrective when
 * k mod N_S == 0 -- which includes the very first step, where no state n-1 exists -- N_S = verlet_steps
 * ("N_S ~ 40 is recommended"); dt is the variable dt of Eq. 35 from this step's pass, used as
 * printed (2 dt^n) although Eq. 30 assumes a constant step; boundary particles integrate rho with the same
 * formulas (as A11) and take r, v from the motion law at t + dt.
 * vel_m1 (n x 3), rho_m1 (n): state n-1, in/out (ignored on corrective steps); *kstep: counter, in/out. */
ORC_API int orc_step_verlet(const orc_params* p, int64_t n, int32_t* cell, float* u, uint8_t* out,
                            double* vel, double* rho, double* vel_m1, double* rho_m1, const uint8_t* type,
                            int nsteps, int verlet_steps, int64_t* kstep, const orc_motion* motions, int nmotions,
                            const double* pos0, const double* normals, double* t, double* dt_hist, int mode) {
  int ncell[3]; double cs;
  orc_grid(p, &cs, ncell, NULL);
  const int mdbc = p->boundary_model == 1;
  double* shift = p->shift_model == 1 ? (double*)calloc(3 * (size_t)(n > 0 ? n : 1), sizeof(double)) : NULL;
  double* pos_n = (double*)malloc(sizeof(double) * 3 * (size_t)n);
  double* F = (double*)malloc(sizeof(double) * 3 * (size_t)n);
  double* R = (double*)malloc(sizeof(double) * (size_t)n);
  uint32_t* nb = (uint32_t*)malloc(sizeof(uint32_t) * (size_t)n);
  double x[3];
  for (int s = 0; s < nsteps; s++) {
    double visc;
    orc_position(p, n, cell, u, pos_n);
    mdbc_before_pass(p, n, cell, u, out, vel, rho, type, normals, motions, nmotions, *t, mode);
    orc_interactions(p, n, cell, u, out, vel, rho, type, mode, F, R, nb, &visc, NULL);   /* F^n, R^n */
    if (shift) shift_after_pass(p, n, cell, u, out, vel, rho, type, mode, shift);       /* of the state n */
    double dt = orc_dt(p, n, F, type, out, visc);
    if (dt_hist) dt_hist[s] = dt;
    const int corrective = (*kstep % verlet_steps) == 0;
    for (int64_t a = 0; a < n; a++) {
      if (out[a]) continue;
      const double rho_n = rho[a];
      if (type[a] == 0) {
        for (int k = 0; k < 3; k++) {
          const double vn = vel[3 * a + k], f = F[3 * a + k];
          x[k] = pos_n[3 * a + k] + dt * vn + 0.5 * dt * dt * f;
          if (shift) x[k] += dt * shift[3 * a + k];      /* Eq. 40-41 (A28) */
          vel[3 * a + k] = corrective ? vn + dt * f : vel_m1[3 * a + k] + 2.0 * dt * f;
          vel_m1[3 * a + k] = vn;
        }
        canon1(p, ncell, cs, x, cell + 3 * a, u + 3 * a, out + a);
      } else if (type[a] >= 2) {          /* boundary with imposed motion: law at t + dt */
        for (int k = 0; k < 3; k++) { x[k] = pos0[3 * a + k]; vel[3 * a + k] = 0.0; }
        for (int j = 0; j < nmotions; j++)
          if (motions[j].group == type[a]) {
            double d, vv; motion_at(&motions[j], *t + dt, &d, &vv);
            x[motions[j].axis] += d; vel[3 * a + motions[j].axis] = vv;
          }
        canon1(p, ncell, cs, x, cell + 3 * a, u + 3 * a, out + a);
      }
      if (!(mdbc && type[a] != 0)) {                 /* mDBC: the boundary density is not integrated (A24) */
        rho[a] = corrective ? rho_n + dt * R[a] : rho_m1[a] + 2.0 * dt * R[a];
        if (type[a] != 0 && p->rho_bound_floor && rho[a] < p->rho0) rho[a] = p->rho0;   /* A10 */
      }
      rho_m1[a] = rho_n;
    }
    *kstep += 1;
    *t += dt;
  }
  free(shift);
  free(pos_n); free(F); free(R); free(nb);
  return 0;
}

ORC_API int orc_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

ORC_API void orc_set_num_threads(int nthreads) {
#ifdef _OPENMP
  omp_set_num_threads(nthreads);
#else
  (void)nthreads;
#endif
}
