/*
 * oracle/bit1_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, single-threaded CPU oracle of the BIT1-style 1D3V electrostatic
 * PIC-MC timestep (gather + Boris push, wall absorption / re-injection,
 * null-collision Monte Carlo, stable counting sort by cell, int64 fixed-point
 * charge deposition, exact integer-scan Poisson solve).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may build, load or call this file.  It shares no code,
 * header, table generator or helper with the CUDA path under
 * paper_2606_28534_b200/csrc/; every constant below is typed here a second
 * time on purpose.
 *
 * What fixes the algorithm.  The paper names the phases of the
 * cycle and their order only -- PAPER.md:33 (Background, "PIC cycle": mover,
 * deposition, field solver, force interpolation, plus MC collisions),
 * PAPER.md:95 (Table 3: walls absorb plasma and take its charge),
 * PAPER.md:111/121 (mover move0/moveb followed by arranger arrj/narrj).  It
 * prints no equation.  Every numerical rule is therefore the reading recorded
 * in SURVEY.md section 8(c) and DESIGN.md "Readings" (A1..A27 and the R-/N- readings added while building), which follow
 * BASELINE.json's north_star and textbook PIC-MCC (Birdsall-Langdon leapfrog
 * and Boris rotation; Vahedi-Surendra null collision; Salmon et al. Philox).
 * Each function cites the reading it implements.
 *
 * Arithmetic policy: every fp64 + - * / sqrt
 * is one IEEE-754 round-to-nearest operation in exactly the order written;
 * compile with -ffp-contract=off; no libm call inside a step (llrint, used
 * once at create time, is the only libm routine).
 *
 * Beyond the hot path: density smoothing and time-averaged diagnostics (NEXT-1, readings N1-a/b),
 * wall recycling and neutral particles as the collision target (NEXT-2, readings N2-a/b), and reading R-thr
 * (ionisation cross-section zero at or below the threshold).
 *
 * Pins: see tests/test_oracle_*.py (moments and density: test_oracle_moments.py; NEXT-1: test_oracle_next1.py;
 * NEXT-2: test_oracle_next2.py).  No function here
 * is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef __int128 i128;
typedef unsigned __int128 u128;

#define ORC_MAX_SPECIES 8

/* species process flags */
#define F_ELASTIC 1u
#define F_IONISE 2u
#define F_CX 4u
#define F_ION_PRODUCT 8u
#define F_ELECTRON_PRODUCT 16u
#define F_TARGET_MAXWELLIAN 32u

#define SRC_NONE 0
#define SRC_SELF 1
#define SRC_PAIR 2

/* sticky flag bits */
#define FLAG_CAPACITY 1u
#define FLAG_ESCAPE 2u

/* physical constants, CODATA 2018 (SURVEY.md 8(d) "Synthetic inputs") */
static const double E_CHARGE = 1.602176634e-19;
static const double EPS0 = 8.8541878128e-12;
static const double TWO_M32 = 2.3283064365386962890625e-10;  /* 2^-32 */
static const double TWO_M52 = 2.220446049250313080847263336181640625e-16; /* 2^-52 */
static const double TWO_M40 = 9.094947017729282379150390625e-13; /* 2^-40 */
static const double TWO_P32 = 4294967296.0;
static const double TWO_P64 = 18446744073709551616.0;

typedef struct {
  /* grid */
  int32_t nc, bc, ng; /* bc 0 periodic, 1 absorbing walls */
  double dx, area, B[3], dt;
  /* species */
  int32_t ns;
  double q[ORC_MAX_SPECIES], m[ORC_MAX_SPECIES], weight[ORC_MAX_SPECIES];
  uint32_t flags[ORC_MAX_SPECIES];
  int32_t src_mode[ORC_MAX_SPECIES], src_partner[ORC_MAX_SPECIES];
  double src_vth[ORC_MAX_SPECIES], pnull[ORC_MAX_SPECIES], numax[ORC_MAX_SPECIES];
  /* derived once */
  double inv_dx, L, h[ORC_MAX_SPECIES], t[ORC_MAX_SPECIES][3], s[ORC_MAX_SPECIES][3];
  double kin_eV[ORC_MAX_SPECIES], two_e_over_m[ORC_MAX_SPECIES], el_loss[ORC_MAX_SPECIES];
  int64_t Q[ORC_MAX_SPECIES];
  int32_t sign[ORC_MAX_SPECIES];
  double Kphi, KE;
  /* options */
  uint64_t seed, capacity;
  double src_lo, src_hi, n0, vth_n, E_ion, m_n, dE_eV;
  int32_t n_sig, n_norm;
  double *sig_el, *sig_ion, *sig_cx, *inv_norm;
  int32_t sp_electron_product, sp_ion_product;
  /* particle state (SoA), capacity entries each */
  double *x, *vx, *vy, *vz;
  int32_t *cell;
  uint32_t *pid;
  uint8_t *sp;
  /* scratch for the sort */
  double *x2, *vx2, *vy2, *vz2;
  int32_t *cell2;
  uint32_t *pid2;
  uint8_t *sp2;
  uint64_t n;       /* live particles (slots 0..n-1) */
  uint64_t n_slots; /* slots in use after the push phase: n + births of the step */
  int64_t *cell_start; /* nc+1 */
  /* grid state */
  int64_t *dens; /* ns * ng, fixed point */
  int64_t *rho;  /* ng */
  double *phi, *E; /* nc+1 each (periodic: ghost copy at nc) */
  /* counters */
  uint64_t step;
  uint32_t next_pid;
  uint64_t wall_count[2][ORC_MAX_SPECIES];
  int64_t wall_charge[2];
  uint32_t flagword;
  uint64_t diag_nu_overflow, diag_dir_fallback, diag_escape, diag_births, diag_reinject;
  uint64_t diag_candidates[ORC_MAX_SPECIES];
  uint64_t diag_events[ORC_MAX_SPECIES][3]; /* elastic, ionise, cx */
  /* NEXT-2: wall recycling, per species: index of the species born at the wall (-1 = none) */
  int32_t recycle_to[ORC_MAX_SPECIES];
  double recycle_vth[ORC_MAX_SPECIES];
  uint64_t diag_recycled;
  int32_t target_species; /* -1: analytic uniform background n0; else the stored species whose density is the target */
  double kn;
  /* NEXT-1: density smoothing and time-averaged diagnostics */
  int32_t smooth_passes; /* 0 = off */
  int64_t *rho_s;        /* ng: 4^passes * smoothed rho, what the field solve used */
  int32_t avg_window, avg_interval; /* mvflag, mvStep; 0 = off */
  int64_t *acc_dens, *avg_dens;     /* ns*ng running / latched sums over the window */
  double *acc_phi, *avg_phi;        /* nc+1 */
  uint64_t acc_count, avg_count, avg_step;
} orc;

/* ------------------------------------------------------------------ */
/* R (random numbers): Philox4x32-10, Salmon et al. SC'11; SURVEY 8(c) "R". */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
  uint32_t k0 = key[0], k1 = key[1];
  for (int r = 0; r < 10; ++r) {
    uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
    uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
    uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
    uint32_t n1 = (uint32_t)p1;
    uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
    uint32_t n3 = (uint32_t)p0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += 0x9E3779B9u;
    k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* Two-word uniform in (0,1): (((a<<32|b)>>12)+0.5)*2^-52, exact in fp64.
 * DESIGN.md reading R-U: SURVEY 8(c) "R" wrote >>11 and 2^-53, but w+0.5 then needs
 * 54 bits and the top value rounds to 1.0; 52 bits keep the stated range (0,1). */
double orc_u53(uint32_t a, uint32_t b) {
  uint64_t w = (((uint64_t)a << 32) | (uint64_t)b) >> 12;
  return ((double)w + 0.5) * TWO_M52;
}
/* 32-bit uniform in (0,1): (a+0.5)*2^-32. */
double orc_u32(uint32_t a) { return ((double)a + 0.5) * TWO_M32; }

/* Counter layout: (pid, step_lo, step_hi, slot), key (seed_lo, seed_hi). */
static void draw(const orc *o, uint32_t pid, uint64_t step, uint32_t slot, uint32_t w[4]) {
  uint32_t ctr[4] = {pid, (uint32_t)step, (uint32_t)(step >> 32), slot};
  uint32_t key[2] = {(uint32_t)o->seed, (uint32_t)(o->seed >> 32)};
  orc_philox4x32_10(ctr, key, w);
}

/* Normal deviate from one 32-bit word by the caller's piecewise-linear inverse
 * CDF table (n_norm+1 entries).  SURVEY 8(c) "R", reading A18. */
static double normal_from_word(const orc *o, uint32_t a) {
  double t = orc_u32(a) * (double)o->n_norm;
  int32_t i = (int32_t)t;
  if (i > o->n_norm - 1) i = o->n_norm - 1;
  return o->inv_norm[i] + (t - (double)i) * (o->inv_norm[i + 1] - o->inv_norm[i]);
}
double orc_normal(const orc *o, uint32_t a) { return normal_from_word(o, a); }

/* Isotropic unit vector without sin/cos: rejection on the unit disc
 * (Marsaglia 1972).  Four Philox blocks first_slot..first_slot+3, two attempts
 * each.  SURVEY 8(c) "R". Returns 1 when all 8 attempts failed. */
static int direction(const orc *o, uint32_t pid, uint64_t step, uint32_t first_slot, double n[3]) {
  for (uint32_t b = 0; b < 4; ++b) {
    uint32_t w[4];
    draw(o, pid, step, first_slot + b, w);
    for (int a = 0; a < 2; ++a) {
      double p = 2.0 * orc_u32(w[2 * a]) - 1.0;
      double q = 2.0 * orc_u32(w[2 * a + 1]) - 1.0;
      double S = p * p + q * q;
      if (S > 0.0 && S < 1.0) {
        double r = sqrt(1.0 - S);
        n[0] = 1.0 - 2.0 * S;
        n[1] = (2.0 * p) * r;
        n[2] = (2.0 * q) * r;
        return 0;
      }
    }
  }
  n[0] = 1.0; n[1] = 0.0; n[2] = 0.0;
  return 1;
}
int orc_direction(const orc *o, uint32_t pid, uint64_t step, uint32_t first_slot, double n[3]) {
  return direction(o, pid, step, first_slot, n);
}

/* Cross-section table lookup, uniform grid in eV, clamped.  SURVEY 8(c) "C". */
static double sigma_lookup(const orc *o, const double *tab, double E_eV) {
  double t = E_eV / o->dE_eV;
  double tmax = (double)(o->n_sig - 1);
  if (t > tmax) t = tmax;
  if (!(t >= 0.0)) t = 0.0;
  int32_t i = (int32_t)t;
  if (i > o->n_sig - 2) i = o->n_sig - 2;
  double fr = t - (double)i;
  if (fr > 1.0) fr = 1.0;
  return tab[i] + fr * (tab[i + 1] - tab[i]);
}
double orc_sigma(const orc *o, int which, double E_eV) {
  const double *tab = which == 0 ? o->sig_el : which == 1 ? o->sig_ion : o->sig_cx;
  return sigma_lookup(o, tab, E_eV);
}

/* ------------------------------------------------------------------ */
static void *xcalloc(size_t n, size_t sz) {
  void *p = calloc(n ? n : 1, sz);
  if (!p) abort();
  return p;
}
static double *dup_table(const double *src, int32_t n) {
  double *d = (double *)xcalloc((size_t)n, sizeof(double));
  if (src) memcpy(d, src, (size_t)n * sizeof(double));
  return d;
}

/* Create.  Derived constants by the expressions in DESIGN.md "Derived
 * constants"; the CUDA library computes the same quantities by its own copy of
 * these expressions. */
orc *orc_create(int32_t nc, double dx, int32_t bc, double area, const double B[3], double dt,
                int32_t ns, const double *q, const double *m, const double *weight,
                const uint32_t *flags, const int32_t *src_mode, const int32_t *src_partner,
                const double *src_vth, const double *pnull, const double *numax,
                uint64_t seed, uint64_t capacity, double src_lo, double src_hi, double n0,
                double vth_n, double E_ion, double m_n, const double *sig_el,
                const double *sig_ion, const double *sig_cx, int32_t n_sig, double dE_eV,
                const double *inv_norm, int32_t n_norm) {
  if (nc < 2 || ns < 1 || ns > ORC_MAX_SPECIES || !(dx > 0.0) || !(dt > 0.0)) return NULL;
  orc *o = (orc *)xcalloc(1, sizeof(orc));
  o->nc = nc; o->bc = bc; o->ng = bc ? nc + 1 : nc;
  o->dx = dx; o->area = area; o->dt = dt;
  o->B[0] = B[0]; o->B[1] = B[1]; o->B[2] = B[2];
  o->ns = ns;
  o->inv_dx = 1.0 / dx;
  o->L = (double)nc * dx;
  o->sp_electron_product = -1; o->sp_ion_product = -1;
  for (int s = 0; s < ns; ++s) {
    o->q[s] = q[s]; o->m[s] = m[s]; o->weight[s] = weight[s]; o->flags[s] = flags[s];
    o->src_mode[s] = src_mode[s]; o->src_partner[s] = src_partner[s];
    o->src_vth[s] = src_vth[s]; o->pnull[s] = pnull[s]; o->numax[s] = numax[s];
    double h = 0.5 * ((q[s] / m[s]) * dt);
    o->h[s] = h;
    double tx = h * B[0], ty = h * B[1], tz = h * B[2];
    double tt = (tx * tx + ty * ty) + tz * tz;
    o->t[s][0] = tx; o->t[s][1] = ty; o->t[s][2] = tz;
    o->s[s][0] = (2.0 * tx) / (1.0 + tt);
    o->s[s][1] = (2.0 * ty) / (1.0 + tt);
    o->s[s][2] = (2.0 * tz) / (1.0 + tt);
    o->kin_eV[s] = (0.5 * m[s]) / E_CHARGE;
    o->two_e_over_m[s] = (2.0 * E_CHARGE) / m[s];
    o->el_loss[s] = (2.0 * m[s]) / m_n;
    o->recycle_to[s] = -1;
    o->target_species = -1;
    o->Q[s] = (int64_t)llrint((E_CHARGE * weight[s]) * 1099511627776.0);
    o->sign[s] = q[s] > 0.0 ? 1 : (q[s] < 0.0 ? -1 : 0);
    if (o->Q[s] < 1 || o->Q[s] >= ((int64_t)1 << 31)) { free(o); return NULL; }
    if ((flags[s] & F_ELECTRON_PRODUCT) && o->sp_electron_product < 0) o->sp_electron_product = s;
    if ((flags[s] & F_ION_PRODUCT) && o->sp_ion_product < 0) o->sp_ion_product = s;
  }
  o->Kphi = (TWO_M40 * dx) / ((area * EPS0) * (double)nc);
  o->KE = TWO_M40 / (((2.0 * (double)nc) * area) * EPS0);
  if (!bc) { o->Kphi = o->Kphi / (double)nc; o->KE = o->KE / (double)nc; }
  o->seed = seed; o->capacity = capacity;
  o->src_lo = src_lo; o->src_hi = src_hi; o->n0 = n0; o->vth_n = vth_n;
  o->E_ion = E_ion; o->m_n = m_n; o->dE_eV = dE_eV; o->n_sig = n_sig; o->n_norm = n_norm;
  o->sig_el = dup_table(sig_el, n_sig > 0 ? n_sig : 2);
  o->sig_ion = dup_table(sig_ion, n_sig > 0 ? n_sig : 2);
  o->sig_cx = dup_table(sig_cx, n_sig > 0 ? n_sig : 2);
  o->inv_norm = dup_table(inv_norm, n_norm + 1);
  size_t cap = (size_t)capacity;
  o->x = xcalloc(cap, 8); o->vx = xcalloc(cap, 8); o->vy = xcalloc(cap, 8); o->vz = xcalloc(cap, 8);
  o->cell = xcalloc(cap, 4); o->pid = xcalloc(cap, 4); o->sp = xcalloc(cap, 1);
  o->x2 = xcalloc(cap, 8); o->vx2 = xcalloc(cap, 8); o->vy2 = xcalloc(cap, 8); o->vz2 = xcalloc(cap, 8);
  o->cell2 = xcalloc(cap, 4); o->pid2 = xcalloc(cap, 4); o->sp2 = xcalloc(cap, 1);
  o->cell_start = xcalloc((size_t)nc + 1, 8);
  o->dens = xcalloc((size_t)ns * (size_t)o->ng, 8);
  o->rho = xcalloc((size_t)o->ng, 8);
  o->phi = xcalloc((size_t)nc + 1, 8);
  o->E = xcalloc((size_t)nc + 1, 8);
  o->rho_s = xcalloc((size_t)o->ng, 8);
  o->acc_dens = xcalloc((size_t)ns * (size_t)o->ng, 8);
  o->avg_dens = xcalloc((size_t)ns * (size_t)o->ng, 8);
  o->acc_phi = xcalloc((size_t)nc + 1, 8);
  o->avg_phi = xcalloc((size_t)nc + 1, 8);
  return o;
}

void orc_destroy(orc *o) {
  if (!o) return;
  free(o->sig_el); free(o->sig_ion); free(o->sig_cx); free(o->inv_norm);
  free(o->x); free(o->vx); free(o->vy); free(o->vz); free(o->cell); free(o->pid); free(o->sp);
  free(o->x2); free(o->vx2); free(o->vy2); free(o->vz2); free(o->cell2); free(o->pid2); free(o->sp2);
  free(o->cell_start); free(o->dens); free(o->rho); free(o->phi); free(o->E);
  free(o->rho_s); free(o->acc_dens); free(o->avg_dens); free(o->acc_phi); free(o->avg_phi);
  free(o);
}

/* Cell of a position: (int)(x*inv_dx) clamped to [0, nc-1].  SURVEY 8(c) "W". */
static int32_t cell_of(const orc *o, double x) {
  double t = x * o->inv_dx;
  if (!(t >= 0.0)) t = 0.0;
  if (t > (double)(o->nc - 1)) t = (double)(o->nc - 1);
  return (int32_t)t;
}

/* ------------------------------------------------------------------ */
/* S (sort / compaction): stable counting sort by cell of slots 0..n_slots-1,
 * slots with cell < 0 (dead) dropped.  SURVEY 8(c) "S", reading A19;
 * PAPER.md:111 arranger arrj/narrj. */
void orc_phase_sort(orc *o) {
  int32_t nc = o->nc;
  int64_t *cs = o->cell_start;
  for (int32_t c = 0; c <= nc; ++c) cs[c] = 0;
  for (uint64_t i = 0; i < o->n_slots; ++i)
    if (o->cell[i] >= 0) cs[o->cell[i] + 1] += 1;
  for (int32_t c = 0; c < nc; ++c) cs[c + 1] += cs[c];
  int64_t *cursor = (int64_t *)xcalloc((size_t)nc, 8);
  for (int32_t c = 0; c < nc; ++c) cursor[c] = cs[c];
  for (uint64_t i = 0; i < o->n_slots; ++i) {
    int32_t c = o->cell[i];
    if (c < 0) continue;
    int64_t d = cursor[c]++;
    o->x2[d] = o->x[i]; o->vx2[d] = o->vx[i]; o->vy2[d] = o->vy[i]; o->vz2[d] = o->vz[i];
    o->cell2[d] = c; o->pid2[d] = o->pid[i]; o->sp2[d] = o->sp[i];
  }
  free(cursor);
  double *td; int32_t *ti; uint32_t *tu; uint8_t *tb;
  td = o->x; o->x = o->x2; o->x2 = td;
  td = o->vx; o->vx = o->vx2; o->vx2 = td;
  td = o->vy; o->vy = o->vy2; o->vy2 = td;
  td = o->vz; o->vz = o->vz2; o->vz2 = td;
  ti = o->cell; o->cell = o->cell2; o->cell2 = ti;
  tu = o->pid; o->pid = o->pid2; o->pid2 = tu;
  tb = o->sp; o->sp = o->sp2; o->sp2 = tb;
  o->n = (uint64_t)cs[nc];
  o->n_slots = o->n;
}

/* D (deposit): CIC weights in int64 fixed point, unit 2^-40 C.
 * "D", reading A4; PAPER.md:33 step (ii). */
void orc_phase_deposit(orc *o) {
  int32_t ng = o->ng, nc = o->nc;
  memset(o->dens, 0, (size_t)o->ns * (size_t)ng * 8);
  for (uint64_t i = 0; i < o->n; ++i) {
    int32_t c = o->cell[i];
    int s = o->sp[i];
    double f = o->x[i] * o->inv_dx - (double)c;
    uint64_t F;
    if (!(f > 0.0)) F = 0;
    else if (f >= 1.0) F = 4294967295ull;
    else {
      F = (uint64_t)(f * TWO_P32);
      if (F > 4294967295ull) F = 4294967295ull;
    }
    uint64_t Qs = (uint64_t)o->Q[s];
    uint64_t a = (Qs * F + 2147483648ull) >> 32;
    int32_t j1 = c + 1;
    if (!o->bc && j1 == nc) j1 = 0;
    o->dens[(size_t)s * ng + c] += (int64_t)(Qs - a);
    o->dens[(size_t)s * ng + j1] += (int64_t)a;
  }
  for (int32_t j = 0; j < ng; ++j) {
    int64_t r = 0;
    for (int s = 0; s < o->ns; ++s) r += (int64_t)o->sign[s] * o->dens[(size_t)s * ng + j];
    o->rho[j] = r;
  }
}

/* dbl(n) of an int128: sign(n) * ((double)hi(|n|) * 2^64 + (double)lo(|n|)), hi/lo the unsigned
 * 64-bit halves of the magnitude.  DESIGN.md reading R-dbl: SURVEY 8(c) "P" converted the two's
 * complement halves, which loses up to 2^11 units of a small negative n (lo is then near 2^64);
 * the tridiagonal-solve pin in tests/test_oracle_grid.py exposed it.  Magnitude first keeps the
 * relative error below 2^-52 for every n. */
static double dbl128(i128 n) {
  int neg = n < 0;
  u128 a = neg ? (u128)0 - (u128)n : (u128)n;
  uint64_t hi = (uint64_t)(a >> 64);
  uint64_t lo = (uint64_t)a;
  double d = (double)hi * TWO_P64 + (double)lo;
  return neg ? -d : d;
}

/* P (Poisson / field): exact integer double prefix sum of rho.
 * "P", readings A8, A22; PAPER.md:33 step (iii), PAPER.md:37 (native Poisson
 * solver).  Standalone so that tests can feed any rho. */
void orc_poisson(int32_t nc, int32_t bc, double Kphi, double KE, const int64_t *rho,
                 double *phi, double *E) {
  i128 *S = (i128 *)xcalloc((size_t)nc + 1, sizeof(i128));
  i128 *T = (i128 *)xcalloc((size_t)nc + 1, sizeof(i128));
  if (bc) {
    /* nodes 0..nc, phi_0 = phi_nc = 0; S_0 = 0, S_j = S_{j-1} + R_j;
     * T_0 = 0, T_j = T_{j-1} + S_{j-1}. */
    S[0] = 0; T[0] = 0;
    for (int32_t j = 1; j <= nc; ++j) {
      S[j] = S[j - 1] + (i128)rho[j];
      T[j] = T[j - 1] + S[j - 1];
    }
    i128 Tn = T[nc];
    for (int32_t j = 0; j <= nc; ++j) phi[j] = Kphi * dbl128((i128)j * Tn - (i128)nc * T[j]);
    for (int32_t j = 1; j < nc; ++j) E[j] = KE * dbl128((i128)nc * (S[j - 1] + S[j]) - 2 * Tn);
    E[0] = KE * dbl128(-2 * Tn - 2 * (i128)nc * (i128)rho[0]);
    E[nc] = KE * dbl128(2 * (i128)nc * S[nc - 1] - 2 * Tn + 2 * (i128)nc * (i128)rho[nc]);
  } else {
    /* nodes 0..nc-1; R'_j = nc*R_j - sum_k R_k (neutralising background);
     * gauge phi_0 = 0; Kphi, KE already carry the extra 1/nc. */
    i128 tot = 0;
    for (int32_t j = 0; j < nc; ++j) tot += (i128)rho[j];
    S[0] = 0; T[0] = 0;
    for (int32_t j = 1; j < nc; ++j) {
      S[j] = S[j - 1] + ((i128)nc * (i128)rho[j] - tot);
      T[j] = T[j - 1] + S[j - 1];
    }
    i128 Tn = T[nc - 1] + S[nc - 1]; /* T_nc = sum_{k=0}^{nc-1} S_k */
    for (int32_t j = 0; j < nc; ++j) phi[j] = Kphi * dbl128((i128)j * Tn - (i128)nc * T[j]);
    for (int32_t j = 0; j < nc; ++j) {
      i128 Sm = j == 0 ? S[nc - 1] : S[j - 1];
      E[j] = KE * dbl128((i128)nc * (Sm + S[j]) - 2 * Tn);
    }
    phi[nc] = phi[0];
    E[nc] = E[0];
  }
  free(S); free(T);
}

/* Density smoothing ("density smoothing ... improve[s] numerical stability", PAPER.md:37
 * "smoothing operators"; reading N1-a).  One pass of the 1-2-1 binomial
 * filter in exact integers: out_j = in_{j-1} + 2 in_j + in_{j+1} = 4 x the smoothed value (the 1/4 is
 * folded into the field constants).  Every node hands 1/4, 1/2, 1/4 of its charge to j-1, j, j+1;
 * periodic: indices wrap; bounded: the quarter that would leave through a wall stays on the wall node
 * (out_0 = 3 in_0 + in_1, out_nc = in_{nc-1} + 3 in_nc), so the total charge is conserved exactly:
 * sum(out) = 4 sum(in), and global Gauss's law keeps holding in the integers. */
void orc_smooth121(int32_t nc, int32_t bc, const int64_t *in, int64_t *out) {
  if (bc) {
    out[0] = 3 * in[0] + in[1];
    for (int32_t j = 1; j < nc; ++j) out[j] = in[j - 1] + 2 * in[j] + in[j + 1];
    out[nc] = in[nc - 1] + 3 * in[nc];
  } else {
    for (int32_t j = 0; j < nc; ++j) {
      int32_t jm = j == 0 ? nc - 1 : j - 1, jp = j == nc - 1 ? 0 : j + 1;
      out[j] = in[jm] + 2 * in[j] + in[jp];
    }
  }
}

/* Field phase: `smooth_passes` passes over rho (the per-species densities stay as deposited), then the
 * Poisson solve with both constants scaled by 4^-passes (an exact power of two). */
void orc_phase_field(orc *o) {
  int32_t p = o->smooth_passes;
  if (p <= 0) {
    orc_poisson(o->nc, o->bc, o->Kphi, o->KE, o->rho, o->phi, o->E);
    return;
  }
  int64_t *tmp = (int64_t *)xcalloc((size_t)o->ng, 8);
  memcpy(o->rho_s, o->rho, (size_t)o->ng * 8);
  for (int32_t k = 0; k < p; ++k) {
    orc_smooth121(o->nc, o->bc, o->rho_s, tmp);
    memcpy(o->rho_s, tmp, (size_t)o->ng * 8);
  }
  free(tmp);
  double scale = 1.0 / (double)((int64_t)1 << (2 * p));
  orc_poisson(o->nc, o->bc, o->Kphi * scale, o->KE * scale, o->rho_s, o->phi, o->E);
}

/* Time-averaged diagnostics (Table 2: `datfile` "time-averaged diagnostics", `mvflag`
 * "snapshot averaged over mvflag time steps", `mvStep` "interval between successive diagnostic outputs";
 * SURVEY 8(f) NEXT-1; reading N1-b).  With window W = mvflag and interval I = mvStep (W <= I):
 * after the step that makes the step counter k, r = k mod I (0 read as I); the grid state of that step
 * (per-species deposited charge, phi) joins the running sums when r > I - W, i.e. over the last W steps
 * of every interval; at r == I the sums are latched as the latest output and cleared.  Densities are
 * summed in int64 (exact), phi in fp64 in step order (one addition per node and step). */
static void phase_average(orc *o) {
  int32_t W = o->avg_window, I = o->avg_interval;
  if (W <= 0) return;
  uint64_t r = o->step % (uint64_t)I;
  if (r == 0) r = (uint64_t)I;
  size_t nd = (size_t)o->ns * (size_t)o->ng;
  if (r > (uint64_t)(I - W)) {
    for (size_t i = 0; i < nd; ++i) o->acc_dens[i] += o->dens[i];
    for (int32_t j = 0; j <= o->nc; ++j) o->acc_phi[j] = o->acc_phi[j] + o->phi[j];
    o->acc_count += 1;
  }
  if (r == (uint64_t)I) {
    memcpy(o->avg_dens, o->acc_dens, nd * 8);
    memcpy(o->avg_phi, o->acc_phi, ((size_t)o->nc + 1) * 8);
    o->avg_count = o->acc_count;
    o->avg_step = o->step;
    memset(o->acc_dens, 0, nd * 8);
    memset(o->acc_phi, 0, ((size_t)o->nc + 1) * 8);
    o->acc_count = 0;
  }
}

/* NEXT-2: species s recycles into species `to` (-1 switches it off) at wall temperature sqrt(e T_w / m_to) = vth */
int orc_set_recycling(orc *o, int32_t s, int32_t to, double vth) {
  if (s < 0 || s >= o->ns || to >= o->ns || (to >= 0 && !(vth >= 0.0))) return 1;
  o->recycle_to[s] = to < 0 ? -1 : to;
  o->recycle_vth[s] = vth;
  return 0;
}
uint64_t orc_recycled(const orc *o) { return o->diag_recycled; }
int orc_set_neutral_target(orc *o, int32_t species) {
  if (species >= o->ns) return 1;
  o->target_species = species < 0 ? -1 : species;
  if (species >= 0) o->kn = (0.5 * o->weight[species]) / (((double)o->Q[species] * o->area) * o->dx);
  return 0;
}

void orc_set_smoothing(orc *o, int32_t passes) { o->smooth_passes = passes < 0 ? 0 : (passes > 8 ? 8 : passes); }
/* (re)arms the averaging: running and latched sums are cleared */
int orc_set_averaging(orc *o, int32_t window, int32_t interval) {
  if (window < 0 || (window > 0 && interval < window)) return 1;
  o->avg_window = window; o->avg_interval = window > 0 ? interval : 0;
  size_t nd = (size_t)o->ns * (size_t)o->ng;
  memset(o->acc_dens, 0, nd * 8); memset(o->avg_dens, 0, nd * 8);
  memset(o->acc_phi, 0, ((size_t)o->nc + 1) * 8); memset(o->avg_phi, 0, ((size_t)o->nc + 1) * 8);
  o->acc_count = 0; o->avg_count = 0; o->avg_step = 0;
  return 0;
}
void orc_get_average(const orc *o, int64_t *dens_sum, double *phi_sum, uint64_t *count, uint64_t *step) {
  memcpy(dens_sum, o->avg_dens, (size_t)o->ns * (size_t)o->ng * 8);
  memcpy(phi_sum, o->avg_phi, ((size_t)o->nc + 1) * 8);
  *count = o->avg_count; *step = o->avg_step;
}
void orc_get_rho_smoothed(const orc *o, int64_t *out) {
  memcpy(out, o->smooth_passes > 0 ? o->rho_s : o->rho, (size_t)o->ng * 8);
}

/* ------------------------------------------------------------------ */
/* Append one birth.  SURVEY 8(c) "A": parent-index order, pid = next_pid + r;
 * beyond capacity the birth is not created and the CAPACITY flag is set. */
static void append_birth(orc *o, uint32_t *births, int s, double x, int32_t c, double vx,
                         double vy, double vz) {
  uint64_t slot = o->n_slots;
  if (slot >= o->capacity) { o->flagword |= FLAG_CAPACITY; return; }
  o->x[slot] = x; o->vx[slot] = vx; o->vy[slot] = vy; o->vz[slot] = vz;
  o->cell[slot] = c; o->sp[slot] = (uint8_t)s;
  o->pid[slot] = o->next_pid + *births;
  *births += 1;
  o->n_slots = slot + 1;
}

/* G, B, M, W, C, A for every particle in array order.  SURVEY 8(c);
 * PAPER.md:33 steps (i),(iv) + "MC routines"; PAPER.md:111 mover move0/moveb. */
void orc_phase_push(orc *o) {
  const double dt = o->dt, L = o->L, inv_dx = o->inv_dx;
  const uint64_t step = o->step;
  uint32_t births = 0;
  uint64_t n = o->n;
  o->n_slots = n;
  for (uint64_t i = 0; i < n; ++i) {
    const int s = o->sp[i];
    const uint32_t pid = o->pid[i];
    double x = o->x[i], vx = o->vx[i], vy = o->vy[i], vz = o->vz[i];
    const int32_t c = o->cell[i];
    /* G: linear gather of E */
    double f = x * inv_dx - (double)c;
    double Ex = o->E[c] + f * (o->E[c + 1] - o->E[c]);
    /* B: Boris half kick, rotation, half kick */
    const double tx = o->t[s][0], ty = o->t[s][1], tz = o->t[s][2];
    const double sx = o->s[s][0], sy = o->s[s][1], sz = o->s[s][2];
    double a = o->h[s] * Ex;
    double ux = vx + a, uy = vy, uz = vz;
    double px = ux + (uy * tz - uz * ty);
    double py = uy + (uz * tx - ux * tz);
    double pz = uz + (ux * ty - uy * tx);
    double wx = ux + (py * sz - pz * sy);
    double wy = uy + (pz * sx - px * sz);
    double wz = uz + (px * sy - py * sx);
    vx = wx + a; vy = wy; vz = wz;
    /* M: move */
    x = x + vx * dt;
    /* W: boundaries */
    int alive = 1;
    int pair_birth = 0;
    double bvx = 0, bvy = 0, bvz = 0;
    int recycled = 0;
    double rx = 0, rvx = 0, rvy = 0, rvz = 0;
    int32_t rc = 0;
    if (!o->bc) {
      if (x < 0.0) x = x + L;
      if (x >= L) x = x - L;
      if (!(x >= 0.0 && x < L)) { /* A21: more than one domain length */
        o->flagword |= FLAG_ESCAPE; o->diag_escape += 1;
        x = 0.0;
      }
    } else {
      int side = -1;
      if (x < 0.0) side = 0;
      else if (x >= L) side = 1;
      else if (!(x >= 0.0)) { /* NaN */
        o->flagword |= FLAG_ESCAPE; o->diag_escape += 1; side = 0;
      }
      if (side >= 0) {
        o->wall_count[side][s] += 1;
        o->wall_charge[side] += (int64_t)o->sign[s] * o->Q[s];
        if (o->recycle_to[s] >= 0) {
          /* Wall recycling ("Plasma is absorbed at the walls ..., recycling D+ ions into D neutrals";
           * SURVEY 8(f) NEXT-2; reading N2-a): the absorbed particle leaves one particle of species
           * recycle_to at the wall it hit -- x = 0 at the left wall, x = L - dx*2^-20 at the right one -- with a
           * half-Maxwellian velocity at the wall temperature pointing into the plasma: slot 14 (RC) of the
           * parent's stream, vx = +-vth*|z0| (away from the wall), vy = vth*z1, vz = vth*z2.  What happens to the
           * absorbed particle itself (death, re-injection, pair source) is unchanged. */
          uint32_t wr[4];
          draw(o, pid, step, 14u, wr); /* slot RC */
          double z0 = normal_from_word(o, wr[0]);
          if (z0 < 0.0) z0 = -z0;
          double vth_r = o->recycle_vth[s];
          rvx = side == 0 ? vth_r * z0 : -(vth_r * z0);
          rvy = vth_r * normal_from_word(o, wr[1]);
          rvz = vth_r * normal_from_word(o, wr[2]);
          rx = side == 0 ? 0.0 : L - o->dx * 9.5367431640625e-07;
          rc = side == 0 ? 0 : o->nc - 1;
          recycled = 1;
        }
        if (o->src_mode[s] == SRC_NONE) {
          alive = 0;
        } else {
          uint32_t w[4];
          draw(o, pid, step, 2u, w); /* slot RJ */
          double u0 = orc_u32(w[0]);
          x = o->src_lo + u0 * (o->src_hi - o->src_lo);
          double z1 = normal_from_word(o, w[1]);
          double z2 = normal_from_word(o, w[2]);
          double z3 = normal_from_word(o, w[3]);
          vx = o->src_vth[s] * z1; vy = o->src_vth[s] * z2; vz = o->src_vth[s] * z3;
          o->diag_reinject += 1;
          if (o->src_mode[s] == SRC_PAIR) {
            int p = o->src_partner[s];
            uint32_t wp[4];
            draw(o, pid, step, 13u, wp); /* slot PB */
            bvx = o->src_vth[p] * normal_from_word(o, wp[0]);
            bvy = o->src_vth[p] * normal_from_word(o, wp[1]);
            bvz = o->src_vth[p] * normal_from_word(o, wp[2]);
            pair_birth = 1;
          }
        }
      }
    }
    int32_t cn = alive ? cell_of(o, x) : -1;
    /* C: null-collision Monte Carlo for live particles of a species with any
     * process flag (re-injected ones included, reading A10). */
    int ionised = 0;
    double e2vx = 0, e2vy = 0, e2vz = 0, ivx = 0, ivy = 0, ivz = 0;
    const uint32_t fl = o->flags[s];
    if (alive && (fl & (F_ELASTIC | F_IONISE | F_CX))) {
      uint32_t w[4];
      draw(o, pid, step, 0u, w); /* slot C0 */
      double u0 = orc_u53(w[0], w[1]);
      double u1 = orc_u53(w[2], w[3]);
      if (u0 < o->pnull[s]) {
        o->diag_candidates[s] += 1;
        double vnx = 0.0, vny = 0.0, vnz = 0.0;
        if (fl & F_TARGET_MAXWELLIAN) {
          uint32_t wn[4];
          draw(o, pid, step, 1u, wn); /* slot NV */
          vnx = o->vth_n * normal_from_word(o, wn[0]);
          vny = o->vth_n * normal_from_word(o, wn[1]);
          vnz = o->vth_n * normal_from_word(o, wn[2]);
        }
        double gx = vx - vnx, gy = vy - vny, gz = vz - vnz;
        double g2 = (gx * gx + gy * gy) + gz * gz;
        double g = sqrt(g2);
        double EeV = o->kin_eV[s] * g2;
        double r = u1 * o->numax[s];
        /* NEXT-2, second half ("neutral particles as the collision target (density from dens_n instead
         * of constant n0)"; reading N2-b): with a target species set, the neutral density a candidate sees is
         * that species' density in the candidate's (new) cell, from the deposit of the previous step: the mean of the
         * cell's two nodes, n = (D[c] + D[c+1]) * kn with kn = (0.5*weight_n) / ((Q_n*area)*dx).  o->dens still holds
         * the previous step's deposit here (this step's comes after the sort).  numax keeps bounding the rate: it is
         * the caller's, computed for the largest density it expects; beyond it nu_overflow counts, as before. */
        double nloc = o->n0;
        if (o->target_species >= 0) {
          int32_t j1 = cn + 1;
          if (!o->bc && j1 == o->nc) j1 = 0;
          const int64_t *D = o->dens + (size_t)o->target_species * (size_t)o->ng;
          nloc = (double)(D[cn] + D[j1]) * o->kn;
        }
        double cum = 0.0;
        int chosen = -1;
        if (fl & F_ELASTIC) {
          cum = cum + (nloc * sigma_lookup(o, o->sig_el, EeV)) * g;
          if (chosen < 0 && r < cum) chosen = 0;
        }
        if (fl & F_IONISE) {
          /* DESIGN.md reading R-thr: the ionisation cross-section is the table value above the threshold and
           * zero at or below it.  A table that is linear between nodes is positive on the whole interval that
           * holds the threshold (13.5..14.0 eV for SURVEY's 0.5 eV table), and an ionisation picked there would
           * share out a negative energy E - E_ion (sqrt of a negative number: NaN velocities). */
          double sig_i = EeV > o->E_ion ? sigma_lookup(o, o->sig_ion, EeV) : 0.0;
          cum = cum + (nloc * sig_i) * g;
          if (chosen < 0 && r < cum) chosen = 1;
        }
        if (fl & F_CX) {
          cum = cum + (nloc * sigma_lookup(o, o->sig_cx, EeV)) * g;
          if (chosen < 0 && r < cum) chosen = 2;
        }
        if (cum > o->numax[s]) o->diag_nu_overflow += 1;
        if (chosen == 0) {
          /* elastic, isotropic in the lab frame, A14 */
          double nn[3];
          o->diag_dir_fallback += (uint64_t)direction(o, pid, step, 4u, nn);
          double dot = (vx * nn[0] + vy * nn[1]) + vz * nn[2];
          double cosx = dot / g;
          double gn = g * sqrt(1.0 - o->el_loss[s] * (1.0 - cosx));
          vx = gn * nn[0]; vy = gn * nn[1]; vz = gn * nn[2];
          o->diag_events[s][0] += 1;
        } else if (chosen == 1) {
          /* ionisation, A16: uniform split of E - E_ion */
          double Er = EeV - o->E_ion;
          uint32_t ws[4];
          draw(o, pid, step, 3u, ws); /* slot SP */
          double u = orc_u53(ws[0], ws[1]);
          double E1 = u * Er;
          double E2 = Er - E1;
          double n1[3], n2[3];
          o->diag_dir_fallback += (uint64_t)direction(o, pid, step, 4u, n1);
          o->diag_dir_fallback += (uint64_t)direction(o, pid, step, 8u, n2);
          double sp1 = sqrt(E1 * o->two_e_over_m[s]);
          vx = sp1 * n1[0]; vy = sp1 * n1[1]; vz = sp1 * n1[2];
          int ep = o->sp_electron_product;
          double sp2 = sqrt(E2 * o->two_e_over_m[ep]);
          e2vx = sp2 * n2[0]; e2vy = sp2 * n2[1]; e2vz = sp2 * n2[2];
          uint32_t wb[4];
          draw(o, pid, step, 12u, wb); /* slot BI */
          ivx = o->vth_n * normal_from_word(o, wb[0]);
          ivy = o->vth_n * normal_from_word(o, wb[1]);
          ivz = o->vth_n * normal_from_word(o, wb[2]);
          ionised = 1;
          o->diag_events[s][1] += 1;
        } else if (chosen == 2) {
          /* charge exchange: the ion takes the neutral's velocity */
          vx = vnx; vy = vny; vz = vnz;
          o->diag_events[s][2] += 1;
        }
      }
    }
    o->x[i] = x; o->vx[i] = vx; o->vy[i] = vy; o->vz[i] = vz; o->cell[i] = cn;
    /* A: births in parent order: source partner, ionisation electron, ion */
    if (pair_birth) append_birth(o, &births, o->src_partner[s], x, cn, bvx, bvy, bvz);
    if (ionised) {
      append_birth(o, &births, o->sp_electron_product, x, cn, e2vx, e2vy, e2vz);
      append_birth(o, &births, o->sp_ion_product, x, cn, ivx, ivy, ivz);
    }
    if (recycled) {   /* a parent's fourth and last birth */
      append_birth(o, &births, o->recycle_to[s], rx, rc, rvx, rvy, rvz);
      o->diag_recycled += 1;   /* recycling events (the birth itself may be dropped at capacity, reading R-W) */
    }
  }
  o->next_pid += births;
  o->diag_births += births;
}

void orc_step(orc *o, uint64_t nsteps, int freeze_field) {
  for (uint64_t k = 0; k < nsteps; ++k) {
    orc_phase_push(o);
    orc_phase_sort(o);
    orc_phase_deposit(o);
    if (!freeze_field) orc_phase_field(o);
    o->step += 1;
    phase_average(o);
  }
}

/* Load: copy, compute cells, stable sort by cell, deposit, solve.  State
 * after load per SURVEY 8(b): sorted, rho/phi/E valid, step 0. */
int orc_load(orc *o, uint64_t n, const double *x, const double *vx, const double *vy,
             const double *vz, const uint8_t *sp, const uint32_t *pid) {
  if (n > o->capacity) return 1;
  uint32_t maxpid = 0;
  for (uint64_t i = 0; i < n; ++i) {
    if (!(x[i] >= 0.0 && x[i] < o->L) || sp[i] >= o->ns) return 2;
    o->x[i] = x[i]; o->vx[i] = vx[i]; o->vy[i] = vy[i]; o->vz[i] = vz[i];
    o->sp[i] = sp[i];
    o->pid[i] = pid ? pid[i] : (uint32_t)i;
    if (o->pid[i] >= maxpid) maxpid = o->pid[i] + 1;
    o->cell[i] = cell_of(o, x[i]);
  }
  o->n = n; o->n_slots = n; o->next_pid = n ? maxpid : 0; o->step = 0;
  orc_phase_sort(o);
  orc_phase_deposit(o);
  orc_phase_field(o);
  return 0;
}

/* Restore (oracle-side checkpoint/restart): arrays are taken as
 * they were read out (already sorted), counters are set, rho/phi/E rebuilt. */
int orc_restore(orc *o, uint64_t n, const double *x, const double *vx, const double *vy,
                const double *vz, const int32_t *cell, const uint32_t *pid, const uint8_t *sp,
                uint64_t step, uint32_t next_pid, const uint64_t *wall_count, const int64_t *wall_charge) {
  if (n > o->capacity) return 1;
  memcpy(o->x, x, n * 8); memcpy(o->vx, vx, n * 8); memcpy(o->vy, vy, n * 8); memcpy(o->vz, vz, n * 8);
  memcpy(o->cell, cell, n * 4); memcpy(o->pid, pid, n * 4); memcpy(o->sp, sp, n);
  o->n = n; o->n_slots = n; o->step = step; o->next_pid = next_pid;
  for (int side = 0; side < 2; ++side)
    for (int s = 0; s < o->ns; ++s) o->wall_count[side][s] = wall_count[side * o->ns + s];
  o->wall_charge[0] = wall_charge[0]; o->wall_charge[1] = wall_charge[1];
  for (int32_t c = 0; c <= o->nc; ++c) o->cell_start[c] = 0;
  for (uint64_t i = 0; i < n; ++i) {
    if (cell[i] < 0 || cell[i] >= o->nc || (i && cell[i] < cell[i - 1])) return 2;
    o->cell_start[cell[i] + 1] += 1;
  }
  for (int32_t c = 0; c < o->nc; ++c) o->cell_start[c + 1] += o->cell_start[c];
  orc_phase_deposit(o);
  orc_phase_field(o);
  return 0;
}

/* ------------------------------------------------------------------ */
/* getters / setters for tests */
uint64_t orc_n(const orc *o) { return o->n; }
uint64_t orc_n_slots(const orc *o) { return o->n_slots; }
uint64_t orc_step_index(const orc *o) { return o->step; }
uint32_t orc_next_pid(const orc *o) { return o->next_pid; }
uint32_t orc_flagword(const orc *o) { return o->flagword; }
void orc_set_step(orc *o, uint64_t s) { o->step = s; }
void orc_set_E(orc *o, const double *E) { memcpy(o->E, E, ((size_t)o->nc + 1) * 8); }

void orc_get_particles(const orc *o, double *x, double *vx, double *vy, double *vz, int32_t *cell,
                       uint32_t *pid, uint8_t *sp) {
  size_t n = (size_t)o->n_slots;
  if (x) memcpy(x, o->x, n * 8);
  if (vx) memcpy(vx, o->vx, n * 8);
  if (vy) memcpy(vy, o->vy, n * 8);
  if (vz) memcpy(vz, o->vz, n * 8);
  if (cell) memcpy(cell, o->cell, n * 4);
  if (pid) memcpy(pid, o->pid, n * 4);
  if (sp) memcpy(sp, o->sp, n);
}
void orc_get_cell_start(const orc *o, int64_t *cs) { memcpy(cs, o->cell_start, ((size_t)o->nc + 1) * 8); }
void orc_get_rho(const orc *o, int64_t *rho) { memcpy(rho, o->rho, (size_t)o->ng * 8); }
void orc_get_dens(const orc *o, int64_t *dens) { memcpy(dens, o->dens, (size_t)o->ns * (size_t)o->ng * 8); }
void orc_get_phi(const orc *o, double *phi) { memcpy(phi, o->phi, ((size_t)o->nc + 1) * 8); }
void orc_get_E(const orc *o, double *E) { memcpy(E, o->E, ((size_t)o->nc + 1) * 8); }
void orc_get_Q(const orc *o, int64_t *Q) { memcpy(Q, o->Q, (size_t)o->ns * 8); }
void orc_get_wall(const orc *o, uint64_t *count /* [2][ns] */, int64_t *charge /* [2] */) {
  for (int side = 0; side < 2; ++side)
    for (int s = 0; s < o->ns; ++s) count[side * o->ns + s] = o->wall_count[side][s];
  charge[0] = o->wall_charge[0]; charge[1] = o->wall_charge[1];
}
/* diag: [nu_overflow, dir_fallback, escape, births, reinject], then per species
 * candidates[ns], events[ns][3] */
void orc_get_diag(const orc *o, uint64_t *d5, uint64_t *cand, uint64_t *events) {
  d5[0] = o->diag_nu_overflow; d5[1] = o->diag_dir_fallback; d5[2] = o->diag_escape;
  d5[3] = o->diag_births; d5[4] = o->diag_reinject;
  for (int s = 0; s < o->ns; ++s) {
    cand[s] = o->diag_candidates[s];
    for (int k = 0; k < 3; ++k) events[s * 3 + k] = o->diag_events[s][k];
  }
}
void orc_get_constants(const orc *o, double *out /* inv_dx, L, Kphi, KE */, double *h, double *t3,
                       double *s3) {
  out[0] = o->inv_dx; out[1] = o->L; out[2] = o->Kphi; out[3] = o->KE;
  for (int s = 0; s < o->ns; ++s) {
    h[s] = o->h[s];
    for (int k = 0; k < 3; ++k) { t3[s * 3 + k] = o->t[s][k]; s3[s * 3 + k] = o->s[s][k]; }
  }
}

/* Per-species number density n_s[j] = dens_s[j]/Q_s * weight_s/(area*dx), doubled
 * at wall nodes (half cells).  SURVEY 8(c) "Moments". */
void orc_get_density(const orc *o, int s, double *out) {
  for (int32_t j = 0; j < o->ng; ++j) {
    double v = (((double)o->dens[(size_t)s * o->ng + j] / (double)o->Q[s]) * o->weight[s]) / (o->area * o->dx);
    if (o->bc && (j == 0 || j == o->nc)) v = 2.0 * v;
    out[j] = v;
  }
}

/* Moments.  SURVEY 8(c) "Moments": index-order compensated (Kahan) sums.
 * count[ns], kinetic_J[ns], px[ns], field_J (1). */
static void kahan_add(double *sum, double *comp, double v) {
  double y = v - *comp;
  double t = *sum + y;
  *comp = (t - *sum) - y;
  *sum = t;
}
void orc_get_moments(const orc *o, uint64_t *count, double *kinetic_J, double *px, double *field_J) {
  double sv2[ORC_MAX_SPECIES] = {0}, cv2[ORC_MAX_SPECIES] = {0};
  double svx[ORC_MAX_SPECIES] = {0}, cvx[ORC_MAX_SPECIES] = {0};
  for (int s = 0; s < o->ns; ++s) count[s] = 0;
  for (uint64_t i = 0; i < o->n; ++i) {
    int s = o->sp[i];
    count[s] += 1;
    double v2 = (o->vx[i] * o->vx[i] + o->vy[i] * o->vy[i]) + o->vz[i] * o->vz[i];
    kahan_add(&sv2[s], &cv2[s], v2);
    kahan_add(&svx[s], &cvx[s], o->vx[i]);
  }
  for (int s = 0; s < o->ns; ++s) {
    kinetic_J[s] = ((0.5 * o->m[s]) * o->weight[s]) * sv2[s];
    px[s] = (o->m[s] * o->weight[s]) * svx[s];
  }
  double se = 0.0, ce = 0.0;
  for (int32_t j = 0; j < o->ng; ++j) {
    double g = (o->bc && (j == 0 || j == o->nc)) ? 0.5 : 1.0;
    kahan_add(&se, &ce, g * (o->E[j] * o->E[j]));
  }
  *field_J = (((0.5 * EPS0) * o->area) * o->dx) * se;
}
