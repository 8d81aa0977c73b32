/* goracle.c — plain, slow FP64 CPU oracle for the G-CoReCCD hot path (arXiv 2203.11043).
 *
 * TEST INFRASTRUCTURE, NOT THE PRODUCT (see goracle.h).  No blocking, no fusion, no
 * reordering beyond what the paper states: eq. 6 is the literal double loop, one step is
 * the sequence of PAPER.md:68.  OpenMP only runs independent targets j on several cores.
 *
 * Units: um, ns, V/cm, cm^2/(V s), K.
 *   v [um/ns]   = 1e-5 * mu * E            (1 cm/s = 1e-5 um/ns)
 *   D [um^2/ns] = 0.1 * (k_B T/q)[V] * mu  (1 cm^2/s = 0.1 um^2/ns)
 *   z [cm]      = 1e-4 * z [um]
 */
#include "goracle.h"
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* exact SI (2019) values; eps0 CODATA 2018 */
#define GO_Q_E   1.602176634e-19    /* C   */
#define GO_K_B   1.380649e-23       /* J/K */
#define GO_EPS0  8.8541878128e-12   /* F/m */
#define GO_PI    3.14159265358979323846

/* ------------------------------------------------------------------ eq. 1 */
/* PAPER.md:29  E(z) = a1 z - a2 ; a1 in V/cm^2, z given in um -> cm. */
double goracle_depletion_field(double z_um, double a1, double a2) {
  return a1 * (z_um * 1e-4) - a2;
}

/* ------------------------------------------------------------------ eq. 2 */
/* PAPER.md:33  mu(E,T) = 1.31e8 T^-2.2 / [1 + (E/(1.24 T^1.68))^(0.46 T^0.17)]^(1/(0.46 T^0.17)) */
double goracle_mobility(double E, double T) {
  double beta = 0.46 * pow(T, 0.17);
  double Ec   = 1.24 * pow(T, 1.68);
  double mu0  = 1.31e8 * pow(T, -2.2);
  return mu0 / pow(1.0 + pow(E / Ec, beta), 1.0 / beta);
}

/* ------------------------------------------------------------------ eqs. 3-4 */
/* PAPER.md:43  D_h = k_B mu_h T / q  ->  thermal voltage k_B T / q in volts */
double goracle_thermal_voltage(double T) { return GO_K_B * T / GO_Q_E; }

/* PAPER.md:39  sigma_D^2 = 2 D_h t_D, t_D = dt (reading R7); result in um */
double goracle_diffusion_sigma(double mu, double T, double dt_ns) {
  double D = 0.1 * goracle_thermal_voltage(T) * mu;   /* um^2/ns */
  return sqrt(2.0 * D * dt_ns);
}

/* ------------------------------------------------------------------ eq. 6 constant */
/* PAPER.md:80  K = q/(4 pi eps0 eps_Si) [V m]; a hole at r um gives K*1e12/r^2 V/m = K*1e10/r^2 V/cm */
double goracle_coulomb_constant(double eps_si) {
  if (eps_si == 0.0) eps_si = 11.7;
  return GO_Q_E / (4.0 * GO_PI * GO_EPS0 * eps_si) * 1e10;
}

/* ------------------------------------------------------------------ Philox4x32-10 */
/* Salmon, Moraes, Dror, Shaw, "Parallel random numbers: as easy as 1, 2, 3" (SC'11):
 * ten rounds of  (c0,c1,c2,c3) <- (hi(M1*c2)^c1^k0, lo(M1*c2), hi(M0*c0)^c3^k1, lo(M0*c0))
 * with the key bumped by the Weyl constants between rounds.  (Reading R13: the paper only
 * says "cuRAND".) */
void goracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
  for (int round = 0; round < 10; ++round) {
    uint64_t p0 = (uint64_t)M0 * c0, p1 = (uint64_t)M1 * c2;
    uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
    uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    uint32_t n0 = hi1 ^ c1 ^ k0, n1 = lo1, n2 = hi0 ^ c3 ^ k1, n3 = lo0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += W0; k1 += W1;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* Reading R13: counter = (id, 0, step_lo, step_hi), key = (seed_lo, seed_hi);
 * u = ((w>>9)+0.5) 2^-23 in (0,1), f = (w>>8) 2^-24 in [0,1); Box-Muller:
 * n = (R_a cos 2 pi f_a, R_a sin 2 pi f_a, R_b cos 2 pi f_b), R = sqrt(-2 ln u). */
void goracle_normals(uint64_t seed, uint32_t id, uint64_t step, double n[3], uint32_t words[4]) {
  uint32_t ctr[4] = { id, 0u, (uint32_t)(step & 0xffffffffu), (uint32_t)(step >> 32) };
  uint32_t key[2] = { (uint32_t)(seed & 0xffffffffu), (uint32_t)(seed >> 32) };
  uint32_t w[4];
  goracle_philox4x32_10(ctr, key, w);
  double ua = ((double)(w[0] >> 9) + 0.5) * (1.0 / 8388608.0);
  double fa = (double)(w[1] >> 8) * (1.0 / 16777216.0);
  double ub = ((double)(w[2] >> 9) + 0.5) * (1.0 / 8388608.0);
  double fb = (double)(w[3] >> 8) * (1.0 / 16777216.0);
  double Ra = sqrt(-2.0 * log(ua)), Rb = sqrt(-2.0 * log(ub));
  n[0] = Ra * cos(2.0 * GO_PI * fa);
  n[1] = Ra * sin(2.0 * GO_PI * fa);
  n[2] = Rb * cos(2.0 * GO_PI * fb);
  if (words) { words[0] = w[0]; words[1] = w[1]; words[2] = w[2]; words[3] = w[3]; }
}

/* ------------------------------------------------------------------ X-ray initial cloud (front end) */
/* "N = E_e / w_e", w_e = 3.77 eV at 140 K; a fraction of a pair is not a carrier: floor. */
uint64_t goracle_xray_hole_count(double E_e_eV, double w_eV) {
  if (!(E_e_eV > 0.0) || !(w_eV > 0.0)) return 0;
  return (uint64_t)floor(E_e_eV / w_eV);
}

/* "the initial cloud ... 3D Gaussian distribution with standard deviation depending solely on
 * E_e" (the sigma(E_e) model is in the paper's refs [11-13], not in its text: sigma is an input here).
 * Hole k = first_index + i gets centre + sigma * n_k, n_k the Box-Muller triple of
 * Philox4x32-10(ctr = (k_lo, 'XRAY', k_hi, 0), key = gen_seed) with the uniform mapping of goracle_normals;
 * z above the back surface is mirrored (R12); the result is rounded to FP32. */
void goracle_xray_cloud(uint64_t gen_seed, uint64_t first_index, uint64_t n, const double centre_um[3],
                        double sigma_um, double thickness_um, float* xyz) {
  uint32_t key[2] = { (uint32_t)(gen_seed & 0xffffffffu), (uint32_t)(gen_seed >> 32) };
  for (uint64_t i = 0; i < n; ++i) {
    const uint64_t k = first_index + i;
    uint32_t ctr[4] = { (uint32_t)(k & 0xffffffffu), 0x58524159u, (uint32_t)(k >> 32), 0u };
    uint32_t w[4];
    goracle_philox4x32_10(ctr, key, w);
    double ua = ((double)(w[0] >> 9) + 0.5) * (1.0 / 8388608.0);
    double fa = (double)(w[1] >> 8) * (1.0 / 16777216.0);
    double ub = ((double)(w[2] >> 9) + 0.5) * (1.0 / 8388608.0);
    double fb = (double)(w[3] >> 8) * (1.0 / 16777216.0);
    double Ra = sqrt(-2.0 * log(ua)), Rb = sqrt(-2.0 * log(ub));
    double x = centre_um[0] + sigma_um * (Ra * cos(2.0 * GO_PI * fa));
    double y = centre_um[1] + sigma_um * (Ra * sin(2.0 * GO_PI * fa));
    double z = centre_um[2] + sigma_um * (Rb * cos(2.0 * GO_PI * fb));
    if (z > thickness_um) z = 2.0 * thickness_um - z;
    xyz[3 * i] = (float)x; xyz[3 * i + 1] = (float)y; xyz[3 * i + 2] = (float)z;
  }
}

/* ------------------------------------------------------------------ eq. 6 */
/* PAPER.md:78  E_j = K sum_{i=1..N} r_ij / (|r_ij|^2 + eps^2)^{3/2},  r_ij = r_j - r_i.
 * The i = j term is included and is exactly zero (r_jj = 0). */
void goracle_coulomb_field(const double* x, const double* y, const double* z, uint64_t n,
                           const uint64_t* tgt, uint64_t m, double eps_um, double Kp,
                           double* Ex, double* Ey, double* Ez) {
  const double eps2 = eps_um * eps_um;
  int64_t mm = (int64_t)m;
#pragma omp parallel for schedule(static)
  for (int64_t t = 0; t < mm; ++t) {
    uint64_t j = tgt ? tgt[t] : (uint64_t)t;
    double sx = 0.0, sy = 0.0, sz = 0.0;
    for (uint64_t i = 0; i < n; ++i) {
      double dx = x[j] - x[i], dy = y[j] - y[i], dz = z[j] - z[i];
      double r2 = dx * dx + dy * dy + dz * dz + eps2;
      if (r2 == 0.0) continue;   /* eps = 0: eq. 5 -- the i = j term (and exact coincidences) drop out */
      double inv3 = 1.0 / (r2 * sqrt(r2));
      sx += dx * inv3; sy += dy * inv3; sz += dz * inv3;
    }
    Ex[t] = Kp * sx; Ey[t] = Kp * sy; Ez[t] = Kp * sz;
  }
}

/* ------------------------------------------------------------------ one carrier, one step */
/* E(z) -> E_Coul -> sum -> |E| -> mu -> v -> dr_D -> dr -> z check. */
int goracle_advance(const goracle_params* p, uint64_t step, uint32_t id,
                    const double r[3], const double Ecoul[3], double r_new[3]) {
  double Ex = 0.0, Ey = 0.0, Ez = 0.0;
  if (!(p->flags & GORACLE_COULOMB_OFF)) { Ex = Ecoul[0]; Ey = Ecoul[1]; Ez = Ecoul[2]; }
  if (!(p->flags & GORACLE_DEPLETION_OFF))
    Ez += goracle_depletion_field(r[2], p->a1_V_per_cm2, p->a2_V_per_cm);   /* eq. 1 */
  double Emag = sqrt(Ex * Ex + Ey * Ey + Ez * Ez);                          /* |E| of the sum (R3) */
  double mu = goracle_mobility(Emag, p->T_K);                               /* eq. 2 */
  double dx = 1e-5 * mu * Ex * p->dt_ns;                                    /* v = mu E */
  double dy = 1e-5 * mu * Ey * p->dt_ns;
  double dz = 1e-5 * mu * Ez * p->dt_ns;
  if (!(p->flags & GORACLE_DIFFUSION_OFF)) {
    double nrm[3];
    goracle_normals(p->seed, id, step, nrm, NULL);
    double sigma = goracle_diffusion_sigma(mu, p->T_K, p->dt_ns);           /* eqs. 3-4, same mu (R4) */
    dx += sigma * nrm[0]; dy += sigma * nrm[1]; dz += sigma * nrm[2];
  }
  double xn = r[0] + dx, yn = r[1] + dy, zn = r[2] + dz;
  if (zn > p->thickness_um) zn = 2.0 * p->thickness_um - zn;                /* R12: specular back surface */
  if (p->flags & GORACLE_FP32_STATE) { xn = (double)(float)xn; yn = (double)(float)yn; zn = (double)(float)zn; }
  r_new[0] = xn; r_new[1] = yn; r_new[2] = zn;
  return zn <= p->z_well_um;                                                /* R9 */
}

/* ------------------------------------------------------------------ simulation object */
struct goracle {
  goracle_params p;
  double Kp;
  uint64_t cap, n_active, n_loaded, step, n_collected, n_overflow, pairs;
  double *x, *y, *z, *Ex, *Ey, *Ez;
  uint32_t* id;
  uint32_t* image;
  /* per-id record of collected carriers */
  uint64_t rec_cap;
  double* fin;          /* 3 per id */
  uint64_t* fin_step;   /* per id */
};

static void go_reserve(goracle_t* s, uint64_t cap) {
  if (cap <= s->cap) return;
  uint64_t c = s->cap ? s->cap : 1024;
  while (c < cap) c *= 2;
  s->x = realloc(s->x, c * sizeof(double)); s->y = realloc(s->y, c * sizeof(double));
  s->z = realloc(s->z, c * sizeof(double)); s->Ex = realloc(s->Ex, c * sizeof(double));
  s->Ey = realloc(s->Ey, c * sizeof(double)); s->Ez = realloc(s->Ez, c * sizeof(double));
  s->id = realloc(s->id, c * sizeof(uint32_t));
  s->cap = c;
}
static void go_reserve_rec(goracle_t* s, uint64_t n) {
  if (n <= s->rec_cap) return;
  uint64_t c = s->rec_cap ? s->rec_cap : 1024;
  while (c < n) c *= 2;
  s->fin = realloc(s->fin, 3 * c * sizeof(double));
  s->fin_step = realloc(s->fin_step, c * sizeof(uint64_t));
  for (uint64_t k = s->rec_cap; k < c; ++k) {
    s->fin[3 * k] = s->fin[3 * k + 1] = s->fin[3 * k + 2] = NAN;
    s->fin_step[k] = UINT64_MAX;
  }
  s->rec_cap = c;
}

/* R10/R11: bin the position after the crossing step; half-open bins, floor; double arithmetic */
static void go_collect(goracle_t* s, uint32_t id, double x, double y, double z) {
  double fx = floor((x - s->p.img_x0_um) / s->p.pixel_pitch_um);
  double fy = floor((y - s->p.img_y0_um) / s->p.pixel_pitch_um);
  if (fx >= 0.0 && fx < (double)s->p.img_nx && fy >= 0.0 && fy < (double)s->p.img_ny)
    s->image[(uint64_t)fy * (uint64_t)s->p.img_nx + (uint64_t)fx] += 1u;
  else
    s->n_overflow += 1;
  s->n_collected += 1;
  if (id < s->rec_cap) {
    s->fin[3 * (uint64_t)id] = x; s->fin[3 * (uint64_t)id + 1] = y; s->fin[3 * (uint64_t)id + 2] = z;
    s->fin_step[id] = s->step;
  }
}

goracle_t* goracle_create(const goracle_params* p) {
  if (!p || !(p->T_K > 0) || !(p->dt_ns > 0) || !(p->pixel_pitch_um > 0) || p->img_nx <= 0 || p->img_ny <= 0
      || !(p->thickness_um > p->z_well_um) || p->softening_um < 0) return NULL;
  goracle_t* s = calloc(1, sizeof(*s));
  s->p = *p;
  if (s->p.eps_si == 0.0) s->p.eps_si = 11.7;
  s->Kp = goracle_coulomb_constant(s->p.eps_si);
  s->image = calloc((size_t)p->img_nx * (size_t)p->img_ny, sizeof(uint32_t));
  return s;
}

void goracle_destroy(goracle_t* s) {
  if (!s) return;
  free(s->x); free(s->y); free(s->z); free(s->Ex); free(s->Ey); free(s->Ez);
  free(s->id); free(s->image); free(s->fin); free(s->fin_step); free(s);
}

/* ids = load order, continuing (R18: z <= z_well collected at load; z > thickness or non-finite invalid) */
int goracle_load(goracle_t* s, const float* xyz, uint64_t n) {
  for (uint64_t k = 0; k < n; ++k) {
    double x = xyz[3 * k], y = xyz[3 * k + 1], z = xyz[3 * k + 2];
    if (!isfinite(x) || !isfinite(y) || !isfinite(z) || z > s->p.thickness_um) return -1;
  }
  go_reserve(s, s->n_active + n);
  go_reserve_rec(s, s->n_loaded + n);
  for (uint64_t k = 0; k < n; ++k) {
    double x = xyz[3 * k], y = xyz[3 * k + 1], z = xyz[3 * k + 2];
    uint32_t id = (uint32_t)(s->n_loaded + k);
    if (z <= s->p.z_well_um) { go_collect(s, id, x, y, z); continue; }
    uint64_t a = s->n_active++;
    s->x[a] = x; s->y[a] = y; s->z[a] = z; s->id[a] = id;
  }
  s->n_loaded += n;
  return 0;
}

/* restart from an exported snapshot: positions (double), ids, step index */
int goracle_load_state(goracle_t* s, const double* xyz, const uint32_t* id, uint64_t n, uint64_t step) {
  go_reserve(s, n);
  uint32_t maxid = 0;
  for (uint64_t k = 0; k < n; ++k) if (id[k] > maxid) maxid = id[k];
  go_reserve_rec(s, (uint64_t)maxid + 1);
  s->n_active = 0;
  for (uint64_t k = 0; k < n; ++k) {
    s->x[k] = xyz[3 * k]; s->y[k] = xyz[3 * k + 1]; s->z[k] = xyz[3 * k + 2]; s->id[k] = id[k];
  }
  s->n_active = n;
  if (s->n_loaded < n) s->n_loaded = n;
  if (n && s->n_loaded < (uint64_t)maxid + 1) s->n_loaded = (uint64_t)maxid + 1; /* records cover every id of the snapshot */
  s->step = step;
  return 0;
}

uint64_t goracle_step(goracle_t* s, uint64_t n_steps) {
  uint64_t done = 0;
  for (; done < n_steps && s->n_active > 0; ++done) {
    const uint64_t n = s->n_active;
    /* 1. Coulomb field of every still-drifting hole from start-of-step positions (R7, R8) */
    if (!(s->p.flags & GORACLE_COULOMB_OFF)) {
      goracle_coulomb_field(s->x, s->y, s->z, n, NULL, n, s->p.softening_um, s->Kp, s->Ex, s->Ey, s->Ez);
      s->pairs += n * n;
    }
    /* 2-6. per-carrier update, then 7. collection + stable compaction */
    uint64_t a = 0;
    for (uint64_t j = 0; j < n; ++j) {
      double r[3] = { s->x[j], s->y[j], s->z[j] }, Ec[3] = { 0.0, 0.0, 0.0 }, rn[3];
      if (!(s->p.flags & GORACLE_COULOMB_OFF)) { Ec[0] = s->Ex[j]; Ec[1] = s->Ey[j]; Ec[2] = s->Ez[j]; }
      int collected = goracle_advance(&s->p, s->step, s->id[j], r, Ec, rn);
      if (collected) { go_collect(s, s->id[j], rn[0], rn[1], rn[2]); continue; }
      s->x[a] = rn[0]; s->y[a] = rn[1]; s->z[a] = rn[2]; s->id[a] = s->id[j]; ++a;
    }
    s->n_active = a;
    s->step += 1;                                                           /* 8. */
  }
  return done;
}

uint64_t goracle_run(goracle_t* s, uint64_t max_steps) { return goracle_step(s, max_steps); }

void goracle_get_state(const goracle_t* s, uint64_t* step, uint64_t* n_active, uint64_t* n_collected,
                       uint64_t* n_out_of_window, uint64_t* pair_interactions) {
  if (step) *step = s->step;
  if (n_active) *n_active = s->n_active;
  if (n_collected) *n_collected = s->n_collected;
  if (n_out_of_window) *n_out_of_window = s->n_overflow;
  if (pair_interactions) *pair_interactions = s->pairs;
}

uint64_t goracle_read_carriers(const goracle_t* s, double* xyz, uint32_t* id, uint64_t cap) {
  uint64_t n = s->n_active < cap ? s->n_active : cap;
  for (uint64_t k = 0; k < n; ++k) {
    if (xyz) { xyz[3 * k] = s->x[k]; xyz[3 * k + 1] = s->y[k]; xyz[3 * k + 2] = s->z[k]; }
    if (id) id[k] = s->id[k];
  }
  return s->n_active;
}

void goracle_read_image(const goracle_t* s, uint32_t* out) {
  memcpy(out, s->image, (size_t)s->p.img_nx * (size_t)s->p.img_ny * sizeof(uint32_t));
}

uint64_t goracle_read_collected(const goracle_t* s, double* xyz, uint64_t* step_collected, uint64_t cap) {
  uint64_t n = s->n_loaded < cap ? s->n_loaded : cap;
  if (n > s->rec_cap) n = s->rec_cap;
  for (uint64_t k = 0; k < n; ++k) {
    if (xyz) { xyz[3 * k] = s->fin[3 * k]; xyz[3 * k + 1] = s->fin[3 * k + 1]; xyz[3 * k + 2] = s->fin[3 * k + 2]; }
    if (step_collected) step_collected[k] = s->fin_step[k];
  }
  return s->n_loaded;
}

int goracle_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}
