/* goracle.h — FP64 CPU oracle for the G-CoReCCD hot path (arXiv 2203.11043).
 *
 * TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may call this.  It shares no code,
 * header, table or helper with the CUDA path under paper_2203_11043_b200/csrc/.
 *
 * Everything is written out from /root/reference/PAPER.md in the paper's order and
 * notation (PAPER.md:68 gives the order of one step).  Citations are "PAPER.md:<line>".
 * Readings of silent/ambiguous points are the ones listed in DESIGN.md §3 (R1..R22).
 *
 * Units: length um, time ns, field V/cm, mobility cm^2/(V s), temperature K.
 *
 * Parity pins (tests/test_oracle_*.py, all "-m 'not gpu'"):
 *   goracle_mobility        eq. 2 special cases, limits, golden values        PINNED
 *   goracle_coulomb_field   2-body closed form, Newton III, shell theorem,
 *                           symmetries, independent long-double brute force   PINNED
 *   goracle_philox4x32_10   Random123 known-answer vectors                    PINNED
 *   goracle_normals         golden words/normals, moments                     PINNED
 *   goracle_step (drift)    low-field closed-form drift time, Euler goldens   PINNED
 *   goracle_step (coulomb)  two-carrier r^3 closed form, dt->0 convergence    PINNED
 *   goracle_step (diffuse)  sigma_xy^2 = 2(kT/q)/a1 ln(a2/(a2-a1 z0))        PINNED
 *   full-run image with Coulomb ON: the paper prints no image or cloud size,
 *                           so only invariants + monotonicity: PARITY UNPINNED
 */
#ifndef GORACLE_H
#define GORACLE_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

enum {
  GORACLE_COULOMB_OFF   = 1u,   /* PAPER.md:88 "whether Coulomb repulsion should be computed" */
  GORACLE_DIFFUSION_OFF = 2u,
  GORACLE_DEPLETION_OFF = 4u,
  GORACLE_FP32_STATE    = 0x100u /* round x,y,z to float after every step ("3N floats") */
};

typedef struct {
  double   T_K;
  double   a1_V_per_cm2, a2_V_per_cm;   /* eq. 1 */
  double   thickness_um;
  double   z_well_um;                   /* PAPER.md:88 "depth of the potential well" */
  double   pixel_pitch_um;
  double   dt_ns;
  double   softening_um;                /* eps of eq. 6 */
  double   eps_si;                      /* relative permittivity; 0 => 11.7 */
  uint64_t seed;
  int32_t  img_nx, img_ny;
  double   img_x0_um, img_y0_um;
  uint32_t flags;
  uint32_t pad_;
} goracle_params;

typedef struct goracle goracle_t;

/* ---- model equations ---- */
double goracle_depletion_field(double z_um, double a1, double a2);          /* eq. 1 */
double goracle_mobility(double E_V_per_cm, double T_K);                     /* eq. 2 */
double goracle_thermal_voltage(double T_K);                                 /* k_B T / q, eq. 4 */
double goracle_diffusion_sigma(double mu, double T_K, double dt_ns);        /* eqs. 3-4, um */
double goracle_coulomb_constant(double eps_si);                             /* K' (V/cm) um^2, eq. 6 */

/* ---- counter-based RNG ---- */
void goracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
void goracle_normals(uint64_t seed, uint32_t id, uint64_t step, double n[3], uint32_t words[4]);
/* X-ray front end: hole count N = floor(E_e / w) and the seeded 3-D Gaussian initial cloud */
uint64_t goracle_xray_hole_count(double E_e_eV, double w_eV);
void goracle_xray_cloud(uint64_t gen_seed, uint64_t first_index, uint64_t n, const double centre_um[3],
                        double sigma_um, double thickness_um, float* xyz);

/* ---- eq. 6: literal double loop.  Targets j = tgt[0..m) (or all if tgt==NULL, m==n);
 *      sources i = 0..n-1.  Output E in V/cm. ---- */
void goracle_coulomb_field(const double* x, const double* y, const double* z, uint64_t n,
                           const uint64_t* tgt, uint64_t m, double eps_um, double Kp,
                           double* Ex, double* Ey, double* Ez);

/* ---- one carrier, one step, given its Coulomb field (steps 2-6 of DESIGN.md §2).
 *      Returns 1 if the carrier is collected (z_new <= z_well). ---- */
int goracle_advance(const goracle_params* p, uint64_t step, uint32_t id,
                    const double r[3], const double Ecoul[3], double r_new[3]);

/* ---- whole simulation ---- */
goracle_t* goracle_create(const goracle_params* p);
void       goracle_destroy(goracle_t* s);
int        goracle_load(goracle_t* s, const float* xyz, uint64_t n);          /* 0 ok, -1 invalid */
int        goracle_load_state(goracle_t* s, const double* xyz, const uint32_t* id, uint64_t n,
                              uint64_t step);                                   /* restart */
uint64_t   goracle_step(goracle_t* s, uint64_t n_steps);                       /* steps done */
uint64_t   goracle_run(goracle_t* s, uint64_t max_steps);                      /* steps done */
void       goracle_get_state(const goracle_t* s, uint64_t* step, uint64_t* n_active,
                             uint64_t* n_collected, uint64_t* n_out_of_window,
                             uint64_t* pair_interactions);
uint64_t   goracle_read_carriers(const goracle_t* s, double* xyz, uint32_t* id, uint64_t cap);
void       goracle_read_image(const goracle_t* s, uint32_t* out);
/* final (x,y,z) and collection step of every carrier collected so far, indexed by id
 * (NaN / UINT64_MAX where still drifting); arrays of length n_loaded */
uint64_t   goracle_read_collected(const goracle_t* s, double* xyz, uint64_t* step_collected,
                                  uint64_t cap);
int        goracle_num_threads(void);

#ifdef __cplusplus
}
#endif
#endif
