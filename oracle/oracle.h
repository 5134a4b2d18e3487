/*
 * oracle.h -- CPU ORACLE of the GPUMCD hot path.  TEST INFRASTRUCTURE ONLY.
 *
 * A plain, slow, fp64, one-history-at-a-time implementation of the coupled
 * photon-electron transport that arxiv 1101.1245 (GPUMCD; /root/reference/PAPER.md)
 * describes, written from the paper and from the readings listed in DESIGN.md.
 * It shares no code with the CUDA library in paper_1101_1245_b200/csrc and may be
 * used only by tests/, by __graft_entry__.smoke() and by bench.py's cpu_baseline /
 * --impl reference legs.  The product path never calls it.
 *
 * The method is a stochastic simulation, so the oracle follows the algorithm step
 * by step (Sec. II.A photons, II.B electrons) on random streams that are
 * a pure function of (seed, history, track, draw counter): any implementation that
 * makes the same draws for the same particle reproduces it up to rounding.
 *
 * Pins (tests/test_oracle_*.py): Philox known-answer vectors; chi-square of the
 * Klein-Nishina / Moller / bremsstrahlung / Sauter / pair / multiple-scattering
 * samplers against the analytic densities; narrow-beam attenuation exp(-mu x);
 * Woodcock invariance under an inflated majorant; CSDA range against
 * numerical integration of the stopping-power table; exact energy conservation;
 * brute-force expectation on a one-voxel phantom; and, for the transport loop itself
 * (tests/test_oracle_pins.py): <cos theta> = exp(-int rho/lambda_1 ds) in uniform media and
 * across a slab stack (martingale identity), the alternate hinge's two energies, momentum
 * and energy conservation of every Compton / Moller / pair / bremsstrahlung vertex as it is
 * pushed, Sauter angles of photo-electrons, distinct track ids within a history, and the
 * kinematic thresholds of Moller and pair events.
 * PARITY UNPINNED: the dose grid as a whole has no external truth here (EGSnrc and
 * its data files are absent); it is pinned only through the pieces above.
 *
 * Units: MeV (kinetic energy for electrons), cm, g/cm^3.
 */
#ifndef GPUMCD_ORACLE_H
#define GPUMCD_ORACLE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define ORC_M_E 0.51099895 /* electron rest energy, MeV */

/* Input tables: float32 arrays exactly as produced by the input generator; see
 * DESIGN.md "Tables".  Layouts: photon[n_mat][3][n_E], electron[n_mat][4][n_E]. */
typedef struct {
    int32_t n_materials;
    int32_t n_energy;
    double e_min, e_max;
    const float *photon;   /* compton, photo, pair                 cm^2/g            */
    const float *electron; /* L_restricted, moller, brems, 1/lambda1  (MeV) cm^2/g    */
    int32_t n_K;
    double lnK_min, lnK_max;
    const float *ms_a;     /* a(K) on a uniform ln K grid                             */
    double e_cut;          /* electron kinetic cutoff = K_cut of the tables           */
    double p_cut;          /* photon cutoff = k_c of the brems tables                 */
} orc_tables;

typedef struct {
    double es_max_cm;      /* e_s-max of Eq. 4                        */
    double f_eloss_max;    /* max fractional energy loss per step (R9)      */
    double boundary_nudge; /* fraction of the voxel size added to d_vox (R10)         */
    int32_t pair_mode;     /* 1: 2m leaves as two 0.511 MeV photons; 0: deposited     */
    int32_t photon_only;   /* 1: every electron is deposited where it is born         */
    double majorant_scale; /* >=1; inflates mu_max and M_e (Woodcock invariance pin)  */
    double hom_tol;        /* 0: Eq. 4 as printed.  > 0: multi-voxel steps (R32): d_vox
                              becomes the distance to the first voxel along d whose material
                              differs or whose density differs by more than hom_tol (relative)
                              from the start voxel's; the step's energy loss goes to the voxel
                              of a point drawn uniformly along the path of its two legs     */
} orc_options;

typedef struct {
    int32_t particle; /* 0 photon, 1 electron */
    int32_t shape;    /* 0 pencil, 1 parallel rectangle, 2 phase space */
    double cx, cy, wx, wy;
    double energy;    /* used when n_spec == 0 */
    int32_t n_spec;
    const float *spec_E; /* n_spec+1 bin edges */
    const float *spec_w; /* n_spec weights */
    /* shape 2, phase space (R35): n_phsp records {x, y, z, u, v, w, E, type};
     * history h starts from record h mod n_phsp exactly as given, no draw, transport from counter 1 */
    int64_t n_phsp;
    const float *phsp;
} orc_source;

typedef struct {
    uint64_t n_histories;
    uint64_t photon_flights, photon_compton, photon_photo, photon_pair, photon_fict;
    uint64_t ch_steps, hard_moller, hard_brems, hard_fict;
    uint64_t pushes_e, pushes_g;
    uint64_t stack_high_water;
    double e_incident, e_dep_continuous, e_dep_cutoff, e_escaped, e_pair_rest;
} orc_counters;

/* ---- random numbers ---- */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
void orc_philox_batch(const uint32_t *in, uint32_t *out, int64_t n);
double orc_uniform(uint32_t w);

/* ---- tables ---- */
double orc_lookup(const float *col, int32_t n, double x_min, double x_max, double x);
/* mu_max[n_E], m_e[n_E] from per-material maximum densities rho_max[n_mat] */
void orc_majorants(const orc_tables *t, const double *rho_max, double *mu_max, double *m_e);

/* ---- samplers, exposed for the distribution pins.  Each call uses the stream
 * (seed, hist=i, track=0, ctr=0...) for sample i.  Outputs have n entries. ---- */
void orc_batch_compton(double E, uint64_t seed, int64_t n, double *eps, double *cost, double *phi);
void orc_batch_sauter(double E, uint64_t seed, int64_t n, double *nu);
void orc_batch_pair(double E, uint64_t seed, int64_t n, double *T1, double *cos1, double *cos2);
void orc_batch_moller(double T, double k_cut, uint64_t seed, int64_t n, double *eps, double *cos_p,
                      double *cos_d);
void orc_batch_brems(double T, double k_c, uint64_t seed, int64_t n, double *k);
void orc_batch_ms(double a, uint64_t seed, int64_t n, double *cost);
void orc_rotate(const double d[3], double cost, double phi, double out[3]);

/* ---- the hot path ----
 * Simulates histories hist_begin .. hist_begin+n_hist-1.
 * edep_out  : double[nx*ny*nz], energy deposited per voxel in MeV, OVERWRITTEN.
 * dose_out  : float [nx*ny*nz] or NULL: edep/(rho h^3)/n_hist, MeV/g per history.
 * trace_out : uint64[n_hist] or NULL: event codes of the primary track, 3 bits each,
 *             first event in the low bits (1 Compton, 2 photo, 3 pair, 4 escaped,
 *             5 absorbed below P_cut), at most 21 events.
 * Returns 0, or a negative error code (-1 invalid argument, -4 stack overflow). */
int orc_run(const float *density, const uint8_t *material, int32_t nx, int32_t ny, int32_t nz,
            double voxel_cm, const orc_tables *t, const orc_options *opt, const orc_source *src,
            uint64_t hist_begin, uint64_t n_hist, uint64_t seed, double *edep_out,
            float *dose_out, uint64_t *trace_out, orc_counters *counters, int32_t n_threads);

/* As orc_run, plus edep_sq_out[nvox]: the sum over histories of the square of the energy one
 * history deposits in the voxel (MeV^2).  With edep_out this gives the history-by-history
 * uncertainty of PAPER.md Eq. 13: Delta D^2 = (<D^2> - <D>^2)/(N - 1). */
int orc_run_moments(const float *density, const uint8_t *material, int32_t nx, int32_t ny, int32_t nz,
                    double voxel_cm, const orc_tables *t, const orc_options *opt, const orc_source *src,
                    uint64_t hist_begin, uint64_t n_hist, uint64_t seed, double *edep_out,
                    double *edep_sq_out, orc_counters *counters, int32_t n_threads);

/* Mean CSDA path length check helper: total path length travelled by each primary
 * electron track (secondaries excluded) accumulated over a run; n entries. */
int orc_run_pathlen(const float *density, const uint8_t *material, int32_t nx, int32_t ny,
                    int32_t nz, double voxel_cm, const orc_tables *t, const orc_options *opt,
                    const orc_source *src, uint64_t n_hist, uint64_t seed, double *pathlen_out);

/* ---- pins of the transport loop itself (tests/test_oracle_pins.py) ---- */
#define ORC_VLOG_COLS 24
/* End state of every history's primary track, and the primary electron's path length per material. */
int orc_run_endstate(const float *density, const uint8_t *material, int32_t nx, int32_t ny, int32_t nz,
                     double voxel_cm, const orc_tables *t, const orc_options *opt, const orc_source *src,
                     uint64_t n_hist, uint64_t seed, int64_t max_steps, double *end_out, double *pathmat_out);
/* Log of every pushed secondary with its vertex (columns: see oracle.c). */
int orc_run_vertices(const float *density, const uint8_t *material, int32_t nx, int32_t ny, int32_t nz,
                     double voxel_cm, const orc_tables *t, const orc_options *opt, const orc_source *src,
                     uint64_t n_hist, uint64_t seed, double *vlog_out, int64_t cap, int64_t *n_out,
                     orc_counters *counters);

#ifdef __cplusplus
}
#endif
#endif
