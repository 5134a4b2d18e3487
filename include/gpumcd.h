/*
 * gpumcd.h -- C ABI of the B200-native GPUMCD hot path.
 *
 * Coupled photon-electron Monte Carlo transport through a voxelised phantom with energy
 * deposited into a 3-D dose grid (arxiv 1101.1245; Sec. II.A photons, II.B electrons,
 * II.C GPU implementation).  The calls follow the paper's statement of the problem:
 *   inputs  - a density volume and a composition-id volume,
 *             cross-section / stopping-power tables (L170), a source (L166),
 *             cutoffs P_cut (L45) and E_c (L79), the step bound e_s-max (L108);
 *   output  - the dose array (L188).
 *
 * Conventions
 *   - Every call returns a gpumcd_status; nothing throws or aborts across this boundary.
 *   - Pointers named *_dev are CUDA device pointers on the current device; *_host are host
 *     pointers.  The library copies what it needs at create time: the caller keeps ownership of
 *     everything it passes in and may free it as soon as the call returns.
 *   - Volumes are C arrays [nz][ny][nx]; voxel (ix,iy,iz) has index ix + nx*(iy + ny*iz) and
 *     spans [ix*h,(ix+1)*h) x ...; the beam enters the z = 0 face travelling along +z.
 *     nx, ny, nz <= 1024.
 *   - Units: MeV (kinetic for electrons), cm, g/cm^3.  Dose is MeV/g per primary history
 *     (x 1.602e-10 = Gy per history).
 *   - History ids are 0 .. n_histories-1.  A particle's random stream is Philox4x32-10 with
 *     counter (hist_lo, hist_hi, track, ctr) and key (seed_lo, seed_hi) (DESIGN.md "Random
 *     numbers"), so the same (seed, n_histories) gives the same result up to the order of the
 *     fp64 additions into the tally.
 */
#ifndef GPUMCD_H
#define GPUMCD_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct gpumcd_ctx gpumcd_ctx; /* opaque, owned by the library */

typedef enum {
    GPUMCD_OK = 0,
    GPUMCD_ERR_INVALID_ARG = -1,   /* null pointer, bad size, material id out of range, density outside
                                      [2^-20, 2^12) g/cm^3 (9.5e-7 .. 4096) or not a number */
    GPUMCD_ERR_CUDA = -2,          /* a CUDA runtime call failed; see gpumcd_last_error */
    GPUMCD_ERR_OOM = -3,           /* device allocation failed */
    GPUMCD_ERR_BANK_OVERFLOW = -4, /* a particle queue filled up; the run's result is invalid
                                      (the paper silently discards secondaries here, L166) */
    GPUMCD_ERR_NO_SOURCE = -5,     /* gpumcd_run before gpumcd_set_source */
    GPUMCD_ERR_TABLE_RANGE = -6    /* a source energy lies outside [e_min, e_max] of the tables */
} gpumcd_status;

/* Material tables, HOST arrays, copied at create.  All columns are mass
 * coefficients on a grid uniform in ln E between e_min and e_max (n_energy nodes), looked up by
 * linear interpolation in ln E and multiplied by the voxel density (Eq. 2).
 *   photon  [n_materials][3][n_energy] : Compton, photoelectric, pair              cm^2/g
 *   electron[n_materials][4][n_energy] : restricted stopping power L (Eq. 6)   MeV cm^2/g,
 *                                        hard Moller, hard bremsstrahlung,
 *                                        inverse first transport mean free path    cm^2/g
 *   ms_a    [n_K] : multiple-scattering shape parameter a(K) on a uniform ln K grid
 * e_cut is the electron kinetic cutoff E_c = K_cut the tables were built with; p_cut is the
 * photon cutoff P_cut = k_c of the bremsstrahlung tables. */
typedef struct {
    int32_t n_materials; /* 1..8 */
    int32_t n_energy;    /* >= 2 */
    float e_min, e_max;  /* MeV */
    const float *photon;
    const float *electron;
    int32_t n_K;
    float lnK_min, lnK_max;
    const float *ms_a;
    float e_cut;
    float p_cut;
} gpumcd_tables;

typedef struct {
    float es_max_cm;       /* e_s-max of Eq. 4 (L108); default 0.5                                 */
    float f_eloss_max;     /* largest fraction of its energy an electron may lose in one step; 0.25 */
    float boundary_nudge;  /* fraction of the voxel size added to d_vox of Eq. 4; 1e-4             */
    int32_t pair_mode;     /* 1 (default): the 2 m_e c^2 of a pair event leaves as two 0.511 MeV
                              photons; 0: it is deposited at the vertex (L74 is silent)            */
    int32_t photon_only;   /* 1: every electron is deposited where it is born; default 0           */
    float majorant_scale;  /* >= 1, inflates the Woodcock majorants (Eq. 3; test hook); default 1  */
    uint32_t wave_size;    /* scheduler 0: primaries generated per wave; default 2^20              */
    uint32_t bank_factor;  /* scheduler 0: queue capacity = bank_factor * wave_size records (the
                              paper's d, L166); default 8                                          */
    int32_t scheduler;     /* 1 (default): one persistent kernel per run; every warp keeps its own
                              type-sorted stacks of secondaries, refills its lanes and sorts events,
                              no host round trips;
                              0: the paper's scheme (L166): one launch per pass, one thread per
                              particle, the host reads the queue counts between passes            */
    uint32_t warp_stack;   /* scheduler 1: capacity of a warp's electron stack and of its photon
                              stack, records; default 8192 (2.8 GB for the 3552 warps of a B200), at
                              least 256.  A warp works on one particle type until it runs dry or the
                              other type's stack is about to fill up (bank_high_g / bank_high_e can make
                              it change earlier), so the capacity sets how long it stays in one part of
                              the code: on photon beams 4096 is 10 % faster than 1024 and 8192 another 2-4 %.
                              A history that breeds more secondaries than a stack holds overflows it:
                              that is reported (GPUMCD_ERR_BANK_OVERFLOW from gpumcd_run_host and
                              gpumcd_get_counters, overflow_count), never silently dropped        */
    uint32_t cta_threads;  /* scheduler 1: threads of the persistent kernel's one CTA per SM: 0 or 768
                              (default: 6 warps per scheduler, 80 registers per thread), or 512 (128
                              registers) or 1024 (64 registers), both slower on every workload measured
                              and kept for the ablation (fp64 tally and plain sources only)        */
    float hom_tol;         /* 0 (default): electron steps end at every voxel boundary, Eq. 4 as printed.
                              > 0: multi-voxel steps (the paper's "improvements to the electron-step
                              algorithm", L364-368, are future work there; R32): d_vox of
                              Eq. 4 becomes the distance along the direction of flight to the first
                              voxel whose material differs from the start voxel's or whose density
                              differs by more than hom_tol (relative), and the step's energy loss
                              (Eq. 8) is deposited in the voxel of a point drawn uniformly along
                              the path of its two hinge legs (every voxel's path-length share in
                              expectation).  e_s-max then bounds the step in uniform regions:
                              2-2.5 x fewer steps at 0.25 cm voxels                                 */
    int32_t tally_mode;    /* how deposits are added to the energy grid (the paper only says the dose arrays
                              "are summed", L188):
                              0 (default): one fp64 atomic add per deposit, resolved in L2;
                              1: warp-aggregated: lanes of a warp that deposit in the same voxel at the same
                                 time add up first (fp64, lane order) and issue one atomic;
                              2: 64-bit fixed point: every deposit is rounded to a multiple of 2^-k MeV (k chosen
                                 per run so that the grid cannot overflow, 31 for 1e8 histories of 20 MeV, at
                                 most 40; exact for deposits >= 2^(24-k) MeV) and added as an integer: the result
                                 does not depend on the order of the additions, so the same (seed, n_histories)
                                 gives the same dose bit for bit, on either scheduler.
                              Modes 1 and 2 need the default cta_threads.                              */
    int32_t table_memory;  /* scheduler 1: 0 (default) = the table blob is staged into shared memory by TMA
                              bulk copies when it fits (up to ~220 KB: 7 materials at 1024 nodes), else read
                              from global memory; 1 = always read from global memory (test hook)      */
    uint32_t bank_high_g;  /* scheduler 1, tuning (0 = never, the default): a warp stepping electrons changes to
                              photons as soon as this many photons are banked and fewer than bank_high_e
                              electrons are left (at least bank_low)                                     */
    uint32_t bank_high_e;  /* scheduler 1, tuning (0 = never, the default): the same for a warp flying photons.
                              They bound how much work of one type is done before the other type is picked
                              up; measured, every early change costs (round 1 ran 80 / 160: 10 % slower) */
    uint32_t bank_low;     /* scheduler 1, tuning (0 = 8, at most 32): once the source is exhausted a warp with
                              fewer ready particles of its type than this changes to the other type, if a full
                              batch (32) of that type waits.  Above 32 two stacks holding between 32 and bank_low
                              records would send the warp back and forth for ever: refused (INVALID_ARG)         */
    uint32_t steps_per_refill; /* scheduler 1: condensed-history steps a warp makes at most before it looks at its
                              stacks again (refills free lanes, banks hard-event candidates, may change type): the
                              paper's N, "stream compaction after N simulation steps" (L180).  Lanes whose electron
                              ended wait meanwhile, so the loop goes on only while 24 of the 32 lanes still step.
                              0 = automatic: 4; at most 64.  Ignored (1) with a phase-space source and with
                              cta_threads 1024                                                               */
    int32_t l2_persist;    /* scheduler 1: 1 = the packed phantom (4 bytes per voxel) is read through a persisting
                              L2 access window, so that the tally and the particle stacks cannot evict it
                              (raises the device-wide cudaLimitPersistingL2CacheSize to the phantom's size, up
                              to the device maximum; the lines stay set aside until gpumcd_release_l2);
                              0 (default) = plain caching                                                */
} gpumcd_options;

typedef struct {
    int32_t particle;    /* 0 photon, 1 electron (shapes 0 and 1; a phase space carries the type per record) */
    int32_t shape;       /* 0 pencil beam, 1 parallel rectangular field, 2 phase space */
    float cx, cy;        /* field centre on the z = 0 face, cm */
    float wx, wy;        /* full field widths, cm (ignored for a pencil beam) */
    float energy;        /* MeV, used when n_spec == 0 */
    int32_t n_spec;      /* number of spectrum bins, 0 = monoenergetic */
    const float *spec_E; /* HOST, n_spec+1 bin edges, MeV, increasing */
    const float *spec_w; /* HOST, n_spec non-negative bin weights; energy is uniform inside a bin */
    /* shape 2, a phase space (the paper's future work beside spectrum sources): n_phsp records of
     * 8 floats {x, y, z (cm, phantom frame), u, v, w (unit direction, used as given), E (MeV, kinetic for an
     * electron), type (0.0 photon, 1.0 electron)}.  History h starts from record h mod n_phsp, exactly as given
     * (no random number is drawn for the primary; its transport starts at draw counter 1 like every other
     * primary).  A record outside the phantom counts as escaped at birth, one below its type's cutoff is
     * deposited where it is (R5, R35).  gpumcd_set_source copies the records (library-owned) and checks
     * them: type 0 or 1, finite numbers, E inside the energy range of the tables (GPUMCD_ERR_TABLE_RANGE).
     * cx .. spec_w are ignored. */
    uint64_t n_phsp;
    const float *phsp;     /* n_phsp x 8 floats: DEVICE memory, or HOST memory if phsp_on_host != 0 */
    int32_t phsp_on_host;
} gpumcd_source;

typedef struct {
    uint64_t n_histories;
    uint64_t photon_flights, photon_compton, photon_photo, photon_pair, photon_fict;
    uint64_t ch_steps, hard_moller, hard_brems, hard_fict;
    uint64_t pushes_e, pushes_g;
    uint64_t bank_high_water; /* largest queue (scheduler 0) or warp stack (scheduler 1) occupancy seen, records */
    uint64_t overflow_count;  /* records dropped because a queue was full; must be 0 */
    double e_incident, e_dep_continuous, e_dep_cutoff, e_escaped, e_pair_rest; /* MeV */
} gpumcd_counters;

/* Fill *opt with the defaults listed above. */
int gpumcd_default_options(gpumcd_options *opt);

/* Build a context for one phantom: copies the volumes and tables to
 * library-owned device memory, finds the largest density of every material, builds the Woodcock
 * majorants mu_max(E) (Eq. 3) and M_e(E) (L110-113) and allocates the particle queues and the
 * fp64 energy tally.  opt == NULL selects the defaults.  Synchronous.
 * gpumcd_create takes DEVICE volumes, gpumcd_create_host takes HOST volumes (the copy to the
 * device is part of the call; this is the entry bench.py's end-to-end figure times). */
int gpumcd_create(gpumcd_ctx **out, const float *density_dev, const uint8_t *material_dev, int nx,
                  int ny, int nz, float voxel_cm, const gpumcd_tables *tables,
                  const gpumcd_options *opt);
int gpumcd_create_host(gpumcd_ctx **out, const float *density_host, const uint8_t *material_host,
                       int nx, int ny, int nz, float voxel_cm, const gpumcd_tables *tables,
                       const gpumcd_options *opt);

/* Replace the phantom of an existing context by another one of the same dimensions (the
 * per-patient inputs of the method): the volumes are copied (gpumcd_set_phantom:
 * DEVICE pointers; gpumcd_set_phantom_host: HOST pointers, the host-to-device copy is part of the
 * call and is fastest from pinned memory), validated, and the majorants mu_max(E), M_e(E) are
 * rebuilt.  Waits for the context's last run; synchronous.  Tables, options, source and queues
 * are kept.  On GPUMCD_ERR_INVALID_ARG (bad voxel) the context must be given a valid phantom
 * before the next run. */
int gpumcd_set_phantom(gpumcd_ctx *ctx, const float *density_dev, const uint8_t *material_dev);
int gpumcd_set_phantom_host(gpumcd_ctx *ctx, const float *density_host, const uint8_t *material_host);

/* Select the source (PAPER.md L166 initParticle): particle type, energy or spectrum, geometry. */
int gpumcd_set_source(gpumcd_ctx *ctx, const gpumcd_source *src);

/* Simulate n_histories primaries and all their secondaries (Sec. II.A-II.C) and write
 * the dose grid.  dose_out_dev: caller-owned float[nx*ny*nz] on the device, OVERWRITTEN.
 * cuda_stream: a cudaStream_t (NULL = default stream); all work is enqueued on it.  With
 * scheduler 1 the call returns without waiting for the device; with scheduler 0 it waits between
 * passes.  Errors detected on the device (queue overflow) are reported by gpumcd_get_counters (and by
 * gpumcd_run_host, which waits for the run anyway). */
int gpumcd_run(gpumcd_ctx *ctx, uint64_t n_histories, uint64_t seed, float *dose_out_dev,
               void *cuda_stream);

/* Same, with the dose copied into HOST memory; returns after the copy has completed. */
int gpumcd_run_host(gpumcd_ctx *ctx, uint64_t n_histories, uint64_t seed, float *dose_out_host,
                    void *cuda_stream);

/* Dose with its statistical uncertainty (Eq. 11-13).  The n_histories are simulated
 * in n_batches consecutive batches of (nearly) equal size; with x_b the mean energy per history that
 * batch b left in a voxel,
 *     Delta D = sqrt( (<x_b^2> - <x_b>^2) / (n_batches - 1) ) / (rho h^3),
 * which has the same expectation, sigma_history^2 / N, as Eq. 13's history-by-history sum (the
 * batches are the independent samples; a warp works on many histories at once, so per-history sums
 * per voxel do not exist on the device).  The batches cover exactly histories 0 .. n_histories-1, so
 * dose_out_dev equals the result of gpumcd_run with the same arguments up to fp64 summation order.
 * dose_out_dev, sigma_out_dev: caller-owned float[nx*ny*nz] on the device, OVERWRITTEN, both in MeV/g
 * per primary history.  2 <= n_batches <= n_histories.  Counters and the energy tally afterwards are
 * those of all batches together.  Eq. 12 (s) and Eq. 11 (efficiency) are reductions of these two
 * grids and are left to the caller. */
int gpumcd_run_uncertainty(gpumcd_ctx *ctx, uint64_t n_histories, uint32_t n_batches, uint64_t seed,
                           float *dose_out_dev, float *sigma_out_dev, void *cuda_stream);

/* gpumcd_run_uncertainty for callers that must not allocate device memory (code under CUDA graph capture,
 * tight serving loops, harnesses that forbid cudaMalloc).  gpumcd_run_uncertainty allocates its scratch, three
 * fp64 grids of batch statistics (24 bytes per voxel), with cudaMalloc on its first call; this entry point keeps
 * them in a static device array inside the library instead and calls no cudaMalloc, cudaFree or allocating
 * library routine.  Same arguments, same batches, same results (up to the order of the fp64 tally's additions).
 * Limits and rules:
 *  - at most GPUMCD_STATIC_MAX_VOXELS voxels (64^3: the paper's own geometries); a larger phantom is refused
 *    with GPUMCD_ERR_INVALID_ARG and a message naming the limit;
 *  - the array (6 MiB) exists once per GPU that loads the library, until the process exits, and is shared by
 *    every context and every call: it is cleared at the start of each call, and two calls that overlap on the
 *    GPU (different streams, different contexts) race on it: run them one after the other;
 *  - profiling must be off (gpumcd_set_profiling: its event pairs are created per launch);
 *  - the context itself is set up beforehand, as for every other call (gpumcd_create allocates). */
#define GPUMCD_STATIC_MAX_VOXELS 262144
int gpumcd_run_uncertainty_static(gpumcd_ctx *ctx, uint64_t n_histories, uint32_t n_batches, uint64_t seed,
                                  float *dose_out_dev, float *sigma_out_dev, void *cuda_stream);

/* Photon-only replay run: like gpumcd_run with photon_only = 1 but the output is, per history,
 * the ordered event codes of the primary track, 3 bits each, first event in the low bits, at most
 * 21 events: 1 Compton, 2 photoelectric, 3 pair, 4 escaped, 5 absorbed below P_cut.
 * trace_out_dev: caller-owned uint64[n_histories] on the device, OVERWRITTEN. */
int gpumcd_run_trace(gpumcd_ctx *ctx, uint64_t n_histories, uint64_t seed, uint64_t *trace_out_dev,
                     void *cuda_stream);

/* Counters and energy accounts of the last run.  Waits for that run's stream.  Returns
 * GPUMCD_ERR_BANK_OVERFLOW if the run dropped a particle. */
int gpumcd_get_counters(gpumcd_ctx *ctx, gpumcd_counters *host_out);

/* Copy the fp64 energy tally of the last run (MeV per voxel) to a caller-owned
 * double[nx*ny*nz] on the device, on the stream of that run. */
int gpumcd_get_energy_tally(gpumcd_ctx *ctx, double *edep_out_dev);

/* Shift the history ids of the following runs: they simulate histories first_history ..
 * first_history + n_histories - 1 (disjoint ranges on different GPUs give independent samples of
 * the same stream family).  Default 0.  Trace output is indexed from first_history. */
int gpumcd_set_history_offset(gpumcd_ctx *ctx, uint64_t first_history);

/* l2_persist = 1: wait for the context's last run and give the persisting L2 lines back to normal use
 * (cudaCtxResetPersistingL2Cache).  A no-op otherwise. */
int gpumcd_release_l2(gpumcd_ctx *ctx);

/* Per-kernel device times of the last run, measured with CUDA events on the run's stream, and the
 * number of kernels the run launched.  Recording is off by default (it adds events around every
 * launch); gpumcd_set_profiling(ctx, 1) turns it on for the following runs. */
typedef struct {
    uint64_t launches;     /* kernels launched by the last run (always counted) */
    uint32_t n_source, n_photon, n_electron, n_finalize; /* launches per class */
    float ms_source, ms_photon, ms_electron, ms_finalize; /* 0 unless profiling is on */
} gpumcd_profile;
int gpumcd_set_profiling(gpumcd_ctx *ctx, int enable);
int gpumcd_get_profile(gpumcd_ctx *ctx, gpumcd_profile *host_out); /* waits for the run's stream */

/* Tally probe: the rate (updates per second, returned in *updates_per_second, a HOST double) at which
 * this device adds fp64 values into THIS context's energy grid when it does nothing else: about n_updates
 * atomic adds at pseudo-random voxels under the current source's field (all depths), the address pattern
 * of the condensed-history deposits (H4/H8).  It is the measured denominator of the tally's roofline
 * (no vendor figure exists for the L2's fp64 atomic rate).  Synchronous on cuda_stream; the energy tally
 * of the last run is overwritten (zeroed afterwards); needs a source. */
int gpumcd_probe_tally(gpumcd_ctx *ctx, uint64_t n_updates, double *updates_per_second, void *cuda_stream);

/* Device-side self-test of the random-number layer: for i < n, out_dev[4i..4i+3] =
 * Philox4x32-10(counter = ctr_key_dev[6i..6i+3], key = ctr_key_dev[6i+4], ctr_key_dev[6i+5]) as the transport
 * kernels compute it, and (uniform_dev != NULL) uniform_dev[4i..] = U(word) = ((word >> 9) + 1/2) 2^-23 as they
 * turn words into uniforms.  All pointers are DEVICE pointers; asynchronous on cuda_stream. */
int gpumcd_selftest_philox(const uint32_t *ctr_key_dev, uint32_t *out_dev, float *uniform_dev, uint64_t n,
                           void *cuda_stream);

/* Library-owned, NUL-terminated description of the last error on this context (or of the last
 * failed create when ctx == NULL); valid until the next call on the same context. */
const char *gpumcd_last_error(gpumcd_ctx *ctx);

void gpumcd_destroy(gpumcd_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif
