/*
 * oracle.c -- CPU ORACLE of the GPUMCD hot path.  TEST INFRASTRUCTURE ONLY.
 * See oracle.h for scope, pins and the rule about who may call this.
 *
 * Plain C, fp64, one history at a time with a LIFO stack of secondaries.  Every
 * function cites the PAPER.md passage (or the DESIGN.md reading "R<n>" where the
 * paper is silent or garbled) that it follows.  No blocking, fusion or reordering.
 */
#include "oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define M_E ORC_M_E
#define TWO_PI 6.283185307179586476925286766559

/* ======================================================================== *
 * Random numbers.  The paper's combined multiply-with-carry generator
 * (Eq. 9-10) is replaced, as BASELINE.json's north_star
 * requires, by the counter-based Philox4x32-10 of Salmon et al. (SC'11) so that
 * a particle's random stream is a pure function of its lineage.
 * ======================================================================== */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
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

/* n blocks at once (test helper): in[6i..6i+3] = counter, in[6i+4], in[6i+5] = key; out[4i..4i+3] */
void orc_philox_batch(const uint32_t *in, uint32_t *out, int64_t n)
{
    for (int64_t i = 0; i < n; ++i) orc_philox4x32_10(in + 6 * i, in + 6 * i + 4, out + 4 * i);
}

/* U(w) = ((w >> 9) + 1/2) 2^-23, in (0,1): Eq. 1 needs zeta in (0,1].
 * 23 bits plus the half: exactly representable in fp32's 24-bit significand, so a
 * single-precision implementation sees the same value.  The low 9 bits of w are unused. */
double orc_uniform(uint32_t w) { return ((double)(w >> 9) + 0.5) * (1.0 / 8388608.0); }
#define U(w) orc_uniform(w)

/* A particle's stream: block(hist, track, ctr) = philox(counter = (hist_lo, hist_hi, track, ctr),
 * key = (seed_lo, seed_hi)).  Every transport step and every sampler trial consumes one
 * fresh block (ctr++); unused words are discarded. */
typedef struct {
    uint32_t key[2];
    uint32_t hist_lo, hist_hi, track, ctr;
} stream_t;

static void draw(stream_t *s, uint32_t w[4])
{
    uint32_t c[4] = { s->hist_lo, s->hist_hi, s->track, s->ctr };
    orc_philox4x32_10(c, s->key, w);
    s->ctr += 1u;
}

/* Track ids of the secondaries born at the parent's current counter: the block at
 * (hist, track, ctr | 2^31), a counter value no transport step reaches.  Child j gets
 * word j and starts at ctr = 0.  The parent's counter is not advanced. */
static void lineage(const stream_t *s, uint32_t w[4])
{
    uint32_t c[4] = { s->hist_lo, s->hist_hi, s->track, s->ctr | 0x80000000u };
    orc_philox4x32_10(c, s->key, w);
}

static stream_t make_stream(uint64_t seed, uint64_t hist, uint32_t track, uint32_t ctr)
{
    stream_t s;
    s.key[0] = (uint32_t)seed;
    s.key[1] = (uint32_t)(seed >> 32);
    s.hist_lo = (uint32_t)hist;
    s.hist_hi = (uint32_t)(hist >> 32);
    s.track = track;
    s.ctr = ctr;
    return s;
}

/* ======================================================================== *
 * Tables.  The paper pre-interpolates its data on a 1 keV grid;
 * here the grid is uniform in ln E and looked up by linear interpolation
 * (DESIGN.md "Tables").  x is ln E (or ln K for the a(K) table).
 * ======================================================================== */
double orc_lookup(const float *col, int32_t n, double x_min, double x_max, double x)
{
    double f = (x - x_min) / ((x_max - x_min) / (double)(n - 1));
    if (f < 0.0) f = 0.0;
    if (f > (double)(n - 1)) f = (double)(n - 1);
    int i = (int)floor(f);
    if (i > n - 2) i = n - 2;
    double t = f - (double)i;
    return (1.0 - t) * (double)col[i] + t * (double)col[i + 1];
}

/* Majorants.  Photons: mu_max of Eq. 3, "the attenuation coefficient of the most
 * attenuating voxel", evaluated per energy node; interpolating node
 * maxima linearly bounds every interpolated mu.  Electrons: L110-113 takes
 * mu_max(E) at the step-start energy "assuming mu decreasing with energy"; the
 * running maximum over lower energies makes that bound rigorous (R16). */
void orc_majorants(const orc_tables *t, const double *rho_max, double *mu_max, double *m_e)
{
    int nE = t->n_energy;
    for (int i = 0; i < nE; ++i) {
        double mu = 0.0, se = 0.0;
        for (int m = 0; m < t->n_materials; ++m) {
            const float *p = t->photon + (size_t)m * 3 * nE;
            const float *e = t->electron + (size_t)m * 4 * nE;
            double a = rho_max[m] * ((double)p[i] + (double)p[nE + i] + (double)p[2 * nE + i]);
            double b = rho_max[m] * ((double)e[nE + i] + (double)e[2 * nE + i]);
            if (a > mu) mu = a;
            if (b > se) se = b;
        }
        mu_max[i] = mu;
        m_e[i] = (i > 0 && m_e[i - 1] > se) ? m_e[i - 1] : se;
    }
}

/* ======================================================================== *
 * Direction change by polar angle theta (cos, sin given) and azimuth phi about
 * the current direction d (standard frame rotation; R-P8).
 * ======================================================================== */
static void rotate(const double d[3], double cost, double sint, double phi, double out[3])
{
    double u = d[0], v = d[1], w = d[2];
    double cp = cos(phi), sp = sin(phi);
    double r2 = u * u + v * v;
    double a, b, c;
    if (r2 < 1e-10) {
        a = sint * cp;
        b = sint * sp;
        c = (w >= 0.0 ? cost : -cost);
    } else {
        double r = sqrt(r2);
        a = u * cost + sint * (u * w * cp - v * sp) / r;
        b = v * cost + sint * (v * w * cp + u * sp) / r;
        c = w * cost - r * sint * cp;
    }
    double n = sqrt(a * a + b * b + c * c);
    out[0] = a / n; out[1] = b / n; out[2] = c / n;
}

void orc_rotate(const double d[3], double cost, double phi, double out[3])
{
    double s2 = 1.0 - cost * cost;
    rotate(d, cost, s2 > 0.0 ? sqrt(s2) : 0.0, phi, out);
}

/* ======================================================================== *
 * Samplers.  One Philox block per trial.
 * ======================================================================== */

/* Compton: Klein-Nishina for a free electron at rest.  The paper uses the
 * Everett-Cashwell fit, whose constants are not available; any exact sampler of the same
 * density is equivalent (R27).  Composition-rejection on eps = E'/E in [eps0, 1]:
 * f(eps) ~ (1/eps + eps) g(eps), g = 1 - eps t (2 - t)/(1 + eps^2), t = 1 - cos(theta). */
static void sample_compton(stream_t *s, double E, double *eps_out, double *cost, double *sint,
                           double *phi)
{
    double k = E / M_E;
    double eps0 = 1.0 / (1.0 + 2.0 * k);
    double a1 = log(1.0 / eps0);
    double a2 = 0.5 * (1.0 - eps0 * eps0);
    uint32_t v[4];
    for (;;) {
        draw(s, v);
        double eps;
        if (U(v[0]) < a1 / (a1 + a2))
            eps = exp(-a1 * U(v[1]));
        else
            eps = sqrt(eps0 * eps0 + (1.0 - eps0 * eps0) * U(v[1]));
        double t = (1.0 - eps) / (k * eps);
        double g = 1.0 - eps * t * (2.0 - t) / (1.0 + eps * eps);
        if (U(v[2]) <= g) {
            *eps_out = eps;
            *cost = 1.0 - t;
            double s2 = t * (2.0 - t);
            *sint = s2 > 0.0 ? sqrt(s2) : 0.0;
            *phi = TWO_PI * U(v[3]);
            return;
        }
    }
}

/* Photo-electron polar angle: Sauter K-shell distribution,
 * p(nu) ~ (2-nu)[1/(A+nu) + B] nu/(A+nu)^3, nu = 1-cos(theta) in [0,2],
 * A = 1/beta - 1, B = beta gamma (gamma-1)(gamma-2)/2.  nu/(A+nu)^3 is inverted exactly,
 * the remaining factor (maximal at nu = 0) is the rejection function. */
static void sample_sauter(stream_t *s, double T, double *nu_out, double *phi)
{
    double gam = 1.0 + T / M_E;
    double beta = sqrt(T * (T + 2.0 * M_E)) / (T + M_E);
    double A = 1.0 / beta - 1.0;
    double B = 0.5 * beta * gam * (gam - 1.0) * (gam - 2.0);
    double g0 = 2.0 * (1.0 / A + B);
    uint32_t v[4];
    for (;;) {
        draw(s, v);
        double q = sqrt(U(v[0])) * 2.0 / (A + 2.0);
        double nu = q * A / (1.0 - q);
        if (U(v[1]) * g0 <= (2.0 - nu) * (1.0 / (A + nu) + B)) {
            *nu_out = nu;
            *phi = TWO_PI * U(v[2]);
            return;
        }
    }
}

/* Pair production: no positron, two electrons; the available kinetic
 * energy E - 2m is "trivially split ... using a uniformly distributed random number";
 * each polar angle from the leading-order density ~ (1 - beta cos(theta))^-2; the two
 * azimuths are opposite. */
static void sample_pair(stream_t *s, double E, double *T1, double *T2, double *c1, double *c2,
                        double *phi)
{
    uint32_t v[4];
    draw(s, v);
    double Tsum = E - 2.0 * M_E;
    *T1 = U(v[0]) * Tsum;
    *T2 = Tsum - *T1;
    double b1 = sqrt(*T1 * (*T1 + 2.0 * M_E)) / (*T1 + M_E);
    double b2 = sqrt(*T2 * (*T2 + 2.0 * M_E)) / (*T2 + M_E);
    double x1 = 2.0 * U(v[1]) - 1.0, x2 = 2.0 * U(v[2]) - 1.0;
    *c1 = (x1 + b1) / (1.0 + b1 * x1);
    *c2 = (x2 + b2) / (1.0 + b2 * x2);
    *phi = TWO_PI * U(v[3]);
}

/* Moller scattering above K_cut: eps = W/T in [K_cut/T, 1/2] from 1/eps^2,
 * rejection with g(eps) = 1 + g2 eps^2 + r (r - g3), r = eps/(1-eps), maximal at 1/2. */
static void sample_moller(stream_t *s, double T, double k_cut, double *eps_out, double *phi)
{
    double tau = T / M_E;
    double g2 = (tau / (tau + 1.0)) * (tau / (tau + 1.0));
    double g3 = (2.0 * tau + 1.0) / ((tau + 1.0) * (tau + 1.0));
    double gmax = 1.0 + g2 * 0.25 + 1.0 * (1.0 - g3);
    double emin = k_cut / T;
    uint32_t v[4];
    for (;;) {
        draw(s, v);
        double eps = emin / (1.0 - U(v[0]) * (1.0 - 2.0 * emin));
        double r = eps / (1.0 - eps);
        double g = 1.0 + g2 * eps * eps + r * (r - g3);
        if (U(v[1]) * gmax <= g) {
            *eps_out = eps;
            *phi = TWO_PI * U(v[2]);
            return;
        }
    }
}

/* Bremsstrahlung photon energy above k_c: k from 1/k on [k_c, T],
 * rejection with the complete-screening shape 4/3 (1-y) + y^2, y = k/(T+m). */
static void sample_brems(stream_t *s, double T, double k_c, double *k_out, double *phi)
{
    uint32_t v[4];
    for (;;) {
        draw(s, v);
        double k = k_c * exp(U(v[0]) * log(T / k_c));
        double y = k / (T + M_E);
        if (U(v[1]) * (4.0 / 3.0) <= (4.0 / 3.0) * (1.0 - y) + y * y) {
            *k_out = k;
            *phi = TWO_PI * U(v[2]);
            return;
        }
    }
}

/* Multiple-scattering deflection (msnew.dat is absent, R13): the
 * one-parameter screened-Rutherford shape p(mu) ~ (a+mu)^-2, mu = (1-cos)/2 in [0,1],
 * whose a(K) is tabulated so that <cos(theta)> = exp(-K), K = path / lambda_1. */
static double ms_mu(double a, double u) { return a * u / (1.0 + a - u); }

/* ---- batch entry points for the distribution pins ---- */
void orc_batch_compton(double E, uint64_t seed, int64_t n, double *eps, double *cost, double *phi)
{
    for (int64_t i = 0; i < n; ++i) {
        stream_t s = make_stream(seed, (uint64_t)i, 0, 0);
        double st;
        sample_compton(&s, E, &eps[i], &cost[i], &st, &phi[i]);
    }
}
void orc_batch_sauter(double E, uint64_t seed, int64_t n, double *nu)
{
    for (int64_t i = 0; i < n; ++i) {
        stream_t s = make_stream(seed, (uint64_t)i, 0, 0);
        double phi;
        sample_sauter(&s, E, &nu[i], &phi);
    }
}
void orc_batch_pair(double E, uint64_t seed, int64_t n, double *T1, double *cos1, double *cos2)
{
    for (int64_t i = 0; i < n; ++i) {
        stream_t s = make_stream(seed, (uint64_t)i, 0, 0);
        double T2, phi;
        sample_pair(&s, E, &T1[i], &T2, &cos1[i], &cos2[i], &phi);
    }
}
void orc_batch_moller(double T, double k_cut, uint64_t seed, int64_t n, double *eps, double *cos_p,
                      double *cos_d)
{
    for (int64_t i = 0; i < n; ++i) {
        stream_t s = make_stream(seed, (uint64_t)i, 0, 0);
        double phi;
        sample_moller(&s, T, k_cut, &eps[i], &phi);
        double W = eps[i] * T;
        cos_p[i] = sqrt((T - W) * (T + 2.0 * M_E) / (T * (T - W + 2.0 * M_E)));
        cos_d[i] = sqrt(W * (T + 2.0 * M_E) / (T * (W + 2.0 * M_E)));
    }
}
void orc_batch_brems(double T, double k_c, uint64_t seed, int64_t n, double *k)
{
    for (int64_t i = 0; i < n; ++i) {
        stream_t s = make_stream(seed, (uint64_t)i, 0, 0);
        double phi;
        sample_brems(&s, T, k_c, &k[i], &phi);
    }
}
void orc_batch_ms(double a, uint64_t seed, int64_t n, double *cost)
{
    for (int64_t i = 0; i < n; ++i) {
        stream_t s = make_stream(seed, (uint64_t)i, 0, 0);
        uint32_t v[4];
        draw(&s, v);
        cost[i] = 1.0 - 2.0 * ms_mu(a, U(v[2]));
    }
}

/* ======================================================================== *
 * Transport
 * ======================================================================== */
typedef struct {
    int type; /* 0 photon, 1 electron */
    double x[3], d[3], E;
    uint32_t track, ctr;
    int primary;
} particle_t;

#define STACK_MAX 4096

typedef struct {
    /* inputs */
    const float *density;
    const uint8_t *material;
    int nx, ny, nz;
    double h;
    const orc_tables *t;
    orc_options opt;
    double ln_emin, ln_emax;
    double *mu_max, *m_e; /* majorants, n_energy each */
    /* outputs of one worker */
    double *edep;
    orc_counters c;
    /* per-history state */
    particle_t stack[STACK_MAX];
    int sp;
    int overflow;
    uint64_t seed, hist;
    uint64_t trace;
    int trace_n;
    int want_trace;
    double *pathlen; /* NULL, or where to accumulate the primary electron's path length */
    /* pins of the transport loop itself (orc_run_endstate, orc_run_vertices): NULL / 0 unless asked for */
    double *end;      /* 8 doubles: where and how the primary track ended (x, d, E, steps taken) */
    double *pathmat;  /* n_materials doubles: the primary electron's path length per material */
    int64_t max_steps; /* > 0: the primary electron is stopped after this many condensed-history steps */
    double *vlog;     /* ORC_VLOG_COLS doubles per pushed secondary */
    int64_t vlog_cap, vlog_n;
    double vtx[12];   /* the vertex being processed: kind, parent track, parent ctr, E0, d0, E1, d1, (pad) */
    /* history-by-history second moment (Eq. 13): NULL unless asked for */
    double *esq;     /* sum over histories of (energy the history left in the voxel)^2 */
    double *etmp;    /* energy the current history has left in each voxel so far */
    size_t *touched; /* voxels the current history has deposited in */
    size_t n_touched, cap_touched;
} world_t;

static double tab_photon(const world_t *W, int m, int col, double lnE)
{
    const orc_tables *t = W->t;
    return orc_lookup(t->photon + ((size_t)m * 3 + col) * t->n_energy, t->n_energy, W->ln_emin,
                      W->ln_emax, lnE);
}
static double tab_electron(const world_t *W, int m, int col, double lnE)
{
    const orc_tables *t = W->t;
    return orc_lookup(t->electron + ((size_t)m * 4 + col) * t->n_energy, t->n_energy, W->ln_emin,
                      W->ln_emax, lnE);
}
static double tab_major(const world_t *W, const double *col, double lnE)
{
    /* majorant columns are double; same interpolation rule as orc_lookup */
    int n = W->t->n_energy;
    double f = (lnE - W->ln_emin) / ((W->ln_emax - W->ln_emin) / (double)(n - 1));
    if (f < 0.0) f = 0.0;
    if (f > (double)(n - 1)) f = (double)(n - 1);
    int i = (int)floor(f);
    if (i > n - 2) i = n - 2;
    double tt = f - (double)i;
    return W->opt.majorant_scale * ((1.0 - tt) * col[i] + tt * col[i + 1]);
}

/* voxel containing x: (ix,iy,iz) = floor(x/h); returns 0 when outside the phantom */
static int locate(const world_t *W, const double x[3], int v[3])
{
    v[0] = (int)floor(x[0] / W->h);
    v[1] = (int)floor(x[1] / W->h);
    v[2] = (int)floor(x[2] / W->h);
    return v[0] >= 0 && v[0] < W->nx && v[1] >= 0 && v[1] < W->ny && v[2] >= 0 && v[2] < W->nz;
}
static size_t vindex(const world_t *W, const int v[3])
{
    return (size_t)v[0] + (size_t)W->nx * ((size_t)v[1] + (size_t)W->ny * (size_t)v[2]);
}

enum { DEP_CONTINUOUS, DEP_CUTOFF };
static void deposit(world_t *W, const int v[3], double e, int kind)
{
    const size_t idx = vindex(W, v);
    W->edep[idx] += e;
    if (W->esq) {
        if (W->etmp[idx] == 0.0) {
            if (W->n_touched == W->cap_touched) {
                W->cap_touched = W->cap_touched ? 2 * W->cap_touched : 1024;
                W->touched = (size_t *)realloc(W->touched, sizeof(size_t) * W->cap_touched);
            }
            W->touched[W->n_touched++] = idx;
        }
        W->etmp[idx] += e;
    }
    if (kind == DEP_CONTINUOUS) W->c.e_dep_continuous += e; else W->c.e_dep_cutoff += e;
}

static void push(world_t *W, int type, const double x[3], const double d[3], double E,
                 uint32_t track)
{
    if (W->sp >= STACK_MAX) { W->overflow = 1; return; }
    particle_t *p = &W->stack[W->sp++];
    p->type = type;
    memcpy(p->x, x, sizeof p->x);
    memcpy(p->d, d, sizeof p->d);
    p->E = E;
    p->track = track;
    p->ctr = 0;
    p->primary = 0;
    if (W->vlog) {
        /* one row per pushed secondary: the vertex (set by the caller) and the child as pushed */
        if (W->vlog_n < W->vlog_cap) {
            double *r = W->vlog + (size_t)W->vlog_n * ORC_VLOG_COLS;
            r[0] = (double)W->hist;
            memcpy(r + 1, W->vtx, sizeof(double) * 11);
            r[12] = (double)type; r[13] = (double)track; r[14] = E;
            r[15] = d[0]; r[16] = d[1]; r[17] = d[2];
            r[18] = x[0]; r[19] = x[1]; r[20] = x[2];
            r[21] = r[22] = r[23] = 0.0;
        }
        W->vlog_n++;
    }
    if (type == 0) W->c.pushes_g++; else W->c.pushes_e++;
    if ((uint64_t)W->sp > W->c.stack_high_water) W->c.stack_high_water = (uint64_t)W->sp;
}

static void trace_event(world_t *W, const particle_t *p, int code)
{
    if (W->want_trace && p->primary && W->trace_n < 21) {
        W->trace |= (uint64_t)code << (3 * W->trace_n);
        W->trace_n++;
    }
}

/* orc_run_vertices: describe the vertex whose secondaries are about to be pushed.  kind: 1 Compton,
 * 2 photoelectric, 3 pair, 4 Moller, 5 bremsstrahlung.  (E0, d0): the parent before the event,
 * (E1, d1): after it (E1 = 0 if it is absorbed). */
static void vertex(world_t *W, int kind, const stream_t *s, double E0, const double d0[3], double E1,
                   const double d1[3])
{
    if (!W->vlog) return;
    W->vtx[0] = (double)kind; W->vtx[1] = (double)s->track; W->vtx[2] = (double)s->ctr;
    W->vtx[3] = E0; W->vtx[4] = d0[0]; W->vtx[5] = d0[1]; W->vtx[6] = d0[2];
    W->vtx[7] = E1; W->vtx[8] = d1[0]; W->vtx[9] = d1[1]; W->vtx[10] = d1[2];
}

/* orc_run_endstate: where and how the primary track ended */
static void end_state(world_t *W, const particle_t *p, int64_t steps)
{
    if (!W->end || !p->primary) return;
    W->end[0] = p->x[0]; W->end[1] = p->x[1]; W->end[2] = p->x[2];
    W->end[3] = p->d[0]; W->end[4] = p->d[1]; W->end[5] = p->d[2];
    W->end[6] = p->E; W->end[7] = (double)steps;
}

/* An electron is born with kinetic energy T at x: transported if T >= E_cut and electrons
 * are transported at all, otherwise deposited on the spot (R5). */
static int electron_is_tracked(const world_t *W, double T)
{
    return !W->opt.photon_only && T >= W->t->e_cut;
}

/* ---------------- photon history: PAPER.md Sec. II.A (L45-74) ---------------- */
static void photon_history(world_t *W, particle_t p)
{
    stream_t s = make_stream(W->seed, W->hist, p.track, p.ctr);
    const double p_cut = W->t->p_cut;
    int v[3];
    for (;;) {
        uint32_t w[4];
        draw(&s, w);
        double lnE = log(p.E);
        double mu_max = tab_major(W, W->mu_max, lnE);
        /* Eq. 1 with the Woodcock majorant (Eq. 3) */
        double dist = -log(U(w[0])) / mu_max;
        for (int a = 0; a < 3; ++a) p.x[a] += dist * p.d[a];
        W->c.photon_flights++;
        if (!locate(W, p.x, v)) {
            W->c.e_escaped += p.E;
            trace_event(W, &p, 4);
            return;
        }
        size_t iv = vindex(W, v);
        int m = W->material[iv];
        double rho = (double)W->density[iv];
        /* Eq. 2 per interaction type; the remainder up to mu_max is the fictitious one */
        double r = U(w[1]) * mu_max;
        double c1 = rho * tab_photon(W, m, 0, lnE);
        double c2 = c1 + rho * tab_photon(W, m, 1, lnE);
        /* pair production needs E > 2 m (L74): the column interpolated between the nodes around the
         * threshold is not zero just below it (R33) */
        double c3 = c2 + (p.E > 2.0 * M_E ? rho * tab_photon(W, m, 2, lnE) : 0.0);
        if (r < c1) {
            /* ---- Compton (L65) ---- */
            W->c.photon_compton++;
            trace_event(W, &p, 1);
            double eps, cost, sint, phi, dnew[3];
            sample_compton(&s, p.E, &eps, &cost, &sint, &phi);
            rotate(p.d, cost, sint, phi, dnew);
            double E1 = eps * p.E;
            double Te = p.E - E1;
            if (electron_is_tracked(W, Te)) {
                /* recoil direction from momentum conservation: E d - E' d' */
                double q[3], n = 0.0;
                for (int a = 0; a < 3; ++a) { q[a] = p.E * p.d[a] - E1 * dnew[a]; n += q[a] * q[a]; }
                n = sqrt(n);
                for (int a = 0; a < 3; ++a) q[a] /= n;
                uint32_t id[4];
                lineage(&s, id);
                vertex(W, 1, &s, p.E, p.d, E1, dnew);
                push(W, 1, p.x, q, Te, id[0]);
            } else {
                deposit(W, v, Te, DEP_CUTOFF);
            }
            p.E = E1;
            memcpy(p.d, dnew, sizeof dnew);
            if (p.E < p_cut) {
                deposit(W, v, p.E, DEP_CUTOFF);
                trace_event(W, &p, 5);
                return;
            }
        } else if (r < c2) {
            /* ---- photoelectric (L67-72): one electron, T = E_phot (R7) ---- */
            W->c.photon_photo++;
            trace_event(W, &p, 2);
            if (electron_is_tracked(W, p.E)) {
                double nu, phi, q[3];
                sample_sauter(&s, p.E, &nu, &phi);
                double s2 = nu * (2.0 - nu);
                rotate(p.d, 1.0 - nu, s2 > 0.0 ? sqrt(s2) : 0.0, phi, q);
                uint32_t id[4];
                lineage(&s, id);
                vertex(W, 2, &s, p.E, p.d, 0.0, p.d);
                push(W, 1, p.x, q, p.E, id[0]);
            } else {
                deposit(W, v, p.E, DEP_CUTOFF);
            }
            return;
        } else if (r < c3) {
            /* ---- pair production (L74) ---- */
            W->c.photon_pair++;
            trace_event(W, &p, 3);
            double T1, T2, ca, cb, phi, q1[3], q2[3];
            sample_pair(&s, p.E, &T1, &T2, &ca, &cb, &phi);
            double sa = 1.0 - ca * ca, sb = 1.0 - cb * cb;
            rotate(p.d, ca, sa > 0.0 ? sqrt(sa) : 0.0, phi, q1);
            rotate(p.d, cb, sb > 0.0 ? sqrt(sb) : 0.0, phi + 0.5 * TWO_PI, q2);
            double qa[3] = { 0, 0, 1 }, qb[3] = { 0, 0, -1 };
            if (W->opt.pair_mode == 1) {
                /* the rest energy 2m leaves the vertex as two back-to-back 0.511 MeV photons,
                 * isotropic (no positron is transported, L74; R6) */
                uint32_t z[4];
                draw(&s, z);
                double cz = 2.0 * U(z[0]) - 1.0;
                double sz = sqrt(1.0 - cz * cz);
                double pz = TWO_PI * U(z[1]);
                qa[0] = sz * cos(pz); qa[1] = sz * sin(pz); qa[2] = cz;
                for (int a = 0; a < 3; ++a) qb[a] = -qa[a];
            }
            int t1 = electron_is_tracked(W, T1), t2 = electron_is_tracked(W, T2);
            uint32_t id[4] = { 0, 0, 0, 0 };
            if (t1 || t2 || W->opt.pair_mode == 1) lineage(&s, id);
            vertex(W, 3, &s, p.E, p.d, 0.0, p.d);
            if (t1) push(W, 1, p.x, q1, T1, id[0]); else deposit(W, v, T1, DEP_CUTOFF);
            if (t2) push(W, 1, p.x, q2, T2, id[1]); else deposit(W, v, T2, DEP_CUTOFF);
            W->c.e_pair_rest += 2.0 * M_E;
            if (W->opt.pair_mode == 1) {
                push(W, 0, p.x, qa, M_E, id[2]);
                push(W, 0, p.x, qb, M_E, id[3]);
            } else {
                deposit(W, v, 2.0 * M_E, DEP_CUTOFF);
            }
            return;
        } else {
            W->c.photon_fict++; /* fictitious interaction: nothing changes (L59) */
        }
    }
}

/* ---------------- multi-voxel steps (R32; the paper's "improvements to the electron-step
 * algorithm", L364-368, are future work there) ---------------- */

/* Distance from x (inside voxel v) along d to the face through which the ray leaves voxel v; *axis
 * receives the axis of that face. */
static double exit_distance(const world_t *W, const double x[3], const double d[3], const int v[3], int *axis)
{
    double best = HUGE_VAL;
    *axis = 0;
    for (int k = 0; k < 3; ++k) {
        double dk = HUGE_VAL;
        if (d[k] > 0.0) dk = ((double)(v[k] + 1) * W->h - x[k]) / d[k];
        else if (d[k] < 0.0) dk = ((double)v[k] * W->h - x[k]) / d[k];
        if (dk < best) { best = dk; *axis = k; }
    }
    return best < 0.0 ? 0.0 : best;
}

/* d_hom: distance along d to the first voxel that does not continue the start voxel's medium (other
 * material, density off by more than hom_tol, or outside the phantom); HUGE_VAL if none within s_max. */
static double hom_distance(const world_t *W, const double x0[3], const double d[3], const int v0[3], double s_max)
{
    const size_t i0 = vindex(W, v0);
    const int m0 = W->material[i0];
    const double rho0 = (double)W->density[i0];
    double x[3] = {x0[0], x0[1], x0[2]};
    int v[3] = {v0[0], v0[1], v0[2]};
    double t = 0.0;
    for (;;) {
        int axis;
        const double te = exit_distance(W, x, d, v, &axis);
        t += te;
        if (t >= s_max) return HUGE_VAL;
        for (int k = 0; k < 3; ++k) x[k] += te * d[k];
        v[axis] += d[axis] > 0.0 ? 1 : -1;
        x[axis] = (double)(d[axis] > 0.0 ? v[axis] : v[axis] + 1) * W->h; /* exactly on the face */
        if (v[0] < 0 || v[0] >= W->nx || v[1] < 0 || v[1] >= W->ny || v[2] < 0 || v[2] >= W->nz) return t;
        const size_t i = vindex(W, v);
        if (W->material[i] != m0 || fabs((double)W->density[i] - rho0) > W->opt.hom_tol * rho0) return t;
    }
}

/* The uniform of the deposit point (R32): 23 bits from the low 9 bits of the step block's words 1-3,
 * which U() does not use (word 0's low bit chooses the hinge alternative). */
static double U_low(const uint32_t a[4])
{
    uint32_t bits = (a[1] & 0x1ffu) | ((a[2] & 0x1ffu) << 9) | ((a[3] & 0x1fu) << 18);
    return ((double)bits + 0.5) * (1.0 / 8388608.0);
}

/* ---------------- electron history: PAPER.md Sec. II.B (L78-139) ---------------- */
static void electron_history(world_t *W, particle_t p)
{
    stream_t s = make_stream(W->seed, W->hist, p.track, p.ctr);
    const orc_tables *t = W->t;
    const double e_cut = t->e_cut, h = W->h;
    int v[3];
    int64_t steps = 0;
    if (!locate(W, p.x, v)) { W->c.e_escaped += p.E; end_state(W, &p, steps); return; }
    if (!electron_is_tracked(W, p.E)) { deposit(W, v, p.E, DEP_CUTOFF); end_state(W, &p, steps); return; }
    for (;;) {
        if (W->max_steps > 0 && p.primary && steps == W->max_steps) {
            /* orc_run_endstate: the primary is taken out of the run here (audited as escaped) */
            W->c.e_escaped += p.E;
            end_state(W, &p, steps);
            return;
        }
        size_t iv = vindex(W, v);
        int m = W->material[iv];
        double rho = (double)W->density[iv];
        double T = p.E, lnT = log(T);
        uint32_t a[4];
        draw(&s, a);
        /* distance to the next hard interaction by Woodcock with the majorant taken at the
         * step-start energy (L110-113), re-sampled every step (R15) */
        double M = tab_major(W, W->m_e, lnT);
        double e_hard = M > 0.0 ? -log(U(a[0])) / M : HUGE_VAL;
        /* distance to the voxel boundary along d, plus the boundary nudge (R10) */
        double d_vox = HUGE_VAL;
        for (int k = 0; k < 3; ++k) {
            double dk = HUGE_VAL;
            if (p.d[k] > 0.0) dk = ((double)(v[k] + 1) * h - p.x[k]) / p.d[k];
            else if (p.d[k] < 0.0) dk = ((double)v[k] * h - p.x[k]) / p.d[k];
            if (dk < d_vox) d_vox = dk;
        }
        d_vox += W->opt.boundary_nudge * h;
        double L0 = rho * tab_electron(W, m, 0, lnT);
        double e_cap = W->opt.f_eloss_max * T / L0; /* R9 */
        if (W->opt.es_max_cm < e_cap) e_cap = W->opt.es_max_cm;
        const int multi = W->opt.hom_tol > 0.0;
        if (multi) { /* R32: the boundary that limits the step is the next change of medium along d */
            d_vox = hom_distance(W, p.x, p.d, v, e_hard < e_cap ? e_hard : e_cap);
            d_vox += W->opt.boundary_nudge * h;
        }
        /* Eq. 4: e_s = min{d_vox, e_s-max, e_hard} */
        int hard = (e_hard <= d_vox && e_hard <= e_cap);
        double es = hard ? e_hard : (d_vox < e_cap ? d_vox : e_cap);
        /* Eq. 8 (de-garbled, R3): dE = s L(E0 - L(E0) s / 2) */
        double Tmid = T - 0.5 * L0 * es;
        if (Tmid < t->e_min) Tmid = t->e_min;
        double dE = es * rho * tab_electron(W, m, 0, log(Tmid));
        W->c.ch_steps++;
        steps++;
        if (T - dE < e_cut) {
            /* end of range: everything left is deposited in the current voxel (R8) */
            if (W->pathlen && p.primary) *W->pathlen += es * (T - e_cut) / dE;
            deposit(W, v, T, DEP_CUTOFF);
            end_state(W, &p, steps);
            return;
        }
        if (W->pathlen && p.primary) *W->pathlen += es;
        if (W->pathmat && p.primary) W->pathmat[m] += es;
        double zeta = U(a[1]);
        /* R32: the loss of a multi-voxel step goes to the voxel of a point drawn uniformly along the
         * step's path (first leg, then second leg): the path-length share of every voxel in expectation */
        const double s_dep = multi ? U_low(a) * es : 0.0;
        if (!multi) {
            deposit(W, v, dE, DEP_CONTINUOUS); /* at the hinge, which lies in the step-start voxel (R11) */
        } else if (s_dep <= zeta * es) {
            double xd[3];
            int vd[3];
            for (int k = 0; k < 3; ++k) xd[k] = p.x[k] + s_dep * p.d[k];
            deposit(W, locate(W, xd, vd) ? vd : v, dE, DEP_CONTINUOUS);
        }
        /* random hinge (L137): first leg zeta e_s */
        for (int k = 0; k < 3; ++k) p.x[k] += zeta * es * p.d[k];
        /* Bielajew's alternate hinge (L139, R12): scattering strength at the energy before
         * or after the loss, chosen by the low bit of a[0] (unused by U) */
        double Tms = (a[0] & 1u) ? T : T - dE;
        double K = es * rho * tab_electron(W, m, 3, log(Tms));
        double lnK = K > 0.0 ? log(K) : -HUGE_VAL;
        if (lnK >= t->lnK_min) {
            double sa = orc_lookup(t->ms_a, t->n_K, t->lnK_min, t->lnK_max, lnK);
            double mu = ms_mu(sa, U(a[2]));
            double dnew[3];
            rotate(p.d, 1.0 - 2.0 * mu, 2.0 * sqrt(mu * (1.0 - mu)), TWO_PI * U(a[3]), dnew);
            memcpy(p.d, dnew, sizeof dnew);
        }
        /* second leg (1 - zeta) e_s (L137 prints (zeta-1): sign garble, R2) */
        if (multi && s_dep > zeta * es) {
            double xd[3];
            int vd[3];
            for (int k = 0; k < 3; ++k) xd[k] = p.x[k] + (s_dep - zeta * es) * p.d[k];
            deposit(W, locate(W, xd, vd) ? vd : v, dE, DEP_CONTINUOUS); /* a point outside: the start voxel */
        }
        for (int k = 0; k < 3; ++k) p.x[k] += (1.0 - zeta) * es * p.d[k];
        p.E = T - dE;
        if (!locate(W, p.x, v)) { W->c.e_escaped += p.E; end_state(W, &p, steps); return; }
        if (!hard) continue;
        /* ---- hard event: real or fictitious (L110-113), at the post-step energy ---- */
        uint32_t b[4];
        draw(&s, b);
        iv = vindex(W, v);
        int m1 = W->material[iv];
        double rho1 = (double)W->density[iv];
        double lnT1 = log(p.E);
        /* a Moller event transfers W in [K_cut, T/2] (L90): none is possible for T <= 2 K_cut, where the
         * column interpolated between the nodes around the threshold is not zero (R33) */
        double sM = p.E > 2.0 * e_cut ? rho1 * tab_electron(W, m1, 1, lnT1) : 0.0;
        double sB = rho1 * tab_electron(W, m1, 2, lnT1);
        double r = U(b[0]) * M;
        if (r < sM) {
            /* Moller (L88-90): scattered and knock-on electrons */
            W->c.hard_moller++;
            double eps, phi, dp[3], dd[3];
            double T1 = p.E;
            sample_moller(&s, T1, e_cut, &eps, &phi);
            double Wd = eps * T1;
            double c2p = (T1 - Wd) * (T1 + 2.0 * M_E) / (T1 * (T1 - Wd + 2.0 * M_E));
            double c2d = Wd * (T1 + 2.0 * M_E) / (T1 * (Wd + 2.0 * M_E));
            rotate(p.d, sqrt(c2p), sqrt(1.0 - c2p > 0.0 ? 1.0 - c2p : 0.0), phi, dp);
            rotate(p.d, sqrt(c2d), sqrt(1.0 - c2d > 0.0 ? 1.0 - c2d : 0.0), phi + 0.5 * TWO_PI, dd);
            uint32_t id[4];
            lineage(&s, id);
            vertex(W, 4, &s, T1, p.d, T1 - Wd, dp);
            push(W, 1, p.x, dd, Wd, id[0]); /* Wd >= K_cut = E_cut: always tracked */
            p.E = T1 - Wd;
            memcpy(p.d, dp, sizeof dp);
        } else if (r < sM + sB) {
            /* bremsstrahlung (L92): electron direction unchanged, photon at theta = m/E (R14) */
            W->c.hard_brems++;
            double k, phi, dg[3];
            double T1 = p.E;
            sample_brems(&s, T1, t->p_cut, &k, &phi);
            double th = M_E / (T1 + M_E);
            rotate(p.d, cos(th), sin(th), phi, dg);
            uint32_t id[4];
            lineage(&s, id);
            vertex(W, 5, &s, T1, p.d, T1 - k, p.d);
            push(W, 0, p.x, dg, k, id[0]); /* k >= k_c = P_cut: always tracked */
            p.E = T1 - k;
            if (p.E < e_cut) { deposit(W, v, p.E, DEP_CUTOFF); end_state(W, &p, steps); return; }
        } else {
            W->c.hard_fict++;
        }
    }
}

/* ---------------- source (PAPER.md L166 initParticle; R17) ---------------- */
static int make_primary(world_t *W, const orc_source *src, const double *cdf, particle_t *p)
{
    if (src->shape == 2) {
        /* phase space (R35): record h mod n, exactly as given; no draw is made
         * for the primary and its transport starts at counter 1 like every other primary's */
        const float *r = src->phsp + 8 * (size_t)(W->hist % (uint64_t)src->n_phsp);
        p->type = r[7] != 0.0f;
        for (int k = 0; k < 3; ++k) { p->x[k] = (double)r[k]; p->d[k] = (double)r[3 + k]; }
        p->E = (double)r[6];
        p->track = 0;
        p->ctr = 1;
        p->primary = 1;
        return 0;
    }
    stream_t s = make_stream(W->seed, W->hist, 0, 0);
    uint32_t w[4];
    draw(&s, w);
    p->type = src->particle;
    p->x[0] = src->cx; p->x[1] = src->cy; p->x[2] = 0.0;
    if (src->shape == 1) {
        p->x[0] = src->cx + (U(w[0]) - 0.5) * src->wx;
        p->x[1] = src->cy + (U(w[1]) - 0.5) * src->wy;
    }
    p->d[0] = 0.0; p->d[1] = 0.0; p->d[2] = 1.0;
    if (src->n_spec > 0) {
        double target = U(w[2]) * cdf[src->n_spec];
        int j = 0;
        while (j < src->n_spec - 1 && cdf[j + 1] <= target) ++j;
        p->E = (double)src->spec_E[j] + U(w[3]) * ((double)src->spec_E[j + 1] - (double)src->spec_E[j]);
    } else {
        p->E = src->energy;
    }
    p->track = 0;
    p->ctr = s.ctr; /* = 1 */
    p->primary = 1;
    return 0;
}

/* outputs of the transport-loop pins (single worker; all NULL / 0 in a plain run) */
typedef struct {
    double *end;      /* [n_hist][8] */
    double *pathmat;  /* [n_hist][n_materials] */
    int64_t max_steps;
    double *vlog;     /* [vlog_cap][ORC_VLOG_COLS] */
    int64_t vlog_cap;
    int64_t *vlog_n;
} pins_t;

static int run_impl(const float *density, const uint8_t *material, int32_t nx, int32_t ny,
                    int32_t nz, double voxel_cm, const orc_tables *t, const orc_options *opt,
                    const orc_source *src, uint64_t hist_begin, uint64_t n_hist, uint64_t seed,
                    double *edep_out, float *dose_out, uint64_t *trace_out, orc_counters *counters,
                    int32_t n_threads, double *pathlen_out, double *edep_sq_out, const pins_t *pins)
{
    if (!density || !material || !t || !opt || !src || !edep_out) return -1;
    if (nx <= 0 || ny <= 0 || nz <= 0 || voxel_cm <= 0.0) return -1;
    if (t->n_materials <= 0 || t->n_energy < 2 || t->e_cut < t->e_min) return -1;
    if (src->shape == 2) {
        if (src->n_phsp <= 0 || !src->phsp) return -1;
        for (int64_t i = 0; i < src->n_phsp; ++i) {
            const float *r = src->phsp + 8 * (size_t)i;
            if (!(r[7] == 0.0f || r[7] == 1.0f)) return -1;
            if (!((double)r[6] >= t->e_min && (double)r[6] <= t->e_max)) return -1;
        }
    } else if (src->n_spec == 0 && (src->energy > t->e_max || src->energy < t->e_min)) return -1;
    if (opt->majorant_scale < 1.0) return -1;
    const size_t nvox = (size_t)nx * ny * nz;

    /* per-material maximum density -> majorants */
    double *rho_max = (double *)calloc((size_t)t->n_materials, sizeof(double));
    for (size_t i = 0; i < nvox; ++i) {
        if (material[i] >= t->n_materials || !(density[i] > 0.0f)) { free(rho_max); return -1; }
        if ((double)density[i] > rho_max[material[i]]) rho_max[material[i]] = (double)density[i];
    }
    double *mu_max = (double *)malloc(sizeof(double) * (size_t)t->n_energy);
    double *m_e = (double *)malloc(sizeof(double) * (size_t)t->n_energy);
    orc_majorants(t, rho_max, mu_max, m_e);
    free(rho_max);

    double *cdf = NULL;
    if (src->n_spec > 0) {
        cdf = (double *)malloc(sizeof(double) * (size_t)(src->n_spec + 1));
        cdf[0] = 0.0;
        for (int j = 0; j < src->n_spec; ++j) cdf[j + 1] = cdf[j] + (double)src->spec_w[j];
    }

#ifdef _OPENMP
    int nthr = n_threads > 0 ? n_threads : omp_get_max_threads();
#else
    int nthr = 1;
#endif
    world_t **workers = (world_t **)calloc((size_t)nthr, sizeof(world_t *));
    int failed = 0;

#ifdef _OPENMP
#pragma omp parallel num_threads(nthr)
#endif
    {
#ifdef _OPENMP
        int tid = omp_get_thread_num();
#else
        int tid = 0;
#endif
        world_t *W = (world_t *)calloc(1, sizeof(world_t));
        workers[tid] = W;
        W->density = density; W->material = material;
        W->nx = nx; W->ny = ny; W->nz = nz; W->h = voxel_cm;
        W->t = t; W->opt = *opt;
        W->ln_emin = log(t->e_min); W->ln_emax = log(t->e_max);
        W->mu_max = mu_max; W->m_e = m_e;
        W->edep = (tid == 0) ? edep_out : (double *)malloc(sizeof(double) * nvox);
        memset(W->edep, 0, sizeof(double) * nvox);
        if (edep_sq_out) {
            W->esq = (tid == 0) ? edep_sq_out : (double *)malloc(sizeof(double) * nvox);
            memset(W->esq, 0, sizeof(double) * nvox);
            W->etmp = (double *)calloc(nvox, sizeof(double));
        }
        W->seed = seed;
        W->want_trace = trace_out != NULL;
        if (pins) { W->max_steps = pins->max_steps; W->vlog = pins->vlog; W->vlog_cap = pins->vlog_cap; }
#ifdef _OPENMP
#pragma omp for schedule(static)
#endif
        for (int64_t ih = 0; ih < (int64_t)n_hist; ++ih) {
            if (W->overflow) continue;
            W->hist = hist_begin + (uint64_t)ih;
            W->sp = 0; W->trace = 0; W->trace_n = 0;
            W->pathlen = pathlen_out ? &pathlen_out[ih] : NULL;
            if (W->pathlen) *W->pathlen = 0.0;
            if (pins && pins->end) { W->end = pins->end + 8 * ih; memset(W->end, 0, 8 * sizeof(double)); }
            if (pins && pins->pathmat) {
                W->pathmat = pins->pathmat + (size_t)t->n_materials * ih;
                memset(W->pathmat, 0, sizeof(double) * (size_t)t->n_materials);
            }
            particle_t p;
            make_primary(W, src, cdf, &p);
            W->c.e_incident += p.E;
            W->c.n_histories++;
            W->stack[W->sp++] = p;
            if (src->shape == 2 && p.type == 0) {
                /* a phase-space photon is treated like a photon pushed at a vertex: outside the phantom it
                 * has escaped, below P_cut it is deposited where it is (R5, R35); electron_history applies
                 * the same two rules to every electron it is handed */
                int v[3];
                if (!locate(W, p.x, v)) { W->c.e_escaped += p.E; W->sp = 0; }
                else if (p.E < t->p_cut) { deposit(W, v, p.E, DEP_CUTOFF); W->sp = 0; }
            }
            while (W->sp > 0 && !W->overflow) {
                particle_t q = W->stack[--W->sp];
                if (q.type == 0) photon_history(W, q); else electron_history(W, q);
            }
            if (trace_out) trace_out[ih] = W->trace;
            /* Eq. 13: the history's contribution to <D^2> is the square of ALL it left in a voxel */
            for (size_t k = 0; k < W->n_touched; ++k) {
                const size_t idx = W->touched[k];
                W->esq[idx] += W->etmp[idx] * W->etmp[idx];
                W->etmp[idx] = 0.0;
            }
            W->n_touched = 0;
        }
    }

    /* reduce workers in thread order */
    orc_counters tot;
    memset(&tot, 0, sizeof tot);
    for (int k = 0; k < nthr; ++k) {
        world_t *W = workers[k];
        if (!W) continue;
        if (W->overflow) failed = 1;
        if (pins && pins->vlog_n) *pins->vlog_n = W->vlog_n;
        if (k > 0) {
            for (size_t i = 0; i < nvox; ++i) edep_out[i] += W->edep[i];
            free(W->edep);
            if (W->esq) {
                for (size_t i = 0; i < nvox; ++i) edep_sq_out[i] += W->esq[i];
                free(W->esq);
            }
        }
        free(W->etmp);
        free(W->touched);
        const orc_counters *c = &W->c;
        tot.n_histories += c->n_histories;
        tot.photon_flights += c->photon_flights; tot.photon_compton += c->photon_compton;
        tot.photon_photo += c->photon_photo; tot.photon_pair += c->photon_pair;
        tot.photon_fict += c->photon_fict; tot.ch_steps += c->ch_steps;
        tot.hard_moller += c->hard_moller; tot.hard_brems += c->hard_brems;
        tot.hard_fict += c->hard_fict; tot.pushes_e += c->pushes_e; tot.pushes_g += c->pushes_g;
        if (c->stack_high_water > tot.stack_high_water) tot.stack_high_water = c->stack_high_water;
        tot.e_incident += c->e_incident; tot.e_dep_continuous += c->e_dep_continuous;
        tot.e_dep_cutoff += c->e_dep_cutoff; tot.e_escaped += c->e_escaped;
        tot.e_pair_rest += c->e_pair_rest;
        free(W);
    }
    free(workers); free(mu_max); free(m_e); free(cdf);
    if (counters) *counters = tot;
    /* dose = energy / mass / number of histories (R24) */
    if (dose_out) {
        double h3 = voxel_cm * voxel_cm * voxel_cm;
        for (size_t i = 0; i < nvox; ++i)
            dose_out[i] = (float)(edep_out[i] / ((double)density[i] * h3) / (double)n_hist);
    }
    return failed ? -4 : 0;
}

int orc_run(const float *density, const uint8_t *material, int32_t nx, int32_t ny, int32_t nz,
            double voxel_cm, const orc_tables *t, const orc_options *opt, const orc_source *src,
            uint64_t hist_begin, uint64_t n_hist, uint64_t seed, double *edep_out, float *dose_out,
            uint64_t *trace_out, orc_counters *counters, int32_t n_threads)
{
    return run_impl(density, material, nx, ny, nz, voxel_cm, t, opt, src, hist_begin, n_hist, seed,
                    edep_out, dose_out, trace_out, counters, n_threads, NULL, NULL, NULL);
}

/* As orc_run, and also the per-voxel sum over histories of the squared energy a history deposits
 * (edep_sq_out, MeV^2): with edep_out these are N <D> and N <D^2> of PAPER.md Eq. 13 in energy units,
 * history by history. */
int orc_run_moments(const float *density, const uint8_t *material, int32_t nx, int32_t ny, int32_t nz,
                    double voxel_cm, const orc_tables *t, const orc_options *opt, const orc_source *src,
                    uint64_t hist_begin, uint64_t n_hist, uint64_t seed, double *edep_out,
                    double *edep_sq_out, orc_counters *counters, int32_t n_threads)
{
    if (!edep_sq_out) return -1;
    return run_impl(density, material, nx, ny, nz, voxel_cm, t, opt, src, hist_begin, n_hist, seed,
                    edep_out, NULL, NULL, counters, n_threads, NULL, edep_sq_out, NULL);
}

int orc_run_pathlen(const float *density, const uint8_t *material, int32_t nx, int32_t ny,
                    int32_t nz, double voxel_cm, const orc_tables *t, const orc_options *opt,
                    const orc_source *src, uint64_t n_hist, uint64_t seed, double *pathlen_out)
{
    size_t nvox = (size_t)nx * ny * nz;
    double *edep = (double *)malloc(sizeof(double) * nvox);
    if (!edep) return -3;
    int rc = run_impl(density, material, nx, ny, nz, voxel_cm, t, opt, src, 0, n_hist, seed, edep,
                      NULL, NULL, NULL, 1, pathlen_out, NULL, NULL);
    free(edep);
    return rc;
}

/* Transport-loop pin: the state in which each history's PRIMARY track ended (end_out[n_hist][8] = position,
 * direction, energy, condensed-history steps taken) and, for an electron primary, its path length per material
 * (pathmat_out[n_hist][n_materials], step lengths booked on the step-start voxel's material; may be NULL).
 * max_steps > 0 takes the primary electron out of the run after that many steps.  One worker. */
int orc_run_endstate(const float *density, const uint8_t *material, int32_t nx, int32_t ny, int32_t nz,
                     double voxel_cm, const orc_tables *t, const orc_options *opt, const orc_source *src,
                     uint64_t n_hist, uint64_t seed, int64_t max_steps, double *end_out, double *pathmat_out)
{
    if (!end_out || max_steps < 0) return -1;
    size_t nvox = (size_t)nx * ny * nz;
    double *edep = (double *)malloc(sizeof(double) * nvox);
    if (!edep) return -3;
    pins_t pins = { end_out, pathmat_out, max_steps, NULL, 0, NULL };
    int rc = run_impl(density, material, nx, ny, nz, voxel_cm, t, opt, src, 0, n_hist, seed, edep, NULL, NULL,
                      NULL, 1, NULL, NULL, &pins);
    free(edep);
    return rc;
}

/* Transport-loop pin: one row of ORC_VLOG_COLS doubles per secondary, in the order they are pushed, as they
 * are pushed (the in-situ kinematics, not a re-typed copy).  Columns: 0 history, 1 vertex kind (1 Compton,
 * 2 photoelectric, 3 pair, 4 Moller, 5 bremsstrahlung), 2 parent track id, 3 parent draw counter at the
 * vertex, 4 parent energy before, 5-7 parent direction before, 8 parent energy after (0: absorbed), 9-11
 * parent direction after, 12 child type (0 photon, 1 electron), 13 child track id, 14 child energy, 15-17
 * child direction, 18-20 vertex position.  At most cap rows are written; *n_out receives the number of
 * secondaries pushed.  One worker. */
int orc_run_vertices(const float *density, const uint8_t *material, int32_t nx, int32_t ny, int32_t nz,
                     double voxel_cm, const orc_tables *t, const orc_options *opt, const orc_source *src,
                     uint64_t n_hist, uint64_t seed, double *vlog_out, int64_t cap, int64_t *n_out,
                     orc_counters *counters)
{
    if (!vlog_out || cap <= 0 || !n_out) return -1;
    size_t nvox = (size_t)nx * ny * nz;
    double *edep = (double *)malloc(sizeof(double) * nvox);
    if (!edep) return -3;
    pins_t pins = { NULL, NULL, 0, vlog_out, cap, n_out };
    int rc = run_impl(density, material, nx, ny, nz, voxel_cm, t, opt, src, 0, n_hist, seed, edep, NULL, NULL,
                      counters, 1, NULL, NULL, &pins);
    free(edep);
    return rc;
}
