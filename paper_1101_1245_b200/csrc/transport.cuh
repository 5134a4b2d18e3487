// transport.cuh -- per-particle transport of the GPUMCD hot path (device code, sm_100a).
//
// photon_step   : PAPER.md Sec. II.A (L45-74)  one Woodcock flight + interaction
// electron_step : PAPER.md Sec. II.B (L104-139) one class-II condensed-history step
// electron_hard : PAPER.md Sec. II.B.1 (L88-92, L110-113) hard-event candidate
// All follow DESIGN.md "Algorithm" draw for draw.  They report what happened through event codes;
// who runs which particle when, and how events are counted, is the schedulers' business
// (gpumcd.cu, persistent.cuh).
#pragma once

#include "physics.cuh"

namespace gpumcd {

// All tables live in one blob (global memory, or its copy in shared memory); the transport
// functions take the blob's base pointer `TB` and these float offsets:
//   [0]      photon   [n_mat][3][nE] compton, photo, pair         (cm^2/g)
//   [off_el] electron [n_mat][4][nE] L, moller, brems, 1/lambda1
//   [off_mu] mu_max   [nE] photon majorant (1/cm), majorant_scale applied
//   [off_me] m_e      [nE] electron hard-event majorant (1/cm)
//   [off_ms] ms_a     [nK]
struct Tables {
    const float *blob; // the global-memory copy
    unsigned off_el, off_mu, off_me, off_ms;
    Grid gE, gK;
    float e_min, e_cut, p_cut;
    int n_mat;
};

struct Geom {
    const uint32_t *phantom; // packed {density, material id}, 4 bytes per voxel (pack_voxel_record)
    const uint8_t *radius;   // multi-voxel steps only (else nullptr): the uniform radius of every voxel
    int nx, ny, nz;
    float h, inv_h;
};

struct Opts {
    float es_max, f_eloss, nudge, hom_tol;
    int pair_mode, photon_only;
};

// Compile-time variant of the transport code: TRACE records the primary track's event codes
// (gpumcd_run_trace), MULTI selects multi-voxel electron steps (R32), TALLY the tally arithmetic
// (gpumcd_options.tally_mode), PHSP a phase-space source (gpumcd_source.shape 2: primaries of both types, possibly
// outside the phantom or below a cutoff; kept out of the other variants, where its code cost 4 % of the run time).
enum : int { TALLY_F64 = 0, TALLY_WARP = 1, TALLY_FIXED = 2 };
// INNER: scheduler 1 makes up to `steps_per_refill` condensed-history steps per look at its stacks (the paper's N,
// L180); a variant of its own because the loop form costs the single-step form 2 % where it does not pay.
template <bool TRACE_, bool MULTI_, int TALLY_, bool PHSP_ = false, bool INNER_ = false>
struct Variant {
    static constexpr bool TRACE = TRACE_, MULTI = MULTI_, PHSP = PHSP_, INNER = INNER_;
    static constexpr int TALLY = TALLY_;
};

// Particle queue: three 16-byte SoA streams -> every push / pop is three 128-bit accesses.
struct Queue {
    float4 *A;        // fx, fy, fz, E
    float4 *B;        // u, v, w, packed voxel (bits)
    uint4 *C;         // hist_lo, track, ctr, -
    unsigned *count;  // device counter
    unsigned cap;
};

constexpr int kEnergySlots = 64;
struct EnergySlot { // energy accounts in global memory, spread over slots so that the flushes do not pile on one address
    double e_esc, e_cut, e_inc;
};
struct DevCounters {
    unsigned long long photon_flights, photon_compton, photon_photo, photon_pair, photon_fict;
    unsigned long long ch_steps, hard_moller, hard_brems, hard_fict;
    unsigned long long pushes_e, pushes_g;
    unsigned long long overflow;
    unsigned long long high_water; // scheduler 1: fullest per-warp stack seen
    double e_dep_total;
    EnergySlot slot[kEnergySlots];
};

struct Params {
    Tables tab;
    Geom geo;
    Opts opt;
    Rng rng;
    double *edep;                 // energy tally; TALLY_FIXED: 64-bit integers in units of 1/fx_scale MeV until finalize
    float fx_scale;               // TALLY_FIXED: a power of two chosen per run so that the grid cannot overflow
    DevCounters *cnt;
    unsigned long long *trace;    // or nullptr
    unsigned long long trace_off; // id of the run's first history
};

// Energy accounts (escaped, deposited below a cutoff): every thread adds into its own two fp64 slots in shared
// memory, and a kernel flushes them once at its end (acc_flush).  They used to be fp64 atomics on 64 slots in
// global memory, one per escape / cutoff deposit: a few 1e8 atomics per run on 2 KB, i.e. on one L2 slice, whose
// queue then held up every other request of the SMs (config 5: the phantom loads waited ~3000 cycles).
constexpr int kAccThreads = 1024; // largest CTA of any kernel that uses the accounts
struct Acc {
    __device__ __forceinline__ explicit Acc(const Params &) {}
    static __device__ __forceinline__ double *slots()
    {
        __shared__ double s_acc[2 * kAccThreads];
        return s_acc;
    }
    __device__ __forceinline__ void esc(float e) const { slots()[threadIdx.x] += static_cast<double>(e); }
    __device__ __forceinline__ void cut(float e) const { slots()[kAccThreads + threadIdx.x] += static_cast<double>(e); }
};
// all threads of the CTA, before any transport code runs
__device__ __forceinline__ void acc_init()
{
    Acc::slots()[threadIdx.x] = 0.0;
    Acc::slots()[kAccThreads + threadIdx.x] = 0.0;
}
__device__ __forceinline__ EnergySlot *energy_slot(const Params &P)
{
    return &P.cnt->slot[((blockIdx.x * blockDim.x + threadIdx.x) >> 5) & (kEnergySlots - 1)];
}

// Phantom record, 4 bytes per voxel (half of {float density, int material}: the phantom is fetched at every move,
// PAPER.md L168, and a warp waits for the slowest of its 32 fetches, so what matters is that the whole phantom
// stays in L2).  Lossless: a density is a positive finite float, so its sign bit is 0, and with its biased
// exponent in [kExpLo, kExpLo + 32), i.e. 2^-20 <= rho < 2^12 g/cm^3 (checked when the phantom is loaded), three
// exponent bits are free too:  bits 0-27 = (exponent - kExpLo) << 23 | mantissa,  bits 28-31 = material id.
constexpr uint32_t kExpLo = 107u;
struct Voxel {
    float x; // density, g/cm^3 (bit for bit the caller's)
    int m;   // material id
};
__host__ __device__ __forceinline__ bool density_packable(uint32_t float_bits)
{
    const uint32_t e = float_bits >> 23; // sign bit included: a negative number fails too
    return e >= kExpLo && e < kExpLo + 32u;
}
__host__ __device__ __forceinline__ uint32_t pack_voxel_record(uint32_t float_bits, int m)
{
    return (float_bits - (kExpLo << 23)) | (static_cast<uint32_t>(m) << 28);
}
__device__ __forceinline__ Voxel unpack_voxel(uint32_t b)
{
    return Voxel{__uint_as_float((b & 0x0fffffffu) + (kExpLo << 23)), static_cast<int>(b >> 28)};
}
__device__ __forceinline__ Voxel fetch_voxel(const Geom &g, unsigned lin) { return unpack_voxel(__ldg(&g.phantom[lin])); }
__device__ __forceinline__ int mat_of(Voxel pv) { return pv.m; }
// Multi-voxel steps: the uniform radius R of a voxel (0-7): every voxel within Chebyshev distance R continues
// its medium (same material, density within hom_tol), so no ray from inside it meets a change of medium before
// R voxel sizes.

__device__ __forceinline__ bool inside(const Geom &g, const Particle &p)
{
    return (static_cast<unsigned>(p.ix) < static_cast<unsigned>(g.nx)) &
           (static_cast<unsigned>(p.iy) < static_cast<unsigned>(g.ny)) &
           (static_cast<unsigned>(p.iz) < static_cast<unsigned>(g.nz));
}
// Internal layout of the library's volumes (phantom, tally, radius): the caller's, x fastest,
// lin = ix + nx (iy + ny iz); <= 2^30 voxels.  These two functions are the only place that knows it.
// (Measured alternative: z fastest, the beam axis, so that consecutive steps of a track share 32-byte sectors:
// 1 % on config 5, nothing on configs 2-4, and a pencil beam (config 1) then piles its deposits onto a few
// sectors of one column, whose atomics serialise: 0.155 -> 0.28 ms.  Dropped.)
__device__ __forceinline__ unsigned lin_of(const Geom &g, int ix, int iy, int iz)
{
    return static_cast<unsigned>(ix) + static_cast<unsigned>(g.nx) * (static_cast<unsigned>(iy) +
           static_cast<unsigned>(g.ny) * static_cast<unsigned>(iz));
}
__device__ __forceinline__ unsigned voxel_index(const Geom &g, const Particle &p) { return lin_of(g, p.ix, p.iy, p.iz); }
// internal index t -> index in the caller's [nz][ny][nx] arrays
__device__ __forceinline__ size_t caller_index(const Geom &, size_t t) { return t; }

// H4/H8 tally into the L2-resident energy grid (the paper only says the dose arrays "are summed", L188):
//   TALLY_F64   one fp64 atomic add per lane (RED.E.ADD.F64, resolved in L2);
//   TALLY_WARP  warp-aggregated: the lanes that are together here and hit the same voxel (match.any on the
//               voxel index) add up in fp64 in lane order and their first lane issues one atomic;
//   TALLY_FIXED 64-bit fixed point: e * 2^k rounded to an integer (exact for e >= 2^(24-k) MeV), integer
//               atomic add: additions commute exactly, so the tally is bitwise reproducible.
template <class V>
__device__ __forceinline__ void deposit(const Params &P, unsigned lin, float e)
{
    if (V::TALLY == TALLY_FIXED) {
        atomicAdd(reinterpret_cast<unsigned long long *>(P.edep) + lin,
                  static_cast<unsigned long long>(__float2ll_rn(e * P.fx_scale)));
    } else if (V::TALLY == TALLY_WARP) {
        const unsigned act = __activemask();
        const unsigned grp = __match_any_sync(act, lin);
        double s = static_cast<double>(e);
        if (grp & (grp - 1u)) { // several lanes on this voxel: every one of them walks the group in lane order
            s = 0.0;
            for (unsigned m = grp; m; m &= m - 1u) s += static_cast<double>(__shfl_sync(grp, e, __ffs(m) - 1));
        }
        if ((threadIdx.x & 31) == __ffs(grp) - 1) atomicAdd(&P.edep[lin], s);
    } else {
        atomicAdd(&P.edep[lin], static_cast<double>(e));
    }
}
// the tally entry as energy in MeV (finalize)
template <int TALLY>
__device__ __forceinline__ double tally_value(const Params &P, size_t i)
{
    if (TALLY == TALLY_FIXED)
        return static_cast<double>(reinterpret_cast<const long long *>(P.edep)[i]) / static_cast<double>(P.fx_scale);
    return P.edep[i];
}

// A record that finds its queue full is counted, never dropped silently (R18).  Out of line: the push code is
// inlined a dozen times and this never runs in a valid run.
__device__ __noinline__ void count_overflow(DevCounters *cnt) { atomicAdd(&cnt->overflow, 1ull); }

// ---- records ---------------------------------------------------------------------------------
__device__ __forceinline__ void store_rec(float4 *A, float4 *B, uint4 *C, size_t i, const Particle &c, uint32_t extra)
{
    A[i] = make_float4(c.fx, c.fy, c.fz, c.E);
    B[i] = make_float4(c.u, c.v, c.w, __uint_as_float(pack_voxel(c.ix, c.iy, c.iz)));
    C[i] = make_uint4(c.hist, c.track, c.ctr, extra);
}
__device__ __forceinline__ Particle load_rec(const float4 *A, const float4 *B, const uint4 *C, size_t i, uint32_t &extra)
{
    // (a popped record is never read again: evict-first loads keep its lines from crowding the phantom and the
    // tally out of the L2; 0.3-0.7 % on the photon configs)
    const float4 a = __ldcs(&A[i]);
    const float4 b = __ldcs(&B[i]);
    const uint4 c = __ldcs(&C[i]);
    Particle p;
    p.fx = a.x; p.fy = a.y; p.fz = a.z; p.E = a.w;
    p.u = b.x; p.v = b.y; p.w = b.z;
    const uint32_t vox = __float_as_uint(b.w);
    p.ix = vox & 1023u; p.iy = (vox >> 10) & 1023u; p.iz = vox >> 20;
    p.hist = c.x; p.track = c.y; p.ctr = c.z;
    extra = c.w;
    return p;
}

// H7 push from divergent code: one atomic per group of converged lanes (activemask + popc prefix),
// then three 16-byte stores per record.
//   Queue     : a global queue shared by the whole grid (scheduler 0); counter in global memory
//   WarpStack : a stack owned by the calling warp (scheduler 1); counter in shared memory.  A lane
//               that finds the stack full gives its claim back, so the counter ends at the number of
//               records stored and never above the capacity.
struct WarpStack {
    float4 *A;
    float4 *B;
    uint4 *C;
    unsigned *count;  // shared memory
    unsigned *pushed; // shared memory: event counter (pushes_e / pushes_g)
    unsigned cap;
};

__device__ __forceinline__ void push(const Params &P, const Queue &q, const Particle &c, unsigned long long *tally)
{
    const unsigned mask = __activemask();
    const int lane = threadIdx.x & 31;
    const int leader = __ffs(mask) - 1;
    unsigned base = 0;
    if (lane == leader) {
        base = atomicAdd(q.count, static_cast<unsigned>(__popc(mask)));
        if (tally) atomicAdd(tally, static_cast<unsigned long long>(__popc(mask)));
    }
    base = __shfl_sync(mask, base, leader);
    const unsigned slot = base + __popc(mask & ((1u << lane) - 1u));
    if (slot < q.cap) store_rec(q.A, q.B, q.C, slot, c, 0u);
    else count_overflow(P.cnt);
}
__device__ __forceinline__ void push(const Params &P, const WarpStack &q, const Particle &c)
{
    const unsigned mask = __activemask();
    const int lane = threadIdx.x & 31;
    const int leader = __ffs(mask) - 1;
    unsigned base = 0;
    if (lane == leader) {
        base = atomicAdd(q.count, static_cast<unsigned>(__popc(mask)));
        atomicAdd(q.pushed, static_cast<unsigned>(__popc(mask)));
    }
    base = __shfl_sync(mask, base, leader);
    const unsigned slot = base + __popc(mask & ((1u << lane) - 1u));
    if (slot < q.cap) {
        store_rec(q.A, q.B, q.C, slot, c, 0u);
    } else {
        atomicSub(q.count, 1u);
        count_overflow(P.cnt);
    }
}
__device__ __forceinline__ void push_e(const Params &P, const Queue &q, const Particle &c) { push(P, q, c, &P.cnt->pushes_e); }
__device__ __forceinline__ void push_g(const Params &P, const Queue &q, const Particle &c) { push(P, q, c, &P.cnt->pushes_g); }
__device__ __forceinline__ void push_e(const Params &P, const WarpStack &q, const Particle &c) { push(P, q, c); }
__device__ __forceinline__ void push_g(const Params &P, const WarpStack &q, const Particle &c) { push(P, q, c); }

__device__ __forceinline__ bool electron_tracked(const Params &P, float T)
{
    return !P.opt.photon_only && T >= P.tab.e_cut;
}

// ---------------------------------------------------------------------------------------------
// Photon transport in two halves, so that a scheduler can run them with different lane sets:
//   photon_flight   (H1 + the selection of H2): one Woodcock flight, then which interaction
//   photon_interact (H2): the interaction itself; secondaries are pushed to qE (electrons) and qG
//                   (annihilation photons)
// photon_step = flight + interaction, for one-thread-per-particle schedulers.  A photon's mode:
// PM_DEAD, PM_FLIGHT (next: a flight), PM_COMPTON / PM_PHOTO / PM_PAIR (next: that interaction at
// the current position).  TRACE records the primary track's event codes (gpumcd_run_trace).
// ---------------------------------------------------------------------------------------------
enum : int { PM_DEAD = 0, PM_FLIGHT = 1, PM_COMPTON = 2, PM_PHOTO = 3, PM_PAIR = 4 };
enum : int { PH_ESCAPE = 0, PH_COMPTON = 1, PH_ABSORBED = 2, PH_PHOTO = 3, PH_PAIR = 4, PH_FICT = 5 };
__device__ __forceinline__ bool photon_alive(int ev) { return ev == PH_COMPTON || ev == PH_FICT; }

// Replay trace (gpumcd_run_trace): the primary track appends its event codes, 3 bits each, to the
// history's word in global memory.  The codes are non-zero, so the number of events recorded so far
// is the index of the highest non-zero group + 1 and no per-particle trace state exists: a photon
// can be parked in a stack and picked up by another lane of its warp (persistent.cuh) in between.
template <class V>
__device__ __forceinline__ void record(const Params &P, const Particle &p, int code)
{
    if (V::TRACE && p.track == 0u) {
        volatile unsigned long long *t =
            P.trace + (((static_cast<unsigned long long>(P.rng.hist_hi) << 32) | p.hist) - P.trace_off);
        const unsigned long long bits = *t;
        const int n = bits ? (66 - __clzll(static_cast<long long>(bits))) / 3 : 0;
        if (n < 21) *t = bits | (static_cast<unsigned long long>(code) << (3 * n));
    }
}

// One flight (Eq. 1 with the Woodcock majorant of Eq. 3) and the choice of the interaction at its
// end (Eq. 2 per type; the remainder up to mu_max is fictitious, L59).  Returns the next mode:
// PM_DEAD (escaped), PM_FLIGHT (fictitious interaction: nothing changes), or the interaction.
template <class V>
__device__ __forceinline__ int photon_flight(const Params &P, const float *__restrict__ TB, Particle &p)
{
    const Tables &tb = P.tab;
    const uint4 w = draw<true>(P.rng, p);
    const Interp iE = locate(tb.gE, flog(p.E));
    const float mu_max = interp(TB + tb.off_mu, iE);
    const float s = fdiv(-flog(u01(w.x)), mu_max);
    advance(p, s * P.geo.inv_h);
    if (!inside(P.geo, p)) {
        Acc(P).esc(p.E);
        record<V>(P, p, 4);
        return PM_DEAD;
    }
    const Voxel pv = fetch_voxel(P.geo, voxel_index(P.geo, p));
    const float rho = pv.x;
    const float *col = TB + mat_of(pv) * 3 * tb.gE.n;
    const float r = u01(w.y) * mu_max;
    const float c1 = rho * interp(col, iE);
    const float c2 = fmaf(rho, interp(col + tb.gE.n, iE), c1);
    // pair production needs E > 2 m (L74; R33: the interpolated column is not zero just below the threshold)
    const float c3 = p.E > 2.0f * kMe ? fmaf(rho, interp(col + 2 * tb.gE.n, iE), c2) : c2;
    if (r >= c3) return PM_FLIGHT;
    return r < c1 ? PM_COMPTON : (r < c2 ? PM_PHOTO : PM_PAIR);
}

// The interaction `kind` (PM_COMPTON / PM_PHOTO / PM_PAIR) at the photon's position.  Returns
// PM_FLIGHT if the photon goes on (Compton above P_cut), else PM_DEAD.
template <class V, class QE, class QG>
__device__ __forceinline__ int photon_interact(const Params &P, Particle &p, int kind, const QE &qE, const QG &qG)
{
    const Tables &tb = P.tab;
    const Acc acc(P);
    const unsigned lin = voxel_index(P.geo, p);
    if (kind == PM_COMPTON) {
        // ---- Compton (L65) ----
        record<V>(P, p, 1);
        float eps, t, uphi, nu, nv, nw, sp, cp;
        sample_compton(P.rng, p, eps, t, uphi);
        sincos2pi(uphi, sp, cp);
        rotate(p.u, p.v, p.w, 1.0f - t, sqrtf(fmaxf(t * (2.0f - t), 0.0f)), cp, sp, nu, nv, nw);
        const float E1 = eps * p.E;
        const float Te = p.E - E1;
        if (electron_tracked(P, Te)) {
            Particle c = p;
            float qx = p.E * p.u - E1 * nu, qy = p.E * p.v - E1 * nv, qz = p.E * p.w - E1 * nw;
            const float inv = rsqrtf(fmaf(qx, qx, fmaf(qy, qy, qz * qz)));
            c.u = qx * inv; c.v = qy * inv; c.w = qz * inv;
            c.E = Te;
            c.track = lineage(P.rng, p).x;
            c.ctr = 0u;
            push_e(P, qE, c);
        } else {
            deposit<V>(P, lin, Te);
            acc.cut(Te);
        }
        p.E = E1;
        p.u = nu; p.v = nv; p.w = nw;
        if (p.E < tb.p_cut) {
            deposit<V>(P, lin, p.E);
            acc.cut(p.E);
            record<V>(P, p, 5);
            return PM_DEAD;
        }
        return PM_FLIGHT;
    }
    if (kind == PM_PHOTO) {
        // ---- photoelectric (L67-72): one electron with T = E_phot ----
        record<V>(P, p, 2);
        if (electron_tracked(P, p.E)) {
            float nu_, uphi, sp, cp;
            sample_sauter(P.rng, p, p.E, nu_, uphi);
            sincos2pi(uphi, sp, cp);
            Particle c = p;
            rotate(p.u, p.v, p.w, 1.0f - nu_, sqrtf(fmaxf(nu_ * (2.0f - nu_), 0.0f)), cp, sp, c.u, c.v, c.w);
            c.track = lineage(P.rng, p).x;
            c.ctr = 0u;
            push_e(P, qE, c);
        } else {
            deposit<V>(P, lin, p.E);
            acc.cut(p.E);
        }
        return PM_DEAD;
    }
    // ---- pair production (L74): two electrons, no positron ----
    record<V>(P, p, 3);
    const uint4 v = draw(P.rng, p);
    const float Tsum = p.E - 2.0f * kMe;
    const float T1 = u01(v.x) * Tsum;
    const float T2 = Tsum - T1;
    float ca, sa, cb, sb, sp, cp;
    pair_angle(T1, u01(v.y), ca, sa);
    pair_angle(T2, u01(v.z), cb, sb);
    sincos2pi(u01(v.w), sp, cp);
    float ax = 0.f, ay = 0.f, az = 1.f;
    if (P.opt.pair_mode == 1) {
        const uint4 z = draw(P.rng, p);
        az = 2.0f * u01(z.x) - 1.0f;
        const float sz = sqrtf(fmaxf(1.0f - az * az, 0.0f));
        float s2, c2_;
        sincos2pi(u01(z.y), s2, c2_);
        ax = sz * c2_;
        ay = sz * s2;
    }
    const bool t1 = electron_tracked(P, T1), t2 = electron_tracked(P, T2);
    uint4 id = make_uint4(0, 0, 0, 0);
    if (t1 || t2 || P.opt.pair_mode == 1) id = lineage(P.rng, p);
    Particle c = p;
    c.ctr = 0u;
    if (t1) {
        rotate(p.u, p.v, p.w, ca, sa, cp, sp, c.u, c.v, c.w);
        c.E = T1; c.track = id.x;
        push_e(P, qE, c);
    } else {
        deposit<V>(P, lin, T1);
        acc.cut(T1);
    }
    if (t2) {
        rotate(p.u, p.v, p.w, cb, sb, -cp, -sp, c.u, c.v, c.w); // opposite azimuth
        c.E = T2; c.track = id.y;
        push_e(P, qE, c);
    } else {
        deposit<V>(P, lin, T2);
        acc.cut(T2);
    }
    if (P.opt.pair_mode == 1) {
        c.E = kMe;
        c.u = ax; c.v = ay; c.w = az; c.track = id.z;
        push_g(P, qG, c);
        c.u = -ax; c.v = -ay; c.w = -az; c.track = id.w;
        push_g(P, qG, c);
    } else {
        deposit<V>(P, lin, 2.0f * kMe);
        acc.cut(2.0f * kMe);
    }
    return PM_DEAD;
}

// flight + interaction; returns the event (the photon is alive afterwards iff photon_alive(event))
template <class V>
__device__ int photon_step(const Params &P, const float *__restrict__ TB, Particle &p, const Queue &qE,
                           const Queue &qG)
{
    const int kind = photon_flight<V>(P, TB, p);
    if (kind == PM_DEAD) return PH_ESCAPE;
    if (kind == PM_FLIGHT) return PH_FICT;
    const int next = photon_interact<V>(P, p, kind, qE, qG);
    if (kind == PM_COMPTON) return next == PM_FLIGHT ? PH_COMPTON : PH_ABSORBED;
    return kind == PM_PHOTO ? PH_PHOTO : PH_PAIR;
}

// ---------------------------------------------------------------------------------------------
// One condensed-history step (H3, H4, H5).  Caller guarantees: inside the phantom, T >= E_cut,
// lnT = ln(p.E).  Returns ST_ALIVE, ST_DEAD, or ST_HARD (the step ended on a hard-event
// candidate; M is the majorant it was sampled with, to be passed to electron_hard).
// ---------------------------------------------------------------------------------------------
enum : int { ST_ALIVE = 0, ST_DEAD = 1, ST_HARD = 2 };

// ---- multi-voxel steps (R32; gpumcd_options.hom_tol > 0) ------------------------------
// Both walk the voxel grid along a direction in the kernels' (voxel, fraction) coordinates, lengths in
// voxel sizes.  kWalkMax bounds the walk (e_s-max / h voxels are crossed at most, a handful).
constexpr int kWalkMax = 256;

// distance to the face through which the ray leaves the voxel, and the axis of that face
__device__ __forceinline__ float exit_distance(float fx, float fy, float fz, float u, float v, float w, int &axis)
{
    const float tx = fdiv((u > 0.0f) ? 1.0f - fx : fx, fabsf(u));
    const float ty = fdiv((v > 0.0f) ? 1.0f - fy : fy, fabsf(v));
    const float tz = fdiv((w > 0.0f) ? 1.0f - fz : fz, fabsf(w));
    const float te = fminf(tx, fminf(ty, tz)); // a zero direction cosine gives +inf or NaN: dropped
    axis = (te == tx) ? 0 : ((te == ty) ? 1 : 2);
    return fmaxf(te, 0.0f);
}

// d_hom: distance along the direction to the first voxel that does not continue the start voxel's
// medium (other material, density off by more than hom_tol, outside the phantom); +inf if none
// within s_max.
__device__ __forceinline__ float hom_distance(const Params &P, const Particle &p, unsigned lin0, Voxel pv0, float s_max)
{
    // the voxel's uniform radius (precomputed per phantom) answers most look-aheads without a walk
    if (s_max < static_cast<float>(__ldg(&P.geo.radius[lin0]))) return __int_as_float(0x7f800000);
    float fx = p.fx, fy = p.fy, fz = p.fz, t = 0.0f;
    int ix = p.ix, iy = p.iy, iz = p.iz;
    const float band = P.opt.hom_tol * pv0.x;
    for (int it = 0; it < kWalkMax; ++it) {
        int axis;
        const float te = exit_distance(fx, fy, fz, p.u, p.v, p.w, axis);
        t += te;
        if (t >= s_max) return __int_as_float(0x7f800000);
        fx = fmaf(te, p.u, fx); fy = fmaf(te, p.v, fy); fz = fmaf(te, p.w, fz);
        if (axis == 0) { const bool up = p.u > 0.0f; ix += up ? 1 : -1; fx = up ? 0.0f : 1.0f; }
        else if (axis == 1) { const bool up = p.v > 0.0f; iy += up ? 1 : -1; fy = up ? 0.0f : 1.0f; }
        else { const bool up = p.w > 0.0f; iz += up ? 1 : -1; fz = up ? 0.0f : 1.0f; }
        if (static_cast<unsigned>(ix) >= static_cast<unsigned>(P.geo.nx) ||
            static_cast<unsigned>(iy) >= static_cast<unsigned>(P.geo.ny) ||
            static_cast<unsigned>(iz) >= static_cast<unsigned>(P.geo.nz)) return t;
        const Voxel pv = fetch_voxel(P.geo, lin_of(P.geo, ix, iy, iz));
        if (mat_of(pv) != mat_of(pv0) || fabsf(pv.x - pv0.x) > band) return t;
    }
    return t;
}

// The voxel of the point a distance t (voxel sizes) along the direction from the particle's position, or
// `fallback` if that point lies outside the phantom.
__device__ __forceinline__ unsigned voxel_ahead(const Geom &g, const Particle &p, float t, unsigned fallback)
{
    const int ix = p.ix + static_cast<int>(floorf(fmaf(t, p.u, p.fx)));
    const int iy = p.iy + static_cast<int>(floorf(fmaf(t, p.v, p.fy)));
    const int iz = p.iz + static_cast<int>(floorf(fmaf(t, p.w, p.fz)));
    const bool in = (static_cast<unsigned>(ix) < static_cast<unsigned>(g.nx)) & (static_cast<unsigned>(iy) < static_cast<unsigned>(g.ny)) &
                    (static_cast<unsigned>(iz) < static_cast<unsigned>(g.nz));
    return in ? lin_of(g, ix, iy, iz) : fallback;
}

template <class V>
__device__ __forceinline__ int electron_step(const Params &P, const float *__restrict__ TB, Particle &p, float &lnT,
                                             float &M)
{
    const Acc acc(P);
    const Tables &tb = P.tab;
    const int nE = tb.gE.n;
    const unsigned lin = voxel_index(P.geo, p);
    const Voxel pv = fetch_voxel(P.geo, lin);
    const float rho = pv.x;
    const float *el = TB + tb.off_el + mat_of(pv) * 4 * nE;
    const float T = p.E;
    const uint4 a = draw<true>(P.rng, p);
    const Interp iT = locate(tb.gE, lnT);
    // distance to the next hard event: Woodcock with the majorant at the step-start energy (L110-113);
    // M = 0 gives +inf (no hard events possible)
    M = interp(TB + tb.off_me, iT);
    const float e_hard = fdiv(-flog(u01(a.x)), M);
    // distance to the voxel boundary along d, in voxel units, plus the nudge: per axis the gap to
    // the face the particle is heading for, over |direction cosine| (u = 0 gives +inf or NaN,
    // both dropped by fminf)
    const float dx = fdiv((p.u > 0.0f) ? 1.0f - p.fx : p.fx, fabsf(p.u));
    const float dy = fdiv((p.v > 0.0f) ? 1.0f - p.fy : p.fy, fabsf(p.v));
    const float dz = fdiv((p.w > 0.0f) ? 1.0f - p.fz : p.fz, fabsf(p.w));
    const float L0 = rho * interp(el, iT);
    const float e_cap = fminf(P.opt.es_max, fdiv(P.opt.f_eloss * T, L0));
    float d_vox;
    if (V::MULTI) // R32: the boundary that limits the step is the next change of medium along d
        d_vox = (hom_distance(P, p, lin, pv, fminf(e_hard, e_cap) * P.geo.inv_h) + P.opt.nudge) * P.geo.h;
    else
        d_vox = (fminf(dx, fminf(dy, dz)) + P.opt.nudge) * P.geo.h;
    // Eq. 4
    const bool hard = (e_hard <= d_vox) && (e_hard <= e_cap);
    const float es = hard ? e_hard : fminf(d_vox, e_cap);
    // Eq. 8: dE = s L(E0 - L(E0) s/2)
    const float Tmid = fmaxf(fmaf(-0.5f * L0, es, T), tb.e_min);
    const float dE = es * rho * interp(el, locate(tb.gE, flog(Tmid)));
    if (T - dE < tb.e_cut) {
        deposit<V>(P, lin, T);
        acc.cut(T);
        return ST_DEAD;
    }
    // random hinge (L137): legs zeta*es and (1-zeta)*es around the deflection
    const float zeta = u01(a.y);
    const float esv = es * P.geo.inv_h;
    const float T1 = T - dE;
    const float lnT1 = flog(T1);
    const float leg1 = zeta * esv;
    // R32: the loss of a multi-voxel step goes to the voxel of a point drawn uniformly along the step's
    // path (first leg, then second leg); its uniform comes from the low bits of a.y, a.z, a.w that u01
    // does not use
    float s_dep = 0.0f;
    if (V::MULTI) {
        const uint32_t bits = (a.y & 0x1ffu) | ((a.z & 0x1ffu) << 9) | ((a.w & 0x1fu) << 18);
        s_dep = fmaf(__uint2float_rz(bits), 1.0f / 8388608.0f, 1.0f / 16777216.0f) * esv;
        if (s_dep <= leg1) deposit<V>(P, voxel_ahead(P.geo, p, s_dep, lin), dE);
    } else {
        deposit<V>(P, lin, dE);
    }
    p.fx = fmaf(leg1, p.u, p.fx);
    p.fy = fmaf(leg1, p.v, p.fy);
    p.fz = fmaf(leg1, p.w, p.fz);
    // Bielajew's alternate hinge (L139): scattering strength before or after the loss
    const float lnTms = (a.x & 1u) ? lnT : lnT1;
    const float K = es * rho * interp(el + 3 * nE, locate(tb.gE, lnTms));
    const float lnK = flog(K); // K = 0 gives -inf: no deflection
    if (lnK >= tb.gK.x_min) {
        const float sa = interp(TB + tb.off_ms, locate(tb.gK, lnK));
        const float um = u01(a.z);
        const float mu = fdiv(sa * um, 1.0f + sa - um);
        float sp, cp;
        sincos2pi(u01(a.w), sp, cp);
        rotate(p.u, p.v, p.w, fmaf(-2.0f, mu, 1.0f), 2.0f * sqrtf(mu * (1.0f - mu)), cp, sp, p.u, p.v, p.w);
    }
    if (V::MULTI && s_dep > leg1) deposit<V>(P, voxel_ahead(P.geo, p, s_dep - leg1, lin), dE);
    advance(p, (1.0f - zeta) * esv);
    p.E = T1;
    lnT = lnT1;
    if (!inside(P.geo, p)) {
        acc.esc(p.E);
        return ST_DEAD;
    }
    return hard ? ST_HARD : ST_ALIVE;
}

// ---------------------------------------------------------------------------------------------
// Hard-event candidate at the post-step energy and position (H6): real (Moller, bremsstrahlung)
// or fictitious.  kind: HK_FICT / HK_MOLLER / HK_BREMS.  A secondary (Moller: electron, brems:
// photon) is returned in `child`; the caller pushes it.  Returns ST_ALIVE or ST_DEAD.
// ---------------------------------------------------------------------------------------------
enum : int { HK_FICT = 0, HK_MOLLER = 1, HK_BREMS = 2 };

template <class V>
__device__ __forceinline__ int electron_hard(const Params &P, const float *__restrict__ TB, Particle &p, float &lnT,
                                             float M, Particle &child, int &kind)
{
    const Acc acc(P);
    const Tables &tb = P.tab;
    const int nE = tb.gE.n;
    const uint4 b = draw(P.rng, p);
    const unsigned lin1 = voxel_index(P.geo, p);
    const Voxel pv1 = fetch_voxel(P.geo, lin1);
    const float *el1 = TB + tb.off_el + mat_of(pv1) * 4 * nE;
    const Interp i1 = locate(tb.gE, lnT);
    const float T1 = p.E;
    // a Moller event transfers W in [K_cut, T/2] (L90): none for T <= 2 K_cut (R33)
    const float sM = T1 > 2.0f * tb.e_cut ? pv1.x * interp(el1 + nE, i1) : 0.0f;
    const float sB = pv1.x * interp(el1 + 2 * nE, i1);
    const float r = u01(b.x) * M;
    kind = HK_FICT;
    if (r >= sM + sB) return ST_ALIVE;
    // One rejection loop serves both samplers (one Philox block per trial, as everywhere): the lanes
    // of a sorted batch stay together through the expensive part, whatever their event kind.
    //   Moller (L90): eps = W/T in [K_cut/T, 1/2] from 1/eps^2, g = 1 + g2 eps^2 + r (r - g3)
    //   brems  (L92): k in [k_c, T] from 1/k, g = 4/3 (1 - y) + y^2, y = k/(T + m)
    const bool mol = r < sM;
    kind = mol ? HK_MOLLER : HK_BREMS;
    const float tau = T1 * (1.0f / kMe);
    const float qq = tau / (tau + 1.0f);
    const float g2 = qq * qq;
    const float g3 = (2.0f * tau + 1.0f) / ((tau + 1.0f) * (tau + 1.0f));
    const float gmax = mol ? 1.0f + 0.25f * g2 + (1.0f - g3) : (4.0f / 3.0f);
    const float emin = tb.e_cut / T1;
    const float lr = logf(T1 / tb.p_cut);
    const float iEt = 1.0f / (T1 + kMe);
    float x, uphi;
    for (;;) {
        const uint4 v = draw(P.rng, p);
        const float u0 = u01(v.x);
        float gg;
        if (mol) {
            x = emin / (1.0f - u0 * (1.0f - 2.0f * emin));
            const float rr = x / (1.0f - x);
            gg = 1.0f + g2 * x * x + rr * (rr - g3);
        } else {
            x = tb.p_cut * expf(u0 * lr);
            const float y = x * iEt;
            gg = fmaf(y, y, (4.0f / 3.0f) * (1.0f - y));
        }
        if (u01(v.y) * gmax <= gg) {
            uphi = u01(v.z);
            break;
        }
    }
    float sp, cp;
    sincos2pi(uphi, sp, cp);
    child = p;
    child.track = lineage(P.rng, p).x;
    child.ctr = 0u;
    if (mol) {
        // Moller kinematics (L88-90): scattered and knock-on electrons at opposite azimuths
        const float W = x * T1;
        const float Tp = T1 - W;
        const float den_p = 1.0f / (T1 * (Tp + 2.0f * kMe));
        const float den_d = 1.0f / (T1 * (W + 2.0f * kMe));
        const float cpo = sqrtf(Tp * (T1 + 2.0f * kMe) * den_p), spo = sqrtf(2.0f * kMe * W * den_p);
        const float cdo = sqrtf(W * (T1 + 2.0f * kMe) * den_d), sdo = sqrtf(2.0f * kMe * Tp * den_d);
        rotate(p.u, p.v, p.w, cdo, sdo, -cp, -sp, child.u, child.v, child.w);
        child.E = W;
        rotate(p.u, p.v, p.w, cpo, spo, cp, sp, p.u, p.v, p.w);
        p.E = Tp;
        lnT = flog(Tp);
        return ST_ALIVE;
    }
    // bremsstrahlung (L92): electron direction unchanged, photon at theta = m/E
    float st, ct;
    sincosf(kMe * iEt, &st, &ct);
    rotate(p.u, p.v, p.w, ct, st, cp, sp, child.u, child.v, child.w);
    child.E = x;
    p.E = T1 - x;
    if (p.E < tb.e_cut) {
        deposit<V>(P, lin1, p.E);
        acc.cut(p.E);
        return ST_DEAD;
    }
    lnT = flog(p.E);
    return ST_ALIVE;
}

// ---------------------------------------------------------------------------------------------
// Scheduler 0 (one thread per particle, run to completion): per-thread event
// counts, flushed once per kernel.
// ---------------------------------------------------------------------------------------------
struct Local {
    unsigned flights = 0, compton = 0, photo = 0, pair = 0, fict = 0;
    unsigned steps = 0, moller = 0, brems = 0, hfict = 0;
};

template <class V>
__device__ void photon_run(const Params &P, Particle p, Local &L, const Queue &qE, const Queue &qG)
{
    const float *TB = P.tab.blob;
    for (;;) {
        const int ev = photon_step<V>(P, TB, p, qE, qG);
        L.flights++;
        L.compton += (ev == PH_COMPTON || ev == PH_ABSORBED);
        L.photo += (ev == PH_PHOTO);
        L.pair += (ev == PH_PAIR);
        L.fict += (ev == PH_FICT);
        if (!photon_alive(ev)) break;
    }
}

template <class V>
__device__ void electron_run(const Params &P, Particle p, Local &L, const Queue &qE, const Queue &qG)
{
    float lnT = flog(p.E), M;
    const float *TB = P.tab.blob;
    for (;;) {
        int st = electron_step<V>(P, TB, p, lnT, M);
        L.steps++;
        if (st == ST_HARD) {
            Particle c;
            int kind;
            st = electron_hard<V>(P, TB, p, lnT, M, c, kind);
            if (kind == HK_MOLLER) { L.moller++; push_e(P, qE, c); }
            else if (kind == HK_BREMS) { L.brems++; push_g(P, qG, c); }
            else L.hfict++;
        }
        if (st == ST_DEAD) return;
    }
}

__device__ __forceinline__ unsigned wsum(unsigned v) { return __reduce_add_sync(0xffffffffu, v); }
__device__ __forceinline__ double wsum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
// all 32 lanes of every warp, after the transport code: the warp's energy accounts (and e_inc, its share of the
// primaries' energy) go to the global slots with one atomic each
__device__ __forceinline__ void acc_flush(const Params &P, double e_inc)
{
    const double esc = wsum(Acc::slots()[threadIdx.x]);
    const double cut = wsum(Acc::slots()[kAccThreads + threadIdx.x]);
    e_inc = wsum(e_inc);
    if ((threadIdx.x & 31) == 0) {
        EnergySlot *s = energy_slot(P);
        if (esc != 0.0) atomicAdd(&s->e_esc, esc);
        if (cut != 0.0) atomicAdd(&s->e_cut, cut);
        if (e_inc != 0.0) atomicAdd(&s->e_inc, e_inc);
    }
}
__device__ __forceinline__ void bump(unsigned long long *c, unsigned v)
{
    if (v) atomicAdd(c, static_cast<unsigned long long>(v));
}
// all 32 lanes of every warp must call this
__device__ void flush(const Params &P, const Local &L, double e_inc = 0.0)
{
    acc_flush(P, e_inc);
    const unsigned f = wsum(L.flights), c = wsum(L.compton), ph = wsum(L.photo), pr = wsum(L.pair), fi = wsum(L.fict);
    const unsigned st = wsum(L.steps), mo = wsum(L.moller), br = wsum(L.brems), hf = wsum(L.hfict);
    if ((threadIdx.x & 31) == 0) {
        DevCounters *k = P.cnt;
        bump(&k->photon_flights, f); bump(&k->photon_compton, c); bump(&k->photon_photo, ph);
        bump(&k->photon_pair, pr); bump(&k->photon_fict, fi);
        bump(&k->ch_steps, st); bump(&k->hard_moller, mo); bump(&k->hard_brems, br); bump(&k->hard_fict, hf);
    }
}

} // namespace gpumcd
