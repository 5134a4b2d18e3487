// transport.cuh -- per-particle transport of the GPUMCD hot path (device code, sm_100a).
//
// photon_run  : PAPER.md Sec. II.A (L45-74)  analogue photon transport with Woodcock tracking
// electron_run: PAPER.md Sec. II.B (L78-139) class-II condensed-history electron transport
// Both follow DESIGN.md "Algorithm" draw for draw; scheduling (who runs which particle when)
// lives in the kernels of gpumcd.cu.
#pragma once

#include "physics.cuh"

namespace gpumcd {

// All tables live in one blob (global memory, or its copy in shared memory); the transport
// functions take the blob's base pointer `T` and these float offsets:
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
    const float2 *phantom; // {density, material id as int bits} per voxel
    int nx, ny, nz;
    float h, inv_h;
};

struct Opts {
    float es_max, f_eloss, nudge;
    int pair_mode, photon_only;
};

// Particle queue: three 16-byte SoA streams -> every push / pop is three 128-bit accesses.
struct Queue {
    float4 *A;        // fx, fy, fz, E
    float4 *B;        // u, v, w, packed voxel (bits)
    uint4 *C;         // hist_lo, track, ctr, -
    unsigned *count;  // device counter
    unsigned cap;
};

struct DevCounters {
    unsigned long long n_histories;
    unsigned long long photon_flights, photon_compton, photon_photo, photon_pair, photon_fict;
    unsigned long long ch_steps, hard_moller, hard_brems, hard_fict;
    unsigned long long pushes_e, pushes_g;
    unsigned long long overflow;
    double e_incident, e_dep_total, e_dep_cutoff, e_escaped, e_pair_rest;
};

struct Params {
    Tables tab;
    Geom geo;
    Opts opt;
    Rng rng;
    double *edep;
    DevCounters *cnt;
    unsigned long long *trace; // or nullptr
    unsigned long long trace_off; // id of the run's first history
};

// per-thread tallies, flushed once per kernel
struct Local {
    unsigned flights = 0, compton = 0, photo = 0, pair = 0, fict = 0;
    unsigned steps = 0, moller = 0, brems = 0, hfict = 0;
    unsigned push_e = 0, push_g = 0;
    double e_esc = 0.0, e_cut = 0.0, e_pair = 0.0, e_inc = 0.0;
};

__device__ __forceinline__ bool inside(const Geom &g, const Particle &p)
{
    return (static_cast<unsigned>(p.ix) < static_cast<unsigned>(g.nx)) &
           (static_cast<unsigned>(p.iy) < static_cast<unsigned>(g.ny)) &
           (static_cast<unsigned>(p.iz) < static_cast<unsigned>(g.nz));
}
__device__ __forceinline__ size_t voxel_index(const Geom &g, const Particle &p)
{
    return static_cast<size_t>(p.ix) + static_cast<size_t>(g.nx) * (static_cast<size_t>(p.iy) +
           static_cast<size_t>(g.ny) * static_cast<size_t>(p.iz));
}

// H4/H8 tally: fp64 atomic add into the L2-resident energy grid
__device__ __forceinline__ void deposit(const Params &P, size_t lin, float e)
{
    atomicAdd(&P.edep[lin], static_cast<double>(e));
}

// H7 push: one atomic per group of converged lanes, then three 16-byte stores per record
__device__ __forceinline__ void push(const Params &P, const Queue &q, const Particle &c)
{
    const unsigned mask = __activemask();
    const int lane = threadIdx.x & 31;
    const int leader = __ffs(mask) - 1;
    unsigned base = 0;
    if (lane == leader) base = atomicAdd(q.count, __popc(mask));
    base = __shfl_sync(mask, base, leader);
    const unsigned slot = base + __popc(mask & ((1u << lane) - 1u));
    if (slot < q.cap) {
        q.A[slot] = make_float4(c.fx, c.fy, c.fz, c.E);
        q.B[slot] = make_float4(c.u, c.v, c.w, __uint_as_float(pack_voxel(c.ix, c.iy, c.iz)));
        q.C[slot] = make_uint4(c.hist, c.track, c.ctr, 0u);
    } else {
        atomicAdd(&P.cnt->overflow, 1ull);
    }
}

__device__ __forceinline__ Particle pop(const Queue &q, unsigned slot)
{
    const float4 a = q.A[slot];
    const float4 b = q.B[slot];
    const uint4 c = q.C[slot];
    Particle p;
    p.fx = a.x; p.fy = a.y; p.fz = a.z; p.E = a.w;
    p.u = b.x; p.v = b.y; p.w = b.z;
    const uint32_t vox = __float_as_uint(b.w);
    p.ix = vox & 1023u; p.iy = (vox >> 10) & 1023u; p.iz = vox >> 20;
    p.hist = c.x; p.track = c.y; p.ctr = c.z;
    return p;
}

__device__ __forceinline__ bool electron_tracked(const Params &P, float T)
{
    return !P.opt.photon_only && T >= P.tab.e_cut;
}

// ---------------------------------------------------------------------------------------------
// One photon flight + interaction (H1, H2).  Returns true while the photon is alive.
// Secondaries are pushed to qE (electrons) and qG (annihilation photons).
// TRACE records the primary track's event codes (gpumcd_run_trace).
// ---------------------------------------------------------------------------------------------
struct Trace {
    unsigned long long bits = 0ull;
    int n = 0;
};

template <bool TRACE>
__device__ __forceinline__ void record(Trace &tr, const Particle &p, int code)
{
    if (TRACE && p.track == 0u && tr.n < 21) {
        tr.bits |= static_cast<unsigned long long>(code) << (3 * tr.n);
        ++tr.n;
    }
}
template <bool TRACE>
__device__ __forceinline__ void write_trace(const Params &P, const Particle &p, const Trace &tr)
{
    if (TRACE && p.track == 0u)
        P.trace[((static_cast<unsigned long long>(P.rng.hist_hi) << 32) | p.hist) - P.trace_off] = tr.bits;
}

template <bool TRACE>
__device__ bool photon_step(const Params &P, const float *__restrict__ TB, Particle &p, Local &L, const Queue &qE, const Queue &qG, Trace &tr)
{
    const Tables &tb = P.tab;
    const uint4 w = draw(P.rng, p);
    const Interp iE = locate(tb.gE, logf(p.E));
    const float mu_max = interp(TB + tb.off_mu, iE);
    // Eq. 1 with the Woodcock majorant of Eq. 3
    const float s = -logf(u01(w.x)) / mu_max;
    advance(p, s * P.geo.inv_h);
    L.flights++;
    if (!inside(P.geo, p)) {
        L.e_esc += static_cast<double>(p.E);
        record<TRACE>(tr, p, 4);
        return false;
    }
    const size_t lin = voxel_index(P.geo, p);
    const float2 pv = __ldg(&P.geo.phantom[lin]);
    const float rho = pv.x;
    const float *col = TB + __float_as_int(pv.y) * 3 * tb.gE.n;
    const float r = u01(w.y) * mu_max;
    const float c1 = rho * interp(col, iE);
    const float c2 = fmaf(rho, interp(col + tb.gE.n, iE), c1);
    const float c3 = fmaf(rho, interp(col + 2 * tb.gE.n, iE), c2);
    if (r < c1) {
        // ---- Compton (L65) ----
        L.compton++;
        record<TRACE>(tr, p, 1);
        float eps, t, uphi, nu, nv, nw;
        sample_compton(P.rng, p, eps, t, uphi);
        rotate(p.u, p.v, p.w, 1.0f - t, sqrtf(fmaxf(t * (2.0f - t), 0.0f)), uphi, 0.0f, nu, nv, nw);
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
            push(P, qE, c);
            L.push_e++;
        } else {
            deposit(P, lin, Te);
            L.e_cut += static_cast<double>(Te);
        }
        p.E = E1;
        p.u = nu; p.v = nv; p.w = nw;
        if (p.E < tb.p_cut) {
            deposit(P, lin, p.E);
            L.e_cut += static_cast<double>(p.E);
            record<TRACE>(tr, p, 5);
            return false;
        }
        return true;
    }
    if (r < c2) {
        // ---- photoelectric (L67-72): one electron with T = E_phot ----
        L.photo++;
        record<TRACE>(tr, p, 2);
        if (electron_tracked(P, p.E)) {
            float nu_, uphi;
            sample_sauter(P.rng, p, p.E, nu_, uphi);
            Particle c = p;
            rotate(p.u, p.v, p.w, 1.0f - nu_, sqrtf(fmaxf(nu_ * (2.0f - nu_), 0.0f)), uphi, 0.0f, c.u, c.v, c.w);
            c.track = lineage(P.rng, p).x;
            c.ctr = 0u;
            push(P, qE, c);
            L.push_e++;
        } else {
            deposit(P, lin, p.E);
            L.e_cut += static_cast<double>(p.E);
        }
        return false;
    }
    if (r < c3) {
        // ---- pair production (L74): two electrons, no positron ----
        L.pair++;
        record<TRACE>(tr, p, 3);
        const uint4 v = draw(P.rng, p);
        const float Tsum = p.E - 2.0f * kMe;
        const float T1 = u01(v.x) * Tsum;
        const float T2 = Tsum - T1;
        float ca, sa, cb, sb;
        pair_angle(T1, u01(v.y), ca, sa);
        pair_angle(T2, u01(v.z), cb, sb);
        const float uphi = u01(v.w);
        float ax = 0.f, ay = 0.f, az = 1.f;
        if (P.opt.pair_mode == 1) {
            const uint4 z = draw(P.rng, p);
            az = 2.0f * u01(z.x) - 1.0f;
            const float sz = sqrtf(fmaxf(1.0f - az * az, 0.0f));
            float sp, cp;
            sincospif(2.0f * u01(z.y), &sp, &cp);
            ax = sz * cp;
            ay = sz * sp;
        }
        const bool t1 = electron_tracked(P, T1), t2 = electron_tracked(P, T2);
        uint4 id = make_uint4(0, 0, 0, 0);
        if (t1 || t2 || P.opt.pair_mode == 1) id = lineage(P.rng, p);
        Particle c = p;
        c.ctr = 0u;
        if (t1) {
            rotate(p.u, p.v, p.w, ca, sa, uphi, 0.0f, c.u, c.v, c.w);
            c.E = T1; c.track = id.x;
            push(P, qE, c);
            L.push_e++;
        } else {
            deposit(P, lin, T1);
            L.e_cut += static_cast<double>(T1);
        }
        if (t2) {
            rotate(p.u, p.v, p.w, cb, sb, uphi, 1.0f, c.u, c.v, c.w);
            c.E = T2; c.track = id.y;
            push(P, qE, c);
            L.push_e++;
        } else {
            deposit(P, lin, T2);
            L.e_cut += static_cast<double>(T2);
        }
        L.e_pair += 2.0 * static_cast<double>(kMe);
        if (P.opt.pair_mode == 1) {
            c.E = kMe;
            c.u = ax; c.v = ay; c.w = az; c.track = id.z;
            push(P, qG, c);
            c.u = -ax; c.v = -ay; c.w = -az; c.track = id.w;
            push(P, qG, c);
            L.push_g += 2;
        } else {
            deposit(P, lin, 2.0f * kMe);
            L.e_cut += 2.0 * static_cast<double>(kMe);
        }
        return false;
    }
    L.fict++; // fictitious interaction (L59): nothing changes
    return true;
}

// ---------------------------------------------------------------------------------------------
// One condensed-history step (H3, H4, H5).  Caller guarantees: inside the phantom, T >= E_cut,
// lnT = ln(p.E).  Returns ST_ALIVE, ST_DEAD, or ST_HARD (the step ended on a hard-event
// candidate; M is the majorant it was sampled with, to be passed to electron_hard).
// ---------------------------------------------------------------------------------------------
enum : int { ST_ALIVE = 0, ST_DEAD = 1, ST_HARD = 2 };

__device__ __forceinline__ int electron_step(const Params &P, const float *__restrict__ TB, Particle &p, float &lnT, float &M, Local &L)
{
    const Tables &tb = P.tab;
    const int nE = tb.gE.n;
    const float inf = __int_as_float(0x7f800000);
    const size_t lin = voxel_index(P.geo, p);
    const float2 pv = __ldg(&P.geo.phantom[lin]);
    const float rho = pv.x;
    const float *el = TB + tb.off_el + __float_as_int(pv.y) * 4 * nE;
    const float T = p.E;
    const uint4 a = draw(P.rng, p);
    const Interp iT = locate(tb.gE, lnT);
    // distance to the next hard event: Woodcock with the majorant at the step-start energy (L110-113)
    M = interp(TB + tb.off_me, iT);
    const float e_hard = (M > 0.0f) ? -logf(u01(a.x)) / M : inf;
    // distance to the voxel boundary along d, in voxel units, plus the nudge
    const float dx = (p.u > 0.0f) ? (1.0f - p.fx) / p.u : ((p.u < 0.0f) ? p.fx / -p.u : inf);
    const float dy = (p.v > 0.0f) ? (1.0f - p.fy) / p.v : ((p.v < 0.0f) ? p.fy / -p.v : inf);
    const float dz = (p.w > 0.0f) ? (1.0f - p.fz) / p.w : ((p.w < 0.0f) ? p.fz / -p.w : inf);
    const float d_vox = (fminf(dx, fminf(dy, dz)) + P.opt.nudge) * P.geo.h;
    const float L0 = rho * interp(el, iT);
    const float e_cap = fminf(P.opt.es_max, P.opt.f_eloss * T / L0);
    // Eq. 4
    const bool hard = (e_hard <= d_vox) && (e_hard <= e_cap);
    const float es = hard ? e_hard : fminf(d_vox, e_cap);
    // Eq. 8: dE = s L(E0 - L(E0) s/2)
    const float Tmid = fmaxf(fmaf(-0.5f * L0, es, T), tb.e_min);
    const float dE = es * rho * interp(el, locate(tb.gE, logf(Tmid)));
    L.steps++;
    if (T - dE < tb.e_cut) {
        deposit(P, lin, T);
        L.e_cut += static_cast<double>(T);
        return ST_DEAD;
    }
    deposit(P, lin, dE);
    // random hinge (L137): legs zeta*es and (1-zeta)*es around the deflection
    const float zeta = u01(a.y);
    const float esv = es * P.geo.inv_h;
    const float T1 = T - dE;
    const float lnT1 = logf(T1);
    const float leg1 = zeta * esv;
    p.fx = fmaf(leg1, p.u, p.fx);
    p.fy = fmaf(leg1, p.v, p.fy);
    p.fz = fmaf(leg1, p.w, p.fz);
    // Bielajew's alternate hinge (L139): scattering strength before or after the loss
    const float lnTms = (a.x & 1u) ? lnT : lnT1;
    const float K = es * rho * interp(el + 3 * nE, locate(tb.gE, lnTms));
    if (K > 0.0f) {
        const float lnK = logf(K);
        if (lnK >= tb.gK.x_min) {
            const float sa = interp(TB + tb.off_ms, locate(tb.gK, lnK));
            const float um = u01(a.z);
            const float mu = sa * um / (1.0f + sa - um);
            rotate(p.u, p.v, p.w, fmaf(-2.0f, mu, 1.0f), 2.0f * sqrtf(mu * (1.0f - mu)), u01(a.w), 0.0f,
                   p.u, p.v, p.w);
        }
    }
    advance(p, (1.0f - zeta) * esv);
    p.E = T1;
    lnT = lnT1;
    if (!inside(P.geo, p)) {
        L.e_esc += static_cast<double>(p.E);
        return ST_DEAD;
    }
    return hard ? ST_HARD : ST_ALIVE;
}

// ---------------------------------------------------------------------------------------------
// Hard-event candidate at the post-step energy and position (H6): real (Moller, bremsstrahlung)
// or fictitious.  A secondary, if any, is returned in `child` with child_type 1 (electron) or
// 2 (photon); the caller pushes it.  Returns ST_ALIVE or ST_DEAD for the primary.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ int electron_hard(const Params &P, const float *__restrict__ TB, Particle &p, float &lnT, float M, Local &L,
                                             Particle &child, int &child_type)
{
    const Tables &tb = P.tab;
    const int nE = tb.gE.n;
    child_type = 0;
    const uint4 b = draw(P.rng, p);
    const size_t lin1 = voxel_index(P.geo, p);
    const float2 pv1 = __ldg(&P.geo.phantom[lin1]);
    const float *el1 = TB + tb.off_el + __float_as_int(pv1.y) * 4 * nE;
    const Interp i1 = locate(tb.gE, lnT);
    const float sM = pv1.x * interp(el1 + nE, i1);
    const float sB = pv1.x * interp(el1 + 2 * nE, i1);
    const float r = u01(b.x) * M;
    const float T1 = p.E;
    if (r < sM) {
        // Moller (L88-90)
        L.moller++;
        float eps, uphi;
        sample_moller(P.rng, p, T1, tb.e_cut, eps, uphi);
        const float W = eps * T1;
        const float Tp = T1 - W;
        const float den_p = 1.0f / (T1 * (Tp + 2.0f * kMe));
        const float den_d = 1.0f / (T1 * (W + 2.0f * kMe));
        const float cp = sqrtf(Tp * (T1 + 2.0f * kMe) * den_p), sp = sqrtf(2.0f * kMe * W * den_p);
        const float cd = sqrtf(W * (T1 + 2.0f * kMe) * den_d), sd = sqrtf(2.0f * kMe * Tp * den_d);
        child = p;
        rotate(p.u, p.v, p.w, cd, sd, uphi, 1.0f, child.u, child.v, child.w);
        child.E = W;
        child.track = lineage(P.rng, p).x;
        child.ctr = 0u;
        child_type = 1;
        L.push_e++;
        rotate(p.u, p.v, p.w, cp, sp, uphi, 0.0f, p.u, p.v, p.w);
        p.E = Tp;
        lnT = logf(Tp);
        return ST_ALIVE;
    }
    if (r < sM + sB) {
        // bremsstrahlung (L92): electron direction unchanged, photon at theta = m/E
        L.brems++;
        float k, uphi;
        sample_brems(P.rng, p, T1, tb.p_cut, k, uphi);
        float st, ct;
        sincosf(kMe / (T1 + kMe), &st, &ct);
        child = p;
        rotate(p.u, p.v, p.w, ct, st, uphi, 0.0f, child.u, child.v, child.w);
        child.E = k;
        child.track = lineage(P.rng, p).x;
        child.ctr = 0u;
        child_type = 2;
        L.push_g++;
        p.E = T1 - k;
        if (p.E < tb.e_cut) {
            deposit(P, lin1, p.E);
            L.e_cut += static_cast<double>(p.E);
            return ST_DEAD;
        }
        lnT = logf(p.E);
        return ST_ALIVE;
    }
    L.hfict++;
    return ST_ALIVE;
}

// ---------------------------------------------------------------------------------------------
// Run-to-completion wrappers used by scheduler 0 (one thread per particle)
// ---------------------------------------------------------------------------------------------
template <bool TRACE>
__device__ void photon_run(const Params &P, Particle p, Local &L, const Queue &qE, const Queue &qG)
{
    Trace tr;
    const float *TB = P.tab.blob;
    while (photon_step<TRACE>(P, TB, p, L, qE, qG, tr)) {}
    write_trace<TRACE>(P, p, tr);
}

__device__ void electron_run(const Params &P, Particle p, Local &L, const Queue &qE, const Queue &qG)
{
    float lnT = logf(p.E), M;
    const float *TB = P.tab.blob;
    for (;;) {
        int st = electron_step(P, TB, p, lnT, M, L);
        if (st == ST_HARD) {
            Particle c;
            int ct;
            st = electron_hard(P, TB, p, lnT, M, L, c, ct);
            if (ct == 1) push(P, qE, c);
            else if (ct == 2) push(P, qG, c);
        }
        if (st == ST_DEAD) return;
    }
}

// warp-reduce the per-thread tallies and add them to the global counters
__device__ __forceinline__ unsigned wsum(unsigned v)
{
    return __reduce_add_sync(0xffffffffu, v);
}
__device__ __forceinline__ double wsum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ void flush(const Params &P, const Local &L)
{
    // all 32 lanes of every warp must call this
    const unsigned f = wsum(L.flights), c = wsum(L.compton), ph = wsum(L.photo), pr = wsum(L.pair), fi = wsum(L.fict);
    const unsigned st = wsum(L.steps), mo = wsum(L.moller), br = wsum(L.brems), hf = wsum(L.hfict);
    const unsigned pe = wsum(L.push_e), pg = wsum(L.push_g);
    const double ee = wsum(L.e_esc), ec = wsum(L.e_cut), ep = wsum(L.e_pair), ei = wsum(L.e_inc);
    if ((threadIdx.x & 31) == 0) {
        DevCounters *k = P.cnt;
        if (f) atomicAdd(&k->photon_flights, (unsigned long long)f);
        if (c) atomicAdd(&k->photon_compton, (unsigned long long)c);
        if (ph) atomicAdd(&k->photon_photo, (unsigned long long)ph);
        if (pr) atomicAdd(&k->photon_pair, (unsigned long long)pr);
        if (fi) atomicAdd(&k->photon_fict, (unsigned long long)fi);
        if (st) atomicAdd(&k->ch_steps, (unsigned long long)st);
        if (mo) atomicAdd(&k->hard_moller, (unsigned long long)mo);
        if (br) atomicAdd(&k->hard_brems, (unsigned long long)br);
        if (hf) atomicAdd(&k->hard_fict, (unsigned long long)hf);
        if (pe) atomicAdd(&k->pushes_e, (unsigned long long)pe);
        if (pg) atomicAdd(&k->pushes_g, (unsigned long long)pg);
        if (ee != 0.0) atomicAdd(&k->e_escaped, ee);
        if (ec != 0.0) atomicAdd(&k->e_dep_cutoff, ec);
        if (ep != 0.0) atomicAdd(&k->e_pair_rest, ep);
        if (ei != 0.0) atomicAdd(&k->e_incident, ei);
    }
}

} // namespace gpumcd
