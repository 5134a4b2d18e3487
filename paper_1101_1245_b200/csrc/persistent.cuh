// persistent.cuh -- scheduler 1: one persistent kernel per gpumcd_run, warp-autonomous (H7).
//
// The paper alternates one launch per particle type until both lists are empty
// and reports small gains from stream compaction and a persistent "pool" (L180-182, Tab. VI).
// Here every warp of one resident CTA per SM is a small event-driven simulator of its own:
//   * it owns four type-sorted stacks of particle records (global memory, L2-resident tops):
//       ES electrons due a condensed-history step      EH electrons waiting for a hard event
//       GS photons due a flight                        GI photons waiting for an interaction
//     so no queue is shared between warps, no push needs a global atomic, and there is no grid-wide
//     barrier between particle types: the only shared counter is the head of the primary source;
//   * its 32 lanes hold particles of one type and run ONE piece of code per iteration: the step /
//     flight code for all lanes, or, once 32 records wait (or nothing else is left), the hard-event /
//     interaction code for 32 waiting records.  A lane whose particle needs the other code swaps it
//     out to the waiting stack and takes the next ready record (stack first, then a primary), so the
//     long step code and the rejection samplers both run with full warps ("grouping particles",
//     L352; compaction by ballot + popc prefix sums);
//   * secondaries of the other type pile up in that type's stack; the warp changes type when its own
//     type runs dry or that stack is about to fill up (or, optionally, passes a high-water mark),
//     parking the particles in flight: the longer it stays with one type, the better;
//   * tables are staged into shared memory once with TMA bulk copies (cp.async.bulk + mbarrier).
// A particle's random stream depends only on its lineage (physics.cuh), so the order in which a
// warp works through its stacks does not change any history.
#pragma once

#include <cooperative_groups.h>

#include "transport.cuh"

namespace gpumcd {

namespace cg = cooperative_groups;

// Threads per persistent CTA (one CTA per SM): 768 by default, i.e. 6 warps per scheduler at 80 registers per
// thread (124 bytes of spills outside the step loop).  Measured once a warp stays with one particle type until it
// has to change (config 5, ms): 512 threads 58.0, 576 60.4, 640 53.8, 704 59.4, 768 53.0, 896 54.7, 1024 54.7 (the
// sizes that give every scheduler the same number of warps win).  512 (128 registers, no spills) and 1024 (64
// registers) are kept as options for the ablation.
constexpr int kPThreadsDefault = 768;
constexpr int kPThreadsMax = 1024;
constexpr unsigned kFull = 0xffffffffu;
constexpr unsigned kChunk = 32;            // primaries a warp claims per atomic on the source head
constexpr unsigned kPend = 64;             // capacity of a waiting stack (EH, GI, GR): < 32 before a move, + 32 after
constexpr unsigned kKeep = 24;             // lanes that must be able to go on for another step inside one iteration
constexpr unsigned kLowDefault = 8;        // own-type particles below which a warp with no source changes type
// Forced type changes.  Between two looks at the rules below photon mode banks at most 96 electrons (one Compton
// batch: 32, one batch of pair events: 64) and electron mode at most 32 photons (one hard-event batch).
//   photon mode leaves once ES holds cap - kRoomE or more (its interactions could overflow it otherwise);
//   electron mode leaves once GS holds cap/2 - 32 or more (in photon mode a photon can at most turn into two,
//     by a pair event, and annihilation photons do not multiply: 2 x cap/2 fits), provided ES + lanes are below
//     cap - kRoomE, i.e. photon mode will not send the warp straight back (no ping-pong: a forced change is only
//     made into a mode that can work);
// if both stacks are that full the warp stays with the electrons, and knock-on electrons pile up on ES without a
// bound other than the history itself: a push that finds a stack full is counted and reported
// (GPUMCD_ERR_BANK_OVERFLOW), never dropped silently.
constexpr unsigned kRoomE = 160;
constexpr unsigned kMinStack = 256;        // smallest ready stack: cap - kRoomE must exceed low + 32

struct SourceDev {
    int particle, shape;
    double cx, cy, wx, wy, energy;
    int n_spec;
    const double *cdf;  // n_spec+1, unnormalised running sum of the weights
    const float *edges; // n_spec+1
    const float4 *phsp; // shape 2: n_phsp records of two float4 {x, y, z, u}, {v, w, E, type}
    unsigned long long n_phsp;
    int has_g, has_e;   // the source makes photons / electrons (a phase space may make both)
};

// H0: primary of one history from block (hist, track 0, ctr 0); transport starts at ctr 1.
// (cdf, edges: the spectrum arrays, S.cdf / S.edges or their copies in shared memory)
// `type` returns the primary's particle type (0 photon, 1 electron).  A phase-space primary (shape 2, PAPER.md
// L389, R35) is record hist mod n_phsp exactly as given: no block is drawn for it, and it may lie
// outside the phantom (the caller checks).
template <bool PHSP>
__device__ __forceinline__ Particle make_primary(const Params &P, const SourceDev &S, unsigned long long hist,
                                                 const double *__restrict__ cdf, const float *__restrict__ edges,
                                                 int &type)
{
    Particle p;
    p.hist = static_cast<uint32_t>(hist);
    p.track = 0u;
    p.ctr = 0u;
    type = S.particle;
    if (PHSP) {
        const unsigned long long r = hist % S.n_phsp;
        const float4 a = __ldg(&S.phsp[2 * r]), b = __ldg(&S.phsp[2 * r + 1]);
        const double hd = static_cast<double>(P.geo.h); // (divisions, as in the oracle's floor(x / h))
        const double vx = static_cast<double>(a.x) / hd, vy = static_cast<double>(a.y) / hd, vz = static_cast<double>(a.z) / hd;
        const double fx = floor(vx), fy = floor(vy), fz = floor(vz);
        // (cells far outside the phantom are clamped to just outside, so that they fit the packed record)
        p.ix = static_cast<int>(fmin(fmax(fx, -1.0), 1024.0));
        p.iy = static_cast<int>(fmin(fmax(fy, -1.0), 1024.0));
        p.iz = static_cast<int>(fmin(fmax(fz, -1.0), 1024.0));
        p.fx = static_cast<float>(vx - fx);
        p.fy = static_cast<float>(vy - fy);
        p.fz = static_cast<float>(vz - fz);
        p.u = a.w; p.v = b.x; p.w = b.y;
        p.E = b.z;
        p.ctr = 1u;
        type = b.w != 0.0f;
        return p;
    }
    const uint4 w = draw(P.rng, p);
    double x = S.cx, y = S.cy;
    if (S.shape == 1) {
        x = S.cx + (static_cast<double>(u01(w.x)) - 0.5) * S.wx;
        y = S.cy + (static_cast<double>(u01(w.y)) - 0.5) * S.wy;
    }
    const double vx = x / static_cast<double>(P.geo.h), vy = y / static_cast<double>(P.geo.h);
    const double fx = floor(vx), fy = floor(vy);
    p.ix = static_cast<int>(fx);
    p.iy = static_cast<int>(fy);
    p.iz = 0;
    p.fx = static_cast<float>(vx - fx);
    p.fy = static_cast<float>(vy - fy);
    p.fz = 0.0f;
    p.u = 0.0f; p.v = 0.0f; p.w = 1.0f;
    double E = S.energy;
    if (S.n_spec > 0) {
        const double target = static_cast<double>(u01(w.z)) * cdf[S.n_spec];
        int lo = 0, hi = S.n_spec - 1; // largest j with cdf[j] <= target, clamped to n_spec-1
        while (lo < hi) {
            const int mid = (lo + hi + 1) >> 1;
            if (cdf[mid] <= target) lo = mid; else hi = mid - 1;
        }
        const double e0 = edges[lo], e1 = edges[lo + 1];
        E = e0 + static_cast<double>(u01(w.w)) * (e1 - e0);
    }
    p.E = static_cast<float>(E);
    return p;
}

template <bool PHSP>
__device__ __forceinline__ Particle make_primary(const Params &P, const SourceDev &S, unsigned long long hist, int &type)
{
    return make_primary<PHSP>(P, S, hist, S.cdf, S.edges, type);
}

// the kernel's dynamic shared memory: [table blob | spectrum cdf (double) | spectrum edges (float)]
__device__ __forceinline__ float *dyn_smem()
{
    extern __shared__ __align__(128) float dyn_smem_base[];
    return dyn_smem_base;
}

// ---- TMA bulk copy of the table blob into shared memory (G7) --------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p)
{
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void stage_tables(float *dst, const float *src, unsigned n_floats, uint64_t *bar)
{
    const uint32_t bar_a = smem_u32(bar);
    if (threadIdx.x == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar_a));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        const unsigned bytes = n_floats * 4u; // multiple of 16 (blob is padded)
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar_a), "r"(bytes) : "memory");
        unsigned off = 0;
        while (off < bytes) {
            const unsigned chunk = min(bytes - off, 32768u);
            asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::
                             "r"(smem_u32(reinterpret_cast<const char *>(dst) + off)),
                         "l"(reinterpret_cast<const char *>(src) + off), "r"(chunk), "r"(bar_a)
                         : "memory");
            off += chunk;
        }
    }
    unsigned done = 0;
    while (!done) {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], 0;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(done)
                     : "r"(bar_a)
                     : "memory");
    }
}


struct PersistArgs {
    Params P;
    SourceDev S;
    unsigned *head;    // next primary of this launch to be claimed (the only counter the warps share)
    float4 *stkA;      // per-warp stacks, `stride` records per warp: [ES cap_r | GS cap_r | EH kPend | GI kPend | GR kPend]
    float4 *stkB;
    uint4 *stkC;
    unsigned cap_r;                // capacity of a ready stack (ES, GS)
    unsigned high_g, high_e;       // banked photons / electrons that make a warp change to that type
    unsigned low;                  // own-type ready particles below which a warp with no source changes type
    unsigned inner;                // condensed-history steps a warp makes at most between two looks at its stacks
    unsigned stride;               // 2 cap_r + 3 kPend
    unsigned long long hist0;      // first history of the launch (low word never wraps inside a launch)
    unsigned n_hist;               // histories of the launch (< 2^32)
    unsigned table_floats;         // length of the table blob, padded to a multiple of 4 floats
    int spec_in_smem;              // the spectrum's cdf and bin edges are copied into shared memory behind the tables
    double inv_h3_n;
    float *dose;                   // or nullptr
    size_t nvox;
    int finalize;                  // 0 for all but the last launch of a run split at a 2^32 history boundary
};

// Event counters of one warp, in shared memory (lane 0 adds ballot counts; flushed once per kernel).
// DevCounters lists its first eleven members in this order.
enum : int { WC_FLIGHT = 0, WC_COMPTON, WC_PHOTO, WC_PAIR, WC_FICT, WC_STEP, WC_MOLLER, WC_BREMS, WC_HFICT,
             WC_PUSH_E, WC_PUSH_G, WC_N };
enum : int { SK_ES = 0, SK_GS = 1, SK_EH = 2, SK_GI = 3, SK_GR = 4 };

struct WarpCtl {          // one per warp, shared memory
    unsigned n_es, n_gs;  // stack counts while divergent code pushes (photon_interact); else in registers
    unsigned wc[WC_N];
};

// This warp's next chunk of the primary source: [next, end) out of [0, n_in); one atomic per chunk.
struct Claim {
    unsigned next = 0, end = 0;
    bool exhausted = false;
    __device__ __forceinline__ bool empty() const { return exhausted && next == end; }
    __device__ __forceinline__ void refill(unsigned *head, unsigned n_in)
    {
        if (next != end || exhausted) return;
        unsigned base = 0;
        if ((threadIdx.x & 31) == 0) base = atomicAdd(head, kChunk);
        base = __shfl_sync(kFull, base, 0);
        next = min(base, n_in);
        end = min(base + kChunk, n_in);
        if (base + kChunk >= n_in) exhausted = true;
    }
};

// The calling warp: its stacks, their counts (warp-uniform registers) and its shared-memory block.
struct Warp {
    float4 *A;
    float4 *B;
    uint4 *C;
    unsigned cap_r;
    unsigned high_g, high_e, low;
    unsigned n[5];
    unsigned lt;   // lanes below this one
    unsigned hw;   // fullest ready stack seen
    WarpCtl *ctl;
    double *e_inc; // this thread's account of the primaries' energy (shared memory)

    __device__ __forceinline__ unsigned off(int s) const
    {
        return s == SK_ES ? 0u : (s == SK_GS ? cap_r : 2u * cap_r + static_cast<unsigned>(s - SK_EH) * kPend);
    }
    __device__ __forceinline__ unsigned cap(int s) const { return s < 2 ? cap_r : kPend; }
    __device__ __forceinline__ void count(int k, unsigned mask) const
    {
        // (a shared-memory atomic by lane 0: one instruction instead of load, add, store; 0.5-1 % of the run)
        if ((threadIdx.x & 31) == 0 && mask) atomicAdd(&ctl->wc[k], static_cast<unsigned>(__popc(mask)));
    }
    // Converged code: the lanes with `on` append their record to stack s (ballot + popc prefix).
    __device__ __forceinline__ unsigned push(const Params &P, int s, bool on, const Particle &c, uint32_t extra)
    {
        const unsigned m = __ballot_sync(kFull, on);
        if (m) {
            if (on) {
                const unsigned slot = n[s] + __popc(m & lt);
                if (slot < cap(s)) store_rec(A, B, C, off(s) + slot, c, extra);
                else count_overflow(P.cnt);
            }
            n[s] = min(n[s] + static_cast<unsigned>(__popc(m)), cap(s));
            __syncwarp(); // the records are read back by other lanes of this warp
        }
        return m;
    }
    // Converged code: the lanes with `want` take the top records of stack s while there are any.
    __device__ __forceinline__ bool pop(int s, bool want, Particle &p, uint32_t &extra)
    {
        const unsigned m = __ballot_sync(kFull, want);
        const unsigned take = min(static_cast<unsigned>(__popc(m)), n[s]);
        const unsigned rank = __popc(m & lt);
        const bool got = want && rank < take;
        if (got) p = load_rec(A, B, C, off(s) + n[s] - 1u - rank, extra);
        n[s] -= take;
        return got;
    }
    // Converged code: the whole warp makes this warp's next (up to 32) primaries at once and banks them on the
    // ready stack of their type (ES electrons, GS photons; a phase space may hold both), from where free lanes pop
    // them like any other ready particle: the source code (H0) then always runs with full lanes.  Returns false if
    // the source is dry or a stack has no room for them right now.
    template <class V>
    __device__ __forceinline__ bool bank_primaries(const PersistArgs &a, Claim &cl, int s_mode)
    {
        cl.refill(a.head, a.n_hist);
        const unsigned k = cl.end - cl.next;
        if (k == 0u) return false;
        if (V::PHSP ? (a.S.has_e && n[SK_ES] + k > cap_r) || (a.S.has_g && n[SK_GS] + k > cap_r)
                    : n[s_mode] + k > cap_r) return false;
        const unsigned lane = threadIdx.x & 31;
        bool on = lane < k;
        int type = a.S.particle;
        Particle q;
        if (on) {
            // the spectrum arrays: their shared-memory copies if the kernel staged them (512 bins: nine dependent
            // look-ups per primary, which were 3 % of config 5's stall samples from global memory)
            const double *cdf = a.S.cdf;
            const float *edges = a.S.edges;
            if (a.spec_in_smem) {
                cdf = reinterpret_cast<const double *>(dyn_smem() + a.table_floats);
                edges = reinterpret_cast<const float *>(cdf + (a.S.n_spec + 1));
            }
            q = make_primary<V::PHSP>(a.P, a.S, a.hist0 + (cl.next + lane), cdf, edges, type);
            *e_inc += static_cast<double>(q.E);
            if (V::PHSP && !inside(a.P.geo, q)) { // a phase-space record outside the phantom: escaped at birth
                Acc(a.P).esc(q.E);
                on = false;
            } else if (type == 1 ? !electron_tracked(a.P, q.E) : (V::PHSP && q.E < a.P.tab.p_cut)) {
                // below its cutoff (or photon_only): deposited where it is born (R5)
                deposit<V>(a.P, voxel_index(a.P.geo, q), q.E);
                Acc(a.P).cut(q.E);
                on = false;
            }
        }
        if (V::PHSP) { // a phase space may hold both types
            if (a.S.has_e) push(a.P, SK_ES, on && type == 1, q, 0u);
            if (a.S.has_g) push(a.P, SK_GS, on && type == 0, q, 0u);
        } else { // s_mode: the ready stack of the calling mode, which is the source's type when it asks for primaries
            push(a.P, s_mode, on, q, 0u);
        }
        cl.next += k;
        return true;
    }
};

// ---------------------------------------------------------------------------------------------
// Electron mode: the lanes hold electrons due a condensed-history step.  Returns the type to go on
// with (0 photons, 1 electrons never, -1 nothing left); on return no lane holds a particle.
// ---------------------------------------------------------------------------------------------
template <class V>
__device__ __forceinline__ int electron_mode(const PersistArgs &a, const float *__restrict__ TB, Warp &w, Claim &cl)
{
    const Params &P = a.P;
    const unsigned lane = threadIdx.x & 31;
    const bool src_is_e = a.S.has_e != 0, src_is_g = a.S.has_g != 0;
    Particle p;
    float lnT = 0.f, M = 0.f;
    bool alive = false;
    for (;;) {
        const unsigned live = __ballot_sync(kFull, alive);
        const bool src_e = src_is_e && !cl.empty();
        // ---- hard events of 32 waiting electrons (or of what is left when nothing else can move)
        if (w.n[SK_EH] >= 32u || (w.n[SK_EH] != 0u && live == 0u && w.n[SK_ES] == 0u && !src_e)) {
            w.push(P, SK_ES, alive, p, 0u); // park the electrons in flight
            alive = false;
            const unsigned nb = min(32u, w.n[SK_EH]);
            Particle c;
            int kind = -1;
            if (lane < nb) {
                uint32_t mbits;
                p = load_rec(w.A, w.B, w.C, w.off(SK_EH) + w.n[SK_EH] - 1u - lane, mbits);
                lnT = flog(p.E);
                alive = electron_hard<V>(P, TB, p, lnT, __uint_as_float(mbits), c, kind) == ST_ALIVE;
            }
            w.n[SK_EH] -= nb;
            __syncwarp();
            const unsigned gm = w.push(P, SK_GS, kind == HK_BREMS, c, 0u);  // bremsstrahlung photons
            const unsigned em = w.push(P, SK_ES, kind == HK_MOLLER, c, 0u); // knock-on electrons
            w.count(WC_MOLLER, em);
            w.count(WC_BREMS, gm);
            w.count(WC_PUSH_E, em);
            w.count(WC_PUSH_G, gm);
            w.count(WC_HFICT, __ballot_sync(kFull, kind == HK_FICT));
            w.hw = max(w.hw, max(w.n[SK_ES], w.n[SK_GS]));
            continue;
        }
        // ---- change of particle type?  (E, G: all electrons / photons this warp holds; both are
        // unchanged by parking, and the two modes' rules exclude each other, so a change is never
        // undone before some work has been done)
        const unsigned ready = static_cast<unsigned>(__popc(live)) + w.n[SK_ES];
        const unsigned E = ready + w.n[SK_EH], G = w.n[SK_GS] + w.n[SK_GI] + w.n[SK_GR];
        const bool src_g = src_is_g && !cl.empty();
        // (only READY photons count towards the high-water mark: photon mode stays while it has kLow of them,
        // so a change made here is never undone before some work has been done)
        const unsigned Gr = w.n[SK_GS];
        // (a change is only made if photon mode will not send the warp straight back: ES + lanes below its forced mark)
        bool leave = ready + kRoomE < w.cap_r && ((Gr >= w.high_g && E < w.high_e) || Gr + 32u >= w.cap_r / 2u);
        if (!src_e) {
            if (ready == 0u) return (G != 0u || src_g) ? 0 : -1; // (EH is empty here)
            leave = leave || (ready < w.low && (src_g || w.n[SK_GS] >= 32u));
        }
        if (leave) {
            w.push(P, SK_ES, alive, p, 0u);
            w.hw = max(w.hw, w.n[SK_ES]);
            return 0;
        }
        // ---- refill the free lanes: the stack first (depth first keeps it short), then primaries
        if (~live) {
            uint32_t extra;
            bool got = w.pop(SK_ES, !alive, p, extra);
            if (src_e && __any_sync(kFull, !alive && !got) && w.template bank_primaries<V>(a, cl, SK_ES))
                got = w.pop(SK_ES, !alive && !got, p, extra) || got;
            if (got) {
                lnT = flog(p.E);
                alive = true;
            }
        }
        const unsigned sm = __ballot_sync(kFull, alive);
        if (sm == 0u) continue;
        int st = alive ? ST_ALIVE : ST_DEAD;
        if (!V::INNER) {
            // ---- one condensed-history step for every lane that holds an electron
            if (alive) st = electron_step<V>(P, TB, p, lnT, M);
            w.count(WC_STEP, sm);
        } else {
            // ---- or several (the paper's N, L180: steps between two compactions): the lanes go on stepping while
            // enough of them still can (kKeep) or nothing could refill the others anyway; a lane whose step ended
            // the electron or on a hard-event candidate waits.  Pays for long tracks (an electron beam in water).
            const bool can_refill = w.n[SK_ES] != 0u || src_e;
            unsigned act = sm, k = 0u;
#pragma unroll 1
            do {
                if (st == ST_ALIVE) st = electron_step<V>(P, TB, p, lnT, M);
                w.count(WC_STEP, act);
                act = __ballot_sync(kFull, st == ST_ALIVE);
            } while (act != 0u && ++k < a.inner && (static_cast<unsigned>(__popc(act)) >= kKeep || !can_refill));
        }
        w.push(P, SK_EH, st == ST_HARD, p, __float_as_uint(M));
        alive = st == ST_ALIVE;
    }
}

// Photon mode, interactions of up to 32 photons waiting in stack sk (H2).  KIND != 0: all of them are of
// that kind (the compiler drops the other branches of photon_interact); else the kind is in the record.
template <class V, int KIND>
__device__ __forceinline__ void interact_batch(const Params &P, Warp &w, int sk, Particle &p, bool &alive)
{
    const unsigned lane = threadIdx.x & 31;
    w.push(P, SK_GS, alive, p, 0u); // park the photons in flight
    alive = false;
    const unsigned nb = min(32u, w.n[sk]);
    // the interaction code pushes from divergent branches: the two ready stacks' counts go through shared
    // memory for its duration
    if (lane == 0) {
        w.ctl->n_es = w.n[SK_ES];
        w.ctl->n_gs = w.n[SK_GS];
    }
    __syncwarp();
    int kind = 0;
    if (lane < nb) {
        uint32_t kbits;
        p = load_rec(w.A, w.B, w.C, w.off(sk) + w.n[sk] - 1u - lane, kbits);
        kind = KIND ? KIND : static_cast<int>(kbits);
        const WarpStack qE{w.A + w.off(SK_ES), w.B + w.off(SK_ES), w.C + w.off(SK_ES), &w.ctl->n_es,
                           &w.ctl->wc[WC_PUSH_E], w.cap_r};
        const WarpStack qG{w.A + w.off(SK_GS), w.B + w.off(SK_GS), w.C + w.off(SK_GS), &w.ctl->n_gs,
                           &w.ctl->wc[WC_PUSH_G], w.cap_r};
        alive = photon_interact<V>(P, p, kind, qE, qG) == PM_FLIGHT;
    }
    __syncwarp();
    w.n[SK_ES] = w.ctl->n_es;
    w.n[SK_GS] = w.ctl->n_gs;
    w.n[sk] -= nb;
    w.hw = max(w.hw, max(w.n[SK_ES], w.n[SK_GS]));
    if (KIND == PM_COMPTON) {
        w.count(WC_COMPTON, __ballot_sync(kFull, kind == PM_COMPTON));
    } else {
        w.count(WC_PHOTO, __ballot_sync(kFull, kind == PM_PHOTO));
        w.count(WC_PAIR, __ballot_sync(kFull, kind == PM_PAIR));
    }
    __syncwarp();
}

// ---------------------------------------------------------------------------------------------
// Photon mode: the lanes hold photons due a flight.  Returns the type to go on with (1 electrons,
// -1 nothing left); on return no lane holds a particle.
// ---------------------------------------------------------------------------------------------
template <class V>
__device__ __forceinline__ int photon_mode(const PersistArgs &a, const float *__restrict__ TB, Warp &w, Claim &cl)
{
    const Params &P = a.P;
    const bool src_is_g = a.S.has_g != 0, src_is_e = a.S.has_e != 0;
    Particle p;
    bool alive = false;
    for (;;) {
        const unsigned live = __ballot_sync(kFull, alive);
        const bool src_g = src_is_g && !cl.empty();
        // ---- interactions of 32 waiting photons (or of what is left when nothing else can move): Compton
        // events wait in GI, the rare photoelectric and pair events in GR, so that a batch of Compton events
        // does not drag the long pair code along for one or two lanes
        const bool stuck = live == 0u && w.n[SK_GS] == 0u && !src_g;
        if (w.n[SK_GI] >= 32u || (w.n[SK_GI] != 0u && stuck)) {
            interact_batch<V, PM_COMPTON>(P, w, SK_GI, p, alive);
            continue;
        }
        if (w.n[SK_GR] >= 32u || (w.n[SK_GR] != 0u && stuck)) {
            interact_batch<V, 0>(P, w, SK_GR, p, alive);
            continue;
        }
        // ---- change of particle type?  (see electron_mode)
        const unsigned ready = static_cast<unsigned>(__popc(live)) + w.n[SK_GS];
        const unsigned G = ready + w.n[SK_GI] + w.n[SK_GR], E = w.n[SK_ES] + w.n[SK_EH];
        const bool src_e = src_is_e && !cl.empty();
        const unsigned Er = w.n[SK_ES];
        bool leave = (Er >= w.high_e && G < w.high_g) || Er + kRoomE >= w.cap_r;
        if (!src_g) {
            if (ready == 0u) return (E != 0u || src_e) ? 1 : -1; // (GI is empty here)
            leave = leave || (ready < w.low && (src_e || w.n[SK_ES] >= 32u));
        }
        if (leave) {
            w.push(P, SK_GS, alive, p, 0u);
            w.hw = max(w.hw, w.n[SK_GS]);
            return 1;
        }
        // ---- refill the free lanes: the stack first, then primaries
        if (~live) {
            uint32_t extra;
            bool got = w.pop(SK_GS, !alive, p, extra);
            if (src_g && __any_sync(kFull, !alive && !got) && w.template bank_primaries<V>(a, cl, SK_GS))
                got = w.pop(SK_GS, !alive && !got, p, extra) || got;
            if (got) alive = true;
        }
        const unsigned fl = __ballot_sync(kFull, alive);
        if (fl == 0u) continue;
        // ---- one flight for every lane that holds a photon
        int mode = PM_DEAD;
        if (alive) mode = photon_flight<V>(P, TB, p);
        w.count(WC_FLIGHT, fl);
        w.count(WC_FICT, __ballot_sync(kFull, mode == PM_FLIGHT));
        w.push(P, SK_GI, mode == PM_COMPTON, p, static_cast<uint32_t>(mode));
        w.push(P, SK_GR, mode > PM_COMPTON, p, static_cast<uint32_t>(mode)); // photoelectric and pair events: rare
        alive = mode == PM_FLIGHT;
    }
}

// ---------------------------------------------------------------------------------------------
// The persistent kernel
// ---------------------------------------------------------------------------------------------
template <class V, bool SMEM_TABLES, int kPThreads>
__global__ void __launch_bounds__(kPThreads, 1) k_persistent(const __grid_constant__ PersistArgs a)
{
    float *smem = dyn_smem();
    constexpr int kPWarps = kPThreads / 32;
    __shared__ uint64_t bar;
    __shared__ WarpCtl s_ctl[kPWarps];
    __shared__ double s_einc[kPThreads];
    cg::grid_group grid = cg::this_grid();

    const Params &P = a.P;
    const float *TB = P.tab.blob;
    if (SMEM_TABLES) {
        stage_tables(smem, P.tab.blob, a.table_floats, &bar);
        TB = smem;
        if (a.spec_in_smem) {
            double *sc = reinterpret_cast<double *>(smem + a.table_floats);
            float *se = reinterpret_cast<float *>(sc + (a.S.n_spec + 1));
            for (int i = threadIdx.x; i <= a.S.n_spec; i += kPThreads) {
                sc[i] = a.S.cdf[i];
                se[i] = a.S.edges[i];
            }
            __syncthreads();
        }
    }
    const unsigned lane = threadIdx.x & 31;
    const size_t gwarp = (blockIdx.x * static_cast<size_t>(blockDim.x) + threadIdx.x) >> 5;
    Warp w;
    w.A = a.stkA + gwarp * a.stride;
    w.B = a.stkB + gwarp * a.stride;
    w.C = a.stkC + gwarp * a.stride;
    w.cap_r = a.cap_r;
    w.high_g = a.high_g;
    w.high_e = a.high_e;
    w.low = a.low;
    w.n[0] = w.n[1] = w.n[2] = w.n[3] = w.n[4] = 0u;
    w.lt = (1u << lane) - 1u;
    w.hw = 0u;
    w.ctl = &s_ctl[threadIdx.x >> 5];
    w.e_inc = &s_einc[threadIdx.x];
    s_einc[threadIdx.x] = 0.0;
    acc_init();
    if (lane < WC_N) w.ctl->wc[lane] = 0u;
    __syncwarp();

    // Each warp works on its own until the source is exhausted and its stacks are empty.
    Claim cl;
    cl.exhausted = (a.n_hist == 0u);
    int type = a.S.has_g ? 0 : 1;
    while (type >= 0) type = (type == 1) ? electron_mode<V>(a, TB, w, cl) : photon_mode<V>(a, TB, w, cl);

    // ---- flush this warp's event counts and accounts
    __syncwarp();
    if (lane < WC_N) {
        const unsigned v = w.ctl->wc[lane];
        if (v) atomicAdd(&P.cnt->photon_flights + lane, static_cast<unsigned long long>(v));
    }
    acc_flush(P, s_einc[threadIdx.x]);
    if (lane == 0 && w.hw) atomicMax(&P.cnt->high_water, static_cast<unsigned long long>(w.hw));
    if (!a.finalize) return;
    grid.sync();
    // ---- H8 finalize: dose = energy / mass / histories, and the total deposited energy
    double s = 0.0;
    for (size_t i = blockIdx.x * static_cast<size_t>(blockDim.x) + threadIdx.x; i < a.nvox;
         i += static_cast<size_t>(gridDim.x) * blockDim.x) {
        const double e = tally_value<V::TALLY>(P, i);
        s += e;
        if (V::TALLY == TALLY_FIXED) P.edep[i] = e; // from here on the tally holds MeV as fp64, whatever the mode
        if (a.dose) a.dose[caller_index(P.geo, i)] = static_cast<float>(e / static_cast<double>(unpack_voxel(P.geo.phantom[i]).x) * a.inv_h3_n);
    }
    s = wsum(s);
    __shared__ double part[kPWarps];
    if (lane == 0) part[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int k = 0; k < kPWarps; ++k) t += part[k];
        atomicAdd(&P.cnt->e_dep_total, t);
    }
}

} // namespace gpumcd
