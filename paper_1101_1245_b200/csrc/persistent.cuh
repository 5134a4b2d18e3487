// persistent.cuh -- scheduler 1: one persistent cooperative kernel per gpumcd_run (H7).
//
// The paper alternates one launch per particle type until both lists are empty
// and reports small gains from stream compaction and a persistent "pool" (L180-182, Tab. VI).
// On B200 the transport kernels are issue-bound with most lanes idle (profiles/r01_*), so the
// scheduler is built around keeping all 32 lanes of a warp in the SAME code:
//   * one CTA per SM stays resident for the whole run; tables are staged into shared memory once
//     with TMA bulk copies (cp.async.bulk + mbarrier);
//   * a warp steps 32 particles in lock step and refills finished lanes at once, first from its
//     private stack of same-type secondaries, then from the phase's input queue (atomic head);
//   * electrons whose step ended on a hard-event candidate are swapped out into a per-warp buffer
//     and processed 32 at a time (event-based sorting), so neither the step code nor the
//     Moller / bremsstrahlung samplers run with a handful of active lanes;
//   * photons born in an electron phase and electrons born in a photon phase go to global queues
//     (ballot + popc prefix, one atomic per warp) that the next phase consumes; phases are separated
//     by grid-wide barriers, so a queue is never read and written at the same time.
#pragma once

#include <cooperative_groups.h>

#include "transport.cuh"

namespace gpumcd {

namespace cg = cooperative_groups;

#ifndef GPUMCD_PTHREADS
#define GPUMCD_PTHREADS 512
#endif
constexpr int kPThreads = GPUMCD_PTHREADS; // threads per persistent CTA (one CTA per SM)
constexpr unsigned kHardCap = 64; // per-warp buffer of pending hard events
constexpr unsigned kFull = 0xffffffffu;
constexpr unsigned kChunk = 32;   // inputs a warp claims per atomic on the phase's head counter

struct SourceDev {
    int particle, shape;
    double cx, cy, wx, wy, energy;
    int n_spec;
    const double *cdf;  // n_spec+1, unnormalised running sum of the weights
    const float *edges; // n_spec+1
};

// H0: primary of one history from block (hist, track 0, ctr 0); transport starts at ctr 1.
__device__ __forceinline__ Particle make_primary(const Params &P, const SourceDev &S, unsigned long long hist)
{
    Particle p;
    p.hist = static_cast<uint32_t>(hist);
    p.track = 0u;
    p.ctr = 0u;
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
        const double target = static_cast<double>(u01(w.z)) * S.cdf[S.n_spec];
        int lo = 0, hi = S.n_spec - 1; // largest j with cdf[j] <= target, clamped to n_spec-1
        while (lo < hi) {
            const int mid = (lo + hi + 1) >> 1;
            if (S.cdf[mid] <= target) lo = mid; else hi = mid - 1;
        }
        const double e0 = S.edges[lo], e1 = S.edges[lo + 1];
        E = e0 + static_cast<double>(u01(w.w)) * (e1 - e0);
    }
    p.E = static_cast<float>(E);
    return p;
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
    Queue qP[3];       // photon queues, rotating: read [i%3], written [(i+1)%3], reset [(i+2)%3]
    Queue qE[3];       // electron queues, same rotation
    unsigned *heads;   // pop heads: [0..2] photon queues, [3..5] electron queues
    float4 *privA;     // per-warp private records: ready stack [priv_ready] then hard buffer [kHardCap]
    float4 *privB;
    uint4 *privC;
    unsigned priv_ready;           // capacity of a warp's ready stack
    unsigned long long hist0;      // first history of the run (low word never wraps inside a launch)
    unsigned long long n_hist;
    unsigned wave;
    unsigned table_floats;         // length of the table blob, padded to a multiple of 4 floats
    double inv_h3_n;
    float *dose;                   // or nullptr
    size_t nvox;
    int finalize;                  // 0 for all but the last launch of a run split at a 2^32 history boundary
};

// ---------------------------------------------------------------------------------------------
// Photon phase: every warp steps 32 photons; finished lanes are refilled from the input.
// SRC: the input is the source itself (primaries generated on the fly), else queue `in`.
// Event counts are warp-level (ballot + popc into warp-uniform counters): no per-lane registers.
// ---------------------------------------------------------------------------------------------
template <bool TRACE, bool SRC>
__device__ void photon_phase(const Params &P, const float *__restrict__ TB, const SourceDev &S,
                             unsigned long long hist_base, const Queue &in, unsigned n_queue, unsigned n_in,
                             unsigned *head, const Queue &qE, const Queue &qG)
{
    const int lane = threadIdx.x & 31;
    const unsigned lt = (1u << lane) - 1u;
    const Acc acc(P);
    Particle p;
    Trace tr;
    bool alive = false, exhausted = (n_in == 0);
    unsigned n_flight = 0, n_compton = 0, n_photo = 0, n_pair = 0, n_fict = 0;
    unsigned w_next = 0, w_end = 0; // this warp's chunk of the input, [w_next, w_end)
    for (;;) {
        const unsigned dead = __ballot_sync(kFull, !alive);
        if (dead && !(exhausted && w_next == w_end)) {
            if (w_next == w_end) { // take the next chunk of kChunk inputs: one atomic per chunk
                unsigned base = 0;
                if (lane == 0) base = atomicAdd(head, kChunk);
                base = __shfl_sync(kFull, base, 0);
                w_next = min(base, n_in);
                w_end = min(base + kChunk, n_in);
                if (base + kChunk >= n_in) exhausted = true;
            }
            const unsigned take = min(static_cast<unsigned>(__popc(dead)), w_end - w_next);
            const unsigned rank = __popc(dead & lt);
            double e_new = 0.0;
            if (!alive && rank < take) {
                const unsigned idx = w_next + rank;
                uint32_t extra;
                if (SRC && idx >= n_queue) {
                    p = make_primary(P, S, hist_base + (idx - n_queue));
                    e_new = static_cast<double>(p.E);
                } else {
                    p = load_rec(in.A, in.B, in.C, idx, extra);
                }
                alive = true;
                tr = Trace{};
            }
            w_next += take;
            if (SRC) {
                e_new = wsum(e_new);
                if (lane == 0 && e_new != 0.0) acc.inc(e_new);
            }
        }
        const unsigned am = __ballot_sync(kFull, alive);
        if (am == 0u) {
            if (exhausted && w_next == w_end) break;
            continue;
        }
        int ev = -1;
        if (alive) {
            ev = photon_step<TRACE>(P, TB, p, acc, qE, qG, tr);
            if (!photon_alive(ev)) {
                write_trace<TRACE>(P, p, tr);
                alive = false;
            }
        }
        n_flight += __popc(am);
        n_compton += __popc(__ballot_sync(kFull, ev == PH_COMPTON || ev == PH_ABSORBED));
        n_photo += __popc(__ballot_sync(kFull, ev == PH_PHOTO));
        n_pair += __popc(__ballot_sync(kFull, ev == PH_PAIR));
        n_fict += __popc(__ballot_sync(kFull, ev == PH_FICT));
    }
    if (lane == 0) {
        DevCounters *c = P.cnt;
        bump(&c->photon_flights, n_flight); bump(&c->photon_compton, n_compton); bump(&c->photon_photo, n_photo);
        bump(&c->photon_pair, n_pair); bump(&c->photon_fict, n_fict);
    }
}

// ---------------------------------------------------------------------------------------------
// Electron phase: lock-step condensed-history steps with lane refill and event-sorted hard events.
// ---------------------------------------------------------------------------------------------
template <bool SRC>
__device__ void electron_phase(const Params &P, const float *__restrict__ TB, const SourceDev &S,
                               unsigned long long hist_base, const Queue &in, unsigned n_queue, unsigned n_in,
                               unsigned *head, const Queue &qG, float4 *pA, float4 *pB, uint4 *pC,
                               unsigned ready_cap)
{
    const int lane = threadIdx.x & 31;
    const unsigned lt = (1u << lane) - 1u;
    const Acc acc(P);
    // private records of this warp: [0, ready_cap) ready stack (extra word = ln T),
    // [ready_cap, ready_cap + kHardCap) pending hard events (extra word = majorant M)
    Particle p;
    float lnT = 0.f, M = 0.f;
    bool alive = false, exhausted = (n_in == 0);
    unsigned n_ready = 0, n_hard = 0;
    unsigned n_step = 0, n_moller = 0, n_brems = 0, n_hfict = 0;
    unsigned w_next = 0, w_end = 0; // this warp's chunk of the input, [w_next, w_end)
    for (;;) {
        // ---- refill dead lanes: private stack first, then the phase input
        const unsigned dead = __ballot_sync(kFull, !alive);
        if (dead) {
            const unsigned k = __popc(dead), rank = __popc(dead & lt);
            const unsigned take = min(k, n_ready);
            if (!alive && rank < take) {
                uint32_t extra;
                p = load_rec(pA, pB, pC, n_ready - 1u - rank, extra);
                lnT = __uint_as_float(extra);
                alive = true;
            }
            n_ready -= take;
            if (k > take && !(exhausted && w_next == w_end)) {
                if (w_next == w_end) { // next chunk of the input: one atomic per kChunk particles
                    unsigned base = 0;
                    if (lane == 0) base = atomicAdd(head, kChunk);
                    base = __shfl_sync(kFull, base, 0);
                    w_next = min(base, n_in);
                    w_end = min(base + kChunk, n_in);
                    if (base + kChunk >= n_in) exhausted = true;
                }
                const unsigned take2 = min(k - take, w_end - w_next);
                double e_new = 0.0;
                if (!alive && rank >= take && rank - take < take2) {
                    const unsigned idx = w_next + rank - take;
                    uint32_t extra;
                    if (SRC && idx >= n_queue) {
                        p = make_primary(P, S, hist_base + (idx - n_queue));
                        e_new = static_cast<double>(p.E);
                        if (electron_tracked(P, p.E)) {
                            alive = true;
                        } else { // below the cutoff (or photon_only): deposited where it is born
                            deposit(P, voxel_index(P.geo, p), p.E);
                            acc.cut(p.E);
                        }
                    } else {
                        p = load_rec(in.A, in.B, in.C, idx, extra);
                        alive = true;
                    }
                    lnT = flog(p.E);
                }
                w_next += take2;
                if (SRC) {
                    e_new = wsum(e_new);
                    if (lane == 0 && e_new != 0.0) acc.inc(e_new);
                }
            }
        }
        const unsigned am = __ballot_sync(kFull, alive);
        // ---- hard events, 32 at a time (or whatever is left when nothing else can run)
        if (n_hard >= 32u || (n_hard > 0u && am == 0u && n_ready == 0u && exhausted && w_next == w_end)) {
            const unsigned nb = min(32u, n_hard);
            Particle q, c;
            float qlnT = 0.f;
            int st = ST_DEAD, kind = -1;
            if (static_cast<unsigned>(lane) < nb) {
                uint32_t mbits;
                q = load_rec(pA, pB, pC, ready_cap + n_hard - 1u - lane, mbits);
                qlnT = flog(q.E);
                st = electron_hard(P, TB, q, qlnT, __uint_as_float(mbits), acc, c, kind);
            }
            n_hard -= nb;
            // bremsstrahlung photons -> global photon queue of the next photon phase
            const unsigned gm = __ballot_sync(kFull, kind == HK_BREMS);
            if (gm) {
                unsigned base = 0;
                if (lane == 0) base = atomicAdd(qG.count, static_cast<unsigned>(__popc(gm)));
                base = __shfl_sync(kFull, base, 0);
                if (kind == HK_BREMS) {
                    const unsigned slot = base + __popc(gm & lt);
                    if (slot < qG.cap) store_rec(qG.A, qG.B, qG.C, slot, c, 0u);
                    else atomicAdd(&P.cnt->overflow, 1ull);
                }
            }
            // knock-on electrons and the surviving primaries -> this warp's ready stack
            const unsigned em = __ballot_sync(kFull, kind == HK_MOLLER);
            if (kind == HK_MOLLER) {
                const unsigned slot = n_ready + __popc(em & lt);
                if (slot < ready_cap) store_rec(pA, pB, pC, slot, c, __float_as_uint(flog(c.E)));
                else atomicAdd(&P.cnt->overflow, 1ull);
            }
            n_ready = min(n_ready + __popc(em), ready_cap);
            const bool cont = (kind >= 0) && st == ST_ALIVE;
            const unsigned cm = __ballot_sync(kFull, cont);
            if (cont) {
                const unsigned slot = n_ready + __popc(cm & lt);
                if (slot < ready_cap) store_rec(pA, pB, pC, slot, q, __float_as_uint(qlnT));
                else atomicAdd(&P.cnt->overflow, 1ull);
            }
            n_ready = min(n_ready + __popc(cm), ready_cap);
            n_moller += __popc(em);
            n_brems += __popc(gm);
            n_hfict += __popc(__ballot_sync(kFull, kind == HK_FICT));
            __syncwarp();
            continue;
        }
        if (am == 0u) {
            if (exhausted && w_next == w_end && n_ready == 0u) break;
            continue;
        }
        // ---- one condensed-history step for every live lane
        int st = ST_ALIVE;
        if (alive) st = electron_step(P, TB, p, lnT, M, acc);
        n_step += __popc(am);
        const bool hard = alive && st == ST_HARD;
        const unsigned hm = __ballot_sync(kFull, hard);
        if (hard) {
            store_rec(pA, pB, pC, ready_cap + n_hard + __popc(hm & lt), p, __float_as_uint(M));
            alive = false;
        }
        n_hard += __popc(hm);
        if (st == ST_DEAD) alive = false;
        __syncwarp();
    }
    if (lane == 0) {
        DevCounters *c = P.cnt;
        bump(&c->ch_steps, n_step); bump(&c->hard_moller, n_moller); bump(&c->hard_brems, n_brems);
        bump(&c->hard_fict, n_hfict); bump(&c->pushes_e, n_moller); bump(&c->pushes_g, n_brems);
    }
}

// ---------------------------------------------------------------------------------------------
// Optional phase timeline (compile with -DGPUMCD_TIMELINE; development aid, not in the default build):
// per phase the input size, start time, the time each CTA finished and the time the barrier opened.
// ---------------------------------------------------------------------------------------------
#ifdef GPUMCD_TIMELINE
constexpr int kTlPhases = 256, kTlBlocks = 160;
struct Timeline {
    unsigned n_phase;
    unsigned type[kTlPhases], n_in[kTlPhases];
    unsigned long long t0[kTlPhases], t1[kTlPhases];
    unsigned long long done[kTlPhases][kTlBlocks];
};
__device__ Timeline g_timeline;
__device__ __forceinline__ unsigned long long gtime()
{
    unsigned long long t;
    asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t));
    return t;
}
#define TL_BEGIN(np, ne) do { if (leader && tl < kTlPhases) { g_timeline.type[tl] = (np); g_timeline.n_in[tl] = (ne); g_timeline.t0[tl] = gtime(); } } while (0)
#define TL_DONE() do { __syncthreads(); if (threadIdx.x == 0 && tl < kTlPhases && blockIdx.x < kTlBlocks) g_timeline.done[tl][blockIdx.x] = gtime(); } while (0)
#define TL_END() do { if (leader && tl < kTlPhases) { g_timeline.t1[tl] = gtime(); g_timeline.n_phase = tl + 1; } ++tl; } while (0)
#else
#define TL_BEGIN(np, ne) do {} while (0)
#define TL_DONE() do {} while (0)
#define TL_END() do {} while (0)
#endif

// ---------------------------------------------------------------------------------------------
// The persistent kernel
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned ld_volatile(const unsigned *p) { return *reinterpret_cast<const volatile unsigned *>(p); }

template <bool TRACE, bool SMEM_TABLES>
__global__ void __launch_bounds__(kPThreads, 1) k_persistent(const PersistArgs a)
{
    extern __shared__ __align__(128) float smem[];
    __shared__ uint64_t bar;
    cg::grid_group grid = cg::this_grid();

    const Params &P = a.P;
    const float *TB = P.tab.blob;
    if (SMEM_TABLES) {
        stage_tables(smem, P.tab.blob, a.table_floats, &bar);
        TB = smem;
    }
    const unsigned gwarp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const size_t stride = static_cast<size_t>(a.priv_ready) + kHardCap;
    float4 *pA = a.privA + gwarp * stride, *pB = a.privB + gwarp * stride;
    uint4 *pC = a.privC + gwarp * stride;
    const bool leader = (blockIdx.x == 0 && threadIdx.x == 0);
#ifdef GPUMCD_TIMELINE
    unsigned tl = 0;
#endif

    // One iteration = one photon phase and one electron phase that do NOT depend on each other:
    // iteration i reads photon queue X[i%3] and electron queue Y[i%3] and writes X[(i+1)%3] /
    // Y[(i+1)%3]; the third pair was read in iteration i-1 and is reset now, to be written in i+1.
    // So one grid barrier per iteration suffices, a warp that runs out of one type's input moves on
    // to the other type without waiting, and odd / even warps start with different types, which
    // keeps latency-bound photon warps and issue-bound electron warps on every SM at the same time.
    // Each iteration also injects the next wave of primaries, so what is left over from a wave
    // rides along with the bulk of the next one; only the very end of the run has a tail.
    unsigned long long done = 0;
    unsigned it = 0;
    unsigned nP = 0, nE = 0; // queued photons in X[it%3] / electrons in Y[it%3]
    const bool e_first = ((threadIdx.x >> 5) & 1) != 0;
    for (;;) {
        const unsigned r = it % 3u, w = (it + 1u) % 3u, z = (it + 2u) % 3u;
        const unsigned n_src = static_cast<unsigned>(min(static_cast<unsigned long long>(a.wave), a.n_hist - done));
        const unsigned long long hist_base = a.hist0 + done;
        const unsigned srcP = (a.S.particle == 0) ? n_src : 0u, srcE = (a.S.particle == 1) ? n_src : 0u;
        if (leader) {
            *a.qP[z].count = 0u; a.heads[z] = 0u;
            *a.qE[z].count = 0u; a.heads[3 + z] = 0u;
        }
        TL_BEGIN(nP + srcP, nE + srcE);
#pragma unroll 1
        for (int t = 0; t < 2; ++t) {
            if ((t == 0) != e_first) {
                // photons: read X[r] and the source, electrons -> Y[w], annihilation photons -> X[w]
                if (nP + srcP) {
                    if (srcP) photon_phase<TRACE, true>(P, TB, a.S, hist_base, a.qP[r], nP, nP + srcP, a.heads + r, a.qE[w], a.qP[w]);
                    else photon_phase<TRACE, false>(P, TB, a.S, hist_base, a.qP[r], nP, nP, a.heads + r, a.qE[w], a.qP[w]);
                }
            } else {
                // electrons: read Y[r] and the source, bremsstrahlung photons -> X[w], knock-ons stay in the warp
                if (nE + srcE) {
                    if (srcE) electron_phase<true>(P, TB, a.S, hist_base, a.qE[r], nE, nE + srcE, a.heads + 3 + r, a.qP[w], pA, pB, pC, a.priv_ready);
                    else electron_phase<false>(P, TB, a.S, hist_base, a.qE[r], nE, nE, a.heads + 3 + r, a.qP[w], pA, pB, pC, a.priv_ready);
                }
            }
        }
        TL_DONE();
        grid.sync();
        TL_END();
        nP = min(ld_volatile(a.qP[w].count), a.qP[w].cap);
        nE = min(ld_volatile(a.qE[w].count), a.qE[w].cap);
        done += n_src;
        ++it;
        if (nP == 0u && nE == 0u && done >= a.n_hist) break;
    }
    if (!a.finalize) return;
    grid.sync();
    // ---- H8 finalize: dose = energy / mass / histories, and the total deposited energy
    double s = 0.0;
    for (size_t i = blockIdx.x * static_cast<size_t>(blockDim.x) + threadIdx.x; i < a.nvox;
         i += static_cast<size_t>(gridDim.x) * blockDim.x) {
        const double e = P.edep[i];
        s += e;
        if (a.dose) a.dose[i] = static_cast<float>(e / static_cast<double>(P.geo.phantom[i].x) * a.inv_h3_n);
    }
    s = wsum(s);
    __shared__ double part[kPThreads / 32];
    if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int k = 0; k < kPThreads / 32; ++k) t += part[k];
        atomicAdd(&P.cnt->e_dep_total, t);
    }
}

} // namespace gpumcd
