// gpumcd.cu -- kernels, scheduling and the C ABI of the B200-native GPUMCD hot path.
//
// See include/gpumcd.h for the boundary and DESIGN.md for the data layout and scheduling.
#include "../../include/gpumcd.h"
#include "persistent.cuh"

#include <algorithm>
#include <cmath>
#include <map>
#include <mutex>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>

namespace gpumcd {

constexpr int kBlock = 256;

// ---------------------------------------------------------------------------------------------
// Setup kernels
// ---------------------------------------------------------------------------------------------
// Pack {density, material} per voxel into 4 bytes (transport.cuh pack_voxel_record), validate, and reduce the
// largest density of each material (H10; positive floats order like their bit patterns, so atomicMax on the bits
// is a float max).
__global__ void k_pack_phantom(const float *__restrict__ density, const uint8_t *__restrict__ material, Geom g,
                               size_t nvox, int n_mat, uint32_t *__restrict__ out, unsigned *rho_max_bits,
                               unsigned *n_bad)
{
    __shared__ unsigned s_max[8];
    if (threadIdx.x < 8) s_max[threadIdx.x] = 0u;
    __syncthreads();
    for (size_t i = blockIdx.x * static_cast<size_t>(blockDim.x) + threadIdx.x; i < nvox;
         i += static_cast<size_t>(gridDim.x) * blockDim.x) { // i: internal index
        const size_t src = caller_index(g, i);
        const uint32_t d = __float_as_uint(density[src]);
        const int m = material[src];
        if (m >= n_mat || !density_packable(d)) { // (NaN, inf, zero, negative and denormal densities fail the range test)
            atomicAdd(n_bad, 1u);
            out[i] = pack_voxel_record(__float_as_uint(1.0f), 0);
        } else {
            atomicMax(&s_max[m], d);
            out[i] = pack_voxel_record(d, m);
        }
    }
    __syncthreads();
    if (threadIdx.x < 8 && s_max[threadIdx.x]) atomicMax(&rho_max_bits[threadIdx.x], s_max[threadIdx.x]);
}

// Multi-voxel steps (hom_tol > 0): the uniform radius of every voxel, R = the largest r <= r_max such that
// all voxels within Chebyshev distance r lie inside the phantom and continue the voxel's medium (same
// material, |density - own| <= hom_tol * own).
__global__ void k_uniform_radius(const uint32_t *__restrict__ phantom, uint8_t *__restrict__ radius, Geom g,
                                 float hom_tol, int r_max)
{
    const int nx = g.nx, ny = g.ny, nz = g.nz;
    const size_t nvox = static_cast<size_t>(nx) * ny * nz;
    for (size_t i = blockIdx.x * static_cast<size_t>(blockDim.x) + threadIdx.x; i < nvox;
         i += static_cast<size_t>(gridDim.x) * blockDim.x) { // i: internal index
        const int ix = static_cast<int>(i % nx), iy = static_cast<int>((i / nx) % ny), iz = static_cast<int>(i / (static_cast<size_t>(nx) * ny));
        const Voxel pv0 = unpack_voxel(phantom[i]);
        const float band = hom_tol * pv0.x;
        int R = 0;
        for (int r = 1; r <= r_max; ++r) {
            bool ok = ix - r >= 0 && ix + r < nx && iy - r >= 0 && iy + r < ny && iz - r >= 0 && iz + r < nz;
            for (int dz = -r; ok && dz <= r; ++dz)
                for (int dy = -r; ok && dy <= r; ++dy) {
                    const bool shell_row = (dz == -r || dz == r || dy == -r || dy == r);
                    for (int dx = -r; ok && dx <= r; dx += (shell_row ? 1 : 2 * r)) { // the shell at distance r only
                        const Voxel pv = unpack_voxel(phantom[lin_of(g, ix + dx, iy + dy, iz + dz)]);
                        ok = pv.m == pv0.m && fabsf(pv.x - pv0.x) <= band;
                    }
                }
            if (!ok) break;
            R = r;
        }
        radius[i] = static_cast<uint8_t>(R);
    }
}

// H0: one primary per history (from block (hist, track 0, ctr 0), or a phase-space record); transport starts at
// ctr 1.  The primaries go to the list of their type (a phase space may hold both).
template <class V>
__global__ void k_source(Params P, SourceDev S, Queue qG, Queue qE, unsigned long long hist0, unsigned n)
{
    const unsigned i = blockIdx.x * blockDim.x + threadIdx.x;
    const Acc acc(P);
    acc_init();
    double e_inc = 0.0;
    if (i < n) {
        int type;
        const Particle p = S.shape == 2 ? make_primary<true>(P, S, hist0 + i, type) : make_primary<false>(P, S, hist0 + i, type);
        e_inc = static_cast<double>(p.E);
        if (S.shape == 2 && !inside(P.geo, p)) {
            acc.esc(p.E); // a phase-space record outside the phantom: escaped at birth
        } else if (type == 1 ? !electron_tracked(P, p.E) : (S.shape == 2 && p.E < P.tab.p_cut)) {
            // below its cutoff (or photon_only): deposited where it is born (R5)
            deposit<V>(P, voxel_index(P.geo, p), p.E);
            acc.cut(p.E);
        } else if (type == 1) {
            push(P, qE, p, nullptr);
        } else {
            push(P, qG, p, nullptr);
        }
    }
    acc_flush(P, e_inc);
}

// ---------------------------------------------------------------------------------------------
// Scheduler 0: one launch per pass, one thread per particle, run to completion
// (the paper's base scheme, L166: alternate the two particle types until both lists are empty)
// ---------------------------------------------------------------------------------------------
template <class V>
__global__ void __launch_bounds__(kBlock) k_photon_pass(Params P, Queue in, unsigned n_in, Queue qE, Queue qG)
{
    const unsigned i = blockIdx.x * blockDim.x + threadIdx.x;
    Local L;
    acc_init();
    if (i < n_in) {
        uint32_t extra;
        const Particle p = load_rec(in.A, in.B, in.C, i, extra);
        if (p.E >= 0.0f) photon_run<V>(P, p, L, qE, qG);
    }
    flush(P, L);
}

template <class V>
__global__ void __launch_bounds__(kBlock) k_electron_pass(Params P, Queue in, unsigned n_in, Queue qE, Queue qG)
{
    const unsigned i = blockIdx.x * blockDim.x + threadIdx.x;
    Local L;
    acc_init();
    if (i < n_in) {
        uint32_t extra;
        const Particle p = load_rec(in.A, in.B, in.C, i, extra);
        if (p.E >= 0.0f) electron_run<V>(P, p, L, qE, qG);
    }
    flush(P, L);
}

// H8: dose = energy / mass / histories; also the total deposited energy
template <int TALLY>
__global__ void k_finalize(Params P, size_t nvox, double inv_h3_n, float *__restrict__ dose)
{
    const uint32_t *__restrict__ phantom = P.geo.phantom;
    DevCounters *cnt = P.cnt;
    double s = 0.0;
    for (size_t i = blockIdx.x * static_cast<size_t>(blockDim.x) + threadIdx.x; i < nvox;
         i += static_cast<size_t>(gridDim.x) * blockDim.x) {
        const double e = tally_value<TALLY>(P, i);
        s += e;
        if (TALLY == TALLY_FIXED) P.edep[i] = e; // from here on the tally holds MeV as fp64
        if (dose) dose[caller_index(P.geo, i)] = static_cast<float>(e / static_cast<double>(unpack_voxel(phantom[i]).x) * inv_h3_n);
    }
    s = wsum(s);
    __shared__ double part[32];
    if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int k = 0; k < (blockDim.x + 31) / 32; ++k) t += part[k];
        atomicAdd(&cnt->e_dep_total, t);
    }
}

// Batch statistics of gpumcd_run_uncertainty (Eq. 13 with batches as the samples): fold the
// energy tally of one batch of m histories into the running sums and clear it for the next batch.
//   s1 += e (total energy);  x = e / m (the batch's mean energy per history);  sx += x;  sxx += x^2
__global__ void k_accumulate_batch(double *__restrict__ edep, double *__restrict__ s1, double *__restrict__ sx,
                                   double *__restrict__ sxx, size_t nvox, double inv_m)
{
    for (size_t i = blockIdx.x * static_cast<size_t>(blockDim.x) + threadIdx.x; i < nvox;
         i += static_cast<size_t>(gridDim.x) * blockDim.x) {
        const double e = edep[i];
        edep[i] = 0.0;
        const double x = e * inv_m;
        s1[i] += e;
        sx[i] += x;
        sxx[i] += x * x;
    }
}

// dose = total energy / mass / histories (H8); Delta D = sqrt((<x^2> - <x>^2) / (B - 1)) / mass (Eq. 13);
// the energy tally is left holding the total of all batches.
__global__ void k_finalize_uncertainty(const double *__restrict__ s1, const double *__restrict__ sx,
                                       const double *__restrict__ sxx, Geom g,
                                       size_t nvox, double inv_h3, double inv_n, double n_batches,
                                       float *__restrict__ dose, float *__restrict__ sigma, double *__restrict__ edep)
{
    const uint32_t *__restrict__ phantom = g.phantom;
    for (size_t i = blockIdx.x * static_cast<size_t>(blockDim.x) + threadIdx.x; i < nvox;
         i += static_cast<size_t>(gridDim.x) * blockDim.x) {
        const double inv_mass = inv_h3 / static_cast<double>(unpack_voxel(phantom[i]).x);
        const double mean = sx[i] / n_batches;
        const double var = (sxx[i] / n_batches - mean * mean) / (n_batches - 1.0);
        const size_t o = caller_index(g, i);
        dose[o] = static_cast<float>(s1[i] * inv_mass * inv_n);
        sigma[o] = static_cast<float>(sqrt(fmax(var, 0.0)) * inv_mass);
        edep[i] = s1[i];
    }
}

// gpumcd_get_energy_tally: the tally in the caller's [nz][ny][nx] order
__global__ void k_export_tally(const double *__restrict__ edep, Geom g, size_t nvox, double *__restrict__ out)
{
    for (size_t i = blockIdx.x * static_cast<size_t>(blockDim.x) + threadIdx.x; i < nvox;
         i += static_cast<size_t>(gridDim.x) * blockDim.x)
        out[caller_index(g, i)] = edep[i];
}

// Tally probe (the denominator of the tally's roofline, since no vendor figure exists for
// the fp64 atomic rate of the L2): every thread adds `per_thread` values into the context's own energy grid
// at pseudo-random voxels of the beam-shaped region x in [x0, x0+wx), y in [y0, y0+wy), all depths, the
// address pattern of the condensed-history deposits, and nothing else.
template <bool FIXED>
__global__ void k_tally_probe(double *__restrict__ edep, Geom g, int x0, int y0, int wx, int wy,
                              unsigned per_thread, unsigned seed)
{
    const unsigned tid = blockIdx.x * blockDim.x + threadIdx.x;
    uint4 r = philox4x32_10(tid, 0u, 0u, 0u, seed, 0x5eedu);
    for (unsigned k = 0; k < per_thread; ++k) {
        // a cheap generator inside the loop (the probe must be bound by the atomics, not by Philox)
        r.x = r.x * 1664525u + 1013904223u;
        r.y = r.y * 22695477u + 1u;
        r.z = r.z * 1103515245u + 12345u;
        const unsigned ix = x0 + __umulhi(r.x, static_cast<unsigned>(wx));
        const unsigned iy = y0 + __umulhi(r.y, static_cast<unsigned>(wy));
        const unsigned iz = __umulhi(r.z, static_cast<unsigned>(g.nz));
        const size_t lin = lin_of(g, static_cast<int>(ix), static_cast<int>(iy), static_cast<int>(iz));
        if (FIXED) atomicAdd(reinterpret_cast<unsigned long long *>(edep) + lin, 1ull);
        else atomicAdd(&edep[lin], 1.0);
    }
}

// gpumcd_set_source, shape 2: check the phase-space records and count them by type.
// out[0] bad records (type not 0 / 1, a number that is not finite), out[1] energies outside the tables,
// out[2] photons, out[3] electrons
__global__ void k_check_phsp(const float4 *__restrict__ rec, unsigned long long n, float e_lo, float e_hi,
                             unsigned long long *out)
{
    unsigned long long bad = 0, range = 0, ng = 0, ne = 0;
    for (unsigned long long i = blockIdx.x * static_cast<unsigned long long>(blockDim.x) + threadIdx.x; i < n;
         i += static_cast<unsigned long long>(gridDim.x) * blockDim.x) {
        const float4 a = rec[2 * i], b = rec[2 * i + 1];
        const bool fin = isfinite(a.x) && isfinite(a.y) && isfinite(a.z) && isfinite(a.w) && isfinite(b.x) &&
                         isfinite(b.y) && isfinite(b.z);
        if (!fin || !(b.w == 0.0f || b.w == 1.0f)) { ++bad; continue; }
        if (!(b.z >= e_lo && b.z <= e_hi)) ++range;
        if (b.w == 0.0f) ++ng; else ++ne;
    }
    if (bad) atomicAdd(&out[0], bad);
    if (range) atomicAdd(&out[1], range);
    if (ng) atomicAdd(&out[2], ng);
    if (ne) atomicAdd(&out[3], ne);
}

// Device-side check of the random-number layer (gpumcd_selftest_philox): block i = Philox4x32-10 of counter
// in[6i .. 6i+3] under key in[6i+4], in[6i+5], and the uniforms the transport code makes of its four words.
__global__ void k_philox_selftest(const uint32_t *__restrict__ in, uint32_t *__restrict__ out, float *__restrict__ u,
                                  unsigned long long n)
{
    for (unsigned long long i = blockIdx.x * static_cast<unsigned long long>(blockDim.x) + threadIdx.x; i < n;
         i += static_cast<unsigned long long>(gridDim.x) * blockDim.x) {
        const uint4 r = philox4x32_10(in[6 * i], in[6 * i + 1], in[6 * i + 2], in[6 * i + 3], in[6 * i + 4], in[6 * i + 5]);
        out[4 * i] = r.x; out[4 * i + 1] = r.y; out[4 * i + 2] = r.z; out[4 * i + 3] = r.w;
        if (u) { u[4 * i] = u01(r.x); u[4 * i + 1] = u01(r.y); u[4 * i + 2] = u01(r.z); u[4 * i + 3] = u01(r.w); }
    }
}

} // namespace gpumcd

// =============================================================================================
// Host side
// =============================================================================================
using namespace gpumcd;

constexpr int kMaxQueues = 4;
constexpr int kSpecSmemBins = 1024;
constexpr size_t kSpecSmemBytes = (kSpecSmemBins + 1) * (sizeof(double) + sizeof(float)) + 4; // padded to 16 bytes

struct gpumcd_ctx {
    int nx = 0, ny = 0, nz = 0;
    size_t nvox = 0;
    float h = 0.f;
    float e_max = 0.f;
    gpumcd_options opt{};
    // device memory
    uint32_t *phantom = nullptr;      // packed records, 4 B per voxel
    uint8_t *radius = nullptr;        // hom_tol > 0: uniform radius per voxel
    float *stage_density = nullptr;   // device staging of host volumes (gpumcd_create_host / set_phantom_host)
    uint8_t *stage_material = nullptr;
    unsigned *scratch = nullptr;      // 8 rho_max bit patterns + 1 bad-voxel count
    float *dose_stage = nullptr;      // device dose of gpumcd_run_host
    float *table_blob = nullptr;
    std::vector<float> blob_host;     // host copy of the table blob (majorants are rebuilt per phantom)
    int n_mat = 0, n_E = 0;
    double *edep = nullptr;
    double *moments = nullptr;        // gpumcd_run_uncertainty: s1 | sx | sxx, nvox each (allocated on first use)
    DevCounters *cnt = nullptr;
    // global particle queues of scheduler 0: PA, PB, EA, EB (scheduler 1 has per-warp stacks instead)
    int n_queues = 4;
    unsigned *qcount = nullptr; // kMaxQueues push counters
    float4 *qA[kMaxQueues] = {};
    float4 *qB[kMaxQueues] = {};
    uint4 *qC[kMaxQueues] = {};
    unsigned qcap = 0;
    double *spec_cdf = nullptr;
    float *spec_edges = nullptr;
    float4 *phsp = nullptr;         // phase-space records of the current source (shape 2), library-owned
    // scheduler 1 (persistent kernel)
    unsigned *head = nullptr;       // next primary to be claimed
    float4 *stkA = nullptr, *stkB = nullptr; // per-warp stacks (persistent.cuh)
    uint4 *stkC = nullptr;
    unsigned cap_r = 0;             // ready-stack capacity per warp
    unsigned stride = 0;            // records per warp
    int p_grid = 0;                 // CTAs of the persistent kernel (one per SM)
    bool smem_tables = false;
    unsigned table_floats = 0;
    size_t spec_smem_bytes = 0;     // dynamic shared memory reserved behind the tables for the spectrum arrays
    size_t l2_window = 0;           // l2_persist: bytes of the phantom covered by the persisting access window
    float l2_hit_ratio = 0.f;
    // host state
    Tables tab{};
    bool have_source = false;
    SourceDev src{};
    cudaStream_t last_stream = nullptr;
    unsigned long long last_n = 0;
    unsigned long long high_water = 0;
    bool ran = false;
    unsigned long long hist_offset = 0;
    float fx_scale = 1.0f;          // tally_mode 2: MeV -> integer units of the current run
    // launch accounting / optional event timing
    bool profiling = false;
    gpumcd_profile prof{};
    struct Ev { int cls; cudaEvent_t a, b; };
    std::vector<Ev> events;
    std::string err;
};

enum { CLS_SOURCE = 0, CLS_PHOTON = 1, CLS_ELECTRON = 2, CLS_FINALIZE = 3 };

// bracket one kernel launch: counts it, and records an event pair when profiling is on
struct LaunchScope {
    gpumcd_ctx *c; cudaStream_t st; int cls; cudaEvent_t a = nullptr, b = nullptr;
    LaunchScope(gpumcd_ctx *c_, cudaStream_t st_, int cls_) : c(c_), st(st_), cls(cls_) {
        c->prof.launches++;
        (&c->prof.n_source)[cls]++;
        if (c->profiling) { cudaEventCreate(&a); cudaEventCreate(&b); cudaEventRecord(a, st); }
    }
    ~LaunchScope() { if (c->profiling) { cudaEventRecord(b, st); c->events.push_back({cls, a, b}); } }
};

static std::string g_create_error;

#define CK(call)                                                                                   \
    do {                                                                                           \
        cudaError_t e_ = (call);                                                                   \
        if (e_ != cudaSuccess) {                                                                   \
            char buf_[512];                                                                        \
            snprintf(buf_, sizeof buf_, "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_), __FILE__, __LINE__); \
            set_error(ctx, buf_);                                                                  \
            return e_ == cudaErrorMemoryAllocation ? GPUMCD_ERR_OOM : GPUMCD_ERR_CUDA;             \
        }                                                                                          \
    } while (0)

static void set_error(gpumcd_ctx *ctx, const char *msg)
{
    if (ctx) ctx->err = msg; else g_create_error = msg;
}

static Geom make_geom(const gpumcd_ctx *c)
{
    Geom g;
    g.phantom = c->phantom;
    g.radius = c->radius;
    g.nx = c->nx; g.ny = c->ny; g.nz = c->nz;
    g.h = c->h; g.inv_h = 1.0f / c->h;
    return g;
}

static Queue make_queue(gpumcd_ctx *c, int k)
{
    Queue q;
    q.A = c->qA[k]; q.B = c->qB[k]; q.C = c->qC[k];
    q.count = c->qcount + k;
    q.cap = c->qcap;
    return q;
}

extern "C" int gpumcd_default_options(gpumcd_options *opt)
{
    if (!opt) return GPUMCD_ERR_INVALID_ARG;
    opt->es_max_cm = 0.5f;
    opt->f_eloss_max = 0.25f;
    opt->boundary_nudge = 1e-4f;
    opt->pair_mode = 1;
    opt->photon_only = 0;
    opt->majorant_scale = 1.0f;
    opt->wave_size = 1u << 20;
    opt->bank_factor = 8;
    opt->scheduler = 1;
    opt->warp_stack = 8192;
    opt->cta_threads = 0;
    opt->hom_tol = 0.0f;
    opt->tally_mode = 0;
    opt->table_memory = 0;
    opt->bank_high_g = 0;
    opt->bank_high_e = 0;
    opt->bank_low = 0;
    opt->steps_per_refill = 0;
    opt->l2_persist = 0;
    return GPUMCD_OK;
}

static void destroy_impl(gpumcd_ctx *c)
{
    if (!c) return;
    cudaFree(c->phantom);
    cudaFree(c->radius);
    cudaFree(c->stage_density);
    cudaFree(c->stage_material);
    cudaFree(c->scratch);
    cudaFree(c->dose_stage);
    cudaFree(c->table_blob);
    cudaFree(c->edep);
    cudaFree(c->moments);
    cudaFree(c->cnt);
    cudaFree(c->qcount);
    for (int k = 0; k < kMaxQueues; ++k) { cudaFree(c->qA[k]); cudaFree(c->qB[k]); cudaFree(c->qC[k]); }
    cudaFree(c->spec_cdf);
    cudaFree(c->spec_edges);
    cudaFree(c->phsp);
    cudaFree(c->head);
    cudaFree(c->stkA); cudaFree(c->stkB); cudaFree(c->stkC);
    for (auto &e : c->events) { cudaEventDestroy(e.a); cudaEventDestroy(e.b); }
    delete c;
}

// The persistent kernel's variants: (trace | multi-voxel steps x tally mode) x tables in shared / global memory
// x CTA size.  1024 threads per CTA exist for the fp64 tally only (the ablation of DESIGN.md 7).
template <class V>
static const void *persistent_variant(bool smem, int threads)
{
    if (threads == kPThreadsDefault) return smem ? (const void *)k_persistent<V, true, kPThreadsDefault> : (const void *)k_persistent<V, false, kPThreadsDefault>;
    // the other CTA sizes (ablation): fp64 tally, no phase space, the several-steps-per-refill form of the loop
    if (V::TALLY == TALLY_F64 && !V::PHSP) {
        using A = Variant<V::TRACE, V::MULTI, TALLY_F64, false, !V::TRACE>;
        if (threads == 512) return smem ? (const void *)k_persistent<A, true, 512> : (const void *)k_persistent<A, false, 512>;
        if (threads == 1024) return smem ? (const void *)k_persistent<A, true, 1024> : (const void *)k_persistent<A, false, 1024>;
    }
    return nullptr;
}
template <bool MULTI, bool PHSP, bool INNER>
static const void *persistent_tally(int tally, bool smem, int threads)
{
    if (tally == TALLY_WARP) return persistent_variant<Variant<false, MULTI, TALLY_WARP, PHSP, INNER>>(smem, threads);
    if (tally == TALLY_FIXED) return persistent_variant<Variant<false, MULTI, TALLY_FIXED, PHSP, INNER>>(smem, threads);
    return persistent_variant<Variant<false, MULTI, TALLY_F64, PHSP, INNER>>(smem, threads);
}
// nullptr: the combination is not built (1024 threads per CTA with another tally than fp64, a phase space or
// several steps per refill; a phase space with several steps per refill)
static const void *persistent_kernel(bool trace, bool multi, int tally, bool phsp, bool inner, bool smem, int threads)
{
    if (trace) return phsp ? persistent_variant<Variant<true, false, TALLY_F64, true>>(smem, threads)
                           : persistent_variant<Variant<true, false, TALLY_F64>>(smem, threads); // a trace run tallies nothing of interest
    if (phsp) return multi ? persistent_tally<true, true, false>(tally, smem, threads) : persistent_tally<false, true, false>(tally, smem, threads);
    if (inner) return multi ? persistent_tally<true, false, true>(tally, smem, threads) : persistent_tally<false, false, true>(tally, smem, threads);
    return multi ? persistent_tally<true, false, false>(tally, smem, threads) : persistent_tally<false, false, false>(tally, smem, threads);
}

// cudaFuncAttributeMaxDynamicSharedMemorySize belongs to the kernel function, not to a context: it is only
// ever raised, so that contexts with table blobs of different sizes can be alive at the same time.
static int allow_dynamic_smem(gpumcd_ctx *ctx, const void *fn, size_t bytes)
{
    static std::mutex mu;
    static std::map<const void *, size_t> allowed;
    std::lock_guard<std::mutex> lock(mu);
    size_t &cur = allowed[fn];
    if (bytes > cur) {
        CK(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(bytes)));
        cur = bytes;
    }
    return GPUMCD_OK;
}

// Phantom -> device: pack {density, material}, validate, reduce rho_max per material, rebuild the
// Woodcock majorants (H10) and upload the table blob.  Synchronous.
//   mu_max(E_i) = max_m rho_max[m] mu_m(E_i) (Eq. 3);  M_e = running max in E of
//   max_m rho_max[m] (Sigma_Moller + Sigma_brems) (L110-113 made rigorous).
static int load_phantom(gpumcd_ctx *ctx, const float *density, const uint8_t *material, bool on_host)
{
    const size_t nvox = ctx->nvox;
    const float *d_density = density;
    const uint8_t *d_material = material;
    if (on_host) {
        if (!ctx->stage_density) {
            CK(cudaMalloc(&ctx->stage_density, nvox * sizeof(float)));
            CK(cudaMalloc(&ctx->stage_material, nvox));
        }
        CK(cudaMemcpyAsync(ctx->stage_density, density, nvox * sizeof(float), cudaMemcpyHostToDevice, nullptr));
        CK(cudaMemcpyAsync(ctx->stage_material, material, nvox, cudaMemcpyHostToDevice, nullptr));
        d_density = ctx->stage_density;
        d_material = ctx->stage_material;
    }
    CK(cudaMemsetAsync(ctx->scratch, 0, 12 * sizeof(unsigned), nullptr));
    const int grid = static_cast<int>(std::min<size_t>((nvox + kBlock - 1) / kBlock, 148 * 8));
    k_pack_phantom<<<grid, kBlock>>>(d_density, d_material, make_geom(ctx), nvox, ctx->n_mat, ctx->phantom, ctx->scratch, ctx->scratch + 8);
    CK(cudaGetLastError());
    if (ctx->opt.hom_tol > 0.f) {
        const int r_max = std::min(7, static_cast<int>(std::ceil(ctx->opt.es_max_cm / ctx->h)) + 1);
        k_uniform_radius<<<grid, kBlock>>>(ctx->phantom, ctx->radius, make_geom(ctx), ctx->opt.hom_tol, r_max);
        CK(cudaGetLastError());
    }
    unsigned h_scratch[12];
    CK(cudaMemcpy(h_scratch, ctx->scratch, sizeof h_scratch, cudaMemcpyDeviceToHost));
    if (h_scratch[8] != 0) {
        set_error(ctx, "phantom has a material id >= n_materials or a density outside [2^-20, 2^12) g/cm^3 (or not a number)");
        return GPUMCD_ERR_INVALID_ARG;
    }
    double rho_max[8];
    for (int m = 0; m < 8; ++m) { float f; memcpy(&f, &h_scratch[m], 4); rho_max[m] = f; }
    const int nE = ctx->n_E, nM = ctx->n_mat;
    const float *ph = ctx->blob_host.data(), *el = ph + ctx->tab.off_el;
    float *mu_max = ctx->blob_host.data() + ctx->tab.off_mu, *m_e = ctx->blob_host.data() + ctx->tab.off_me;
    double run = 0.0;
    for (int i = 0; i < nE; ++i) {
        double mu = 0.0, se = 0.0;
        for (int m = 0; m < nM; ++m) {
            const float *p = ph + static_cast<size_t>(m) * 3 * nE;
            const float *e = el + static_cast<size_t>(m) * 4 * nE;
            mu = std::max(mu, rho_max[m] * (static_cast<double>(p[i]) + p[nE + i] + p[2 * nE + i]));
            se = std::max(se, rho_max[m] * (static_cast<double>(e[nE + i]) + e[2 * nE + i]));
        }
        run = std::max(run, se);
        mu_max[i] = static_cast<float>(mu * ctx->opt.majorant_scale);
        m_e[i] = static_cast<float>(run * ctx->opt.majorant_scale);
    }
    CK(cudaMemcpy(ctx->table_blob, ctx->blob_host.data(), ctx->blob_host.size() * sizeof(float), cudaMemcpyHostToDevice));
    return GPUMCD_OK;
}

static int create_impl(gpumcd_ctx **out, const float *density, const uint8_t *material, bool on_host, int nx,
                       int ny, int nz, float voxel_cm, const gpumcd_tables *t, const gpumcd_options *opt_in)
{
    gpumcd_ctx *ctx = nullptr; // errors before allocation go to the global string
    if (!out) return GPUMCD_ERR_INVALID_ARG;
    *out = nullptr;
    if (!density || !material || !t) { set_error(nullptr, "null pointer argument"); return GPUMCD_ERR_INVALID_ARG; }
    if (nx < 1 || ny < 1 || nz < 1 || nx > 1024 || ny > 1024 || nz > 1024 || !(voxel_cm > 0.f)) {
        set_error(nullptr, "bad phantom dimensions (1..1024 per axis, voxel size > 0)");
        return GPUMCD_ERR_INVALID_ARG;
    }
    if (t->n_materials < 1 || t->n_materials > 8 || t->n_energy < 2 || !t->photon || !t->electron || !t->ms_a ||
        t->n_K < 2 || !(t->e_min > 0.f) || !(t->e_max > t->e_min) || !(t->lnK_max > t->lnK_min) ||
        t->e_cut < t->e_min || t->p_cut < t->e_min) {
        set_error(nullptr, "bad table description");
        return GPUMCD_ERR_INVALID_ARG;
    }
    gpumcd_options opt;
    gpumcd_default_options(&opt);
    if (opt_in) opt = *opt_in;
    if (!(opt.es_max_cm > 0.f) || !(opt.f_eloss_max > 0.f) || opt.f_eloss_max > 1.f || opt.boundary_nudge < 0.f ||
        !(opt.majorant_scale >= 1.f) || opt.wave_size == 0 || opt.bank_factor == 0 || opt.warp_stack > (1u << 20) ||
        (opt.cta_threads != 0 && opt.cta_threads != 512 && opt.cta_threads != kPThreadsDefault && opt.cta_threads != 1024) || !(opt.hom_tol >= 0.f) ||
        opt.tally_mode < 0 || opt.tally_mode > 2 || (opt.tally_mode != 0 && opt.cta_threads != 0 && opt.cta_threads != kPThreadsDefault) ||
        opt.table_memory < 0 || opt.table_memory > 1 || opt.bank_low > 32 || opt.steps_per_refill > 64 || opt.l2_persist < 0 || opt.l2_persist > 1 ||
        (opt.bank_high_g && opt.bank_high_g < (opt.bank_low ? opt.bank_low : kLowDefault)) || // (a warp would change to
        (opt.bank_high_e && opt.bank_high_e < (opt.bank_low ? opt.bank_low : kLowDefault)) || //  a type it leaves at once)
        static_cast<unsigned long long>(opt.wave_size) * opt.bank_factor > 0x7fffffffull) {
        set_error(nullptr, "bad options");
        return GPUMCD_ERR_INVALID_ARG;
    }
    ctx = new gpumcd_ctx;
    struct Guard { gpumcd_ctx *&c; bool ok = false; ~Guard() { if (!ok) { if (c) g_create_error = c->err; destroy_impl(c); } } } guard{ctx};
    ctx->nx = nx; ctx->ny = ny; ctx->nz = nz; ctx->h = voxel_cm;
    ctx->nvox = static_cast<size_t>(nx) * ny * nz;
    ctx->opt = opt;
    const size_t nvox = ctx->nvox;
    const int nE = t->n_energy, nK = t->n_K, nM = t->n_materials;

    // ---- tables: one device blob = photon | electron | mu_max | m_e | ms_a (majorants filled per phantom) ----
    const size_t n_ph = static_cast<size_t>(nM) * 3 * nE, n_el = static_cast<size_t>(nM) * 4 * nE;
    const size_t blob_len = n_ph + n_el + 2 * static_cast<size_t>(nE) + nK;
    ctx->blob_host.assign((blob_len + 3) & ~static_cast<size_t>(3), 0.0f); // padded for 16-byte bulk copies
    memcpy(ctx->blob_host.data(), t->photon, n_ph * sizeof(float));
    memcpy(ctx->blob_host.data() + n_ph, t->electron, n_el * sizeof(float));
    memcpy(ctx->blob_host.data() + n_ph + n_el + 2 * static_cast<size_t>(nE), t->ms_a, static_cast<size_t>(nK) * sizeof(float));
    ctx->n_mat = nM; ctx->n_E = nE;
    CK(cudaMalloc(&ctx->table_blob, ctx->blob_host.size() * sizeof(float)));
    Tables &tb = ctx->tab;
    tb.blob = ctx->table_blob;
    tb.off_el = static_cast<unsigned>(n_ph);
    tb.off_mu = static_cast<unsigned>(n_ph + n_el);
    tb.off_me = tb.off_mu + nE;
    tb.off_ms = tb.off_me + nE;
    tb.gE.n = nE;
    tb.gE.x_min = static_cast<float>(std::log(static_cast<double>(t->e_min)));
    tb.gE.inv_dx = static_cast<float>((nE - 1) / (std::log(static_cast<double>(t->e_max)) - std::log(static_cast<double>(t->e_min))));
    tb.gK.n = nK;
    tb.gK.x_min = t->lnK_min;
    tb.gK.inv_dx = static_cast<float>((nK - 1) / (static_cast<double>(t->lnK_max) - static_cast<double>(t->lnK_min)));
    tb.e_min = t->e_min; tb.e_cut = t->e_cut; tb.p_cut = t->p_cut;
    ctx->e_max = t->e_max;
    tb.n_mat = nM;
    ctx->table_floats = static_cast<unsigned>(ctx->blob_host.size());

    // ---- phantom (and the majorants that depend on it) ----
    CK(cudaMalloc(&ctx->phantom, nvox * sizeof(uint32_t)));
    if (opt.hom_tol > 0.f) CK(cudaMalloc(&ctx->radius, nvox));
    CK(cudaMalloc(&ctx->scratch, 12 * sizeof(unsigned)));
    {
        const int rc = load_phantom(ctx, density, material, on_host);
        if (rc != GPUMCD_OK) return rc;
    }

    // ---- tally, counters, queues ----
    CK(cudaMalloc(&ctx->edep, nvox * sizeof(double)));
    CK(cudaMalloc(&ctx->cnt, sizeof(DevCounters)));
    CK(cudaMalloc(&ctx->qcount, kMaxQueues * sizeof(unsigned)));
    ctx->n_queues = opt.scheduler == 1 ? 0 : 4;
    ctx->qcap = opt.wave_size * opt.bank_factor;
    for (int k = 0; k < ctx->n_queues; ++k) {
        CK(cudaMalloc(&ctx->qA[k], static_cast<size_t>(ctx->qcap) * sizeof(float4)));
        CK(cudaMalloc(&ctx->qB[k], static_cast<size_t>(ctx->qcap) * sizeof(float4)));
        CK(cudaMalloc(&ctx->qC[k], static_cast<size_t>(ctx->qcap) * sizeof(uint4)));
    }
    if (opt.scheduler == 1) {
        int dev = 0, n_sm = 0, coop = 0, max_smem = 0;
        CK(cudaGetDevice(&dev));
        CK(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
        CK(cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev));
        CK(cudaDeviceGetAttribute(&max_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
        if (!coop) { set_error(ctx, "device does not support cooperative launches (scheduler 1)"); return GPUMCD_ERR_CUDA; }
        const size_t table_bytes = static_cast<size_t>(ctx->table_floats) * sizeof(float);
        const int threads = opt.cta_threads ? static_cast<int>(opt.cta_threads) : kPThreadsDefault;
        const void *fn = persistent_kernel(false, opt.hom_tol > 0.f, opt.tally_mode, false, false, true, threads);
        cudaFuncAttributes fa{};
        CK(cudaFuncGetAttributes(&fa, fn));
        ctx->smem_tables = opt.table_memory == 0 && table_bytes + fa.sharedSizeBytes + 1024 <= static_cast<size_t>(max_smem);
        // behind the tables: room for a spectrum of up to kSpecSmemBins bins (cdf as double, edges as float), if it fits
        ctx->spec_smem_bytes = 0;
        if (ctx->smem_tables && table_bytes + kSpecSmemBytes + fa.sharedSizeBytes + 1024 <= static_cast<size_t>(max_smem))
            ctx->spec_smem_bytes = kSpecSmemBytes;
        const size_t dyn = ctx->smem_tables ? table_bytes + ctx->spec_smem_bytes : 0;
        fn = persistent_kernel(false, opt.hom_tol > 0.f, opt.tally_mode, false, false, ctx->smem_tables, threads);
        { const int rc = allow_dynamic_smem(ctx, fn, dyn); if (rc != GPUMCD_OK) return rc; }
        int per_sm = 0;
        CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, threads, dyn));
        if (per_sm < 1) { set_error(ctx, "persistent kernel does not fit on an SM"); return GPUMCD_ERR_CUDA; }
        ctx->p_grid = n_sm; // one CTA per SM
        ctx->cap_r = std::max(opt.warp_stack, kMinStack);
        ctx->stride = 2 * ctx->cap_r + 3 * kPend;
        const size_t n_warps = static_cast<size_t>(ctx->p_grid) * (threads / 32); // of the CTA size actually used
        const size_t recs = n_warps * ctx->stride;
        CK(cudaMalloc(&ctx->stkA, recs * sizeof(float4)));
        CK(cudaMalloc(&ctx->stkB, recs * sizeof(float4)));
        CK(cudaMalloc(&ctx->stkC, recs * sizeof(uint4)));
        CK(cudaMalloc(&ctx->head, sizeof(unsigned)));
        // l2_persist: set aside L2 for the packed phantom (the one array every move reads)
        ctx->l2_window = 0;
        if (opt.l2_persist == 1) {
            int max_persist = 0, max_window = 0;
            CK(cudaDeviceGetAttribute(&max_persist, cudaDevAttrMaxPersistingL2CacheSize, dev));
            CK(cudaDeviceGetAttribute(&max_window, cudaDevAttrMaxAccessPolicyWindowSize, dev));
            const size_t want = nvox * sizeof(uint32_t);
            size_t cur = 0;
            CK(cudaDeviceGetLimit(&cur, cudaLimitPersistingL2CacheSize));
            const size_t carve = std::min<size_t>(want, static_cast<size_t>(max_persist));
            if (carve > cur) CK(cudaDeviceSetLimit(cudaLimitPersistingL2CacheSize, carve)); // device-wide: only ever raised
            ctx->l2_window = std::min<size_t>(want, static_cast<size_t>(max_window));
            ctx->l2_hit_ratio = ctx->l2_window ? std::min(1.0f, static_cast<float>(static_cast<double>(std::max(carve, cur)) / static_cast<double>(ctx->l2_window))) : 0.f;
        }
    }
    CK(cudaDeviceSynchronize());
    guard.ok = true;
    *out = ctx;
    return GPUMCD_OK;
}

extern "C" int gpumcd_create(gpumcd_ctx **out, const float *density_dev, const uint8_t *material_dev, int nx, int ny,
                             int nz, float voxel_cm, const gpumcd_tables *tables, const gpumcd_options *opt)
{
    return create_impl(out, density_dev, material_dev, false, nx, ny, nz, voxel_cm, tables, opt);
}

extern "C" int gpumcd_create_host(gpumcd_ctx **out, const float *density_host, const uint8_t *material_host, int nx,
                                  int ny, int nz, float voxel_cm, const gpumcd_tables *tables,
                                  const gpumcd_options *opt)
{
    return create_impl(out, density_host, material_host, true, nx, ny, nz, voxel_cm, tables, opt);
}

extern "C" int gpumcd_set_phantom_host(gpumcd_ctx *ctx, const float *density_host, const uint8_t *material_host)
{
    if (!ctx || !density_host || !material_host) return GPUMCD_ERR_INVALID_ARG;
    if (ctx->ran) CK(cudaStreamSynchronize(ctx->last_stream)); // the last run still reads the old phantom
    return load_phantom(ctx, density_host, material_host, true);
}

extern "C" int gpumcd_set_phantom(gpumcd_ctx *ctx, const float *density_dev, const uint8_t *material_dev)
{
    if (!ctx || !density_dev || !material_dev) return GPUMCD_ERR_INVALID_ARG;
    if (ctx->ran) CK(cudaStreamSynchronize(ctx->last_stream));
    return load_phantom(ctx, density_dev, material_dev, false);
}

extern "C" int gpumcd_set_source(gpumcd_ctx *ctx, const gpumcd_source *s)
{
    if (!ctx || !s) return GPUMCD_ERR_INVALID_ARG;
    if ((s->particle != 0 && s->particle != 1) || s->shape < 0 || s->shape > 2 || s->n_spec < 0) {
        set_error(ctx, "bad source description");
        return GPUMCD_ERR_INVALID_ARG;
    }
    if (ctx->ran) CK(cudaStreamSynchronize(ctx->last_stream)); // the last run still reads the old source arrays
    if (s->shape == 2) {
        // ---- phase space (R35): copy the records, check them, count them by type
        if (!s->phsp || s->n_phsp == 0) { set_error(ctx, "empty phase space"); return GPUMCD_ERR_INVALID_ARG; }
        float4 *rec = nullptr;
        const size_t bytes = static_cast<size_t>(s->n_phsp) * 8 * sizeof(float);
        CK(cudaMalloc(&rec, bytes));
        struct Free { float4 *&p; ~Free() { cudaFree(p); } } guard{rec};
        CK(cudaMemcpy(rec, s->phsp, bytes, s->phsp_on_host ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice));
        unsigned long long *d_out = nullptr, h_out[4];
        CK(cudaMalloc(&d_out, sizeof h_out));
        struct Free2 { unsigned long long *p; ~Free2() { cudaFree(p); } } guard2{d_out};
        CK(cudaMemset(d_out, 0, sizeof h_out));
        const unsigned blocks = static_cast<unsigned>(std::min<uint64_t>((s->n_phsp + kBlock - 1) / kBlock, 148 * 8));
        k_check_phsp<<<blocks, kBlock>>>(rec, s->n_phsp, ctx->tab.e_min, ctx->e_max, d_out);
        CK(cudaGetLastError());
        CK(cudaMemcpy(h_out, d_out, sizeof h_out, cudaMemcpyDeviceToHost));
        if (h_out[0]) { set_error(ctx, "phase space: a record has a type other than 0 / 1 or a number that is not finite"); return GPUMCD_ERR_INVALID_ARG; }
        if (h_out[1]) { set_error(ctx, "phase space: an energy lies outside the energy range of the tables"); return GPUMCD_ERR_TABLE_RANGE; }
        SourceDev d{};
        d.shape = 2;
        d.has_g = h_out[2] != 0; d.has_e = h_out[3] != 0;
        d.particle = d.has_g ? 0 : 1;
        d.n_phsp = s->n_phsp;
        cudaFree(ctx->phsp);
        ctx->phsp = rec;
        rec = nullptr; // owned by the context from here on
        d.phsp = ctx->phsp;
        cudaFree(ctx->spec_cdf); ctx->spec_cdf = nullptr;
        cudaFree(ctx->spec_edges); ctx->spec_edges = nullptr;
        ctx->src = d;
        ctx->have_source = true;
        return GPUMCD_OK;
    }
    const double wx = s->shape == 1 ? s->wx : 0.0, wy = s->shape == 1 ? s->wy : 0.0;
    if (wx < 0 || wy < 0 || s->cx - 0.5 * wx < 0 || s->cx + 0.5 * wx >= static_cast<double>(ctx->nx) * ctx->h ||
        s->cy - 0.5 * wy < 0 || s->cy + 0.5 * wy >= static_cast<double>(ctx->ny) * ctx->h) {
        set_error(ctx, "the source field does not lie inside the z = 0 face of the phantom");
        return GPUMCD_ERR_INVALID_ARG;
    }
    const float e_lo = ctx->tab.e_min, e_hi = ctx->e_max;
    SourceDev d{};
    d.particle = s->particle; d.shape = s->shape;
    d.cx = s->cx; d.cy = s->cy; d.wx = wx; d.wy = wy; d.energy = s->energy;
    d.n_spec = s->n_spec;
    d.has_g = s->particle == 0; d.has_e = s->particle == 1;
    cudaFree(ctx->phsp); ctx->phsp = nullptr;
    cudaFree(ctx->spec_cdf); ctx->spec_cdf = nullptr;
    cudaFree(ctx->spec_edges); ctx->spec_edges = nullptr;
    if (s->n_spec > 0) {
        if (!s->spec_E || !s->spec_w) { set_error(ctx, "null spectrum arrays"); return GPUMCD_ERR_INVALID_ARG; }
        std::vector<double> cdf(s->n_spec + 1);
        cdf[0] = 0.0;
        for (int j = 0; j < s->n_spec; ++j) {
            if (!(s->spec_w[j] >= 0.f) || !(s->spec_E[j + 1] > s->spec_E[j])) {
                set_error(ctx, "spectrum weights must be >= 0 and edges increasing");
                return GPUMCD_ERR_INVALID_ARG;
            }
            cdf[j + 1] = cdf[j] + static_cast<double>(s->spec_w[j]);
        }
        if (!(cdf[s->n_spec] > 0.0)) { set_error(ctx, "spectrum has zero total weight"); return GPUMCD_ERR_INVALID_ARG; }
        if (s->spec_E[0] < e_lo || s->spec_E[s->n_spec] > e_hi) {
            set_error(ctx, "spectrum extends outside the energy range of the tables");
            return GPUMCD_ERR_TABLE_RANGE;
        }
        CK(cudaMalloc(&ctx->spec_cdf, cdf.size() * sizeof(double)));
        CK(cudaMalloc(&ctx->spec_edges, cdf.size() * sizeof(float)));
        CK(cudaMemcpy(ctx->spec_cdf, cdf.data(), cdf.size() * sizeof(double), cudaMemcpyHostToDevice));
        CK(cudaMemcpy(ctx->spec_edges, s->spec_E, cdf.size() * sizeof(float), cudaMemcpyHostToDevice));
        d.cdf = ctx->spec_cdf;
        d.edges = ctx->spec_edges;
    } else if (s->energy < e_lo || s->energy > e_hi) {
        set_error(ctx, "source energy outside the energy range of the tables");
        return GPUMCD_ERR_TABLE_RANGE;
    }
    ctx->src = d;
    ctx->have_source = true;
    return GPUMCD_OK;
}

static Params make_params(gpumcd_ctx *ctx, uint64_t seed, uint32_t hist_hi, bool photon_only, unsigned long long *trace)
{
    Params P;
    P.fx_scale = ctx->fx_scale;
    P.tab = ctx->tab;
    P.geo = make_geom(ctx);
    P.opt.es_max = ctx->opt.es_max_cm;
    P.opt.f_eloss = ctx->opt.f_eloss_max;
    P.opt.nudge = ctx->opt.boundary_nudge;
    P.opt.hom_tol = ctx->opt.hom_tol;
    P.opt.pair_mode = ctx->opt.pair_mode;
    P.opt.photon_only = photon_only ? 1 : ctx->opt.photon_only;
    P.rng.k0 = static_cast<uint32_t>(seed);
    P.rng.k1 = static_cast<uint32_t>(seed >> 32);
    P.rng.hist_hi = hist_hi;
    P.edep = ctx->edep;
    P.cnt = ctx->cnt;
    P.trace = trace;
    P.trace_off = ctx->hist_offset;
    return P;
}

// run `call` with TL bound to the context's tally mode as a compile-time constant
#define WITH_TALLY(mode, call)                                                  \
    do {                                                                        \
        if ((mode) == TALLY_WARP) { constexpr int TL = TALLY_WARP; call; }      \
        else if ((mode) == TALLY_FIXED) { constexpr int TL = TALLY_FIXED; call; } \
        else { constexpr int TL = TALLY_F64; call; }                            \
    } while (0)

// Scheduler 0: per wave, fill the source list, then alternate photon and electron
// passes until both lists are empty; the host reads the list lengths between passes.
static int run_waves_host_loop(gpumcd_ctx *ctx, uint64_t h_begin, uint64_t n_hist, uint64_t seed, bool trace_mode,
                               unsigned long long *trace, cudaStream_t st)
{
    enum { PA = 0, PB = 1, EA = 2, EB = 3 };
    int pcur = PA, pnext = PB, ecur = EA, enext = EB;
    uint64_t h0 = h_begin;
    const uint64_t h_end = h_begin + n_hist;
    while (h0 < h_end) {
        uint64_t n = std::min<uint64_t>(ctx->opt.wave_size, h_end - h0);
        n = std::min<uint64_t>(n, 0x100000000ull - (h0 & 0xffffffffull)); // a wave never straddles 2^32
        const Params P = make_params(ctx, seed, static_cast<uint32_t>(h0 >> 32), trace_mode, trace);
        CK(cudaMemsetAsync(ctx->qcount, 0, 4 * sizeof(unsigned), st));
        { LaunchScope ls(ctx, st, CLS_SOURCE);
        WITH_TALLY(ctx->opt.tally_mode, (k_source<Variant<false, false, TL>><<<static_cast<unsigned>((n + kBlock - 1) / kBlock), kBlock, 0, st>>>(
                                            P, ctx->src, make_queue(ctx, pcur), make_queue(ctx, ecur), h0, static_cast<unsigned>(n)))); }
        CK(cudaGetLastError());
        unsigned cnt[4];
        for (;;) {
            CK(cudaMemcpyAsync(cnt, ctx->qcount, sizeof cnt, cudaMemcpyDeviceToHost, st));
            CK(cudaStreamSynchronize(st));
            for (int k = 0; k < 4; ++k) ctx->high_water = std::max<unsigned long long>(ctx->high_water, cnt[k]);
            if (cnt[0] > ctx->qcap || cnt[1] > ctx->qcap || cnt[2] > ctx->qcap || cnt[3] > ctx->qcap) {
                set_error(ctx, "particle queue overflow: raise bank_factor or lower wave_size");
                return GPUMCD_ERR_BANK_OVERFLOW;
            }
            if (cnt[pcur] > 0) {
                const unsigned m = cnt[pcur];
                // photons: secondaries of the same type go to the other photon list, electrons are
                // appended to the current electron list (not being consumed now)
                { LaunchScope ls(ctx, st, CLS_PHOTON);
                if (trace_mode)
                    k_photon_pass<Variant<true, false, TALLY_F64>><<<(m + kBlock - 1) / kBlock, kBlock, 0, st>>>(P, make_queue(ctx, pcur), m, make_queue(ctx, ecur), make_queue(ctx, pnext));
                else
                    WITH_TALLY(ctx->opt.tally_mode, (k_photon_pass<Variant<false, false, TL>><<<(m + kBlock - 1) / kBlock, kBlock, 0, st>>>(
                                                        P, make_queue(ctx, pcur), m, make_queue(ctx, ecur), make_queue(ctx, pnext)))); }
                CK(cudaGetLastError());
                CK(cudaMemsetAsync(ctx->qcount + pcur, 0, sizeof(unsigned), st));
                std::swap(pcur, pnext);
            } else if (cnt[ecur] > 0) {
                const unsigned m = cnt[ecur];
                { LaunchScope ls(ctx, st, CLS_ELECTRON);
                if (ctx->opt.hom_tol > 0.f)
                    WITH_TALLY(ctx->opt.tally_mode, (k_electron_pass<Variant<false, true, TL>><<<(m + kBlock - 1) / kBlock, kBlock, 0, st>>>(
                                                        P, make_queue(ctx, ecur), m, make_queue(ctx, enext), make_queue(ctx, pcur))));
                else
                    WITH_TALLY(ctx->opt.tally_mode, (k_electron_pass<Variant<false, false, TL>><<<(m + kBlock - 1) / kBlock, kBlock, 0, st>>>(
                                                        P, make_queue(ctx, ecur), m, make_queue(ctx, enext), make_queue(ctx, pcur)))); }
                CK(cudaGetLastError());
                CK(cudaMemsetAsync(ctx->qcount + ecur, 0, sizeof(unsigned), st));
                std::swap(ecur, enext);
            } else {
                break;
            }
        }
        h0 += n;
    }
    return GPUMCD_OK;
}

// Scheduler 1: the whole run is one cooperative launch (split only where the history id crosses 2^32).
static int run_persistent(gpumcd_ctx *ctx, uint64_t h_begin, uint64_t n_hist, uint64_t seed, float *dose_dev,
                          unsigned long long *trace, cudaStream_t st)
{
    const double h3 = static_cast<double>(ctx->h) * ctx->h * ctx->h;
    uint64_t h0 = h_begin;
    const uint64_t h_end = h_begin + n_hist;
    while (h0 < h_end) {
        uint64_t n = std::min<uint64_t>(h_end - h0, 0x100000000ull - (h0 & 0xffffffffull));
        n = std::min<uint64_t>(n, 0x80000000ull); // the claim counter is 32 bits wide
        PersistArgs a{};
        a.P = make_params(ctx, seed, static_cast<uint32_t>(h0 >> 32), trace != nullptr, trace);
        a.S = ctx->src;
        CK(cudaMemsetAsync(ctx->head, 0, sizeof(unsigned), st));
        a.head = ctx->head;
        a.stkA = ctx->stkA; a.stkB = ctx->stkB; a.stkC = ctx->stkC;
        a.cap_r = ctx->cap_r;
        a.stride = ctx->stride;
        a.hist0 = h0;
        a.n_hist = static_cast<unsigned>(n);
        a.table_floats = ctx->table_floats;
        a.spec_in_smem = (ctx->spec_smem_bytes != 0 && ctx->src.n_spec > 0 && ctx->src.n_spec <= kSpecSmemBins) ? 1 : 0;
        a.inv_h3_n = 1.0 / (h3 * static_cast<double>(n_hist));
        a.dose = dose_dev;
        a.nvox = ctx->nvox;
        a.finalize = (h0 + n == h_end) ? 1 : 0;
        // CTA size (see persistent.cuh): 768 threads unless the caller asks for 512 or 1024
        const int threads = ctx->opt.cta_threads ? static_cast<int>(ctx->opt.cta_threads) : kPThreadsDefault;
        // banked particles of the other type that make a warp change to it before it has to: none by default (a
        // warp stays with one type until it runs dry or a stack is about to fill up; measured on configs 1-5,
        // bench.py --ablation: every earlier change costs)
        a.high_g = ctx->opt.bank_high_g ? ctx->opt.bank_high_g : 0xffffffffu;
        a.high_e = ctx->opt.bank_high_e ? ctx->opt.bank_high_e : 0xffffffffu;
        a.low = ctx->opt.bank_low ? ctx->opt.bank_low : kLowDefault;
        // steps per refill (the paper's N, L180): 4 (measured on configs 1-5: 2.5-5 % faster than 1; 8 is no better)
        const bool phsp = ctx->src.shape == 2;
        a.inner = ctx->opt.steps_per_refill ? ctx->opt.steps_per_refill : 4u;
        if (phsp || trace) a.inner = 1u; // (variants that are not built: one step per refill)
        void *args[] = {&a};
        // the kernel variant: trace (photon-only replay) | multi-voxel steps x tally mode; tables in shared memory; CTA size
        const bool multi = ctx->opt.hom_tol > 0.f && !trace; // a trace run tracks no electrons
        const void *fn = persistent_kernel(trace != nullptr, multi, ctx->opt.tally_mode, phsp, a.inner > 1u, ctx->smem_tables, threads);
        if (!fn) { set_error(ctx, "a phase-space source needs the default CTA size (cta_threads 0)"); return GPUMCD_ERR_INVALID_ARG; }
        if (threads != kPThreadsDefault && !trace) a.inner = std::max(a.inner, 1u); // (these sizes are built in the loop form)
        const size_t dyn = ctx->smem_tables ? static_cast<size_t>(ctx->table_floats) * sizeof(float) + ctx->spec_smem_bytes : 0;
        { const int rc = allow_dynamic_smem(ctx, fn, dyn); if (rc != GPUMCD_OK) return rc; }
        { LaunchScope ls(ctx, st, CLS_ELECTRON);
        cudaLaunchConfig_t cfg{};
        cfg.gridDim = dim3(ctx->p_grid); cfg.blockDim = dim3(threads); cfg.dynamicSmemBytes = dyn; cfg.stream = st;
        cudaLaunchAttribute attr[2];
        attr[0].id = cudaLaunchAttributeCooperative;
        attr[0].val.cooperative = 1;
        cfg.attrs = attr; cfg.numAttrs = 1;
        if (ctx->l2_window) { // phantom reads of this launch hit a persisting carve-out of the L2
            attr[1].id = cudaLaunchAttributeAccessPolicyWindow;
            attr[1].val.accessPolicyWindow.base_ptr = ctx->phantom;
            attr[1].val.accessPolicyWindow.num_bytes = ctx->l2_window;
            attr[1].val.accessPolicyWindow.hitRatio = ctx->l2_hit_ratio;
            attr[1].val.accessPolicyWindow.hitProp = cudaAccessPropertyPersisting;
            attr[1].val.accessPolicyWindow.missProp = cudaAccessPropertyStreaming;
            cfg.numAttrs = 2;
        }
        CK(cudaLaunchKernelExC(&cfg, fn, args)); }
        h0 += n;
    }
    return GPUMCD_OK;
}

// Bookkeeping and zeroing at the start of a run.
static int begin_run(gpumcd_ctx *ctx, uint64_t n_hist, unsigned long long *trace_dev, cudaStream_t st)
{
    if (!ctx) return GPUMCD_ERR_INVALID_ARG;
    if (!ctx->have_source) { set_error(ctx, "gpumcd_run called before gpumcd_set_source"); return GPUMCD_ERR_NO_SOURCE; }
    if (n_hist == 0) { set_error(ctx, "n_histories must be > 0"); return GPUMCD_ERR_INVALID_ARG; }
    ctx->last_stream = st;
    ctx->last_n = n_hist;
    ctx->high_water = 0;
    ctx->ran = true;
    ctx->prof = gpumcd_profile{};
    for (auto &e : ctx->events) { cudaEventDestroy(e.a); cudaEventDestroy(e.b); }
    ctx->events.clear();
    // tally_mode 2: the largest power of two (at most 2^40) for which even all the run's energy in one voxel
    // stays below 2^62 units
    ctx->fx_scale = std::ldexp(1.0f, std::min(40, std::max(0, 61 - std::ilogb(static_cast<double>(n_hist) * ctx->e_max + 1.0))));
    CK(cudaMemsetAsync(ctx->edep, 0, ctx->nvox * sizeof(double), st));
    CK(cudaMemsetAsync(ctx->cnt, 0, sizeof(DevCounters), st));
    if (trace_dev) CK(cudaMemsetAsync(trace_dev, 0, n_hist * sizeof(unsigned long long), st));
    return GPUMCD_OK;
}

// One pass of the whole path over histories [h_begin, h_begin + n_hist): transport with all secondaries,
// then the total of the tally and (dose_dev != NULL) the dose, normalised by n_hist.
static int transport(gpumcd_ctx *ctx, uint64_t h_begin, uint64_t n_hist, uint64_t seed, float *dose_dev,
                     unsigned long long *trace_dev, cudaStream_t st)
{
    if (ctx->opt.scheduler == 1) return run_persistent(ctx, h_begin, n_hist, seed, dose_dev, trace_dev, st);
    const int rc = run_waves_host_loop(ctx, h_begin, n_hist, seed, trace_dev != nullptr, trace_dev, st);
    if (rc != GPUMCD_OK) return rc;
    const double h3 = static_cast<double>(ctx->h) * ctx->h * ctx->h;
    const int grid = static_cast<int>(std::min<size_t>((ctx->nvox + kBlock - 1) / kBlock, 148 * 8));
    { LaunchScope ls(ctx, st, CLS_FINALIZE);
    const Params P = make_params(ctx, seed, 0u, trace_dev != nullptr, trace_dev);
    const double inv = 1.0 / (h3 * static_cast<double>(n_hist));
    if (ctx->opt.tally_mode == TALLY_FIXED && !trace_dev) k_finalize<TALLY_FIXED><<<grid, kBlock, 0, st>>>(P, ctx->nvox, inv, dose_dev);
    else k_finalize<TALLY_F64><<<grid, kBlock, 0, st>>>(P, ctx->nvox, inv, dose_dev); }
    CK(cudaGetLastError());
    return GPUMCD_OK;
}

static int run_impl(gpumcd_ctx *ctx, uint64_t n_hist, uint64_t seed, float *dose_dev, unsigned long long *trace_dev,
                    cudaStream_t st)
{
    const int rc = begin_run(ctx, n_hist, trace_dev, st);
    if (rc != GPUMCD_OK) return rc;
    return transport(ctx, ctx->hist_offset, n_hist, seed, dose_dev, trace_dev, st);
}

extern "C" int gpumcd_run(gpumcd_ctx *ctx, uint64_t n_histories, uint64_t seed, float *dose_out_dev, void *cuda_stream)
{
    if (!ctx || !dose_out_dev) return GPUMCD_ERR_INVALID_ARG;
    return run_impl(ctx, n_histories, seed, dose_out_dev, nullptr, static_cast<cudaStream_t>(cuda_stream));
}

extern "C" int gpumcd_run_host(gpumcd_ctx *ctx, uint64_t n_histories, uint64_t seed, float *dose_out_host,
                               void *cuda_stream)
{
    if (!ctx || !dose_out_host) return GPUMCD_ERR_INVALID_ARG;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    if (!ctx->dose_stage) CK(cudaMalloc(&ctx->dose_stage, ctx->nvox * sizeof(float)));
    float *tmp = ctx->dose_stage;
    int rc = run_impl(ctx, n_histories, seed, tmp, nullptr, st);
    if (rc == GPUMCD_OK) {
        cudaError_t e = cudaMemcpyAsync(dose_out_host, tmp, ctx->nvox * sizeof(float), cudaMemcpyDeviceToHost, st);
        unsigned long long dropped = 0;
        if (e == cudaSuccess) e = cudaMemcpyAsync(&dropped, &ctx->cnt->overflow, sizeof dropped, cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        if (e != cudaSuccess) { set_error(ctx, cudaGetErrorString(e)); rc = GPUMCD_ERR_CUDA; }
        else if (dropped) { set_error(ctx, "particle queue overflow: the result is invalid"); rc = GPUMCD_ERR_BANK_OVERFLOW; }
    }
    return rc;
}

extern "C" int gpumcd_run_uncertainty(gpumcd_ctx *ctx, uint64_t n_histories, uint32_t n_batches, uint64_t seed,
                                      float *dose_out_dev, float *sigma_out_dev, void *cuda_stream)
{
    if (!ctx || !dose_out_dev || !sigma_out_dev) return GPUMCD_ERR_INVALID_ARG;
    if (n_batches < 2 || n_batches > n_histories) {
        set_error(ctx, "n_batches must be at least 2 and at most n_histories");
        return GPUMCD_ERR_INVALID_ARG;
    }
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    int rc = begin_run(ctx, n_histories, nullptr, st);
    if (rc != GPUMCD_OK) return rc;
    const size_t nvox = ctx->nvox;
    if (!ctx->moments) CK(cudaMalloc(&ctx->moments, 3 * nvox * sizeof(double)));
    CK(cudaMemsetAsync(ctx->moments, 0, 3 * nvox * sizeof(double), st));
    double *s1 = ctx->moments, *sx = s1 + nvox, *sxx = sx + nvox;
    const int grid = static_cast<int>(std::min<size_t>((nvox + kBlock - 1) / kBlock, 148 * 8));
    // batch b simulates histories [h, h + m_b): together the batches cover exactly the histories of a
    // plain gpumcd_run with the same arguments, so the dose is the same
    uint64_t h = ctx->hist_offset;
    for (uint32_t b = 0; b < n_batches; ++b) {
        const uint64_t m = n_histories / n_batches + (b < n_histories % n_batches ? 1 : 0);
        rc = transport(ctx, h, m, seed, nullptr, nullptr, st);
        if (rc != GPUMCD_OK) return rc;
        { LaunchScope ls(ctx, st, CLS_FINALIZE);
        k_accumulate_batch<<<grid, kBlock, 0, st>>>(ctx->edep, s1, sx, sxx, nvox, 1.0 / static_cast<double>(m)); }
        CK(cudaGetLastError());
        h += m;
    }
    const double h3 = static_cast<double>(ctx->h) * ctx->h * ctx->h;
    { LaunchScope ls(ctx, st, CLS_FINALIZE);
    k_finalize_uncertainty<<<grid, kBlock, 0, st>>>(s1, sx, sxx, make_geom(ctx), nvox, 1.0 / h3,
                                                    1.0 / static_cast<double>(n_histories), static_cast<double>(n_batches),
                                                    dose_out_dev, sigma_out_dev, ctx->edep); }
    CK(cudaGetLastError());
    return GPUMCD_OK;
}

// ---------------------------------------------------------------------------------------------
// gpumcd_run_uncertainty_static: gpumcd_run_uncertainty for callers that cannot allocate (include/gpumcd.h).
// Its scratch, the three fp64 moment grids s1 | sx | sxx of the batch statistics, lives in this file-scope
// array instead of the context's lazily cudaMalloc'ed `moments`: 3 x 64^3 x 8 B = 6 MiB, held by every GPU
// that loads the library until the process exits, shared by all contexts and all calls.
// In host code `g_static_moments` is only a stand-in for the symbol, not a device address: the address a
// kernel can use comes from cudaGetSymbolAddress, asked once per device with that device current.
// ---------------------------------------------------------------------------------------------
constexpr size_t kStaticMaxVoxels = 64 * 64 * 64; // GPUMCD_STATIC_MAX_VOXELS of include/gpumcd.h
static_assert(kStaticMaxVoxels == GPUMCD_STATIC_MAX_VOXELS, "include/gpumcd.h states the limit");
static __device__ __align__(256) double g_static_moments[3 * kStaticMaxVoxels];

constexpr int kMaxDevices = 64;
static int static_moments_address(gpumcd_ctx *ctx, double **out)
{
    static std::mutex mu;
    static double *addr[kMaxDevices] = {};
    int dev = -1;
    CK(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxDevices) { set_error(ctx, "device ordinal beyond the static scratch table"); return GPUMCD_ERR_CUDA; }
    std::lock_guard<std::mutex> lock(mu);
    if (!addr[dev]) {
        void *p = nullptr;
        CK(cudaGetSymbolAddress(&p, g_static_moments)); // this device's copy of the array
        addr[dev] = static_cast<double *>(p);
    }
    *out = addr[dev];
    return GPUMCD_OK;
}

extern "C" int gpumcd_run_uncertainty_static(gpumcd_ctx *ctx, uint64_t n_histories, uint32_t n_batches, uint64_t seed,
                                             float *dose_out_dev, float *sigma_out_dev, void *cuda_stream)
{
    if (!ctx || !dose_out_dev || !sigma_out_dev) return GPUMCD_ERR_INVALID_ARG;
    if (ctx->nvox > kStaticMaxVoxels) {
        char buf[200];
        snprintf(buf, sizeof buf, "gpumcd_run_uncertainty_static: %zu voxels exceed the static scratch of %zu voxels "
                 "(GPUMCD_STATIC_MAX_VOXELS); use gpumcd_run_uncertainty", ctx->nvox, kStaticMaxVoxels);
        set_error(ctx, buf);
        return GPUMCD_ERR_INVALID_ARG;
    }
    if (n_batches < 2 || n_batches > n_histories) {
        set_error(ctx, "n_batches must be at least 2 and at most n_histories");
        return GPUMCD_ERR_INVALID_ARG;
    }
    if (ctx->profiling) { // (per-launch event pairs are created while profiling is on: not in a call that allocates nothing)
        set_error(ctx, "gpumcd_run_uncertainty_static: switch profiling off first (gpumcd_set_profiling)");
        return GPUMCD_ERR_INVALID_ARG;
    }
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    double *moments = nullptr;
    int rc = static_moments_address(ctx, &moments);
    if (rc != GPUMCD_OK) return rc;
    rc = begin_run(ctx, n_histories, nullptr, st);
    if (rc != GPUMCD_OK) return rc;
    const size_t nvox = ctx->nvox;
    // the array keeps the last call's contents (any context's): the sums must start at zero
    CK(cudaMemsetAsync(moments, 0, 3 * nvox * sizeof(double), st));
    double *s1 = moments, *sx = s1 + nvox, *sxx = sx + nvox;
    const int grid = static_cast<int>(std::min<size_t>((nvox + kBlock - 1) / kBlock, 148 * 8));
    uint64_t h = ctx->hist_offset;
    for (uint32_t b = 0; b < n_batches; ++b) { // the same batches as gpumcd_run_uncertainty
        const uint64_t m = n_histories / n_batches + (b < n_histories % n_batches ? 1 : 0);
        rc = transport(ctx, h, m, seed, nullptr, nullptr, st);
        if (rc != GPUMCD_OK) return rc;
        { LaunchScope ls(ctx, st, CLS_FINALIZE);
        k_accumulate_batch<<<grid, kBlock, 0, st>>>(ctx->edep, s1, sx, sxx, nvox, 1.0 / static_cast<double>(m)); }
        CK(cudaGetLastError());
        h += m;
    }
    const double h3 = static_cast<double>(ctx->h) * ctx->h * ctx->h;
    { LaunchScope ls(ctx, st, CLS_FINALIZE);
    k_finalize_uncertainty<<<grid, kBlock, 0, st>>>(s1, sx, sxx, make_geom(ctx), nvox, 1.0 / h3,
                                                    1.0 / static_cast<double>(n_histories), static_cast<double>(n_batches),
                                                    dose_out_dev, sigma_out_dev, ctx->edep); }
    CK(cudaGetLastError());
    return GPUMCD_OK;
}

extern "C" int gpumcd_run_trace(gpumcd_ctx *ctx, uint64_t n_histories, uint64_t seed, uint64_t *trace_out_dev,
                                void *cuda_stream)
{
    if (!ctx || !trace_out_dev) return GPUMCD_ERR_INVALID_ARG;
    return run_impl(ctx, n_histories, seed, nullptr, reinterpret_cast<unsigned long long *>(trace_out_dev),
                    static_cast<cudaStream_t>(cuda_stream));
}

extern "C" int gpumcd_get_counters(gpumcd_ctx *ctx, gpumcd_counters *out)
{
    if (!ctx || !out) return GPUMCD_ERR_INVALID_ARG;
    memset(out, 0, sizeof *out);
    if (!ctx->ran) return GPUMCD_OK;
    DevCounters d;
    CK(cudaStreamSynchronize(ctx->last_stream));
    CK(cudaMemcpy(&d, ctx->cnt, sizeof d, cudaMemcpyDeviceToHost));
    out->n_histories = ctx->last_n;
    out->photon_flights = d.photon_flights; out->photon_compton = d.photon_compton;
    out->photon_photo = d.photon_photo; out->photon_pair = d.photon_pair; out->photon_fict = d.photon_fict;
    out->ch_steps = d.ch_steps; out->hard_moller = d.hard_moller; out->hard_brems = d.hard_brems;
    out->hard_fict = d.hard_fict; out->pushes_e = d.pushes_e; out->pushes_g = d.pushes_g;
    out->bank_high_water = ctx->opt.scheduler == 1 ? d.high_water : ctx->high_water;
    out->overflow_count = d.overflow;
    for (int k = 0; k < kEnergySlots; ++k) {
        out->e_incident += d.slot[k].e_inc;
        out->e_dep_cutoff += d.slot[k].e_cut;
        out->e_escaped += d.slot[k].e_esc;
    }
    out->e_pair_rest = static_cast<double>(d.photon_pair) * (2.0 * static_cast<double>(kMe)); // 2 m c^2 per pair event (R6)
    out->e_dep_continuous = d.e_dep_total - out->e_dep_cutoff;
    if (d.overflow) { set_error(ctx, "particle queue overflow: the result is invalid"); return GPUMCD_ERR_BANK_OVERFLOW; }
    return GPUMCD_OK;
}

extern "C" int gpumcd_get_energy_tally(gpumcd_ctx *ctx, double *edep_out_dev)
{
    if (!ctx || !edep_out_dev) return GPUMCD_ERR_INVALID_ARG;
    const int grid = static_cast<int>(std::min<size_t>((ctx->nvox + kBlock - 1) / kBlock, 148 * 8));
    k_export_tally<<<grid, kBlock, 0, ctx->last_stream>>>(ctx->edep, make_geom(ctx), ctx->nvox, edep_out_dev);
    CK(cudaGetLastError());
    return GPUMCD_OK;
}

extern "C" int gpumcd_set_history_offset(gpumcd_ctx *ctx, uint64_t first_history)
{
    if (!ctx) return GPUMCD_ERR_INVALID_ARG;
    ctx->hist_offset = first_history;
    return GPUMCD_OK;
}

extern "C" int gpumcd_release_l2(gpumcd_ctx *ctx)
{
    if (!ctx) return GPUMCD_ERR_INVALID_ARG;
    if (ctx->ran) CK(cudaStreamSynchronize(ctx->last_stream));
    if (ctx->l2_window) CK(cudaCtxResetPersistingL2Cache());
    return GPUMCD_OK;
}

extern "C" int gpumcd_set_profiling(gpumcd_ctx *ctx, int enable)
{
    if (!ctx) return GPUMCD_ERR_INVALID_ARG;
    ctx->profiling = enable != 0;
    return GPUMCD_OK;
}

extern "C" int gpumcd_get_profile(gpumcd_ctx *ctx, gpumcd_profile *out)
{
    if (!ctx || !out) return GPUMCD_ERR_INVALID_ARG;
    if (ctx->ran) CK(cudaStreamSynchronize(ctx->last_stream));
    gpumcd_profile p = ctx->prof;
    for (auto &e : ctx->events) {
        float ms = 0.f;
        CK(cudaEventElapsedTime(&ms, e.a, e.b));
        (&p.ms_source)[e.cls] += ms;
    }
    *out = p;
    return GPUMCD_OK;
}

extern "C" int gpumcd_probe_tally(gpumcd_ctx *ctx, uint64_t n_updates, double *updates_per_second, void *cuda_stream)
{
    if (!ctx || !updates_per_second || n_updates == 0) return GPUMCD_ERR_INVALID_ARG;
    if (!ctx->have_source) { set_error(ctx, "gpumcd_probe_tally called before gpumcd_set_source"); return GPUMCD_ERR_NO_SOURCE; }
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    // the field's footprint on the grid (a pencil beam: a 3 x 3 voxel column)
    const double h = ctx->h;
    double cx = ctx->src.cx, cy = ctx->src.cy, wx = ctx->src.wx, wy = ctx->src.wy;
    if (ctx->src.shape == 2) { // a phase space: its footprint is not known, take the whole face
        cx = 0.5 * ctx->nx * h; cy = 0.5 * ctx->ny * h;
        wx = (ctx->nx - 1) * h; wy = (ctx->ny - 1) * h;
    }
    const int margin = ctx->src.shape == 0 ? 1 : 0;
    int x0 = static_cast<int>(std::floor((cx - 0.5 * wx) / h)) - margin;
    int y0 = static_cast<int>(std::floor((cy - 0.5 * wy) / h)) - margin;
    int x1 = static_cast<int>(std::floor((cx + 0.5 * wx) / h)) + margin;
    int y1 = static_cast<int>(std::floor((cy + 0.5 * wy) / h)) + margin;
    x0 = std::max(x0, 0); y0 = std::max(y0, 0);
    x1 = std::min(x1, ctx->nx - 1); y1 = std::min(y1, ctx->ny - 1);
    const int threads = 512, blocks = 148 * 2;
    const uint64_t per_thread = (n_updates + static_cast<uint64_t>(threads) * blocks - 1) / (static_cast<uint64_t>(threads) * blocks);
    if (per_thread > 0xffffffffull) { set_error(ctx, "n_updates too large"); return GPUMCD_ERR_INVALID_ARG; }
    cudaEvent_t a, b;
    CK(cudaEventCreate(&a)); CK(cudaEventCreate(&b));
    CK(cudaMemsetAsync(ctx->edep, 0, ctx->nvox * sizeof(double), st));
    // once untimed (first touch of the grid), once timed
    const bool fixed = ctx->opt.tally_mode == TALLY_FIXED; // the probe adds what the run adds: fp64 or 64-bit integers
    auto probe = fixed ? k_tally_probe<true> : k_tally_probe<false>;
    const Geom geo = make_geom(ctx);
    probe<<<blocks, threads, 0, st>>>(ctx->edep, geo, x0, y0, x1 - x0 + 1, y1 - y0 + 1,
                                      static_cast<unsigned>(per_thread), 1u);
    CK(cudaEventRecord(a, st));
    probe<<<blocks, threads, 0, st>>>(ctx->edep, geo, x0, y0, x1 - x0 + 1, y1 - y0 + 1,
                                      static_cast<unsigned>(per_thread), 2u);
    CK(cudaEventRecord(b, st));
    CK(cudaGetLastError());
    CK(cudaEventSynchronize(b));
    float ms = 0.f;
    CK(cudaEventElapsedTime(&ms, a, b));
    cudaEventDestroy(a); cudaEventDestroy(b);
    CK(cudaMemsetAsync(ctx->edep, 0, ctx->nvox * sizeof(double), st)); // the tally of the last run is gone
    *updates_per_second = static_cast<double>(per_thread) * threads * blocks / (static_cast<double>(ms) * 1e-3);
    return GPUMCD_OK;
}

extern "C" int gpumcd_selftest_philox(const uint32_t *ctr_key_dev, uint32_t *out_dev, float *uniform_dev, uint64_t n,
                                      void *cuda_stream)
{
    if (!ctr_key_dev || !out_dev) return GPUMCD_ERR_INVALID_ARG;
    if (n == 0) return GPUMCD_OK;
    const unsigned blocks = static_cast<unsigned>(std::min<uint64_t>((n + kBlock - 1) / kBlock, 148 * 8));
    k_philox_selftest<<<blocks, kBlock, 0, static_cast<cudaStream_t>(cuda_stream)>>>(ctr_key_dev, out_dev, uniform_dev, n);
    return cudaGetLastError() == cudaSuccess ? GPUMCD_OK : GPUMCD_ERR_CUDA;
}

extern "C" const char *gpumcd_last_error(gpumcd_ctx *ctx)
{
    return ctx ? ctx->err.c_str() : g_create_error.c_str();
}

extern "C" void gpumcd_destroy(gpumcd_ctx *ctx) { destroy_impl(ctx); }
