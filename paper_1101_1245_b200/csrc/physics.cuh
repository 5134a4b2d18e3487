// physics.cuh -- device-side building blocks of the GPUMCD hot path (sm_100a).
//
// Single-precision transport, one particle per thread.  Everything here is
// written from the paper and DESIGN.md; nothing is shared with oracle/.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

namespace gpumcd {

constexpr float kMe = 0.51099895f;       // electron rest energy, MeV
constexpr float kTwoPi = 6.283185307179586f;

// ---------------------------------------------------------------------------------------------
// Random numbers (H9).  Philox4x32-10, counter = (hist_lo, hist_hi, track, ctr), key = seed.
// Replaces the paper's multiply-with-carry generator so that a particle's
// stream depends only on its lineage, never on which thread runs it.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ uint4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                               uint32_t k0, uint32_t k1)
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t lo0 = 0xD2511F53u * c0, hi0 = __umulhi(0xD2511F53u, c0);
        const uint32_t lo1 = 0xCD9E8D57u * c2, hi1 = __umulhi(0xCD9E8D57u, c2);
        c0 = hi1 ^ c1 ^ k0;
        c1 = lo1;
        c2 = hi0 ^ c3 ^ k1;
        c3 = lo0;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    return make_uint4(c0, c1, c2, c3);
}
// The same as ONE out-of-line copy, for the call sites outside the step / flight code (rejection loops, vertices,
// lineage, primaries): a dozen inlined copies of the 75-instruction block made the persistent kernel 90 KB of
// SASS, more than the 32 KB instruction cache of an SM holds when its warps work on different event kinds
// (config 5: `no_instruction` was 17 % of the stall cycles).
__device__ __noinline__ uint4 philox4x32_10_call(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                                 uint32_t k0, uint32_t k1)
{
    return philox4x32_10(c0, c1, c2, c3, k0, k1);
}

// U(w) = ((w >> 9) + 1/2) 2^-23 in (0,1); exact in fp32 (Eq. 1 needs zeta in (0,1], L53).
__device__ __forceinline__ float u01(uint32_t w)
{
    // as 1.m - (1 - 2^-24) = m 2^-23 + 2^-24: exact (an odd multiple of 2^-24 below 1), and without the integer-to-
    // float conversion, which shares the quarter-rate XU pipe with the transcendentals (1-2 % of the run time)
    return __uint_as_float(0x3f800000u | (w >> 9)) - 0.99999994f;
}

// ---------------------------------------------------------------------------------------------
// Math policy.  The transport kernels are issue-bound, so the transcendental and division
// sequences matter.  With GPUMCD_FAST_MATH (default) the step code uses the SFU forms
// (MUFU.LG2 / MUFU.RCP / MUFU.SIN,COS): absolute errors of a few 1e-7, the same size as fp32
// rounding of the quantities they feed.  -DGPUMCD_FAST_MATH=0 selects the IEEE library forms.
// ---------------------------------------------------------------------------------------------
#ifndef GPUMCD_FAST_MATH
#define GPUMCD_FAST_MATH 1
#endif
__device__ __forceinline__ float flog(float x)
{
#if GPUMCD_FAST_MATH
    return __logf(x);
#else
    return logf(x);
#endif
}
__device__ __forceinline__ float fdiv(float a, float b)
{
#if GPUMCD_FAST_MATH
    return __fdividef(a, b);
#else
    return a / b;
#endif
}
// sin and cos of 2*pi*u, u in (0,1)
__device__ __forceinline__ void sincos2pi(float u, float &s, float &c)
{
#if GPUMCD_FAST_MATH
    // keep the SFU argument inside (-pi, pi), where its absolute error is 2^-21.4: u - 1/2 is exact
    __sincosf(kTwoPi * (u - 0.5f), &s, &c);
    s = -s;
    c = -c;
#else
    sincospif(2.0f * u, &s, &c);
#endif
}

// ---------------------------------------------------------------------------------------------
// Tables (G7): grids uniform in ln E (or ln K), linear interpolation.
// ---------------------------------------------------------------------------------------------
struct Grid {
    float x_min, inv_dx;
    int n;
};
struct Interp {
    int i;
    float t;
};
__device__ __forceinline__ Interp locate(const Grid &g, float x)
{
    float f = (x - g.x_min) * g.inv_dx;
    f = fminf(fmaxf(f, 0.0f), static_cast<float>(g.n - 1));
    int i = min(static_cast<int>(f), g.n - 2);
    return Interp{i, f - static_cast<float>(i)};
}
__device__ __forceinline__ float interp(const float *__restrict__ col, Interp it)
{
    const float a = col[it.i], b = col[it.i + 1];
    return fmaf(it.t, b - a, a);
}

// ---------------------------------------------------------------------------------------------
// Particle state in registers.  Position = voxel index (ix,iy,iz) + fractional offset in [0,1)
// in units of the voxel size: voxel lookup needs no division and boundary distances need no
// subtraction of large numbers.
// ---------------------------------------------------------------------------------------------
struct Particle {
    float fx, fy, fz;
    int ix, iy, iz;
    float u, v, w;
    float E;
    uint32_t hist, track, ctr;
};

__device__ __forceinline__ uint32_t pack_voxel(int ix, int iy, int iz)
{
    return static_cast<uint32_t>(ix) | (static_cast<uint32_t>(iy) << 10) | (static_cast<uint32_t>(iz) << 20);
}

// move by t voxel sizes along the direction and renormalise (cell, frac)
__device__ __forceinline__ void advance(Particle &p, float t)
{
    p.fx = fmaf(t, p.u, p.fx);
    p.fy = fmaf(t, p.v, p.fy);
    p.fz = fmaf(t, p.w, p.fz);
    const float cx = floorf(p.fx), cy = floorf(p.fy), cz = floorf(p.fz);
    p.ix += static_cast<int>(cx);
    p.iy += static_cast<int>(cy);
    p.iz += static_cast<int>(cz);
    p.fx -= cx;
    p.fy -= cy;
    p.fz -= cz;
}

// Rotate direction d by polar angle (cost, sint) and azimuth (cp, sp) about itself (R-P8).
__device__ __forceinline__ void rotate(float u, float v, float w, float cost, float sint, float cp, float sp,
                                       float &ou, float &ov, float &ow)
{
    const float r2 = fmaf(u, u, v * v);
    float a, b, c;
    if (r2 < 1e-10f) {
        a = sint * cp;
        b = sint * sp;
        c = (w >= 0.0f) ? cost : -cost;
    } else {
        const float ir = rsqrtf(r2);
        const float r = r2 * ir;
        a = fmaf(u, cost, sint * (u * w * cp - v * sp) * ir);
        b = fmaf(v, cost, sint * (v * w * cp + u * sp) * ir);
        c = fmaf(w, cost, -r * sint * cp);
    }
    const float inv = rsqrtf(fmaf(a, a, fmaf(b, b, c * c)));
    ou = a * inv;
    ov = b * inv;
    ow = c * inv;
}

struct Rng {
    uint32_t k0, k1, hist_hi;
};
// the particle's next block; HOT: the inlined copy (step and flight code), else the shared out-of-line one
template <bool HOT = false>
__device__ __forceinline__ uint4 draw(const Rng &g, Particle &p)
{
    const uint4 r = HOT ? philox4x32_10(p.hist, g.hist_hi, p.track, p.ctr, g.k0, g.k1)
                        : philox4x32_10_call(p.hist, g.hist_hi, p.track, p.ctr, g.k0, g.k1);
    p.ctr += 1u;
    return r;
}
// track ids of the children born at the parent's current counter
__device__ __forceinline__ uint4 lineage(const Rng &g, const Particle &p)
{
    return philox4x32_10_call(p.hist, g.hist_hi, p.track, p.ctr | 0x80000000u, g.k0, g.k1);
}

// ---------------------------------------------------------------------------------------------
// Samplers: one Philox block per trial.
// ---------------------------------------------------------------------------------------------

// Klein-Nishina.  Returns eps = E'/E; t = 1 - cos(theta); uphi in (0,1).
__device__ __forceinline__ void sample_compton(const Rng &g, Particle &p, float &eps, float &t, float &uphi)
{
    const float k = p.E * (1.0f / kMe);
    const float eps0 = 1.0f / fmaf(2.0f, k, 1.0f);
    const float a1 = flog(fmaf(2.0f, k, 1.0f)); // (k >= 0.02, the photon cutoff: 1 + 2k keeps all the bits that matter)
    const float one_m_e02 = (1.0f - eps0) * (1.0f + eps0);
    const float a2 = 0.5f * one_m_e02;
    const float pa = a1 / (a1 + a2);
    for (;;) {
        const uint4 v = draw(g, p);
        const float u1 = u01(v.y);
        float e, one_m_e;
        if (u01(v.x) < pa) {
            const float x = -a1 * u1;
            e = expf(x);
            // 1 - e^x without expm1f (a long sequence run by a third of the lanes of a Compton batch: 2 % of the run):
            // the series below |x| = 1/8 (relative error < 1e-7), else the difference (e < 0.89)
            const float ser = -x * fmaf(x, fmaf(x, fmaf(x, fmaf(x, 1.0f / 120.0f, 1.0f / 24.0f), 1.0f / 6.0f), 0.5f), 1.0f);
            one_m_e = x > -0.125f ? ser : 1.0f - e;
        } else {
            e = sqrtf(fmaf(one_m_e02, u1, eps0 * eps0));
            one_m_e = one_m_e02 * (1.0f - u1) / (1.0f + e);
        }
        const float tt = one_m_e / (k * e);
        const float gg = 1.0f - e * tt * (2.0f - tt) / fmaf(e, e, 1.0f);
        if (u01(v.z) <= gg) {
            eps = e;
            t = tt;
            uphi = u01(v.w);
            return;
        }
    }
}

// Sauter photo-electron angle.  Returns nu = 1 - cos(theta).
__device__ __forceinline__ void sample_sauter(const Rng &g, Particle &p, float T, float &nu, float &uphi)
{
    const float gam = 1.0f + T * (1.0f / kMe);
    const float beta = sqrtf(T * (T + 2.0f * kMe)) / (T + kMe);
    const float A = 1.0f / beta - 1.0f;
    const float B = 0.5f * beta * gam * (gam - 1.0f) * (gam - 2.0f);
    const float g0 = 2.0f * (1.0f / A + B);
    for (;;) {
        const uint4 v = draw(g, p);
        const float q = sqrtf(u01(v.x)) * 2.0f / (A + 2.0f);
        const float n = q * A / (1.0f - q);
        if (u01(v.y) * g0 <= (2.0f - n) * (1.0f / (A + n) + B)) {
            nu = n;
            uphi = u01(v.z);
            return;
        }
    }
}

// cos and sin of the pair-electron polar angle, density ~ (1 - beta cos)^-2
__device__ __forceinline__ void pair_angle(float T, float ur, float &c, float &s)
{
    const float Et = T + kMe;
    const float beta = sqrtf(T * (T + 2.0f * kMe)) / Et;
    const float x = 2.0f * ur - 1.0f;
    const float den = fmaf(beta, x, 1.0f);
    c = (x + beta) / den;
    // 1 - c = (1 - beta)(1 - x)/den with 1 - beta = (m/E)^2/(1 + beta): no cancellation
    const float omb = (kMe / Et) * (kMe / Et) / (1.0f + beta);
    const float omc = omb * (1.0f - x) / den;
    s = sqrtf(fmaxf(omc * (1.0f + c), 0.0f));
}

} // namespace gpumcd
