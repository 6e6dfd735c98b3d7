// metropolis_common.cuh -- device code shared by the Metropolis translation units (metropolis_kernels.cu: the
// checkerboard half-sweep; sublattice_kernels.cu: the paper's stride-l schedule): Philox4x32-10, the uniform map,
// the uniform-on-S^2 trial and the scalar Metropolis decision.  Everything here is inline and has internal
// linkage per translation unit.
#pragma once
#include "dsmc_internal.cuh"

namespace {


struct RoundKeys {
    uint32_t k[10][2];
};

// Philox4x32-10 (Salmon et al., SC'11) with precomputed round keys
__host__ __device__ __forceinline__ uint4 philox4x32_10(uint4 c, const RoundKeys &rk) {
#pragma unroll
    for (int round = 0; round < 10; ++round) {
        const uint64_t p0 = (uint64_t)0xD2511F53u * c.x;
        const uint64_t p1 = (uint64_t)0xCD9E8D57u * c.z;
        c = make_uint4((uint32_t)(p1 >> 32) ^ c.y ^ rk.k[round][0], (uint32_t)p1,
                       (uint32_t)(p0 >> 32) ^ c.w ^ rk.k[round][1], (uint32_t)p0);
    }
    return c;
}

// 32 bits -> odd multiple of 2^-24 strictly inside (0,1): exact in fp32 (R9)
__device__ __forceinline__ float unit24(uint32_t x) {
    return (float)(2u * (x >> 9) + 1u) * 5.9604644775390625e-8f;
}

// Uniform point on S^2 from two words (R10): z = 2 u0 - 1, azimuth 2 pi u1.
// u1 = m / 2^24 (m odd): quadrant = top two bits of m, f = remaining 22 bits / 2^22 in (0,1);
// sin(pi f / 2) = f P(f^2), cos(pi f / 2) = Q(f^2) (least-squares fits on Chebyshev nodes, fp32
// Horner: max abs error 1.5e-7), then a quarter-turn rotation by sign/swap.
__device__ __forceinline__ void sphere_point(uint32_t x0, uint32_t x1, float &sx, float &sy, float &sz) {
    const uint32_t m0 = 2u * (x0 >> 9) + 1u;
    const float z = (float)m0 * 1.1920928955078125e-7f - 1.0f;  // exact
    const uint32_t m1 = 2u * (x1 >> 9) + 1u;
    const uint32_t quad = m1 >> 22;
    const float f = (float)(m1 & 0x3FFFFFu) * 2.384185791015625e-7f;  // exact
    const float t = f * f;
    float ps = 1.516751217423007e-4f;
    ps = fmaf(ps, t, -4.674150608479977e-3f);
    ps = fmaf(ps, t, 7.968991994857788e-2f);
    ps = fmaf(ps, t, -6.459637880325317e-1f);
    ps = fmaf(ps, t, 1.5707963705062866f);
    const float s1 = ps * f;
    float pc = -2.3824535674066283e-5f;
    pc = fmaf(pc, t, 9.177238680422306e-4f);
    pc = fmaf(pc, t, -2.086268737912178e-2f);
    pc = fmaf(pc, t, 2.536693215370178e-1f);
    pc = fmaf(pc, t, -1.2337005138397217f);
    pc = fmaf(pc, t, 1.0f);
    // quadrant 0: (c, s); 1: (-s, c); 2: (-c, -s); 3: (s, -c)
    const bool swap = quad & 1u;
    const float cb = swap ? s1 : pc, sb = swap ? pc : s1;
    const float cs = __uint_as_float(__float_as_uint(cb) ^ (((quad + 1u) & 2u) << 30));
    const float sn = __uint_as_float(__float_as_uint(sb) ^ ((quad & 2u) << 30));
    const float w = (1.0f - z) * (1.0f + z);  // > 0: |z| <= 1 - 2^-23
    const float rho = w * rsqrtf(w);
    sx = rho * cs;
    sy = rho * sn;
    sz = z;
}

// the step words of the Philox counter: kernel parameters, or the device-resident counter of dsmc_run
__device__ __forceinline__ void step_words(const MetropolisArgs &p, uint32_t &lo, uint32_t &hi) {
    lo = p.step_lo;
    hi = p.step_hi;
    if (p.step_dev) {
        const unsigned long long st = *p.step_dev + p.step_off;
        lo = (uint32_t)(st & 0xFFFFFFFFull);
        hi = (uint32_t)(st >> 32) & 0x7FFFFFFFu;
    }
}

struct Trial {
    float tx, ty, tz, margin;
    bool acc;
};

// the random part of one Metropolis trial: Philox words -> trial spin and ln u.  It depends on the
// counter only (and on the current spin for the Ising move), not on the field.
struct Draw {
    float tx, ty, tz, lnu;
};
__device__ __forceinline__ Draw draw_from_words(const MetropolisArgs &p, uint4 rnd, float sx, float sy, float sz) {
    Draw d;
    if (p.flip) {                                             // Ising move of App. B: complete reversal
        d.tx = -sx, d.ty = -sy, d.tz = -sz;
    } else {
        sphere_point(rnd.x, rnd.y, d.tx, d.ty, d.tz);
    }
    d.lnu = __logf(unit24(rnd.z));
    return d;
}

// the deterministic part: current spin s, neighbour sum nb, frozen field h  (R12-R14)
__device__ __forceinline__ Trial decide_drawn(const MetropolisArgs &p, const Draw &d, float sx, float sy, float sz,
                                              float nx, float ny, float nz, float hx, float hy, float hz, float invT,
                                              float K2, float K4) {
    Trial t;
    t.tx = d.tx, t.ty = d.ty, t.tz = d.tz;
    const float dx = t.tx - sx, dy = t.ty - sy, dz = t.tz - sz;
    const float dz2 = dz * (t.tz + sz);                       // s'_z^2 - s_z^2
    const float z2sum = fmaf(t.tz, t.tz, sz * sz);
    float dE = -p.J * fmaf(dx, nx, fmaf(dy, ny, dz * nz));    // exchange with the 4 neighbours
    dE = fmaf(-dz2, fmaf(K4, z2sum, K2), dE);                 // -K2 d(z^2) - K4 d(z^4)
    float self = fmaf(p.w0xx * dx, dx, fmaf(p.w0yy * dy, dy, p.w0zz * dz * dz));
    self = fmaf(0.5f, self, p.w0xy * dx * dy);
    dE = fmaf(p.g, fmaf(dx, hx, fmaf(dy, hy, fmaf(dz, hz, self))), dE);
    t.margin = fmaf(dE, invT, d.lnu);
    t.acc = t.margin < 0.0f;
    return t;
}

// one Metropolis decision of site n, replica r
__device__ __forceinline__ Trial decide(const MetropolisArgs &p, const RoundKeys &rk, uint32_t n, uint32_t r, float sx,
                                        float sy, float sz, float nx, float ny, float nz, float hx, float hy, float hz,
                                        float invT, float K2, float K4) {
    uint32_t step_lo, step_hi;
    step_words(p, step_lo, step_hi);
    const uint4 rnd = philox4x32_10(make_uint4(n, r, step_lo, step_hi), rk);
    return decide_drawn(p, draw_from_words(p, rnd, sx, sy, sz), sx, sy, sz, nx, ny, nz, hx, hy, hz, invT, K2, K4);
}

inline RoundKeys make_round_keys(uint32_t lo, uint32_t hi) {
    RoundKeys rk;
    for (int i = 0; i < 10; ++i) {
        rk.k[i][0] = lo + (uint32_t)i * 0x9E3779B9u;
        rk.k[i][1] = hi + (uint32_t)i * 0xBB67AE85u;
    }
    return rk;
}

}  // namespace
