// metropolis_pair.cuh -- the Metropolis decision of one replica pair (two replicas of one site at once, packed f32x2
// arithmetic): Philox words -> trial spins and ln u (trial2), dE / T + ln u (margin2).  Shared by the checkerboard
// half-sweep kernel (metropolis_kernels.cu) and by the FFT field's fused row kernel (field_fft.cu), so that both take
// bit-identical decisions from identical inputs (eq. 7; R12-R14, section 5.3).
#pragma once
#include "metropolis_common.cuh"
#include "packed_f32x2.cuh"

namespace {

__device__ __forceinline__ float rsqrt_approx(float x) {
    float r;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
__device__ __forceinline__ float lg2_approx(float x) {
    float r;
    asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}

// word -> y = 1 + (x >> 9) 2^-23 in [1, 2) by writing the mantissa field (no int->float conversion)
__device__ __forceinline__ float mant(uint32_t x) { return __uint_as_float(0x3F800000u | (x >> 9)); }

// Two Metropolis decisions at once (replicas r, r+1 of one site).  Same arithmetic as decide() with
// two differences, both within the parity tolerances:
//   * u = (2k+1) 2^-24 with k = x >> 9: z = 2u0 - 1 = 2 (y - 1.5) + 2^-23 and v = 2u1 - 1 likewise are
//     exact in fp32 (y - 1.5 is a multiple of 2^-23 in [-1/2, 1/2); the fma rounds once to a
//     representable odd multiple of 2^-23), so the trial z carries no rounding error at all;
//   * azimuth phi = 2 pi u1 = pi v + pi.  With S = sin(pi v / 2) = v P(v^2), C = cos(pi v / 2) = Q(v^2)
//     (the polynomials of sphere_point, valid on [-1, 1] by parity):
//       cos phi = -cos(pi v) = (S - C)(S + C),   sin phi = -sin(pi v) = (-2 S) C,
//     no quadrant selects; max abs error 4.5e-7.
struct Trial2 {
    f2 tx, ty, tz, lnu;   // trial spins and ln u of two replicas: functions of the random words only
};
__device__ __forceinline__ Trial2 trial2(uint4 ra, uint4 rb) {
    Trial2 t;
    const f2 c2 = f2_bc(2.0f), cm15 = f2_bc(-1.5f), ulp = f2_bc(1.1920928955078125e-7f);
    const f2 z = f2_fma(c2, f2_add(f2_make(mant(ra.x), mant(rb.x)), cm15), ulp);
    const f2 v = f2_fma(c2, f2_add(f2_make(mant(ra.y), mant(rb.y)), cm15), ulp);
    // u = (y - 1) + 2^-24, exact
    const f2 u = f2_add(f2_add(f2_make(mant(ra.z), mant(rb.z)), f2_bc(-1.0f)), f2_bc(5.9604644775390625e-8f));
    const f2 q = f2_mul(v, v);
    f2 ps = f2_fma(f2_bc(1.516751217423007e-4f), q, f2_bc(-4.674150608479977e-3f));
    ps = f2_fma(ps, q, f2_bc(7.968991994857788e-2f));
    ps = f2_fma(ps, q, f2_bc(-6.459637880325317e-1f));
    ps = f2_fma(ps, q, f2_bc(1.5707963705062866f));
    const f2 S = f2_mul(ps, v);
    f2 C = f2_fma(f2_bc(-2.3824535674066283e-5f), q, f2_bc(9.177238680422306e-4f));
    C = f2_fma(C, q, f2_bc(-2.086268737912178e-2f));
    C = f2_fma(C, q, f2_bc(2.536693215370178e-1f));
    C = f2_fma(C, q, f2_bc(-1.2337005138397217f));
    C = f2_fma(C, q, f2_bc(1.0f));
    const f2 cs = f2_mul(f2_sub(S, C), f2_add(S, C));
    const f2 sn = f2_mul(f2_mul(S, f2_bc(-2.0f)), C);
    const f2 w = f2_mul(f2_sub(f2_bc(1.0f), z), f2_add(z, f2_bc(1.0f)));  // > 0: |z| <= 1 - 2^-23
    float w0, w1;
    f2_split(w, w0, w1);
    const f2 rho = f2_mul(w, f2_make(rsqrt_approx(w0), rsqrt_approx(w1)));
    t.tx = f2_mul(rho, cs);
    t.ty = f2_mul(rho, sn);
    t.tz = z;
    float u0, u1;
    f2_split(u, u0, u1);
    t.lnu = f2_mul(f2_make(lg2_approx(u0), lg2_approx(u1)), f2_bc(0.693147180559945f));
    return t;
}
// margin = dE / T + ln u for the two trials (eq. 7; R12-R14)
__device__ __forceinline__ f2 margin2(const MetropolisArgs &p, const Trial2 &t, f2 sx, f2 sy, f2 sz, f2 nx, f2 ny, f2 nz,
                                      f2 hx, f2 hy, f2 hz, f2 invT, f2 K2, f2 K4) {
    const f2 z = t.tz;
    const f2 dx = f2_sub(t.tx, sx), dy = f2_sub(t.ty, sy), dz = f2_sub(z, sz);
    const f2 dz2 = f2_mul(dz, f2_add(z, sz));                              // s'_z^2 - s_z^2
    const f2 z2sum = f2_fma(z, z, f2_mul(sz, sz));
    f2 dE = f2_mul(f2_fma(dx, nx, f2_fma(dy, ny, f2_mul(dz, nz))), f2_bc(-p.J));
    dE = f2_fma(f2_mul(dz2, f2_bc(-1.0f)), f2_fma(K4, z2sum, K2), dE);     // -K2 d(z^2) - K4 d(z^4)
    // g [ delta.h + (1/2) delta.W(0).delta ] = g delta.(h + W(0) delta / 2)
    const f2 ex = f2_fma(f2_bc(p.w0xy), dy, f2_fma(f2_bc(0.5f * p.w0xx), dx, hx));
    const f2 ey = f2_fma(f2_bc(0.5f * p.w0yy), dy, hy);
    const f2 ez = f2_fma(f2_bc(0.5f * p.w0zz), dz, hz);
    const f2 dip = f2_fma(dx, ex, f2_fma(dy, ey, f2_mul(dz, ez)));
    dE = f2_fma(f2_bc(p.g), dip, dE);
    return f2_fma(dE, invT, t.lnu);
}
__device__ __forceinline__ void ld2(const float4 *ptr, f2 &lo, f2 &hi) {
    const ulonglong2 v = __ldg(reinterpret_cast<const ulonglong2 *>(ptr));
    lo = v.x;
    hi = v.y;
}

}  // namespace
