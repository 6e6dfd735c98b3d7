// metropolis_kernels.cu -- a2: fused checkerboard Metropolis half-sweep, and a4: spin init.
// Philox4x32-10 trial + exchange + anisotropy + frozen-field dipole dE + accept, all in registers
// (PAPER.md:60-72 eq. 7, :98, :102-118).  The kernel is co-limited by HBM bandwidth (48 B per
// update) and instruction issue, so the per-update instruction count is kept near 130:
//   * one thread updates 4 consecutive replicas of one site: every global access is a 128-bit
//     load/store and the index arithmetic is shared by 4 updates;
//   * Philox round keys are precomputed on the host (kernel parameters = constant bank);
//   * the azimuth 2 pi u1 is reduced to a quadrant exactly in integer arithmetic and sin/cos come
//     from two short polynomials (abs error 1.5e-7); sqrt and log use the MUFU units.
#include "dsmc_internal.cuh"
#include "packed_f32x2.cuh"
#include <algorithm>

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

// R % 4 == 0: one thread = one active site x 4 consecutive replicas (two packed pairs); grid.y =
// lattice row.  All 18 128-bit loads are issued first; the four Philox chains and the trial spins
// do not depend on them and run while they are in flight.  HOOKS = parity outputs requested.
// FLIP: 0 = uniform-sphere trial, 1 = Ising reversal (App. B), 2 = decided at run time from p.flip (parity-hook
// variant only: a run-time branch here splits the block the scheduler interleaves the two pairs in, +5 %)
template <bool HOOKS, bool DEVSTEP, int FLIP>
__global__ void __launch_bounds__(128, 7) metropolis4_kernel(const MetropolisArgs p, const RoundKeys rk) {
    const int Lh = p.L >> 1, RQ = p.R >> 2;
    const int y = blockIdx.y;
    const uint32_t row4 = (uint32_t)(Lh * RQ);
    const uint32_t e = blockIdx.x * blockDim.x + threadIdx.x;   // (i, replica quad) within the row
    if (e >= row4) return;
    const int i = p.rq_shift >= 0 ? (int)(e >> p.rq_shift) : (int)(e / (uint32_t)RQ);
    const int rq = (int)e - i * RQ;
    const int par = (y + p.colour) & 1;
    const size_t plane4 = ((size_t)p.L * Lh * p.R) >> 2;      // float4 per [a][r] plane
    const int yn = (y + 1 == p.L) ? 0 : y + 1, ys = (y == 0) ? p.L - 1 : y - 1;

    // Addresses = three per-thread pointers (S + e, H + e, S + e1) plus offsets that depend only on
    // blockIdx and the parameters (uniform registers).  The four neighbours have the other colour:
    // rows y+-1 at the same in-row index i (offset e), row y at i (e) and i+-1 (e1).
    const int i1 = par ? (i + 1 == Lh ? 0 : i + 1) : (i == 0 ? Lh - 1 : i - 1);
    const uint32_t e1 = (uint32_t)(i1 * RQ + rq);
    float4 *const Se = reinterpret_cast<float4 *>(p.S) + e;
    const float4 *const He = reinterpret_cast<const float4 *>(p.H) + e;
    const float4 *const Se1 = reinterpret_cast<const float4 *>(p.S) + e1;
    const size_t u_own = (size_t)p.colour * 3 * plane4 + (size_t)y * row4;
    const size_t u_oth = (size_t)(1 - p.colour) * 3 * plane4;
    const size_t u_o0 = u_oth + (size_t)y * row4, u_on = u_oth + (size_t)yn * row4, u_os = u_oth + (size_t)ys * row4;
    float4 *own = Se + u_own;
    const float4 *hf = He + u_own, *o0 = Se + u_o0, *o1 = Se1 + u_o0, *on = Se + u_on, *os = Se + u_os;

    f2 s[3][2], h[3][2], nb[3][2];
    {
        f2 a[3][2], b[3][2], c[3][2], d[3][2];
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            ld2(own + k * plane4, s[k][0], s[k][1]);
            ld2(hf + k * plane4, h[k][0], h[k][1]);
            ld2(o0 + k * plane4, a[k][0], a[k][1]);
            ld2(o1 + k * plane4, b[k][0], b[k][1]);
            ld2(on + k * plane4, c[k][0], c[k][1]);
            ld2(os + k * plane4, d[k][0], d[k][1]);
        }
#pragma unroll
        for (int k = 0; k < 3; ++k)
#pragma unroll
            for (int j = 0; j < 2; ++j) nb[k][j] = f2_add(f2_add(a[k][j], b[k][j]), f2_add(c[k][j], d[k][j]));
    }
    f2 invT[2], K2[2], K4[2];
    ld2(reinterpret_cast<const float4 *>(p.invT) + rq, invT[0], invT[1]);
    ld2(reinterpret_cast<const float4 *>(p.K2) + rq, K2[0], K2[1]);
    ld2(reinterpret_cast<const float4 *>(p.K4) + rq, K4[0], K4[1]);

    const uint32_t n = (uint32_t)(y * p.L + 2 * i + par);
    const uint32_t r0 = 4u * (uint32_t)rq;
    uint32_t step_lo = p.step_lo, step_hi = p.step_hi;
    if (DEVSTEP) step_words(p, step_lo, step_hi);
    uint4 rnd[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) rnd[k] = philox4x32_10(make_uint4(n, r0 + p.r_off + k, step_lo, step_hi), rk);

    bool any = false;
    float mg[4];
#pragma unroll
    for (int j = 0; j < 2; ++j) {
        Trial2 tr = trial2(rnd[2 * j], rnd[2 * j + 1]);
        if (FLIP == 1 || (FLIP == 2 && p.flip)) {             // Ising move of App. B: complete reversal
            tr.tx = f2_mul(s[0][j], f2_bc(-1.0f));
            tr.ty = f2_mul(s[1][j], f2_bc(-1.0f));
            tr.tz = f2_mul(s[2][j], f2_bc(-1.0f));
        }
        const f2 margin = margin2(p, tr, s[0][j], s[1][j], s[2][j], nb[0][j], nb[1][j], nb[2][j], h[0][j], h[1][j],
                                  h[2][j], invT[j], K2[j], K4[j]);
        float m0, m1, a0, a1, b0, b1;
        f2_split(margin, m0, m1);
        const bool acc0 = m0 < 0.0f, acc1 = m1 < 0.0f;
        const f2 tv[3] = {tr.tx, tr.ty, tr.tz};
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            f2_split(tv[k], a0, a1);
            f2_split(s[k][j], b0, b1);
            s[k][j] = f2_make(acc0 ? a0 : b0, acc1 ? a1 : b1);
        }
        any |= acc0 | acc1;
        mg[2 * j] = m0;
        mg[2 * j + 1] = m1;
    }
    if (any) {
#pragma unroll
        for (int k = 0; k < 3; ++k)
            *reinterpret_cast<ulonglong2 *>(own + k * plane4) = make_ulonglong2(s[k][0], s[k][1]);
    }
    if (HOOKS) {
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const size_t o = (size_t)(r0 + k) * p.L * p.L + n;
            if (p.accept_out) p.accept_out[o] = mg[k] < 0.0f ? 1 : 0;
            if (p.margin_out) p.margin_out[o] = mg[k];
        }
    }
}

// any R: one thread per (active site, replica), replica fastest
__global__ void __launch_bounds__(256) metropolis1_kernel(const MetropolisArgs p, const RoundKeys rk) {
    const int Lh = p.L >> 1;
    const size_t Nh = (size_t)p.L * Lh;
    const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= Nh * (size_t)p.R) return;
    const int r = (int)(t % (size_t)p.R);
    const int a = (int)(t / (size_t)p.R);
    const int y = a / Lh, i = a - y * Lh;
    const int par = (y + p.colour) & 1;
    const size_t plane = Nh * (size_t)p.R;
    float *own = p.S + (size_t)p.colour * 3 * plane + (size_t)a * p.R + r;
    const float *oth = p.S + (size_t)(1 - p.colour) * 3 * plane + r;
    const float *hf = p.H + (size_t)p.colour * 3 * plane + (size_t)a * p.R + r;
    const int ie = par ? (i + 1 == Lh ? 0 : i + 1) : i;
    const int iw = par ? i : (i == 0 ? Lh - 1 : i - 1);
    const int yn = (y + 1 == p.L) ? 0 : y + 1, ys = (y == 0) ? p.L - 1 : y - 1;
    const size_t ae = ((size_t)y * Lh + ie) * p.R, aw = ((size_t)y * Lh + iw) * p.R;
    const size_t an = ((size_t)yn * Lh + i) * p.R, as = ((size_t)ys * Lh + i) * p.R;
    const float sx = own[0], sy = own[plane], sz = own[2 * plane];
    const float nx = (oth[ae] + oth[aw]) + (oth[an] + oth[as]);
    const float ny = (oth[plane + ae] + oth[plane + aw]) + (oth[plane + an] + oth[plane + as]);
    const float nz = (oth[2 * plane + ae] + oth[2 * plane + aw]) + (oth[2 * plane + an] + oth[2 * plane + as]);
    const uint32_t n = (uint32_t)(y * p.L + 2 * i + par);
    const Trial tr = decide(p, rk, n, (uint32_t)r + p.r_off, sx, sy, sz, nx, ny, nz, hf[0], hf[plane], hf[2 * plane], p.invT[r],
                            p.K2[r], p.K4[r]);
    if (tr.acc) {
        own[0] = tr.tx;
        own[plane] = tr.ty;
        own[2 * plane] = tr.tz;
    }
    if (p.accept_out) p.accept_out[(size_t)r * 2 * Nh + n] = tr.acc ? 1 : 0;
    if (p.margin_out) p.margin_out[(size_t)r * 2 * Nh + n] = tr.margin;
}

// ---------------------------------------------------------------------------------------------
// The paper's own schedule (section 3.1, App. A): one pass updates the n = (L/l)^2 sites
// (ox + a l, oy + b l) of a stride-l sub-lattice simultaneously, every one of them seeing the dipole
// field of the state at entry to the pass.  Two launches per pass, as the paper's dipole kernel and
// flip kernel (a grid-wide barrier separates "all fields computed" from "first spin replaced"):
//   sublattice_field_kernel: one CTA per update site and 32 replicas.  The paper's "P threads per
//     update site, each a strip of the lattice" becomes 8 warps that each sum the source rows
//     y = g, g + 8, ... for 32 replicas (lanes = replicas, so the spin loads are coalesced and the four
//     W values of a source are a warp-wide broadcast), row sums first (two-level fp32 accumulation),
//     then a fixed-order shared-memory reduction; h goes to the site's slot of the field array H.
//   sublattice_flip_kernel: one thread per (update site, replica): exchange, anisotropy, self-term,
//     frozen-field dE and the decision (the paper's exchange and flip kernels fused).
__device__ __forceinline__ size_t site_index(int x, int y, int Lh, int R, size_t plane, int &q) {
    q = (x + y) & 1;
    return (size_t)q * 3 * plane + ((size_t)y * Lh + (x >> 1)) * R;
}

// grid (n sites, replica chunks of 32, KS source slabs); part[ks][site][c][r] receives the slab's sum
// offset of pass `pass` (R21): words x0, x1 of Philox4x32-10(seed; 0xFFFFFFFF, 0xFFFFFFFF, pass) mod l
__host__ __device__ __forceinline__ void pass_offset(const RoundKeys &rk, unsigned long long pass, int l, int &ox,
                                                     int &oy) {
    const uint4 x = philox4x32_10(make_uint4(0xFFFFFFFFu, 0xFFFFFFFFu, (uint32_t)(pass & 0xFFFFFFFFull),
                                             (uint32_t)(pass >> 32) & 0x7FFFFFFFu), rk);
    ox = (int)(x.x % (uint32_t)l);
    oy = (int)(x.y % (uint32_t)l);
}

// pass_dev (nullable): the pass counter on the device; the offset is then recomputed here, so that a
// captured graph of one pass can be replayed (dsmc_sublattice_run)
__global__ void __launch_bounds__(256) sublattice_field_kernel(const float *__restrict__ S, float *__restrict__ part_out,
                                                               const float *__restrict__ Wc, int L, int R, int l,
                                                               int ox, int oy, int rows_per_slab, int segs,
                                                               const unsigned long long *__restrict__ pass_dev,
                                                               const RoundKeys rk) {
    if (pass_dev) pass_offset(rk, *pass_dev, l, ox, oy);
    __shared__ float part[8][3][32];
    const int Lh = L >> 1;
    const size_t N = (size_t)L * L, plane = (size_t)L * Lh * R;
    const int nl = L / l;
    const int xt = ox + l * (int)(blockIdx.x % nl), yt = oy + l * (int)(blockIdx.x / nl);
    const int lane = threadIdx.x & 31, grp = threadIdx.x >> 5;
    const int r = blockIdx.y * 32 + lane;
    const int rr = r < R ? r : R - 1;                          // idle lanes load a valid replica
    const int y0 = blockIdx.z * rows_per_slab, y1 = min(L, y0 + rows_per_slab);
    const int iseg = Lh / segs;                                // in-row indices per work item
    float hx = 0.0f, hy = 0.0f, hz = 0.0f;
    for (int item = grp; item < (y1 - y0) * segs; item += 8) { // a warp takes (source row, row segment) items
        const int ys = y0 + item / segs, i0 = (item % segs) * iseg;
        int ry = ys - yt;
        ry += ry < 0 ? L : 0;
        const float *Wrow = Wc + (size_t)ry * L;
        // sources of row ys in internal order: colour q, in-row index i  ->  x = 2 i + ((ys + q) & 1)
        float ax = 0.0f, ay = 0.0f, az = 0.0f;
#pragma unroll
        for (int q = 0; q < 2; ++q) {
            const float *row = S + (size_t)q * 3 * plane + ((size_t)ys * Lh + i0) * R + rr;
            const int x0 = 2 * i0 + ((ys + q) & 1);
#pragma unroll 4
            for (int i = 0; i < iseg; ++i) {
                int rx = 2 * i + x0 - xt;
                rx += rx < 0 ? L : 0;
                const float sx = row[(size_t)i * R], sy = row[plane + (size_t)i * R], sz = row[2 * plane + (size_t)i * R];
                const float wxx = __ldg(Wrow + rx), wxy = __ldg(Wrow + N + rx), wyy = __ldg(Wrow + 2 * N + rx),
                            wzz = __ldg(Wrow + 3 * N + rx);
                ax = fmaf(wxx, sx, fmaf(wxy, sy, ax));
                ay = fmaf(wxy, sx, fmaf(wyy, sy, ay));
                az = fmaf(wzz, sz, az);
            }
        }
        hx += ax;                                              // item sums first: two-level fp32 accumulation
        hy += ay;
        hz += az;
    }
    part[grp][0][lane] = hx;
    part[grp][1][lane] = hy;
    part[grp][2][lane] = hz;
    __syncthreads();
    if (grp != 0 || r >= R) return;
    hx = hy = hz = 0.0f;
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        hx += part[k][0][lane];
        hy += part[k][1][lane];
        hz += part[k][2][lane];
    }
    float *dst = part_out + (((size_t)blockIdx.z * gridDim.x + blockIdx.x) * 3) * R + r;
    dst[0] = hx;
    dst[R] = hy;
    dst[2 * R] = hz;
}

__global__ void __launch_bounds__(128) sublattice_flip_kernel(const MetropolisArgs p, const RoundKeys rk,
                                                              const float *__restrict__ part, int KS, int l, int ox,
                                                              int oy) {
    if (p.step_dev) pass_offset(rk, *p.step_dev + p.step_off, l, ox, oy);
    const int L = p.L, Lh = L >> 1, R = p.R;
    const size_t N = (size_t)L * L, plane = (size_t)L * Lh * R;
    const int nl = L / l;
    const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= (size_t)nl * nl * R) return;
    const int r = (int)(t % (size_t)R), k = (int)(t / (size_t)R);
    const int xt = ox + l * (k % nl), yt = oy + l * (k / nl);
    int q;
    const size_t at = site_index(xt, yt, Lh, R, plane, q) + r;
    float *own = p.S + at;
    float hx = 0.0f, hy = 0.0f, hz = 0.0f;                     // slab partials in fixed order
    if (KS == 0) {                                             // the field array holds h (FFT route)
        hx = p.H[at];
        hy = p.H[at + plane];
        hz = p.H[at + 2 * plane];
    }
#pragma unroll 8
    for (int ks = 0; ks < KS; ++ks) {                          // unrolled: the loads of 8 slabs are in flight together
        const float *ph = part + (((size_t)ks * nl * nl + k) * 3) * R + r;
        hx += __ldg(ph);
        hy += __ldg(ph + R);
        hz += __ldg(ph + 2 * R);
    }
    const int xe = xt + 1 == L ? 0 : xt + 1, xw = xt == 0 ? L - 1 : xt - 1;
    const int yn = yt + 1 == L ? 0 : yt + 1, ys = yt == 0 ? L - 1 : yt - 1;
    const float *ne = p.S + site_index(xe, yt, Lh, R, plane, q) + r, *nw = p.S + site_index(xw, yt, Lh, R, plane, q) + r;
    const float *nn = p.S + site_index(xt, yn, Lh, R, plane, q) + r, *ns = p.S + site_index(xt, ys, Lh, R, plane, q) + r;
    const float sx = own[0], sy = own[plane], sz = own[2 * plane];
    const float nx = (ne[0] + nw[0]) + (nn[0] + ns[0]);
    const float ny = (ne[plane] + nw[plane]) + (nn[plane] + ns[plane]);
    const float nz = (ne[2 * plane] + nw[2 * plane]) + (nn[2 * plane] + ns[2 * plane]);
    const uint32_t n = (uint32_t)(yt * L + xt);
    const Trial tr = decide(p, rk, n, (uint32_t)r + p.r_off, sx, sy, sz, nx, ny, nz, hx, hy, hz, p.invT[r], p.K2[r], p.K4[r]);
    if (tr.acc) {
        own[0] = tr.tx;
        own[plane] = tr.ty;
        own[2 * plane] = tr.tz;
    }
    if (p.accept_out) p.accept_out[(size_t)r * N + n] = tr.acc ? 1 : 0;
    if (p.margin_out) p.margin_out[(size_t)r * N + n] = tr.margin;
}

// ---------------------------------------------------------------------------------------------
// The same schedule with the lattice resident in shared memory (sublattice_resident_kernel).
// One pass is tiny (n = 4 update sites at the paper's L = 64, l = 32: 4 x 4096 x 5 FMAs per replica) and
// consecutive passes depend on one another, so a launch per pass leaves the run bound by launch
// latency.  Here one CTA owns two replicas for the WHOLE run of passes: their spins (24 N bytes)
// and W (16 N bytes) live in shared memory, a pass costs two __syncthreads and no global access, and
// the R/2 CTAs run side by side on their own SMs.
//   * 8 summing warps.  For L/l = NL the n = NL^2 update sites are the translates of the offset by
//     multiples of l, so the sources are taken in cosets {c + (a l, b l)} of the same n translations: the
//     n x n (source, target) pairs of a coset need only n distinct W entries, rho = c - offset + (u l, v l).
//     Per coset (NL = 2): 4 LDS.128 of W + 12 LDS.64 of spins feed 80 FFMA2 (two replicas packed, the W
//     value as broadcast operand) -- 1 byte of shared-memory traffic per FMA, which balances the FMA pipe.
//   * per-thread sums of a few cosets first, then a fixed-order reduction (two-level fp32 accumulation,
//     deterministic): a halving exchange over the warp (each step trades half of the values for the
//     partner's partial sums of the other half: 18 packed shuffles instead of 60), then 8 warp partials.
//   * one extra warp draws while the others sum: lanes < 2n run Philox for (site, replica, pass) and the
//     trial spin, lane 31 runs the same Philox code on the offset counter of the NEXT pass (no divergence),
//     so after the barrier only the 8-term sums, dE and the store of an accepted spin remain.
// Needs L/l in {1, 2} and 40 N bytes + partials within the 227 KB of one CTA (L <= 74).
#ifndef DSMC_RES_WARPS
#define DSMC_RES_WARPS 8
#endif
constexpr int kResSumWarps = DSMC_RES_WARPS;
constexpr int kResThreads = 32 * (kResSumWarps + 1);

__host__ __device__ constexpr size_t resident_smem_bytes(int L, int NL) {
    return (size_t)40 * L * L + 16 + sizeof(f2) * kResSumWarps * NL * NL * 3 + 64;
}

// Reduction helpers for values held as packed pairs.  halve_exchange: lanes with the mask bit clear keep
// v[0 .. V/2) and receive the partner's partial sums of them, the others keep v[V/2 .. V) (moved to
// v[0 .. V/2)); butterfly_sum: plain xor butterfly over masks first, first/2, ..., 1.
template <int V>
__device__ __forceinline__ void halve_exchange(f2 *v, int lane, int mask) {
    const bool upper = lane & mask;
#pragma unroll
    for (int i = 0; i < V / 2; ++i) {
        const f2 keep = upper ? v[i + V / 2] : v[i], send = upper ? v[i] : v[i + V / 2];
        v[i] = f2_add(keep, __shfl_xor_sync(0xFFFFFFFFu, send, mask));
    }
}
template <int V>
__device__ __forceinline__ void butterfly_sum(f2 *v, int first) {
#pragma unroll
    for (int mask = first; mask >= 1; mask >>= 1)
#pragma unroll
        for (int i = 0; i < V; ++i) v[i] = f2_add(v[i], __shfl_xor_sync(0xFFFFFFFFu, v[i], mask));
}

template <int NL, int CPT, int LC>
__global__ void __launch_bounds__(kResThreads, 1) sublattice_resident_kernel(const MetropolisArgs p, const RoundKeys rk,
                                                                             const float *__restrict__ Wc, int l_arg,
                                                                             unsigned long long first_pass,
                                                                             unsigned n_passes) {
    constexpr int NN = NL * NL;
    extern __shared__ __align__(16) unsigned char rsm[];
    // LC > 0: lattice size (and with it l = L / NL) known at compile time, index arithmetic in shifts
    const int L = LC > 0 ? LC : p.L, l = LC > 0 ? LC / NL : l_arg, Lh = L >> 1, R = p.R, N = L * L;
    float4 *Wsm = reinterpret_cast<float4 *>(rsm);                     // [N + 1]  (xx, xy, yy, zz) at rho = ry L + rx; [N] = 0
    f2 *Ssm = reinterpret_cast<f2 *>(rsm + (size_t)16 * (N + 1));      // [N][3]  replicas (r0, r1) of site n = y L + x
    float *Sf = reinterpret_cast<float *>(Ssm);                        // the same as [N][3][2] floats
    f2 *part = Ssm + 3 * (size_t)N;                                    // [warp][target][c]
    int *off = reinterpret_cast<int *>(part + kResSumWarps * NN * 3);  // [2][2]: offsets of this and the next pass
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int r0 = 2 * blockIdx.x, r1 = min(r0 + 1, R - 1);            // odd R: the last CTA carries its replica twice
    const size_t plane = (size_t)L * Lh * R;

    for (int n = tid; n < N; n += kResThreads) {
        Wsm[n] = make_float4(__ldg(Wc + n), __ldg(Wc + (size_t)N + n), __ldg(Wc + 2 * (size_t)N + n),
                             __ldg(Wc + 3 * (size_t)N + n));
        const int x = n % L, y = n / L;
        int q;
        const float *src = p.S + site_index(x, y, Lh, R, plane, q);
        Ssm[3 * n] = f2_make(src[r0], src[r1]);
        Ssm[3 * n + 1] = f2_make(src[plane + r0], src[plane + r1]);
        Ssm[3 * n + 2] = f2_make(src[2 * plane + r0], src[2 * plane + r1]);
    }
    if (tid == 0) {
        Wsm[N] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
        pass_offset(rk, first_pass, l, off[0], off[1]);
    }
    __syncthreads();

    // the drawing warp's lanes: update site k = lane >> 1, replica half rb = lane & 1
    const bool flipper = warp == kResSumWarps && lane < 2 * NN;
    const int fk = lane >> 1, rb = lane & 1, fr = rb ? r1 : r0;
    float invT = 0.0f, K2 = 0.0f, K4 = 0.0f;
    if (flipper) invT = p.invT[fr], K2 = p.K2[fr], K4 = p.K4[fr];
    MetropolisArgs q = p;
    q.step_dev = nullptr;
    const int cy0 = tid / l, cx0 = tid - cy0 * l;                      // this thread's first coset and the stride to the next
    const int step_y = (32 * kResSumWarps) / l, step_x = 32 * kResSumWarps - step_y * l;

    for (unsigned it = 0; it < n_passes; ++it) {
        const unsigned long long pass = first_pass + it;
        const int cur = (int)(it & 1u);
        const int ox = off[2 * cur], oy = off[2 * cur + 1];
        Draw dr;
        float sx = 0.0f, sy = 0.0f, sz = 0.0f, nx = 0.0f, ny = 0.0f, nz = 0.0f;
        int nt = 0;
        if (warp < kResSumWarps) {
            f2 acc[NN][3];
#pragma unroll
            for (int k = 0; k < NN; ++k) acc[k][0] = acc[k][1] = acc[k][2] = f2_bc(0.0f);
            // UN cosets per trip, all their loads issued before the first FMA.  Measured (us per pass at L = 64,
            // l = 32 / l = 64, run-time trip count): NL = 2 with UN = 1: 1.66, UN = 2: 1.70; NL = 1 with UN = 4: 1.36,
            // UN = 8: 1.29.  With the trip count (CPT) and the lattice size (LC) as template parameters: 1.46 / 1.10.
            constexpr int UN = NL == 2 ? 1 : 8;
            // CPT > 0: the trip count is a compile-time constant and the loop unrolls, so the coset coordinates and
            // spin addresses become invariants of the pass loop
            constexpr int UNR = CPT > 0 ? CPT : 1;
            const int ntrip = CPT > 0 ? CPT : (l * l + UN * 32 * kResSumWarps - 1) / (UN * 32 * kResSumWarps);
            int cx = cx0, cy = cy0;                            // coset c = tid, tid + 256, ...: coordinates stepped, not divided
#pragma unroll UNR
            for (int trip = 0; trip < ntrip; ++trip) {
                const int c = tid + trip * UN * 32 * kResSumWarps;
                float4 w[UN][NL][NL];
                f2 sp[UN][NL][NL][3];
#pragma unroll
                for (int j = 0; j < UN; ++j) {
                    if (cx >= l) cx -= l, ++cy;
                    // past the last coset: W entry N (zeros) and site 0, so the trip contributes exact zeros
                    const bool valid = c + j * 32 * kResSumWarps < l * l;
                    int dx[NL], dy[NL];
                    dx[0] = cx - ox + (cx < ox ? L : 0);
                    dy[0] = cy - oy + (cy < oy ? L : 0);
#pragma unroll
                    for (int u = 1; u < NL; ++u) {
                        dx[u] = dx[u - 1] + l - (dx[u - 1] + l >= L ? L : 0);
                        dy[u] = dy[u - 1] + l - (dy[u - 1] + l >= L ? L : 0);
                    }
                    const int m0 = valid ? cy * L + cx : 0;
#pragma unroll
                    for (int v = 0; v < NL; ++v)
#pragma unroll
                        for (int u = 0; u < NL; ++u) {
                            w[j][v][u] = Wsm[valid ? dy[v] * L + dx[u] : N];
                            const f2 *src = Ssm + 3 * (m0 + v * l * L + u * l);
                            sp[j][v][u][0] = src[0], sp[j][v][u][1] = src[1], sp[j][v][u][2] = src[2];
                        }
                    cx += step_x, cy += step_y;
                }
#pragma unroll
                for (int j = 0; j < UN; ++j)
#pragma unroll
                    for (int k = 0; k < NN; ++k)               // target (a', b') = (k % NL, k / NL)
#pragma unroll
                        for (int b = 0; b < NL; ++b)
#pragma unroll
                            for (int a = 0; a < NL; ++a) {     // source (a, b): rho = c - offset + ((a - a') l, (b - b') l)
                                const float4 ww = w[j][(b - k / NL + NL) % NL][(a - k % NL + NL) % NL];
                                const f2 ax = sp[j][b][a][0], ay = sp[j][b][a][1], az = sp[j][b][a][2];
                                acc[k][0] = f2_fma(f2_bc(ww.x), ax, f2_fma(f2_bc(ww.y), ay, acc[k][0]));
                                acc[k][1] = f2_fma(f2_bc(ww.y), ax, f2_fma(f2_bc(ww.z), ay, acc[k][1]));
                                acc[k][2] = f2_fma(f2_bc(ww.w), az, acc[k][2]);
                            }
            }
            // warp reduction of the 3 NN packed values in fixed order
            f2 *v = &acc[0][0];
            if constexpr (NL == 2) {
                halve_exchange<12>(v, lane, 16);
                halve_exchange<6>(v, lane, 8);
                butterfly_sum<3>(v, 4);
                if ((lane & 7) == 0) {                         // lane bits 4, 3 say which 3 of the 12 values it holds
#pragma unroll
                    for (int i = 0; i < 3; ++i) part[warp * 12 + (lane >> 3) * 3 + i] = v[i];
                }
            } else {
                butterfly_sum<3>(v, 16);
                if (lane == 0) {
#pragma unroll
                    for (int i = 0; i < 3; ++i) part[warp * 3 + i] = v[i];
                }
            }
        } else {
            // the drawing warp: lanes < 2 NN take their site's counter, lane 31 the offset counter of the next pass
            const int xt = ox + l * (fk % NL), yt = oy + l * (fk / NL);
            nt = yt * L + xt;
            uint4 ctr = make_uint4((uint32_t)nt, (uint32_t)fr + p.r_off, (uint32_t)(pass & 0xFFFFFFFFull),
                                   (uint32_t)(pass >> 32) & 0x7FFFFFFFu);
            if (lane == 31)
                ctr = make_uint4(0xFFFFFFFFu, 0xFFFFFFFFu, (uint32_t)((pass + 1) & 0xFFFFFFFFull),
                                 (uint32_t)((pass + 1) >> 32) & 0x7FFFFFFFu);
            const uint4 rnd = philox4x32_10(ctr, rk);
            if (lane == 31) {
                off[2 * (cur ^ 1)] = (int)(rnd.x % (uint32_t)l);
                off[2 * (cur ^ 1) + 1] = (int)(rnd.y % (uint32_t)l);
            }
            if (flipper) {
                const int xe = xt + 1 == L ? 0 : xt + 1, xw = xt == 0 ? L - 1 : xt - 1;
                const int yn = yt + 1 == L ? 0 : yt + 1, ys = yt == 0 ? L - 1 : yt - 1;
                const float *sc = Sf + 6 * nt + rb, *se = Sf + 6 * (yt * L + xe) + rb, *sw = Sf + 6 * (yt * L + xw) + rb,
                            *sn = Sf + 6 * (yn * L + xt) + rb, *ss = Sf + 6 * (ys * L + xt) + rb;
                sx = sc[0], sy = sc[2], sz = sc[4];
                nx = (se[0] + sw[0]) + (sn[0] + ss[0]);
                ny = (se[2] + sw[2]) + (sn[2] + ss[2]);
                nz = (se[4] + sw[4]) + (sn[4] + ss[4]);
                dr = draw_from_words(q, rnd, sx, sy, sz);
            }
        }
        __syncthreads();
        if (flipper) {
            float h[3] = {0.0f, 0.0f, 0.0f};
            const float *pf = reinterpret_cast<const float *>(part) + rb;
#pragma unroll
            for (int w = 0; w < kResSumWarps; ++w)             // warp partials in fixed order
#pragma unroll
                for (int c = 0; c < 3; ++c) h[c] += pf[2 * ((w * NN + fk) * 3 + c)];
            const Trial tr = decide_drawn(q, dr, sx, sy, sz, nx, ny, nz, h[0], h[1], h[2], invT, K2, K4);
            if (tr.acc) {
                Sf[6 * nt + rb] = tr.tx;
                Sf[6 * nt + 2 + rb] = tr.ty;
                Sf[6 * nt + 4 + rb] = tr.tz;
            }
            if (r0 + rb < R) {
                if (p.accept_out) p.accept_out[(size_t)fr * N + nt] = tr.acc ? 1 : 0;
                if (p.margin_out) p.margin_out[(size_t)fr * N + nt] = tr.margin;
            }
        }
        __syncthreads();
    }

    for (int n = tid; n < N; n += kResThreads) {
        const int x = n % L, y = n / L;
        int qc;
        float *dst = p.S + site_index(x, y, Lh, R, plane, qc);
        float a0, a1, b0, b1, c0, c1;
        f2_split(Ssm[3 * n], a0, a1);
        f2_split(Ssm[3 * n + 1], b0, b1);
        f2_split(Ssm[3 * n + 2], c0, c1);
        dst[r0] = a0, dst[plane + r0] = b0, dst[2 * plane + r0] = c0;
        if (r0 + 1 < R) dst[r1] = a1, dst[plane + r1] = b1, dst[2 * plane + r1] = c1;
    }
}

__global__ void __launch_bounds__(256) init_spins_kernel(float *__restrict__ S, int L, int R, int mode, uint32_t r_off,
                                                         const RoundKeys rk) {
    const int Lh = L >> 1;
    const size_t Nh = (size_t)L * Lh;
    const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= 2 * Nh * (size_t)R) return;
    const int r = (int)(t % (size_t)R);
    const size_t qa = t / (size_t)R;
    const int q = (int)(qa / Nh);
    const int a = (int)(qa - (size_t)q * Nh);
    const int y = a / Lh, i = a - y * Lh;
    const int x = 2 * i + ((y + q) & 1);
    float sx = 0.0f, sy = 0.0f, sz = 1.0f;
    if (mode == DSMC_INIT_RANDOM) {
        const uint4 rnd = philox4x32_10(make_uint4((uint32_t)(y * L + x), (uint32_t)r + r_off, 0u, 0x80000000u), rk);
        sphere_point(rnd.x, rnd.y, sx, sy, sz);
    }
    const size_t plane = Nh * (size_t)R;
    float *dst = S + (size_t)q * 3 * plane + (size_t)a * R + r;
    dst[0] = sx;
    dst[plane] = sy;
    dst[2 * plane] = sz;
}

__global__ void step_update_kernel(unsigned long long *step, unsigned long long value, int add) {
    *step = add ? *step + value : value;
}

RoundKeys make_round_keys(uint32_t lo, uint32_t hi) {
    RoundKeys rk;
    for (int i = 0; i < 10; ++i) {
        rk.k[i][0] = lo + (uint32_t)i * 0x9E3779B9u;
        rk.k[i][1] = hi + (uint32_t)i * 0xBB67AE85u;
    }
    return rk;
}

}  // namespace

cudaError_t launch_metropolis(const MetropolisArgs &a, cudaStream_t st, uint64_t *launches) {
    const RoundKeys rk = make_round_keys(a.seed_lo, a.seed_hi);
    cudaError_t err = cudaSuccess;
    if (a.R % 4 == 0 && a.L <= 65535) {
        MetropolisArgs b = a;
        const int RQ = a.R / 4;
        b.rq_shift = -1;
        if ((RQ & (RQ - 1)) == 0) {
            b.rq_shift = 0;
            while ((1 << b.rq_shift) < RQ) ++b.rq_shift;
        }
        const unsigned per_row = (unsigned)((a.L / 2) * RQ);
        dim3 grid((per_row + 127) / 128, a.L);
        if (a.accept_out || a.margin_out) metropolis4_kernel<true, false, 2><<<grid, 128, 0, st>>>(b, rk);
        else if (a.step_dev && a.flip) metropolis4_kernel<false, true, 1><<<grid, 128, 0, st>>>(b, rk);
        else if (a.step_dev) metropolis4_kernel<false, true, 0><<<grid, 128, 0, st>>>(b, rk);
        else if (a.flip) metropolis4_kernel<false, false, 1><<<grid, 128, 0, st>>>(b, rk);
        else metropolis4_kernel<false, false, 0><<<grid, 128, 0, st>>>(b, rk);
        err = cudaGetLastError();
    } else {
        const size_t total = (size_t)a.L * (a.L / 2) * a.R;
        metropolis1_kernel<<<(unsigned)((total + 255) / 256), 256, 0, st>>>(a, rk);
        err = cudaGetLastError();
    }
    ++*launches;
    return err;
}

cudaError_t launch_init_spins(float *S, int L, int R, int mode, uint64_t seed, uint32_t r_off, cudaStream_t st,
                              uint64_t *launches) {
    const size_t total = (size_t)L * L * R;
    const unsigned grid = (unsigned)((total + 255) / 256);
    init_spins_kernel<<<grid, 256, 0, st>>>(S, L, R, mode, r_off,
                                             make_round_keys((uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32)));
    ++*launches;
    return cudaGetLastError();
}

void dsmc_sublattice_offset(uint64_t seed, uint64_t pass, int l, int *ox, int *oy) {
    const RoundKeys rk = make_round_keys((uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32));
    pass_offset(rk, pass, l, *ox, *oy);
}

cudaError_t launch_sublattice_pass(const MetropolisArgs &a, const float *Wc, float *scratch, int sm_count, int l, int ox,
                                   int oy, bool field_in_H, cudaStream_t st, uint64_t *launches) {
    const RoundKeys rk = make_round_keys(a.seed_lo, a.seed_hi);
    const int nl = a.L / l, n = nl * nl, chunks = (a.R + 31) / 32;
    int KS = 0;
    if (!field_in_H) {
        // A CTA's 8 warps share (source row, row segment) items; a row is cut in 4 segments when L allows.
        // Source slabs: enough CTAs to fill the GPU about four times over, at least 8 items per slab, and
        // KS * n <= N so that the partials fit the 3 N R floats of the staging buffer.
        const int segs = (a.L % 8 == 0 && a.L >= 32) ? 4 : 1;
        const int ks_target = std::max(1, (4 * sm_count + n * chunks - 1) / (n * chunks));
        int rows = std::max(8 / segs, (a.L + ks_target - 1) / ks_target);
        rows = std::max(rows, (n + a.L - 1) / a.L);
        KS = (a.L + rows - 1) / rows;
        sublattice_field_kernel<<<dim3((unsigned)n, (unsigned)chunks, (unsigned)KS), 256, 0, st>>>(
            a.S, scratch, Wc, a.L, a.R, l, ox, oy, rows, segs, a.step_dev, rk);
        ++*launches;
    }
    const size_t total = (size_t)n * a.R;
    sublattice_flip_kernel<<<(unsigned)((total + 127) / 128), 128, 0, st>>>(a, rk, scratch, KS, l, ox, oy);
    ++*launches;
    return cudaGetLastError();
}

bool dsmc_resident_supported(int L, int l) {
    const int nl = L / l;
    return (nl == 1 || nl == 2) && resident_smem_bytes(L, nl) <= 227 * 1024;
}

cudaError_t launch_sublattice_resident(const MetropolisArgs &a, const float *Wc, int l, uint64_t first_pass, uint64_t n_passes,
                                       cudaStream_t st, uint64_t *launches) {
    const RoundKeys rk = make_round_keys(a.seed_lo, a.seed_hi);
    const int nl = a.L / l;
    const size_t smem = resident_smem_bytes(a.L, nl);
    // trips of the summing loop per pass: a compile-time constant for the common shapes (0 = run-time count)
    const int un = nl == 2 ? 1 : 8, trips = (l * l + un * 32 * kResSumWarps - 1) / (un * 32 * kResSumWarps);
    void (*kern)(const MetropolisArgs, const RoundKeys, const float *, int, unsigned long long, unsigned) = nullptr;
    if (nl == 2) kern = a.L == 64 ? sublattice_resident_kernel<2, 4, 64> : trips == 4 ? sublattice_resident_kernel<2, 4, 0> : trips == 1 ? sublattice_resident_kernel<2, 1, 0> : sublattice_resident_kernel<2, 0, 0>;
    else kern = a.L == 64 ? sublattice_resident_kernel<1, 2, 64> : trips == 2 ? sublattice_resident_kernel<1, 2, 0> : trips == 1 ? sublattice_resident_kernel<1, 1, 0> : sublattice_resident_kernel<1, 0, 0>;
    if (cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024)) return e;
    const unsigned grid = (unsigned)((a.R + 1) / 2);
    // one launch per 65536 passes keeps a single kernel well under a second
    for (uint64_t done = 0; done < n_passes;) {
        const unsigned chunk = (unsigned)std::min<uint64_t>(n_passes - done, 65536);
        kern<<<grid, kResThreads, smem, st>>>(a, rk, Wc, l, first_pass + done, chunk);
        ++*launches;
        done += chunk;
    }
    return cudaGetLastError();
}

cudaError_t launch_step_update(unsigned long long *step, unsigned long long value, int add, cudaStream_t st,
                               uint64_t *launches) {
    step_update_kernel<<<1, 1, 0, st>>>(step, value, add);
    ++*launches;
    return cudaGetLastError();
}
