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

namespace {

struct RoundKeys {
    uint32_t k[10][2];
};

// Philox4x32-10 (Salmon et al., SC'11) with precomputed round keys
__device__ __forceinline__ uint4 philox4x32_10(uint4 c, const RoundKeys &rk) {
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

struct Trial {
    float tx, ty, tz, margin;
    bool acc;
};

// one Metropolis decision: current spin s, neighbour sum nb, frozen field h  (R12-R14)
__device__ __forceinline__ Trial decide(const MetropolisArgs &p, const RoundKeys &rk, uint32_t n, uint32_t r, float sx,
                                        float sy, float sz, float nx, float ny, float nz, float hx, float hy, float hz,
                                        float invT, float K2, float K4) {
    const uint4 rnd = philox4x32_10(make_uint4(n, r, p.step_lo, p.step_hi), rk);
    Trial t;
    sphere_point(rnd.x, rnd.y, t.tx, t.ty, t.tz);
    const float u = unit24(rnd.z);
    const float dx = t.tx - sx, dy = t.ty - sy, dz = t.tz - sz;
    const float dz2 = dz * (t.tz + sz);                       // s'_z^2 - s_z^2
    const float z2sum = fmaf(t.tz, t.tz, sz * sz);
    float dE = -p.J * fmaf(dx, nx, fmaf(dy, ny, dz * nz));    // exchange with the 4 neighbours
    dE = fmaf(-dz2, fmaf(K4, z2sum, K2), dE);                 // -K2 d(z^2) - K4 d(z^4)
    float self = fmaf(p.w0xx * dx, dx, fmaf(p.w0yy * dy, dy, p.w0zz * dz * dz));
    self = fmaf(0.5f, self, p.w0xy * dx * dy);
    dE = fmaf(p.g, fmaf(dx, hx, fmaf(dy, hy, fmaf(dz, hz, self))), dE);
    t.margin = fmaf(dE, invT, __logf(u));
    t.acc = t.margin < 0.0f;
    return t;
}

// R % 4 == 0: one thread = one active site x 4 consecutive replicas.  grid.y = lattice row.
__global__ void __launch_bounds__(128) metropolis4_kernel(const MetropolisArgs p, const RoundKeys rk) {
    const int Lh = p.L >> 1, RQ = p.R >> 2;
    const int y = blockIdx.y;
    const uint32_t e = blockIdx.x * blockDim.x + threadIdx.x;   // (i, replica quad) within the row
    if (e >= (uint32_t)(Lh * RQ)) return;
    const int i = p.rq_shift >= 0 ? (int)(e >> p.rq_shift) : (int)(e / (uint32_t)RQ);
    const int rq = (int)e - i * RQ;
    const int par = (y + p.colour) & 1;
    const size_t plane4 = ((size_t)p.L * Lh * p.R) >> 2;      // float4 per [a][r] plane
    const size_t row4 = (size_t)Lh * RQ;

    float4 *own = reinterpret_cast<float4 *>(p.S) + (size_t)p.colour * 3 * plane4 + (size_t)y * row4 + e;
    const float4 *oth = reinterpret_cast<const float4 *>(p.S) + (size_t)(1 - p.colour) * 3 * plane4 + rq;
    const float4 *hf = reinterpret_cast<const float4 *>(p.H) + (size_t)p.colour * 3 * plane4 + (size_t)y * row4 + e;

    // the four neighbours all have the other colour (internal layout: same row i or i+-1, rows y+-1 same i)
    const int ie = par ? (i + 1 == Lh ? 0 : i + 1) : i;
    const int iw = par ? i : (i == 0 ? Lh - 1 : i - 1);
    const int yn = (y + 1 == p.L) ? 0 : y + 1, ys = (y == 0) ? p.L - 1 : y - 1;
    const size_t ae = (size_t)y * row4 + (size_t)ie * RQ, aw = (size_t)y * row4 + (size_t)iw * RQ;
    const size_t an = (size_t)yn * row4 + (size_t)i * RQ, as = (size_t)ys * row4 + (size_t)i * RQ;

    float4 s[3], h[3], nb[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        s[c] = own[c * plane4];
        h[c] = __ldg(hf + c * plane4);
        const float4 a = __ldg(oth + c * plane4 + ae), b = __ldg(oth + c * plane4 + aw);
        const float4 cc = __ldg(oth + c * plane4 + an), d = __ldg(oth + c * plane4 + as);
        nb[c] = make_float4((a.x + b.x) + (cc.x + d.x), (a.y + b.y) + (cc.y + d.y), (a.z + b.z) + (cc.z + d.z),
                            (a.w + b.w) + (cc.w + d.w));
    }
    const float4 invT = __ldg(reinterpret_cast<const float4 *>(p.invT) + rq);
    const float4 K2 = __ldg(reinterpret_cast<const float4 *>(p.K2) + rq);
    const float4 K4 = __ldg(reinterpret_cast<const float4 *>(p.K4) + rq);

    const uint32_t n = (uint32_t)(y * p.L + 2 * i + par);
    const uint32_t r0 = 4u * (uint32_t)rq;
    float *sxp = &s[0].x, *syp = &s[1].x, *szp = &s[2].x;
    const float *hxp = &h[0].x, *hyp = &h[1].x, *hzp = &h[2].x;
    const float *nxp = &nb[0].x, *nyp = &nb[1].x, *nzp = &nb[2].x;
    const float *tp = &invT.x, *k2p = &K2.x, *k4p = &K4.x;
    bool any = false;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const Trial t = decide(p, rk, n, r0 + k, sxp[k], syp[k], szp[k], nxp[k], nyp[k], nzp[k], hxp[k], hyp[k], hzp[k],
                               tp[k], k2p[k], k4p[k]);
        if (t.acc) {
            sxp[k] = t.tx;
            syp[k] = t.ty;
            szp[k] = t.tz;
        }
        any |= t.acc;
        if (p.accept_out) p.accept_out[(size_t)(r0 + k) * p.L * p.L + n] = t.acc ? 1 : 0;
        if (p.margin_out) p.margin_out[(size_t)(r0 + k) * p.L * p.L + n] = t.margin;
    }
    if (any) {
#pragma unroll
        for (int c = 0; c < 3; ++c) own[c * plane4] = s[c];
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
    const Trial tr = decide(p, rk, n, (uint32_t)r, sx, sy, sz, nx, ny, nz, hf[0], hf[plane], hf[2 * plane], p.invT[r],
                            p.K2[r], p.K4[r]);
    if (tr.acc) {
        own[0] = tr.tx;
        own[plane] = tr.ty;
        own[2 * plane] = tr.tz;
    }
    if (p.accept_out) p.accept_out[(size_t)r * 2 * Nh + n] = tr.acc ? 1 : 0;
    if (p.margin_out) p.margin_out[(size_t)r * 2 * Nh + n] = tr.margin;
}

__global__ void __launch_bounds__(256) init_spins_kernel(float *__restrict__ S, int L, int R, int mode, const RoundKeys rk) {
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
        const uint4 rnd = philox4x32_10(make_uint4((uint32_t)(y * L + x), (uint32_t)r, 0u, 0x80000000u), rk);
        sphere_point(rnd.x, rnd.y, sx, sy, sz);
    }
    const size_t plane = Nh * (size_t)R;
    float *dst = S + (size_t)q * 3 * plane + (size_t)a * R + r;
    dst[0] = sx;
    dst[plane] = sy;
    dst[2 * plane] = sz;
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
        metropolis4_kernel<<<grid, 128, 0, st>>>(b, rk);
    } else {
        const size_t total = (size_t)a.L * (a.L / 2) * a.R;
        metropolis1_kernel<<<(unsigned)((total + 255) / 256), 256, 0, st>>>(a, rk);
    }
    ++*launches;
    return cudaGetLastError();
}

cudaError_t launch_init_spins(float *S, int L, int R, int mode, uint64_t seed, cudaStream_t st,
                              uint64_t *launches) {
    const size_t total = (size_t)L * L * R;
    const unsigned grid = (unsigned)((total + 255) / 256);
    init_spins_kernel<<<grid, 256, 0, st>>>(S, L, R, mode,
                                             make_round_keys((uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32)));
    ++*launches;
    return cudaGetLastError();
}
