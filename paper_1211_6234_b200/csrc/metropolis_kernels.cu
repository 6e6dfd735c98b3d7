// metropolis_kernels.cu -- a2: fused checkerboard Metropolis half-sweep, and a4: spin init.
// One thread per (active site, replica): Philox4x32-10 trial + exchange + anisotropy +
// frozen-field dipole dE + accept, all in registers (PAPER.md:60-72 eq. 7, :98, :102-118).
#include "dsmc_internal.cuh"

namespace {

// Philox4x32-10 (Salmon et al., SC'11): counter-based, 10 rounds.
__device__ __forceinline__ uint4 philox4x32_10(uint4 c, uint2 k) {
#pragma unroll
    for (int round = 0; round < 10; ++round) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c.x), lo0 = 0xD2511F53u * c.x;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c.z), lo1 = 0xCD9E8D57u * c.z;
        c = make_uint4(hi1 ^ c.y ^ k.x, lo1, hi0 ^ c.w ^ k.y, lo0);
        k.x += 0x9E3779B9u;
        k.y += 0xBB67AE85u;
    }
    return c;
}

// 32 bits -> odd multiple of 2^-24 strictly inside (0,1): exact in fp32 (R9)
__device__ __forceinline__ float unit24(uint32_t x) {
    return (float)(2u * (x >> 9) + 1u) * 5.9604644775390625e-8f;
}

// uniform point on S^2 from two words (R10): z = 2 u0 - 1, azimuth 2 pi u1
__device__ __forceinline__ void sphere_point(uint32_t x0, uint32_t x1, float &sx, float &sy, float &sz) {
    const float z = 2.0f * unit24(x0) - 1.0f;  // exact
    float sn, cs;
    sincospif(2.0f * unit24(x1), &sn, &cs);
    const float rho = sqrtf((1.0f - z) * (1.0f + z));
    sx = rho * cs;
    sy = rho * sn;
    sz = z;
}

// Thread t -> (colour-site a = t / R, replica r = t % R): a warp reads R-contiguous runs.
__global__ void __launch_bounds__(256) metropolis_kernel(const MetropolisArgs p) {
    const int Lh = p.L >> 1;
    const size_t Nh = (size_t)p.L * Lh;
    const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= Nh * (size_t)p.R) return;
    const int r = (int)(t % (size_t)p.R);
    const int a = (int)(t / (size_t)p.R);
    const int y = a / Lh, i = a - y * Lh;
    const int par = (y + p.colour) & 1;
    const int x = 2 * i + par;
    const size_t plane = Nh * (size_t)p.R;

    float *own = p.S + (size_t)p.colour * 3 * plane + (size_t)a * p.R + r;
    const float *oth = p.S + (size_t)(1 - p.colour) * 3 * plane + r;
    const float *hf = p.H + (size_t)p.colour * 3 * plane + (size_t)a * p.R + r;

    // the four neighbours all have the other colour
    const int ie = par ? (i + 1 == Lh ? 0 : i + 1) : i;
    const int iw = par ? i : (i == 0 ? Lh - 1 : i - 1);
    const int yn = (y + 1 == p.L) ? 0 : y + 1, ys = (y == 0) ? p.L - 1 : y - 1;
    const size_t ae = ((size_t)y * Lh + ie) * p.R, aw = ((size_t)y * Lh + iw) * p.R;
    const size_t an = ((size_t)yn * Lh + i) * p.R, as = ((size_t)ys * Lh + i) * p.R;

    const float sx = own[0], sy = own[plane], sz = own[2 * plane];
    const float hx = hf[0], hy = hf[plane], hz = hf[2 * plane];
    const float nx = (oth[ae] + oth[aw]) + (oth[an] + oth[as]);
    const float ny = (oth[plane + ae] + oth[plane + aw]) + (oth[plane + an] + oth[plane + as]);
    const float nz = (oth[2 * plane + ae] + oth[2 * plane + aw]) + (oth[2 * plane + an] + oth[2 * plane + as]);

    const uint32_t n = (uint32_t)(y * p.L + x);
    const uint4 rnd = philox4x32_10(make_uint4(n, (uint32_t)r, p.step_lo, p.step_hi),
                                    make_uint2(p.seed_lo, p.seed_hi));
    float tx, ty, tz;
    sphere_point(rnd.x, rnd.y, tx, ty, tz);
    const float u = unit24(rnd.z);

    const float dx = tx - sx, dy = ty - sy, dz = tz - sz;
    const float K2 = p.K2[r], K4 = p.K4[r];
    const float z2n = tz * tz, z2o = sz * sz;
    const float dz2 = dz * (tz + sz);  // s'_z^2 - s_z^2
    float dE = -p.J * (dx * nx + dy * ny + dz * nz);
    dE -= dz2 * (K2 + K4 * (z2n + z2o));  // -K2 d(z^2) - K4 d(z^4)
    const float self = 0.5f * (p.w0xx * dx * dx + p.w0yy * dy * dy + p.w0zz * dz * dz) + p.w0xy * dx * dy;
    dE += p.g * ((dx * hx + dy * hy + dz * hz) + self);
    const float margin = dE * p.invT[r] + logf(u);
    const bool acc = margin < 0.0f;
    if (acc) {
        own[0] = tx;
        own[plane] = ty;
        own[2 * plane] = tz;
    }
    if (p.accept_out) p.accept_out[(size_t)r * 2 * Nh + n] = acc ? 1 : 0;
    if (p.margin_out) p.margin_out[(size_t)r * 2 * Nh + n] = margin;
}

__global__ void __launch_bounds__(256) init_spins_kernel(float *__restrict__ S, int L, int R, int mode,
                                                         uint32_t seed_lo, uint32_t seed_hi) {
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
        const uint4 rnd = philox4x32_10(make_uint4((uint32_t)(y * L + x), (uint32_t)r, 0u, 0x80000000u),
                                        make_uint2(seed_lo, seed_hi));
        sphere_point(rnd.x, rnd.y, sx, sy, sz);
    }
    const size_t plane = Nh * (size_t)R;
    float *dst = S + (size_t)q * 3 * plane + (size_t)a * R + r;
    dst[0] = sx;
    dst[plane] = sy;
    dst[2 * plane] = sz;
}

}  // namespace

cudaError_t launch_metropolis(const MetropolisArgs &a, cudaStream_t st, uint64_t *launches) {
    const size_t total = (size_t)a.L * (a.L / 2) * a.R;
    const unsigned grid = (unsigned)((total + 255) / 256);
    metropolis_kernel<<<grid, 256, 0, st>>>(a);
    ++*launches;
    return cudaGetLastError();
}

cudaError_t launch_init_spins(float *S, int L, int R, int mode, uint64_t seed, cudaStream_t st,
                              uint64_t *launches) {
    const size_t total = (size_t)L * L * R;
    const unsigned grid = (unsigned)((total + 255) / 256);
    init_spins_kernel<<<grid, 256, 0, st>>>(S, L, R, mode, (uint32_t)(seed & 0xFFFFFFFFu),
                                             (uint32_t)(seed >> 32));
    ++*launches;
    return cudaGetLastError();
}
