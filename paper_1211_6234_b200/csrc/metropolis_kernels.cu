// metropolis_kernels.cu -- a2: fused checkerboard Metropolis half-sweep, and a4: spin init.
// Philox4x32-10 trial + exchange + anisotropy + frozen-field dipole dE + accept, all in registers
// (PAPER.md:60-72 eq. 7, :98, :102-118).  The kernel is co-limited by HBM bandwidth (48 B per
// update) and instruction issue, so the per-update instruction count is kept near 130:
//   * one thread updates 4 consecutive replicas of one site: every global access is a 128-bit
//     load/store and the index arithmetic is shared by 4 updates;
//   * Philox round keys are precomputed on the host (kernel parameters = constant bank);
//   * the azimuth 2 pi u1 is reduced to a quadrant exactly in integer arithmetic and sin/cos come
//     from two short polynomials (abs error 1.5e-7); sqrt and log use the MUFU units.
#include "metropolis_pair.cuh"
#include <algorithm>

namespace {

// R % 4 == 0: one thread = one active site x 4 consecutive replicas (two packed pairs); grid.y =
// lattice row.  All 18 128-bit loads are issued first; the four Philox chains and the trial spins
// do not depend on them and run while they are in flight.  HOOKS = parity outputs requested.
// FLIP: 0 = uniform-sphere trial, 1 = Ising reversal (App. B), 2 = decided at run time from p.flip (parity-hook
// variant only: a run-time branch here splits the block the scheduler interleaves the two pairs in, +5 %)
// TY = lattice rows per CTA: the 128 threads are TY groups of 128 / TY consecutive (i, replica quad) entries, one group
// per row y0 .. y0 + TY - 1.  The neighbour rows of adjacent update rows coincide (row y + 1 of the other colour is
// "north" for row y, "same row" for row y + 1 and "south" for row y + 2), so with TY > 1 those loads hit in L1
// instead of going to L2 three times.  MINB = CTAs per SM the register allocation is held to.
template <bool HOOKS, bool DEVSTEP, int FLIP, int TY, int MINB>
__global__ void __launch_bounds__(128, MINB) metropolis4_kernel(const MetropolisArgs p, const RoundKeys rk) {
    constexpr int EX = 128 / TY;
    const int Lh = p.L >> 1, RQ = p.R >> 2;
    const int y = blockIdx.y * TY + (TY > 1 ? (int)(threadIdx.x / EX) : 0);
    const uint32_t row4 = (uint32_t)(Lh * RQ);
    const uint32_t e = blockIdx.x * EX + (TY > 1 ? threadIdx.x % EX : threadIdx.x);   // (i, replica quad) within the row
    if (!p.pdl_late) pdl_trigger();
    if (e >= row4) return;
    pdl_wait();                                                 // spins, field and step counter come from earlier kernels
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

    if (p.pdl_late) pdl_trigger();
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

// The memory traffic of metropolis4_kernel without its arithmetic (dsmc_stream_footprint: the measured denominator of
// that kernel's roofline): same grid, same 18 128-bit loads per thread at the same addresses, the 3 stores of the
// thread's own spins (unchanged bits) ALWAYS issued -- so it moves at least the bytes of a half-sweep in which every
// move is accepted -- and no Philox, trial or dE.  The store is guarded by a condition on the loaded values that is never
// false for finite inputs, which keeps the loads alive.
template <int TY, int MINB>
__global__ void __launch_bounds__(128, MINB) metropolis_stream_kernel(const MetropolisArgs p) {
    constexpr int EX = 128 / TY;
    const int Lh = p.L >> 1, RQ = p.R >> 2;
    const int y = blockIdx.y * TY + (TY > 1 ? (int)(threadIdx.x / EX) : 0);
    const uint32_t row4 = (uint32_t)(Lh * RQ);
    const uint32_t e = blockIdx.x * EX + (TY > 1 ? threadIdx.x % EX : threadIdx.x);
    pdl_trigger();
    if (e >= row4) return;
    pdl_wait();
    const int i = (int)(e / (uint32_t)RQ), rq = (int)e - i * RQ;
    const int par = (y + p.colour) & 1;
    const size_t plane4 = ((size_t)p.L * Lh * p.R) >> 2;
    const int yn = (y + 1 == p.L) ? 0 : y + 1, ys = (y == 0) ? p.L - 1 : y - 1;
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
    f2 s[3][2], h[3][2], a[3][2], b[3][2], c[3][2], d[3][2];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        ld2(own + k * plane4, s[k][0], s[k][1]);
        ld2(hf + k * plane4, h[k][0], h[k][1]);
        ld2(o0 + k * plane4, a[k][0], a[k][1]);
        ld2(o1 + k * plane4, b[k][0], b[k][1]);
        ld2(on + k * plane4, c[k][0], c[k][1]);
        ld2(os + k * plane4, d[k][0], d[k][1]);
    }
    f2 sum = f2_bc(0.0f);
#pragma unroll
    for (int k = 0; k < 3; ++k)
#pragma unroll
        for (int j = 0; j < 2; ++j) sum = f2_add(f2_add(sum, h[k][j]), f2_add(f2_add(a[k][j], b[k][j]), f2_add(c[k][j], d[k][j])));
    float s0, s1;
    f2_split(sum, s0, s1);
    if (s0 + s1 != 1.2345678e30f) {
#pragma unroll
        for (int k = 0; k < 3; ++k)
            *reinterpret_cast<ulonglong2 *>(own + k * plane4) = make_ulonglong2(s[k][0], s[k][1]);
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
    pdl_trigger();
    pdl_wait();                                                 // the Metropolis kernel before it reads *step
    *step = add ? *step + value : value;
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
        // two lattice rows per CTA (L is even): measured at config 5 over 24 cold launches, 18.6 us for one row per CTA,
        // 18.4 for two, 18.45 for four; 64 registers for 8 CTAs per SM spill and lose (19.3-19.8 us)
        constexpr int TY = 2, MINB = 7;
        dim3 grid((per_row + 128 / TY - 1) / (128 / TY), a.L / TY);
        // measured: a one-wave grid gains from triggering its successor late (L = 128, R = 4:
        // 18.9 -> 20.8 k sweeps/s), a many-wave grid from triggering at the top (L = 256, R = 64)
        b.pdl_late = (size_t)grid.x * grid.y <= 1024 ? 1 : 0;
        if (a.accept_out || a.margin_out) err = launch_pdl(metropolis4_kernel<true, false, 2, TY, MINB>, grid, dim3(128), 0, st, b, rk);
        else if (a.step_dev && a.flip) err = launch_pdl(metropolis4_kernel<false, true, 1, TY, MINB>, grid, dim3(128), 0, st, b, rk);
        else if (a.step_dev) err = launch_pdl(metropolis4_kernel<false, true, 0, TY, MINB>, grid, dim3(128), 0, st, b, rk);
        else if (a.flip) err = launch_pdl(metropolis4_kernel<false, false, 1, TY, MINB>, grid, dim3(128), 0, st, b, rk);
        else err = launch_pdl(metropolis4_kernel<false, false, 0, TY, MINB>, grid, dim3(128), 0, st, b, rk);
        if (err == cudaSuccess) err = cudaGetLastError();
    } else {
        const size_t total = (size_t)a.L * (a.L / 2) * a.R;
        metropolis1_kernel<<<(unsigned)((total + 255) / 256), 256, 0, st>>>(a, rk);
        err = cudaGetLastError();
    }
    ++*launches;
    return err;
}

cudaError_t launch_metropolis_stream(const MetropolisArgs &a, cudaStream_t st, uint64_t *launches) {
    if (a.R % 4 != 0 || a.L > 65535) return cudaErrorInvalidValue;
    constexpr int TY = 2, MINB = 7;                             // the launch shape of launch_metropolis
    const unsigned per_row = (unsigned)((a.L / 2) * (a.R / 4));
    dim3 grid((per_row + 128 / TY - 1) / (128 / TY), a.L / TY);
    cudaError_t err = launch_pdl(metropolis_stream_kernel<TY, MINB>, grid, dim3(128), 0, st, a);
    ++*launches;
    return err != cudaSuccess ? err : cudaGetLastError();
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

cudaError_t launch_step_update(unsigned long long *step, unsigned long long value, int add, cudaStream_t st,
                               uint64_t *launches) {
    const cudaError_t err = launch_pdl(step_update_kernel, dim3(1), dim3(1), 0, st, step, value, add);
    ++*launches;
    return err != cudaSuccess ? err : cudaGetLastError();
}
