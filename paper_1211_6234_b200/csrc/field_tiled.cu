// field_tiled.cu -- a1, the hot kernel: dipole field h = W (*) s as a register-tiled direct sum
// (App. A :331-350; the paper's "2Pn threads, one strip each" becomes a
// split-K grid of CTAs whose threads each own an 8-target x 4-replica outer-product tile).
//
// Shape: L % 16 == 0, R % 4 == 0.  Work decomposition:
//   * targets of the active colour are grouped 8 consecutive same-colour sites of a row
//     (x_t = 2 (8 g + j) + p_t, j = 0..7); a thread owns one group and 4 consecutive replicas:
//     96 fp32 accumulators (8 targets x 3 components x 4 replicas), 160 FFMA per source site.
//   * a CTA is NG groups x RT replica-quads (NG * RT <= 256 threads); the grid is
//     (target tiles) x (source-row chunks KS) x (replica chunks); each CTA writes a partial field
//     for its source chunk, a second kernel adds the KS partials in fixed order (this is also the
//     second level of the two-level fp32 accumulation).
//   * sources stream through shared memory in stages of one (row, colour, segment): the spins of
//     SEG same-colour sites x 3 components x RCH replicas, and for every target row of the CTA the
//     4 x L block of the pre-shifted table Wk.  Stages are filled by TMA bulk copies
//     (cp.async.bulk, completion on an mbarrier) issued by warp 0, double buffered.
//   * because both targets and sources are walked in steps of one same-colour site, the W values a
//     thread needs form a sliding window: one new value per component per source step, kept in an
//     8-deep register ring (fully unrolled by 8), fetched as 128-bit shared loads every 4 steps.
//   * the FMAs are issued as packed FFMA2 over pairs of replicas (W value duplicated in a register
//     pair): 80 FFMA2 per source step per thread.
//
// Wk[cl][pt][dy][c][kk] = W[c][dy][(2 (kk - Lh) + ((pt + dy + cl) & 1) - pt) mod L], kk in [0, L):
//   cl = source colour != target colour, pt = parity offset of the target row, dy = (y_s - y_t) mod L,
//   kk - Lh = i_s - i_t (difference of in-row indices).  All periodic wrapping and the
//   checkerboard parity bookkeeping are folded into this table, so the inner loop has none.
#include "dsmc_internal.cuh"
#include "bulk_copy.cuh"

namespace {

constexpr int TT = 8;          // targets per thread
constexpr int MAX_THREADS = 256;
constexpr int NSTAGE = 2;

struct TiledParams {
    const float *S;
    const float *Wk;
    float *out;        // Hpart base (KS > 1) or H colour base (KS == 1), layout [ks][c][a][r]
    int L, R, colour;
    int RT;            // replica quads per CTA (threads along replicas)
    int NG;            // target groups per CTA
    int RCH;           // replicas per CTA = 4 * RT
    int SEG;           // source sites per stage
    int nrows_max;     // target rows a CTA can touch
    int rows_per_chunk;  // source rows per K chunk = L / KS
    int total_groups;  // L * (L/16)
};

__global__ void __launch_bounds__(MAX_THREADS, 1) field_tiled_kernel(const TiledParams p) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int L = p.L, Lh = L >> 1, R = p.R, RCH = p.RCH, SEG = p.SEG;
    const int GPR = Lh / TT;  // groups per row
    const size_t Nh = (size_t)L * Lh, plane = Nh * (size_t)R;

    const int w_stage_floats = p.nrows_max * 4 * L;
    const int s_stage_floats = 3 * SEG * RCH;
    const int stage_floats = w_stage_floats + s_stage_floats;
    float *buf = reinterpret_cast<float *>(smem_raw);
    uint64_t *bars = reinterpret_cast<uint64_t *>(buf + (size_t)NSTAGE * stage_floats);

    const int tid = threadIdx.x;
    const int rt = tid % p.RT, gl = tid / p.RT;
    const int G0 = blockIdx.x * p.NG;
    const int Gmine = min(G0 + min(gl, p.NG - 1), p.total_groups - 1);
    const bool live = gl < p.NG && (G0 + gl) < p.total_groups;
    const int y_first = G0 / GPR;
    const int y_last = min(G0 + p.NG - 1, p.total_groups - 1) / GPR;
    const int nrows = y_last - y_first + 1;
    const int yt = Gmine / GPR, g = Gmine - yt * GPR;
    const int trow = yt - y_first;
    const int ks = blockIdx.y;
    const int r0 = blockIdx.z * RCH;
    const int nseg = Lh / SEG;
    const int nstages = p.rows_per_chunk * 2 * nseg;

    if (tid == 0) {
        for (int s = 0; s < NSTAGE; ++s) mbar_init(&bars[s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    // producer: warp 0 fills stage `st` into buffer st % NSTAGE
    auto produce = [&](int st) {
        const int b = st % NSTAGE;
        float *wdst = buf + (size_t)b * stage_floats;
        float *sdst = wdst + w_stage_floats;
        const int rr = st / (2 * nseg), rem = st - rr * 2 * nseg;
        const int q = rem / nseg, seg = rem - q * nseg;
        const int i0 = seg * SEG;
        // Source rows in the order far -> near (relative to the CTA's first target row): entry j of the sequence
        // d = -L/2, +(L/2-1), -(L/2-1), ..., +1, -1, 0, dealt out to the KS chunks in turn (chunk ks takes j = ks,
        // ks + KS, ...).  Every chunk then adds its many small far-field terms while its accumulators are still small
        // -- the rounding error of an fp32 add scales with the accumulator, and a term below half an ulp of it is
        // lost altogether -- and ends with ONE of the near rows, so no accumulator ever holds more than one row's
        // worth (<= 2 zeta(3) = 2.4) of the 9.03 the z-aligned state sums to.
        const int j = ks + (int)gridDim.y * rr, mm = (j + 1) >> 1;
        const int d = j == 0 ? -(L >> 1) : ((j & 1) ? (L >> 1) - mm : mm - (L >> 1));
        int ys = y_first + d;
        ys += ys < 0 ? L : 0;
        ys -= ys >= L ? L : 0;
        const int cl = q ^ p.colour;
        const int lane = tid;  // tid < 32 here
        const bool whole = (RCH == R);
        if (lane == 0) {
            const uint32_t bytes = (uint32_t)(nrows * 4 * L + s_stage_floats) * 4u;
            mbar_expect_tx(&bars[b], bytes);
        }
        __syncwarp();
        for (int tr = lane; tr < nrows; tr += 32) {
            const int y = y_first + tr;
            const int ptr_ = (y + p.colour) & 1;
            int dy = ys - y;
            dy += dy < 0 ? L : 0;
            const float *src = p.Wk + ((((size_t)cl * 2 + ptr_) * L + dy) * 4) * L;
            bulk_g2s(wdst + (size_t)tr * 4 * L, src, (uint32_t)(4 * L * 4), &bars[b]);
        }
        if (whole) {
            if (lane < 3) {
                const float *src = p.S + ((size_t)q * 3 + lane) * plane + ((size_t)ys * Lh + i0) * R;
                bulk_g2s(sdst + (size_t)lane * SEG * RCH, src, (uint32_t)(SEG * RCH * 4), &bars[b]);
            }
        } else {
            for (int k = lane; k < 3 * SEG; k += 32) {
                const int c = k / SEG, u = k - c * SEG;
                const float *src = p.S + ((size_t)q * 3 + c) * plane + ((size_t)ys * Lh + i0 + u) * R + r0;
                bulk_g2s(sdst + (size_t)k * RCH, src, (uint32_t)(RCH * 4), &bars[b]);
            }
        }
    };

    if (tid < 32) {
        for (int s = 0; s < NSTAGE && s < nstages; ++s) produce(s);
    }

    // accumulators as packed pairs of replicas: acc[j][c][kp] = (replica 2kp, replica 2kp+1).
    // The inner product is issued as FFMA2 (fma.rn.f32x2): 64-bit register pairs read one word from
    // each register bank, so the operand fetch has no bank conflicts by construction, and one issue
    // slot carries two FMAs per lane (measured 114 vs 102 FMA/clk/SM for the scalar form of this loop).
    float2 acc[TT][3][2];
#pragma unroll
    for (int j = 0; j < TT; ++j)
#pragma unroll
        for (int c = 0; c < 3; ++c)
#pragma unroll
            for (int k = 0; k < 2; ++k) acc[j][c][k] = make_float2(0.0f, 0.0f);

    const int RCH4 = RCH >> 2;
    for (int st = 0; st < nstages; ++st) {
        const int b = st % NSTAGE;
        mbar_wait(&bars[b], (uint32_t)((st / NSTAGE) & 1));
        const float *wsm = buf + (size_t)b * stage_floats;
        const float4 *ssm = reinterpret_cast<const float4 *>(wsm + w_stage_floats) + rt;
        const int rem = st % (2 * nseg);
        const int seg = rem % nseg;
        const int base = seg * SEG + Lh - TT * g;  // multiple of 8
        const float *wr = wsm + (size_t)trow * 4 * L + base;

        // register ring of the sliding W window: slot (u & 7) holds (W[base + u], W[base + u])
        float2 w[4][8];
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            const float4 a = *reinterpret_cast<const float4 *>(wr + c * L - 8);
            const float4 bq = *reinterpret_cast<const float4 *>(wr + c * L - 4);
            w[c][0] = make_float2(a.x, a.x);  // W[base - 8]: never used, overwritten at u = 0
            w[c][1] = make_float2(a.y, a.y); w[c][2] = make_float2(a.z, a.z); w[c][3] = make_float2(a.w, a.w);
            w[c][4] = make_float2(bq.x, bq.x); w[c][5] = make_float2(bq.y, bq.y);
            w[c][6] = make_float2(bq.z, bq.z); w[c][7] = make_float2(bq.w, bq.w);
        }
        for (int ub = 0; ub < SEG; ub += 8) {
            float4 wn[4];
#pragma unroll
            for (int uu = 0; uu < 8; ++uu) {
                const int u = ub + uu;
                if ((uu & 3) == 0) {
#pragma unroll
                    for (int c = 0; c < 4; ++c) wn[c] = *reinterpret_cast<const float4 *>(wr + c * L + u);
                }
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    const float v = (uu & 3) == 0 ? wn[c].x : (uu & 3) == 1 ? wn[c].y : (uu & 3) == 2 ? wn[c].z : wn[c].w;
                    w[c][uu] = make_float2(v, v);
                }
                const float4 sx = ssm[(size_t)(0 * SEG + u) * RCH4];
                const float4 sy = ssm[(size_t)(1 * SEG + u) * RCH4];
                const float4 sz = ssm[(size_t)(2 * SEG + u) * RCH4];
                const float2 sx2[2] = {make_float2(sx.x, sx.y), make_float2(sx.z, sx.w)};
                const float2 sy2[2] = {make_float2(sy.x, sy.y), make_float2(sy.z, sy.w)};
                const float2 sz2[2] = {make_float2(sz.x, sz.y), make_float2(sz.z, sz.w)};
#pragma unroll
                for (int j = 0; j < TT; ++j) {
                    const int slot = (uu - j) & 7;
                    const float2 wxx = w[0][slot], wxy = w[1][slot], wyy = w[2][slot], wzz = w[3][slot];
#pragma unroll
                    for (int k = 0; k < 2; ++k) {
                        acc[j][0][k] = __ffma2_rn(wxx, sx2[k], acc[j][0][k]);
                        acc[j][0][k] = __ffma2_rn(wxy, sy2[k], acc[j][0][k]);
                        acc[j][1][k] = __ffma2_rn(wxy, sx2[k], acc[j][1][k]);
                        acc[j][1][k] = __ffma2_rn(wyy, sy2[k], acc[j][1][k]);
                        acc[j][2][k] = __ffma2_rn(wzz, sz2[k], acc[j][2][k]);
                    }
                }
            }
        }
        __syncthreads();  // everyone is done reading buffer b
        if (tid < 32 && st + NSTAGE < nstages) produce(st + NSTAGE);
    }

    if (live) {
        float *out = p.out + (size_t)ks * 3 * plane;
        const size_t a0 = (size_t)yt * Lh + (size_t)TT * g;
#pragma unroll
        for (int j = 0; j < TT; ++j)
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                float4 v = make_float4(acc[j][c][0].x, acc[j][c][0].y, acc[j][c][1].x, acc[j][c][1].y);
                *reinterpret_cast<float4 *>(out + (size_t)c * plane + (a0 + j) * R + r0 + 4 * rt) = v;
            }
    }
}

// H[c][a][r] = sum over ks of Hpart[ks][c][a][r], fixed order
__global__ void __launch_bounds__(256) reduce_partials_kernel(const float4 *__restrict__ part, float4 *__restrict__ out,
                                                              size_t n4, int KS) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n4) return;
    float4 s = part[i];
    for (int k = 1; k < KS; ++k) {
        const float4 v = part[(size_t)k * n4 + i];
        s.x += v.x; s.y += v.y; s.z += v.z; s.w += v.w;
    }
    out[i] = s;
}

__global__ void __launch_bounds__(256) make_wk_kernel(const float *__restrict__ Wc, float *__restrict__ Wk, int L) {
    const size_t total = (size_t)16 * L * L;
    const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= total) return;
    const int Lh = L >> 1;
    const int kk = (int)(t % L);
    size_t rest = t / L;
    const int c = (int)(rest % 4); rest /= 4;
    const int dy = (int)(rest % L); rest /= L;
    const int pt = (int)(rest % 2);
    const int cl = (int)(rest / 2);
    int dx = 2 * (kk - Lh) + ((pt + dy + cl) & 1) - pt;
    dx %= L;
    dx += dx < 0 ? L : 0;
    Wk[t] = Wc[(size_t)c * L * L + (size_t)dy * L + dx];
}

struct TiledPlan {
    int RT, NG, RCH, SEG, nrows_max, KS, tiles, rchunks;
    size_t smem;
};

bool make_plan(int L, int R, int sm_count, TiledPlan &pl) {
    if (L % 16 != 0 || R % 4 != 0 || L > DSMC_TILED_MAX_L) return false;
    const int Lh = L / 2, GPR = Lh / TT;
    const int rq = R / 4;
    int RT = 1;
    for (int d = 1; d <= 16; ++d)
        if (rq % d == 0) RT = d;
    pl.RT = RT;
    pl.RCH = 4 * RT;
    pl.rchunks = rq / RT;
    pl.NG = MAX_THREADS / RT;
    const int total_groups = L * GPR;
    if (pl.NG > total_groups) pl.NG = total_groups;
    pl.tiles = (total_groups + pl.NG - 1) / pl.NG;
    pl.nrows_max = (pl.NG + GPR - 1) / GPR + ((pl.NG % GPR) ? 1 : 0);
    if (pl.nrows_max > L) pl.nrows_max = L;
    // stage size: largest SEG (multiple of 8 dividing Lh) whose double-buffered footprint fits
    int seg = 0;
    for (int s = Lh; s >= 8; s -= 8) {
        if (Lh % s) continue;
        const size_t stage = (size_t)(pl.nrows_max * 4 * L + 3 * s * pl.RCH) * 4;
        if ((size_t)3 * s * pl.RCH * 4 <= 48 * 1024 && NSTAGE * stage + 64 <= 200 * 1024) { seg = s; break; }
    }
    if (!seg) return false;
    pl.SEG = seg;
    pl.smem = (size_t)NSTAGE * (pl.nrows_max * 4 * L + 3 * seg * pl.RCH) * 4 + 64;
    // source split: enough CTAs for ~8 waves, rows per chunk integral
    int KS = 1;
    while (KS < DSMC_KS_MAX && (L % (2 * KS) == 0) && (long)pl.tiles * pl.rchunks * KS < 8L * sm_count) KS *= 2;
    pl.KS = KS;
    return true;
}

}  // namespace

size_t dsmc_wk_floats(int L) { return (L % 16 == 0 && L <= DSMC_TILED_MAX_L) ? (size_t)16 * L * L : 64; }

bool dsmc_tiled_supported(int L, int R) {
    TiledPlan pl;
    return make_plan(L, R, 148, pl);
}

cudaError_t launch_make_wk(const float *Wc, float *Wk, int L, cudaStream_t st, uint64_t *launches) {
    const size_t total = (size_t)16 * L * L;
    make_wk_kernel<<<(unsigned)((total + 255) / 256), 256, 0, st>>>(Wc, Wk, L);
    ++*launches;
    return cudaGetLastError();
}

cudaError_t launch_field_tiled(const float *S, const float *Wk, float *Hpart, float *H, int L, int R, int colour,
                               int sm_count, bool *configured, cudaStream_t st, uint64_t *launches) {
    TiledPlan pl;
    if (!make_plan(L, R, sm_count, pl)) return cudaErrorInvalidValue;
    const size_t plane = (size_t)L * (L / 2) * R;
    float *Hc = H + (size_t)colour * 3 * plane;
    TiledParams p;
    p.S = S;
    p.Wk = Wk;
    p.out = pl.KS > 1 ? Hpart : Hc;
    p.L = L;
    p.R = R;
    p.colour = colour;
    p.RT = pl.RT;
    p.NG = pl.NG;
    p.RCH = pl.RCH;
    p.SEG = pl.SEG;
    p.nrows_max = pl.nrows_max;
    p.rows_per_chunk = L / pl.KS;
    p.total_groups = L * (L / 16);
    if (!*configured) {                                          // per context, hence per device: no process-global state
        cudaError_t e = cudaFuncSetAttribute(field_tiled_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 210 * 1024);
        if (e != cudaSuccess) return e;
        *configured = true;
    }
    dim3 grid(pl.tiles, pl.KS, pl.rchunks);
    field_tiled_kernel<<<grid, (pl.NG * pl.RT + 31) / 32 * 32, pl.smem, st>>>(p);
    ++*launches;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    if (pl.KS > 1) {
        const size_t n4 = 3 * plane / 4;
        reduce_partials_kernel<<<(unsigned)((n4 + 255) / 256), 256, 0, st>>>(reinterpret_cast<const float4 *>(Hpart),
                                                                             reinterpret_cast<float4 *>(Hc), n4, pl.KS);
        ++*launches;
        e = cudaGetLastError();
    }
    return e;
}
