// sublattice_kernels.cu -- the paper's own update schedule (section 3.1, App. A):
// stride-l sub-lattice passes, as two launches per pass (any shape) and with the lattice resident in shared
// memory for the whole run (L/l in {1, 2, 4}, L <= 74: the paper's L = 64, l = 32).
#include "metropolis_common.cuh"
#include "packed_f32x2.cuh"
#include <algorithm>

namespace {

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
    pdl_trigger();
    pdl_wait();                                                // spins and pass counter come from earlier kernels (section 5.8)
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
    pdl_trigger();
    pdl_wait();                                                // partial fields, spins and pass counter come from earlier kernels
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
//   * L/l = 4 (n = 16): the 16 W entries of a coset stay in registers and its 16 sources are streamed against all 16
//     targets; every lane of the drawing warp then has a site, so lane 0 draws the next offset with a second call.
// Needs L/l in {1, 2, 4} and 40 N bytes + partials within the 227 KB of one CTA (L <= 74).
constexpr int kResSumWarps = 8;   // measured at L = 64, l = 32: 8 warps 1.67, 12 warps 1.78, 16 warps 1.98 us per pass
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
            if constexpr (NL > 2) {
                // n = NL^2 > 4 update sites: the NL^2 distinct W entries of a coset stay in registers and its sources are
                // streamed one at a time against all n targets (3 LDS.64 per 5 n FFMA2)
                for (int c = tid; c < l * l; c += 32 * kResSumWarps) {
                    const int cy = c / l, cx = c - cy * l;
                    int dx[NL], dy[NL];
                    dx[0] = cx - ox + (cx < ox ? L : 0);
                    dy[0] = cy - oy + (cy < oy ? L : 0);
#pragma unroll
                    for (int u = 1; u < NL; ++u) {
                        dx[u] = dx[u - 1] + l - (dx[u - 1] + l >= L ? L : 0);
                        dy[u] = dy[u - 1] + l - (dy[u - 1] + l >= L ? L : 0);
                    }
                    float4 w[NL][NL];
#pragma unroll
                    for (int v = 0; v < NL; ++v)
#pragma unroll
                        for (int u = 0; u < NL; ++u) w[v][u] = Wsm[dy[v] * L + dx[u]];
                    const f2 *src0 = Ssm + 3 * (cy * L + cx);
#pragma unroll
                    for (int b = 0; b < NL; ++b)
#pragma unroll
                        for (int a = 0; a < NL; ++a) {
                            const f2 *src = src0 + 3 * (b * l * L + a * l);
                            const f2 ax = src[0], ay = src[1], az = src[2];
#pragma unroll
                            for (int k = 0; k < NN; ++k) {
                                const float4 ww = w[(b - k / NL + NL) % NL][(a - k % NL + NL) % NL];
                                acc[k][0] = f2_fma(f2_bc(ww.x), ax, f2_fma(f2_bc(ww.y), ay, acc[k][0]));
                                acc[k][1] = f2_fma(f2_bc(ww.y), ax, f2_fma(f2_bc(ww.z), ay, acc[k][1]));
                                acc[k][2] = f2_fma(f2_bc(ww.w), az, acc[k][2]);
                            }
                        }
                }
            } else {
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
            }
            // warp reduction of the 3 NN packed values in fixed order
            f2 *v = &acc[0][0];
            if constexpr (NL == 4) {
                halve_exchange<48>(v, lane, 16);
                halve_exchange<24>(v, lane, 8);
                halve_exchange<12>(v, lane, 4);
                halve_exchange<6>(v, lane, 2);
                butterfly_sum<3>(v, 1);
                if ((lane & 1) == 0) {                         // lane bits 4 .. 1 say which 3 of the 48 values it holds
#pragma unroll
                    for (int i = 0; i < 3; ++i) part[warp * 48 + (lane >> 1) * 3 + i] = v[i];
                }
            } else if constexpr (NL == 2) {
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
            if (2 * NN < 32 && lane == 31)
                ctr = make_uint4(0xFFFFFFFFu, 0xFFFFFFFFu, (uint32_t)((pass + 1) & 0xFFFFFFFFull),
                                 (uint32_t)((pass + 1) >> 32) & 0x7FFFFFFFu);
            const uint4 rnd = philox4x32_10(ctr, rk);
            if (2 * NN < 32 && lane == 31) {
                off[2 * (cur ^ 1)] = (int)(rnd.x % (uint32_t)l);
                off[2 * (cur ^ 1) + 1] = (int)(rnd.y % (uint32_t)l);
            }
            if constexpr (2 * NN >= 32) {                      // every lane has a site: lane 0 draws the next offset as well
                if (lane == 0) pass_offset(rk, pass + 1, l, off[2 * (cur ^ 1)], off[2 * (cur ^ 1) + 1]);
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

// ---------------------------------------------------------------------------------------------
// The same schedule with an INCREMENTAL field (section 3.2, eq. 8 read the
// other way round): after a pass only the accepted update sites have changed, so the dipole field of EVERY site
// changes by exactly  h_t += W(c - t) . delta_c  summed over the accepted sites c (delta = s' - s).  One CTA owns a
// replica pair as in sublattice_resident_kernel, but the 256 field threads keep the field of all N sites in registers
// (site t = tid + 256 j, j < 16: 48 packed values per thread) instead of summing over all N sources for the n update
// sites of every pass:
//   pass:  every field thread adds W(c - t) delta_c of the pass before to its 16 sites (for the c that were accepted),
//          then the owners publish h of this pass's n update sites | one drawing warp reads its sites' neighbours
//          -- barrier --  that warp decides and publishes delta_c (zero when rejected) | the OTHER drawing warp runs
//                         Philox for the next pass (offset, trial spins, ln u: none of it depends on the state)
//          -- barrier --
// Work per pass is 5 n N FMAs per replica pair only for accepted moves (the full sum costs 5 n N always), there is
// no reduction across threads, and a pass in which nothing was accepted costs two barriers.  The field is taken from
// the field array H at entry (the caller computes it with a field kernel) and written back at exit; rounding
// accumulates with every update, so the caller refreshes H every few thousand passes (dsmc_api.cu).
// Needs N <= 4096 (16 sites per thread) and L / l in {1, 2, 4}.
constexpr int kIncThreads = 256;
constexpr int kIncSpt = 16;       // sites per field thread

constexpr int kIncDraw = 3;      // drawing warps
__host__ __device__ constexpr size_t incremental_smem_bytes(int L, int NL) {
    return (size_t)40 * L * L + 16 + 2 * sizeof(f2) * NL * NL * 3 + 64 * 2 * sizeof(int) + 64;
}

template <int NL, int LC>
__global__ void __launch_bounds__(kIncThreads + 32 * kIncDraw, 1) sublattice_incremental_kernel(const MetropolisArgs p, const RoundKeys rk,
                                                                                  const float *__restrict__ Wc,
                                                                                  float *__restrict__ Hio, int l_arg,
                                                                                  unsigned long long first_pass,
                                                                                  unsigned n_passes,
                                                                                  float *__restrict__ margin_log) {
    constexpr int NN = NL * NL;
    constexpr int NT = kIncThreads + 32 * kIncDraw;                    // 8 field warps + 3 drawing warps
    extern __shared__ __align__(16) unsigned char rsm[];
    const int L = LC > 0 ? LC : p.L, l = LC > 0 ? LC / NL : l_arg, Lh = L >> 1, R = p.R, N = L * L;
    float4 *Wsm = reinterpret_cast<float4 *>(rsm);                     // [N + 1]  (xx, xy, yy, zz) at rho = ry L + rx
    f2 *Ssm = reinterpret_cast<f2 *>(rsm + (size_t)16 * (N + 1));      // [N][3]  replicas (r0, r1) of site n = y L + x
    float *Sf = reinterpret_cast<float *>(Ssm);
    f2 *hpub = Ssm + 3 * (size_t)N;                                    // [NN][3] field of the update sites
    float *dlf = reinterpret_cast<float *>(hpub + NN * 3);             // [NN][3][2] delta of the update sites (0 = rejected)
    int *offtab = reinterpret_cast<int *>(dlf + NN * 6);               // [64][2]: offsets of the passes it .. it + 63, slot it & 63
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int r0 = 2 * blockIdx.x, r1 = min(r0 + 1, R - 1);            // odd R: the last CTA carries its replica twice
    const size_t plane = (size_t)L * Lh * R;

    for (int n = tid; n < N; n += NT) {
        Wsm[n] = make_float4(__ldg(Wc + n), __ldg(Wc + (size_t)N + n), __ldg(Wc + 2 * (size_t)N + n),
                             __ldg(Wc + 3 * (size_t)N + n));
        const int x = n % L, y = n / L;
        int q;
        const float *src = p.S + site_index(x, y, Lh, R, plane, q);
        Ssm[3 * n] = f2_make(src[r0], src[r1]);
        Ssm[3 * n + 1] = f2_make(src[plane + r0], src[plane + r1]);
        Ssm[3 * n + 2] = f2_make(src[2 * plane + r0], src[2 * plane + r1]);
    }
    // the field of this thread's sites, from the field array
    f2 h[kIncSpt][3];
    int txy[kIncSpt];                                                  // x | y << 16 of the sites (-1: none)
#pragma unroll
    for (int j = 0; j < kIncSpt; ++j) {
        const int n = tid + kIncThreads * j;
        txy[j] = -1;
        h[j][0] = h[j][1] = h[j][2] = f2_bc(0.0f);
        if (tid < kIncThreads && n < N) {
            const int x = n % L, y = n / L;
            txy[j] = x | (y << 16);
            int q;
            const float *src = Hio + site_index(x, y, Lh, R, plane, q);
            h[j][0] = f2_make(src[r0], src[r1]);
            h[j][1] = f2_make(src[plane + r0], src[plane + r1]);
            h[j][2] = f2_make(src[2 * plane + r0], src[2 * plane + r1]);
        }
    }

    // Three drawing warps take the passes in turn.  The warp that decides pass k then has two whole passes to run Philox
    // for pass k + 3 (the trial spins and ln u of its sites: none of that depends on the state); the offsets of the next
    // 32-64 passes come from a table that one warp refills 32 at a time (one pass per lane), so the serial part of a
    // pass is only "read the neighbours, dE, accept".  Lanes: update site fk = lane >> 1, replica rb = lane & 1.
    // Barriers: A(it) = "h of this pass's sites is published", B(it) = "decisions and deltas of this pass are out":
    // named barriers 1..8 (A and B of pass it & 3) over all threads.  A drawing warp syncs on the barriers of its own
    // passes and only ARRIVES at those of the two passes in between (it has nothing to wait for there); four phases of
    // barrier ids keep an early arrival from ever landing in a phase that is still open.
    const bool drawer = warp >= kIncThreads / 32;
    const int dw = warp - kIncThreads / 32;
    const bool flipper = drawer && lane < 2 * NN;
    const int fk = lane >> 1, rb = lane & 1, fr = rb ? r1 : r0;
    float invT = 0.0f, K2 = 0.0f, K4 = 0.0f;
    if (flipper) invT = p.invT[fr], K2 = p.K2[fr], K4 = p.K4[fr];
    auto fill_offsets = [&](unsigned it0) {                            // passes it0 .. it0 + 31, one per lane
        int ox, oy;
        pass_offset(rk, first_pass + it0 + lane, l, ox, oy);
        offtab[2 * ((it0 + lane) & 63)] = ox, offtab[2 * ((it0 + lane) & 63) + 1] = oy;
    };
    if (drawer && dw == 0) fill_offsets(0), fill_offsets(32);
    __syncthreads();
    Draw dr = {0.0f, 0.0f, 0.0f, 0.0f};
    int my_ox = 0, my_oy = 0;
    auto predraw = [&](unsigned it) {                                  // trial spins and ln u of pass `it`
        my_ox = offtab[2 * (it & 63)], my_oy = offtab[2 * (it & 63) + 1];
        const unsigned long long ps = first_pass + it;
        const int nt = (my_oy + l * (fk / NL)) * L + my_ox + l * (fk % NL);
        const uint4 rnd = philox4x32_10(make_uint4((uint32_t)nt, (uint32_t)fr + p.r_off, (uint32_t)(ps & 0xFFFFFFFFull),
                                                   (uint32_t)(ps >> 32) & 0x7FFFFFFFu), rk);
        sphere_point(rnd.x, rnd.y, dr.tx, dr.ty, dr.tz);              // (the reversal move replaces it at decision time)
        dr.lnu = __logf(unit24(rnd.z));
    };
    auto bar_sync = [&](int id) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(NT) : "memory"); };
    auto bar_arrive = [&](int id) { asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(NT) : "memory"); };

    if (!drawer) {
        int pox = 0, poy = 0;                                          // the offsets of the pass before
        for (unsigned it = 0; it < n_passes; ++it) {
            const int ox = offtab[2 * (it & 63)], oy = offtab[2 * (it & 63) + 1];
            if (it > 0) {
                // rank-n update of the field of this thread's sites by the moves of the pass before:
                // h_t += W(c - t) . delta_c for the accepted c
                const f2 *dl = reinterpret_cast<const f2 *>(dlf);
#pragma unroll 1
                for (int k = 0; k < NN; ++k) {
                    const f2 dxp = dl[3 * k], dyp = dl[3 * k + 1], dzp = dl[3 * k + 2];
                    if ((dxp | dyp | dzp) == 0ull) continue;       // all six components +0: rejected in both replicas (uniform over the CTA)
                    const int xc = pox + l * (k % NL), yc = poy + l * (k / NL);
                    if constexpr (LC == 64) {
                        // site j of this thread is (tid & 63, (tid >> 6) + 4 j): rho_x is the same for all of them and
                        // the table index steps back by 4 rows = 256 entries from one to the next
                        const int idx0 = (((yc - (tid >> 6)) & 63) << 6) | ((xc - tid) & 63);
#pragma unroll
                        for (int j = 0; j < kIncSpt; ++j) {
                            const float4 w = Wsm[(idx0 - 256 * j) & 4095];
                            h[j][0] = f2_fma(f2_bc(w.x), dxp, f2_fma(f2_bc(w.y), dyp, h[j][0]));
                            h[j][1] = f2_fma(f2_bc(w.y), dxp, f2_fma(f2_bc(w.z), dyp, h[j][1]));
                            h[j][2] = f2_fma(f2_bc(w.w), dzp, h[j][2]);
                        }
                    } else {
#pragma unroll
                        for (int j = 0; j < kIncSpt; ++j) {
                            if (txy[j] < 0) continue;
                            int rx = xc - (txy[j] & 0xFFFF), ry = yc - (txy[j] >> 16);
                            rx += rx < 0 ? L : 0;
                            ry += ry < 0 ? L : 0;
                            const float4 w = Wsm[ry * L + rx];
                            h[j][0] = f2_fma(f2_bc(w.x), dxp, f2_fma(f2_bc(w.y), dyp, h[j][0]));
                            h[j][1] = f2_fma(f2_bc(w.y), dxp, f2_fma(f2_bc(w.z), dyp, h[j][1]));
                            h[j][2] = f2_fma(f2_bc(w.w), dzp, h[j][2]);
                        }
                    }
                }
            }
            // the owners publish the field of this pass's update sites (a register array cannot be indexed: compare and select)
#pragma unroll
            for (int k = 0; k < NN; ++k) {
                const int nk = (oy + l * (k / NL)) * L + ox + l * (k % NL);
                if ((nk % kIncThreads) == tid) {
                    const int jj = nk / kIncThreads;
                    f2 v0 = h[0][0], v1 = h[0][1], v2 = h[0][2];
#pragma unroll
                    for (int j = 1; j < kIncSpt; ++j)
                        if (j == jj) v0 = h[j][0], v1 = h[j][1], v2 = h[j][2];
                    hpub[3 * k] = v0, hpub[3 * k + 1] = v1, hpub[3 * k + 2] = v2;
                }
            }
            pox = ox, poy = oy;
            bar_sync(1 + 2 * (int)(it & 3u));
            bar_sync(2 + 2 * (int)(it & 3u));
        }
        // the moves of the last pass are still to be applied to the field that is handed back
        if (n_passes > 0) {
            const f2 *dl = reinterpret_cast<const f2 *>(dlf);
#pragma unroll 1
            for (int k = 0; k < NN; ++k) {
                const f2 dxp = dl[3 * k], dyp = dl[3 * k + 1], dzp = dl[3 * k + 2];
                if ((dxp | dyp | dzp) == 0ull) continue;
                const int xc = pox + l * (k % NL), yc = poy + l * (k / NL);
#pragma unroll
                for (int j = 0; j < kIncSpt; ++j) {
                    if (txy[j] < 0) continue;
                    int rx = xc - (txy[j] & 0xFFFF), ry = yc - (txy[j] >> 16);
                    rx += rx < 0 ? L : 0;
                    ry += ry < 0 ? L : 0;
                    const float4 w = Wsm[ry * L + rx];
                    h[j][0] = f2_fma(f2_bc(w.x), dxp, f2_fma(f2_bc(w.y), dyp, h[j][0]));
                    h[j][1] = f2_fma(f2_bc(w.y), dxp, f2_fma(f2_bc(w.z), dyp, h[j][1]));
                    h[j][2] = f2_fma(f2_bc(w.w), dzp, h[j][2]);
                }
            }
        }
    } else {
        // the passes before this warp's first one: nothing to wait for
        for (unsigned it = 0; it < (unsigned)dw && it < n_passes; ++it) bar_arrive(1 + 2 * (int)(it & 3u)), bar_arrive(2 + 2 * (int)(it & 3u));
        if ((unsigned)dw < n_passes) predraw((unsigned)dw);
        for (unsigned it = (unsigned)dw; it < n_passes; it += kIncDraw) {
            bar_sync(1 + 2 * (int)(it & 3u));
            // the deciding warp: everything that depends on the state, after the barrier that orders it behind the pass before
            if (flipper) {
                const int xt = my_ox + l * (fk % NL), yt = my_oy + l * (fk / NL);
                const int nt = yt * L + xt;
                const int xe = xt + 1 == L ? 0 : xt + 1, xw = xt == 0 ? L - 1 : xt - 1;
                const int yn = yt + 1 == L ? 0 : yt + 1, ys = yt == 0 ? L - 1 : yt - 1;
                const float *sc = Sf + 6 * nt + rb, *se = Sf + 6 * (yt * L + xe) + rb, *sw = Sf + 6 * (yt * L + xw) + rb,
                            *sn = Sf + 6 * (yn * L + xt) + rb, *ss = Sf + 6 * (ys * L + xt) + rb;
                const float sx = sc[0], sy = sc[2], sz = sc[4];
                const float nx = (se[0] + sw[0]) + (sn[0] + ss[0]);
                const float ny = (se[2] + sw[2]) + (sn[2] + ss[2]);
                const float nz = (se[4] + sw[4]) + (sn[4] + ss[4]);
                if (p.flip) dr.tx = -sx, dr.ty = -sy, dr.tz = -sz;     // Ising move of App. B: complete reversal
                const float *pf = reinterpret_cast<const float *>(hpub) + rb;
                const Trial tr = decide_drawn(p, dr, sx, sy, sz, nx, ny, nz, pf[6 * fk], pf[6 * fk + 2], pf[6 * fk + 4], invT, K2, K4);
                const bool live = r0 + rb < R;                         // the duplicate of an odd R's last replica stays silent
                float dx = 0.0f, dy = 0.0f, dz = 0.0f;
                if (tr.acc) {
                    dx = tr.tx - sx, dy = tr.ty - sy, dz = tr.tz - sz;
                    Sf[6 * nt + rb] = tr.tx;
                    Sf[6 * nt + 2 + rb] = tr.ty;
                    Sf[6 * nt + 4 + rb] = tr.tz;
                }
                dlf[6 * fk + rb] = dx, dlf[6 * fk + 2 + rb] = dy, dlf[6 * fk + 4 + rb] = dz;
                if (live) {
                    if (p.accept_out) p.accept_out[(size_t)fr * N + nt] = tr.acc ? 1 : 0;
                    if (p.margin_out) p.margin_out[(size_t)fr * N + nt] = tr.margin;
                    if (margin_log) margin_log[((size_t)it * R + fr) * NN + fk] = tr.margin;
                }
            }
            bar_sync(2 + 2 * (int)(it & 3u));
            // the two passes the other drawing warps decide
            for (unsigned j = it + 1; j < it + kIncDraw && j < n_passes; ++j) bar_arrive(1 + 2 * (int)(j & 3u)), bar_arrive(2 + 2 * (int)(j & 3u));
            // refill duty: whoever decided the first pass of a block of 32 computes the offsets of the block after the next
            // (the table holds passes it .. it + 63 then; the slots it overwrites belong to passes that are done)
            if ((it & 31u) == 0u && it > 0u) {
                fill_offsets(it + 32u);
                __threadfence_block();
            }
            if (it + kIncDraw < n_passes) predraw(it + kIncDraw);
        }
    }
    __syncthreads();
    for (int n = tid; n < N; n += NT) {
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
#pragma unroll
    for (int j = 0; j < kIncSpt; ++j) {
        if (txy[j] < 0) continue;
        int qc;
        float *dst = Hio + site_index(txy[j] & 0xFFFF, txy[j] >> 16, Lh, R, plane, qc);
        float a0, a1, b0, b1, c0, c1;
        f2_split(h[j][0], a0, a1);
        f2_split(h[j][1], b0, b1);
        f2_split(h[j][2], c0, c1);
        dst[r0] = a0, dst[plane + r0] = b0, dst[2 * plane + r0] = c0;
        if (r0 + 1 < R) dst[r1] = a1, dst[plane + r1] = b1, dst[2 * plane + r1] = c1;
    }
}

}  // namespace

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
        const cudaError_t e = launch_pdl(sublattice_field_kernel, dim3((unsigned)n, (unsigned)chunks, (unsigned)KS), dim3(256), 0,
                                         st, (const float *)a.S, scratch, Wc, a.L, a.R, l, ox, oy, rows, segs, a.step_dev, rk);
        ++*launches;
        if (e != cudaSuccess) return e;
    }
    const size_t total = (size_t)n * a.R;
    const cudaError_t e = launch_pdl(sublattice_flip_kernel, dim3((unsigned)((total + 127) / 128)), dim3(128), 0, st, a, rk,
                                     (const float *)scratch, KS, l, ox, oy);
    ++*launches;
    return e != cudaSuccess ? e : cudaGetLastError();
}

bool dsmc_resident_supported(int L, int l) {
    const int nl = L / l;
    return (nl == 1 || nl == 2 || nl == 4) && resident_smem_bytes(L, nl) <= 227 * 1024;
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
    else if (nl == 4) kern = a.L == 64 ? sublattice_resident_kernel<4, 0, 64> : sublattice_resident_kernel<4, 0, 0>;
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

bool dsmc_incremental_supported(int L, int l) {
    const int nl = L / l;
    return (nl == 1 || nl == 2 || nl == 4) && L * L <= kIncThreads * kIncSpt && incremental_smem_bytes(L, nl) <= 227 * 1024;
}

cudaError_t launch_sublattice_incremental(const MetropolisArgs &a, const float *Wc, float *H, int l, uint64_t first_pass,
                                          uint64_t n_passes, float *margin_log, cudaStream_t st, uint64_t *launches) {
    const RoundKeys rk = make_round_keys(a.seed_lo, a.seed_hi);
    const int nl = a.L / l;
    const size_t smem = incremental_smem_bytes(a.L, nl);
    void (*kern)(const MetropolisArgs, const RoundKeys, const float *, float *, int, unsigned long long, unsigned, float *) = nullptr;
    if (nl == 2) kern = a.L == 64 ? sublattice_incremental_kernel<2, 64> : sublattice_incremental_kernel<2, 0>;
    else if (nl == 4) kern = a.L == 64 ? sublattice_incremental_kernel<4, 64> : sublattice_incremental_kernel<4, 0>;
    else kern = a.L == 64 ? sublattice_incremental_kernel<1, 64> : sublattice_incremental_kernel<1, 0>;
    if (cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024)) return e;
    kern<<<(unsigned)((a.R + 1) / 2), kIncThreads + 32 * kIncDraw, smem, st>>>(a, rk, Wc, H, l, first_pass, (unsigned)n_passes, margin_log);
    ++*launches;
    return cudaGetLastError();
}
