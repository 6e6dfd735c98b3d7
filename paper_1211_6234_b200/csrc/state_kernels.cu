// state_kernels.cu -- canonical <-> internal layout transposes and a3: observables.
#include "dsmc_internal.cuh"

namespace {

// canonical s[r][c][y][x]  <->  internal S[q][c][a][r].  One block handles, for a fixed (c, y),
// a tile of 32 x-values by 32 replicas through a padded shared tile, so that both the canonical
// side (contiguous in x) and the internal side (contiguous in r) are coalesced.
template <bool TO_INTERNAL>
__global__ void __launch_bounds__(256) transpose_kernel(float *__restrict__ canon, float *__restrict__ S,
                                                        int L, int R, int colour) {
    __shared__ float tile[32][33];
    const int Lh = L >> 1;
    const size_t Nh = (size_t)L * Lh, N = 2 * Nh, plane = Nh * (size_t)R;
    const int x0 = blockIdx.x * 32, r0 = blockIdx.y * 32;
    const int c = blockIdx.z % 3, y = blockIdx.z / 3;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;  // 32 x 8
    if (TO_INTERNAL) {
        for (int k = ty; k < 32; k += 8) {  // k = replica within tile, tx = x within tile
            const int r = r0 + k, x = x0 + tx;
            if (r < R && x < L) tile[k][tx] = canon[((size_t)r * 3 + c) * N + (size_t)y * L + x];
        }
        __syncthreads();
        for (int k = ty; k < 32; k += 8) {  // k = x within tile, tx = replica within tile
            const int r = r0 + tx, x = x0 + k;
            if (r < R && x < L) {
                const int q = (x + y) & 1;
                S[((size_t)q * 3 + c) * plane + ((size_t)y * Lh + (x >> 1)) * R + r] = tile[tx][k];
            }
        }
    } else {
        for (int k = ty; k < 32; k += 8) {
            const int r = r0 + tx, x = x0 + k;
            if (r < R && x < L) {
                const int q = (x + y) & 1;
                tile[tx][k] = S[((size_t)q * 3 + c) * plane + ((size_t)y * Lh + (x >> 1)) * R + r];
            }
        }
        __syncthreads();
        for (int k = ty; k < 32; k += 8) {
            const int r = r0 + k, x = x0 + tx;
            if (r < R && x < L && (colour < 0 || ((x + y) & 1) == colour))
                canon[((size_t)r * 3 + c) * N + (size_t)y * L + x] = tile[k][tx];
        }
    }
}

// ---------------------------------------------------------------------------------------------
// Deterministic per-replica reductions (a3; north_star "warp-shuffle reductions for the observables").
// The walks below give every thread ONE replica (replica-innermost layout: a warp reads 32 consecutive replicas of
// one site, coalesced) and a fixed list of sites, so a thread's running sums have a fixed order.  What is left is
// to add, for every replica, the partial sums of the threads that own it -- in an order that does not depend on
// scheduling, so that two runs give the same bits (no floating-point atomics anywhere):
//   1. inside a warp, when R divides 32, lanes l, l + R, ... own the same replica: xor-butterfly over the masks
//      16, ..., R (warp shuffles); every lane of a class ends with the same value, the order is fixed by the masks;
//   2. across the warps (or, for other R, across all threads) of the CTA through shared memory, in index order;
//   3. across CTAs: per-CTA partials go to a scratch array part[cta][slot][K]; the last CTA to arrive (ticket from
//      an integer atomic, which only decides WHO sums, not in which order) adds them in CTA-index order and writes
//      out[r][8].  The ticket counter is left at zero for the next launch.
// slot = the replica for R <= block (every CTA starts at replica 0), else the thread index (each replica at most
// once per CTA).
// ---------------------------------------------------------------------------------------------
constexpr int kWalkBlockMax = 256;
constexpr int kWalkGridMax = 592;  // 4 CTAs per SM

template <typename T>
__device__ __forceinline__ T shfl_xor_any(T v, int mask) {
    return __shfl_xor_sync(0xFFFFFFFFu, v, mask);
}

// acc[K]: this thread's sums for replica (gid % R).  sm: blockDim.x * K values of T.
template <int K, typename T>
__device__ __forceinline__ void replica_reduce(T (&acc)[K], T *sm, T *__restrict__ part, T *__restrict__ out,
                                               unsigned int *__restrict__ ticket, int R) {
    const int tid = threadIdx.x, nthr = blockDim.x, lane = tid & 31, warp = tid >> 5;
    const bool pow2_in_warp = R < 32 && (R & (R - 1)) == 0 && (nthr & 31) == 0;
    int E;  // entries in shared memory after step 1; entry e belongs to replica (first_replica_of_cta + e) % R
    if (pow2_in_warp) {
        for (int mask = 16; mask >= R; mask >>= 1)
#pragma unroll
            for (int k = 0; k < K; ++k) acc[k] += shfl_xor_any(acc[k], mask);
        if (lane < R)
#pragma unroll
            for (int k = 0; k < K; ++k) sm[(warp * R + lane) * K + k] = acc[k];
        E = (nthr >> 5) * R;
    } else {
#pragma unroll
        for (int k = 0; k < K; ++k) sm[tid * K + k] = acc[k];
        E = nthr;
    }
    __syncthreads();
    const int slots = R < E ? R : E;
    if (tid < slots) {
        T tot[K];
#pragma unroll
        for (int k = 0; k < K; ++k) tot[k] = T(0);
        for (int e = tid; e < E; e += R)                        // index order
#pragma unroll
            for (int k = 0; k < K; ++k) tot[k] += sm[e * K + k];
        T *dst = part + ((size_t)blockIdx.x * slots + tid) * K;
#pragma unroll
        for (int k = 0; k < K; ++k) dst[k] = tot[k];
    }
    __threadfence();
    __syncthreads();
    __shared__ unsigned int s_last;
    if (tid == 0) s_last = atomicAdd(ticket, 1u) == gridDim.x - 1 ? 1u : 0u;
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    for (int r = tid; r < R; r += nthr) {
        T tot[K];
#pragma unroll
        for (int k = 0; k < K; ++k) tot[k] = T(0);
        for (unsigned b = 0; b < gridDim.x; ++b) {             // CTA-index order
            int slot = r;
            if (R > nthr) {                                     // CTA b holds replicas (b nthr + t) % R, t < nthr
                const long long first = ((long long)b * nthr) % R;
                slot = (int)((r - first + R) % R);
                if (slot >= nthr) continue;
            }
            const T *src = part + ((size_t)b * slots + slot) * K;
#pragma unroll
            for (int k = 0; k < K; ++k) tot[k] += __ldcg(src + k);
        }
#pragma unroll
        for (int k = 0; k < K; ++k) out[(size_t)r * 8 + k] = tot[k];
    }
    if (tid == 0) *ticket = 0u;
}

// Observables (PAPER.md:150 eq. 11, :225 eq. 16, :232 eq. 17).  Per replica seven sums:
//   0 sum s_x, 1 sum s_y, 2 sum s_z, 3 sum (arccos s_z - pi/2)^2,
//   4 sum_bonds s.s (each bond once: east and north), 5 sum K2 s_z^2 + K4 s_z^4, 6 sum s.h
// fp32 per-site terms added into fp64 running sums; reduced by replica_reduce (deterministic).
__global__ void __launch_bounds__(kWalkBlockMax) observables_kernel(const float *__restrict__ S, const float *__restrict__ H,
                                                                    const float *__restrict__ K2, const float *__restrict__ K4,
                                                                    double *__restrict__ obs, double *__restrict__ part,
                                                                    unsigned int *__restrict__ ticket, int L, int R) {
    extern __shared__ double sm[];  // [blockDim.x][7]
    pdl_wait();                     // spins and field come from earlier kernels (dependent launch in the record chain)
    const int Lh = L >> 1;
    const size_t Nh = (size_t)L * Lh, plane = Nh * (size_t)R;
    const size_t nthreads = (size_t)gridDim.x * blockDim.x;
    const size_t gid = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int r = (int)(gid % (size_t)R);
    double acc[7] = {0, 0, 0, 0, 0, 0, 0};
    const float k2 = K2[r], k4 = K4[r];
    for (size_t t = gid; t < 2 * plane; t += nthreads) {  // t % R == r for every iteration
        const size_t qa = t / (size_t)R;
        const int q = (int)(qa / Nh);
        const int a = (int)(qa - (size_t)q * Nh);
        const int y = a / Lh, i = a - y * Lh;
        const int par = (y + q) & 1;
        const float *own = S + (size_t)q * 3 * plane + (size_t)a * R + r;
        const float *oth = S + (size_t)(1 - q) * 3 * plane + r;
        const float *hf = H + (size_t)q * 3 * plane + (size_t)a * R + r;
        const int ie = par ? (i + 1 == Lh ? 0 : i + 1) : i;
        const int yn = (y + 1 == L) ? 0 : y + 1;
        const size_t ae = ((size_t)y * Lh + ie) * R, an = ((size_t)yn * Lh + i) * R;
        const float sx = own[0], sy = own[plane], sz = own[2 * plane];
        const float bond = sx * (oth[ae] + oth[an]) + sy * (oth[plane + ae] + oth[plane + an]) +
                           sz * (oth[2 * plane + ae] + oth[2 * plane + an]);
        const float z2 = sz * sz;
        const float th = acosf(fminf(1.0f, fmaxf(-1.0f, sz))) - 1.57079632679489662f;
        acc[0] += sx;
        acc[1] += sy;
        acc[2] += sz;
        acc[3] += th * th;
        acc[4] += bond;
        acc[5] += z2 * (k2 + k4 * z2);
        acc[6] += sx * hf[0] + sy * hf[plane] + sz * hf[2 * plane];
    }
    pdl_trigger();
    replica_reduce<7, double>(acc, sm, part, obs, ticket, R);
}

// Domain-wall counts (eq. 14): per replica and component a,
//   n_h^a = sum_i 1 - sgn(s_i^a) sgn(s_{i+x}^a),   n_v^a = sum_i 1 - sgn(s_i^a) sgn(s_{i+y}^a),
// every bond once (east and north neighbour of every site), sgn(0) = 0: integer terms 0, 1, 2.
// Same thread-owns-a-replica walk and the same reduction (exact integers in any order; 64-bit partials).
__device__ __forceinline__ int sgnf(float v) { return (v > 0.0f) - (v < 0.0f); }

__global__ void __launch_bounds__(kWalkBlockMax) wall_counts_kernel(const float *__restrict__ S,
                                                                    unsigned long long *__restrict__ counts,
                                                                    unsigned long long *__restrict__ part,
                                                                    unsigned int *__restrict__ ticket, int L, int R) {
    extern __shared__ unsigned long long wsm[];  // [blockDim.x][6]
    pdl_wait();
    const int Lh = L >> 1;
    const size_t Nh = (size_t)L * Lh, plane = Nh * (size_t)R;
    const size_t nthreads = (size_t)gridDim.x * blockDim.x;
    const size_t gid = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int r = (int)(gid % (size_t)R);
    unsigned long long acc[6] = {0, 0, 0, 0, 0, 0};
    for (size_t t = gid; t < 2 * plane; t += nthreads) {
        const size_t qa = t / (size_t)R;
        const int q = (int)(qa / Nh);
        const int a = (int)(qa - (size_t)q * Nh);
        const int y = a / Lh, i = a - y * Lh;
        const int par = (y + q) & 1;
        const float *own = S + (size_t)q * 3 * plane + (size_t)a * R + r;
        const float *oth = S + (size_t)(1 - q) * 3 * plane + r;
        const int ie = par ? (i + 1 == Lh ? 0 : i + 1) : i;
        const int yn = (y + 1 == L) ? 0 : y + 1;
        const size_t ae = ((size_t)y * Lh + ie) * R, an = ((size_t)yn * Lh + i) * R;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const int si = sgnf(own[c * plane]);
            acc[2 * c + 0] += (unsigned long long)(1 - si * sgnf(oth[c * plane + ae]));
            acc[2 * c + 1] += (unsigned long long)(1 - si * sgnf(oth[c * plane + an]));
        }
    }
    pdl_trigger();
    replica_reduce<6, unsigned long long>(acc, wsm, part, counts, ticket, R);
}

// Sub-lattice sums of s_z over the 2 x 2 plaquette (App. B): per replica four fp64 sums,
// index 0 = (x even, y even), 1 = (x odd, y even), 2 = (x odd, y odd), 3 = (x even, y odd).
__global__ void __launch_bounds__(kWalkBlockMax) staggered_kernel(const float *__restrict__ S, double *__restrict__ sums,
                                                                  double *__restrict__ part,
                                                                  unsigned int *__restrict__ ticket, int L, int R) {
    extern __shared__ double ssm[];  // [blockDim.x][4]
    const int Lh = L >> 1;
    const size_t Nh = (size_t)L * Lh, plane = Nh * (size_t)R;
    const size_t nthreads = (size_t)gridDim.x * blockDim.x;
    const size_t gid = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int r = (int)(gid % (size_t)R);
    double acc[4] = {0, 0, 0, 0};
    for (size_t t = gid; t < 2 * plane; t += nthreads) {
        const size_t qa = t / (size_t)R;
        const int q = (int)(qa / Nh);
        const int a = (int)(qa - (size_t)q * Nh);
        const int y = a / Lh, i = a - y * Lh;
        const int x = 2 * i + ((y + q) & 1);
        const int lambda = (y & 1) ? ((x & 1) ? 2 : 3) : ((x & 1) ? 1 : 0);
        const float sz = S[((size_t)q * 3 + 2) * plane + (size_t)a * R + r];
#pragma unroll
        for (int k = 0; k < 4; ++k) acc[k] += (k == lambda) ? (double)sz : 0.0;
    }
    replica_reduce<4, double>(acc, ssm, part, sums, ticket, R);
}

// Debug check of dsmc_set_spins: the largest | |s|^2 - 1 | over every site and replica.  Warp-shuffle
// maximum, then one integer atomicMax per warp on the bit pattern (non-negative floats order like unsigned integers,
// and a maximum does not depend on the order it is taken in).  *out is zero on entry.
__global__ void __launch_bounds__(256) norm_check_kernel(const float *__restrict__ S, unsigned int *__restrict__ out, size_t plane) {
    float worst = 0.0f;
    for (size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x; t < 2 * plane; t += (size_t)gridDim.x * blockDim.x) {
        const size_t q = t / plane, ar = t - q * plane;
        const float *p = S + q * 3 * plane + ar;
        const float sx = p[0], sy = p[plane], sz = p[2 * plane];
        const float dev = fabsf(fmaf(sx, sx, fmaf(sy, sy, sz * sz)) - 1.0f);
        worst = fmaxf(worst, dev == dev ? dev : 3.0e38f);      // a NaN spin counts as a violation
    }
#pragma unroll
    for (int mask = 16; mask >= 1; mask >>= 1) worst = fmaxf(worst, __shfl_xor_sync(0xFFFFFFFFu, worst, mask));
    if ((threadIdx.x & 31) == 0) atomicMax(out, __float_as_uint(worst));
}

// Ensemble accumulator (PAPER.md:175-177 eq. 13; :265 eq. 18): one thread per replica turns the raw sums
// of observables_kernel and the counts of wall_counts_kernel into the eight per-snapshot quantities
//   E/N, m_z, M_par, eta, wall density, O_x, O_y, O_z
// and adds x and x^2 to the running sums stats[r][k][2] (fp64), all on the device.
__global__ void ensemble_add_kernel(const double *__restrict__ obs, const unsigned long long *__restrict__ walls,
                                    double *__restrict__ stats, int L, int R, double J, double g) {
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    pdl_trigger();
    if (r >= R) return;
    pdl_wait();
    const double N = (double)L * L;
    const double *s = obs + 8 * (size_t)r;
    const unsigned long long *n = walls + 8 * (size_t)r;
    double x[8];
    const double mx = s[0] / N, my = s[1] / N;
    x[0] = (-J * s[4] - s[5] + 0.5 * g * s[6]) / N;
    x[1] = s[2] / N;
    x[2] = sqrt(mx * mx + my * my);
    x[3] = (2.0 / 3.14159265358979323846) * sqrt(s[3] / N);
    x[4] = (double)(n[4] + n[5]) / (4.0 * N);
    for (int c = 0; c < 3; ++c) {
        const unsigned long long nh = n[2 * c], nv = n[2 * c + 1];
        x[5 + c] = nh + nv ? (double)(nh > nv ? nh - nv : nv - nh) / (double)(nh + nv) : 0.0;
    }
    double *dst = stats + 16 * (size_t)r;
    for (int k = 0; k < 8; ++k) {
        dst[2 * k] += x[k];
        dst[2 * k + 1] += x[k] * x[k];
    }
}

}  // namespace

cudaError_t launch_canon_to_internal(const float *canon, float *S, int L, int R, cudaStream_t st,
                                     uint64_t *launches) {
    dim3 grid((L + 31) / 32, (R + 31) / 32, 3 * L);
    transpose_kernel<true><<<grid, 256, 0, st>>>(const_cast<float *>(canon), S, L, R, -1);
    ++*launches;
    return cudaGetLastError();
}

cudaError_t launch_internal_to_canon(const float *S, float *canon, int L, int R, int colour, cudaStream_t st,
                                     uint64_t *launches) {
    dim3 grid((L + 31) / 32, (R + 31) / 32, 3 * L);
    transpose_kernel<false><<<grid, 256, 0, st>>>(canon, const_cast<float *>(S), L, R, colour);
    ++*launches;
    return cudaGetLastError();
}

// launch shape of the thread-owns-a-replica walks: grid * block is a multiple of R and at least R
void dsmc_replica_walk_shape(int L, int R, int *block_out, unsigned *grid_out) {
    // block size: a multiple of R when R <= 256 (every block then starts at replica 0), else 256 with a grid that
    // is a multiple of R / gcd(R, 256) so that gid % R stays aligned over the grid-stride walk
    int block = kWalkBlockMax;
    if (R <= kWalkBlockMax) block = (kWalkBlockMax / R) * R;
    size_t total = (size_t)L * L * R;
    size_t want = (total + block - 1) / block;
    unsigned grid = (unsigned)(want < (size_t)kWalkGridMax ? want : (size_t)kWalkGridMax);
    if (R > kWalkBlockMax) {
        int g = R, b = kWalkBlockMax;
        while (b) { int t = g % b; g = b; b = t; }
        const unsigned step = (unsigned)(R / g);
        grid = ((grid + step - 1) / step) * step;
    }
    *block_out = block;
    *grid_out = grid;
}

// bytes of the per-CTA partial-sum scratch of the walks (8 values of 8 bytes per slot)
size_t dsmc_walk_scratch_bytes(int L, int R) {
    int block;
    unsigned grid;
    dsmc_replica_walk_shape(L, R, &block, &grid);
    const size_t slots = (size_t)(R < block ? R : block);
    return (size_t)grid * slots * 8 * sizeof(double);
}

cudaError_t launch_observables(const float *S, const float *H, const float *K2, const float *K4, double *obs, double *part,
                               unsigned int *ticket, int L, int R, cudaStream_t st, uint64_t *launches) {
    int block;
    unsigned grid;
    dsmc_replica_walk_shape(L, R, &block, &grid);
    const cudaError_t e = launch_pdl(observables_kernel, dim3(grid), dim3(block), sizeof(double) * 7 * block, st, S, H, K2, K4,
                                     obs, part, ticket, L, R);
    ++*launches;
    return e != cudaSuccess ? e : cudaGetLastError();
}

cudaError_t launch_wall_counts(const float *S, unsigned long long *counts, unsigned long long *part, unsigned int *ticket,
                               int L, int R, cudaStream_t st, uint64_t *launches) {
    int block;
    unsigned grid;
    dsmc_replica_walk_shape(L, R, &block, &grid);
    const cudaError_t e = launch_pdl(wall_counts_kernel, dim3(grid), dim3(block), sizeof(unsigned long long) * 6 * block, st, S,
                                     counts, part, ticket, L, R);
    ++*launches;
    return e != cudaSuccess ? e : cudaGetLastError();
}

cudaError_t launch_staggered(const float *S, double *sums, double *part, unsigned int *ticket, int L, int R, cudaStream_t st,
                             uint64_t *launches) {
    int block;
    unsigned grid;
    dsmc_replica_walk_shape(L, R, &block, &grid);
    staggered_kernel<<<grid, block, sizeof(double) * 4 * block, st>>>(S, sums, part, ticket, L, R);
    ++*launches;
    return cudaGetLastError();
}

cudaError_t launch_ensemble_add(const double *obs, const unsigned long long *walls, double *stats, int L, int R, double J,
                                double g, cudaStream_t st, uint64_t *launches) {
    const cudaError_t e = launch_pdl(ensemble_add_kernel, dim3((R + 127) / 128), dim3(128), 0, st, obs, walls, stats, L, R, J, g);
    ++*launches;
    return e != cudaSuccess ? e : cudaGetLastError();
}

cudaError_t launch_norm_check(const float *S, float *out, int L, int R, cudaStream_t st, uint64_t *launches) {
    const size_t plane = (size_t)L * (L / 2) * R;
    cudaError_t e = cudaMemsetAsync(out, 0, sizeof(float), st);
    if (e != cudaSuccess) return e;
    const size_t want = (2 * plane + 255) / 256;
    norm_check_kernel<<<(unsigned)(want < 1184 ? want : 1184), 256, 0, st>>>(S, reinterpret_cast<unsigned int *>(out), plane);
    ++*launches;
    return cudaGetLastError();
}
