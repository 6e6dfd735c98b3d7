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

// Observables (PAPER.md:150 eq. 11, :225 eq. 16, :232 eq. 17).  Per replica eight sums:
//   0 sum s_x, 1 sum s_y, 2 sum s_z, 3 sum (arccos s_z - pi/2)^2,
//   4 sum_bonds s.s (each bond once: east and north), 5 sum K2 s_z^2 + K4 s_z^4, 6 sum s.h
// Every thread owns one replica (total threads is a multiple of R), accumulates its sites in
// fp32 per-site terms added into fp64 running sums, then the block folds equal replicas in shared
// memory and issues one fp64 atomicAdd per (replica, sum).
__global__ void __launch_bounds__(256) observables_kernel(const float *__restrict__ S, const float *__restrict__ H,
                                                          const float *__restrict__ K2, const float *__restrict__ K4,
                                                          double *__restrict__ obs, int L, int R) {
    extern __shared__ double sm[];  // [blockDim.x][7] then folded
    pdl_wait();                     // spins and field come from earlier kernels (launch_pdl in the record chain)
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
    for (int k = 0; k < 7; ++k) sm[threadIdx.x * 7 + k] = acc[k];
    __syncthreads();
    // threads with the same replica inside the block are R apart (blockDim.x*blockIdx.x % R == 0)
    if ((int)threadIdx.x < R && threadIdx.x < blockDim.x) {
        double tot[7] = {0, 0, 0, 0, 0, 0, 0};
        for (int j = threadIdx.x; j < (int)blockDim.x; j += R)
            for (int k = 0; k < 7; ++k) tot[k] += sm[j * 7 + k];
        for (int k = 0; k < 7; ++k) atomicAdd(&obs[(size_t)r * 8 + k], tot[k]);
    }
}

// Domain-wall counts (eq. 14): per replica and component a,
//   n_h^a = sum_i 1 - sgn(s_i^a) sgn(s_{i+x}^a),   n_v^a = sum_i 1 - sgn(s_i^a) sgn(s_{i+y}^a),
// every bond once (east and north neighbour of every site), sgn(0) = 0: integer terms 0, 1, 2.
// Same thread-owns-a-replica walk as observables_kernel; 32-bit per-thread counts, folded per
// block in shared memory, one 64-bit integer atomicAdd per (replica, count).
__device__ __forceinline__ int sgnf(float v) { return (v > 0.0f) - (v < 0.0f); }

__global__ void __launch_bounds__(256) wall_counts_kernel(const float *__restrict__ S,
                                                          unsigned long long *__restrict__ counts, int L, int R) {
    extern __shared__ unsigned int wsm[];  // [blockDim.x][6]
    pdl_wait();
    const int Lh = L >> 1;
    const size_t Nh = (size_t)L * Lh, plane = Nh * (size_t)R;
    const size_t nthreads = (size_t)gridDim.x * blockDim.x;
    const size_t gid = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int r = (int)(gid % (size_t)R);
    unsigned int acc[6] = {0, 0, 0, 0, 0, 0};
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
            acc[2 * c + 0] += (unsigned int)(1 - si * sgnf(oth[c * plane + ae]));
            acc[2 * c + 1] += (unsigned int)(1 - si * sgnf(oth[c * plane + an]));
        }
    }
    pdl_trigger();
    for (int k = 0; k < 6; ++k) wsm[threadIdx.x * 6 + k] = acc[k];
    __syncthreads();
    if ((int)threadIdx.x < R) {
        unsigned long long tot[6] = {0, 0, 0, 0, 0, 0};
        for (int j = threadIdx.x; j < (int)blockDim.x; j += R)
            for (int k = 0; k < 6; ++k) tot[k] += wsm[j * 6 + k];
        for (int k = 0; k < 6; ++k) atomicAdd(&counts[(size_t)r * 8 + k], tot[k]);
    }
}

// Sub-lattice sums of s_z over the 2 x 2 plaquette (App. B): per replica four fp64 sums,
// index 0 = (x even, y even), 1 = (x odd, y even), 2 = (x odd, y odd), 3 = (x even, y odd).
__global__ void __launch_bounds__(256) staggered_kernel(const float *__restrict__ S, double *__restrict__ sums, int L,
                                                        int R) {
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
    for (int k = 0; k < 4; ++k) ssm[threadIdx.x * 4 + k] = acc[k];
    __syncthreads();
    if ((int)threadIdx.x < R) {
        double tot[4] = {0, 0, 0, 0};
        for (int j = threadIdx.x; j < (int)blockDim.x; j += R)
            for (int k = 0; k < 4; ++k) tot[k] += ssm[j * 4 + k];
        for (int k = 0; k < 4; ++k) atomicAdd(&sums[(size_t)r * 8 + k], tot[k]);
    }
}

// Ensemble accumulator (PAPER.md:175-177 eq. 13; :265 eq. 18): one thread per replica turns the raw sums
// of observables_kernel and the counts of wall_counts_kernel into the eight per-snapshot quantities
//   E/N, m_z, M_par, eta, wall density, O_x, O_y, O_z
// and adds x and x^2 to the running sums stats[r][k][2] (fp64), all on the device.
__global__ void ensemble_add_kernel(double *__restrict__ obs, unsigned long long *__restrict__ walls,
                                    double *__restrict__ stats, int L, int R, double J, double g) {
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    pdl_trigger();
    if (r >= R) return;
    pdl_wait();
    const double N = (double)L * L;
    double *s = obs + 8 * (size_t)r;
    unsigned long long *n = walls + 8 * (size_t)r;
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
    // the raw sums are consumed: leave them zero for the next record, which then needs no memset in front of the
    // atomics of observables_kernel / wall_counts_kernel (a memset node would cut the dependent-launch chain)
    for (int k = 0; k < 8; ++k) {
        s[k] = 0.0;
        n[k] = 0ull;
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

// launch shape of the thread-owns-a-replica walks: grid * block is a multiple of R
static void replica_walk_shape(int L, int R, int *block_out, unsigned *grid_out) {
    // block size: a multiple of R when R <= 256 (so that every block starts at replica 0),
    // else R threads-per-replica-row blocks of 256 with a grid that keeps gid % R aligned
    int block = 256;
    if (R <= 256) block = (256 / R) * R;
    size_t total = (size_t)L * L * R;
    size_t want = (total + block - 1) / block;
    unsigned grid = (unsigned)(want < 1184 ? want : 1184);
    if (R > 256) {  // make grid*block a multiple of R: use block = 256 and grid multiple of R/gcd(R,256)
        int g = R, b = 256;
        while (b) { int t = g % b; g = b; b = t; }
        const unsigned step = (unsigned)(R / g);
        grid = ((grid + step - 1) / step) * step;
    }
    *block_out = block;
    *grid_out = grid;
}

cudaError_t launch_observables(const float *S, const float *H, const float *K2, const float *K4, double *obs,
                               int L, int R, float, float, bool chained, cudaStream_t st, uint64_t *launches) {
    int block;
    unsigned grid;
    replica_walk_shape(L, R, &block, &grid);
    cudaError_t e;
    if (chained) {  // obs is zero on entry (ensemble_add_kernel leaves it so): dependent launch, no memset
        e = launch_pdl(observables_kernel, dim3(grid), dim3(block), sizeof(double) * 7 * block, st, S, H, K2, K4, obs, L, R);
    } else {
        e = cudaMemsetAsync(obs, 0, sizeof(double) * 8 * (size_t)R, st);
        if (e != cudaSuccess) return e;
        observables_kernel<<<grid, block, sizeof(double) * 7 * block, st>>>(S, H, K2, K4, obs, L, R);
    }
    ++*launches;
    return e != cudaSuccess ? e : cudaGetLastError();
}

cudaError_t launch_wall_counts(const float *S, unsigned long long *counts, int L, int R, bool chained, cudaStream_t st,
                               uint64_t *launches) {
    int block;
    unsigned grid;
    replica_walk_shape(L, R, &block, &grid);
    cudaError_t e;
    if (chained) {
        e = launch_pdl(wall_counts_kernel, dim3(grid), dim3(block), sizeof(unsigned int) * 6 * block, st, S, counts, L, R);
    } else {
        e = cudaMemsetAsync(counts, 0, sizeof(unsigned long long) * 8 * (size_t)R, st);
        if (e != cudaSuccess) return e;
        wall_counts_kernel<<<grid, block, sizeof(unsigned int) * 6 * block, st>>>(S, counts, L, R);
    }
    ++*launches;
    return e != cudaSuccess ? e : cudaGetLastError();
}

cudaError_t launch_staggered(const float *S, double *sums, int L, int R, cudaStream_t st, uint64_t *launches) {
    cudaError_t e = cudaMemsetAsync(sums, 0, sizeof(double) * 8 * (size_t)R, st);
    if (e != cudaSuccess) return e;
    int block;
    unsigned grid;
    replica_walk_shape(L, R, &block, &grid);
    staggered_kernel<<<grid, block, sizeof(double) * 4 * block, st>>>(S, sums, L, R);
    ++*launches;
    return cudaGetLastError();
}

cudaError_t launch_ensemble_add(double *obs, unsigned long long *walls, double *stats, int L, int R, double J,
                                double g, cudaStream_t st, uint64_t *launches) {
    const cudaError_t e = launch_pdl(ensemble_add_kernel, dim3((R + 127) / 128), dim3(128), 0, st, obs, walls, stats, L, R, J, g);
    ++*launches;
    return e != cudaSuccess ? e : cudaGetLastError();
}
