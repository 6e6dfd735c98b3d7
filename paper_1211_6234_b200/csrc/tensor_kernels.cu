// tensor_kernels.cu -- a0: lattice-summed dipole interaction table W (eq. 1-5).
// Run once per context; fp64 arithmetic on the device, one rounding to fp32 at the store.
#include "dsmc_internal.cuh"

namespace {

constexpr double kPi = 3.141592653589793238462643383279502884;

// Ewald parameters (R5): alpha = kAlphaL / L; with these cutoffs the neglected
// terms are below exp(-200) in both sums.
constexpr double kAlphaL = 2.5;
constexpr int kNReal = 6;
constexpr int kNK = 12;

__device__ __forceinline__ int sym_reduce(int rho, int L) { return rho <= L / 2 ? rho : rho - L; }

// One thread block per table entry rho; the threads of the block split the image / k sums and
// reduce in shared memory in a fixed order (deterministic).
template <int BLOCK>
__global__ void __launch_bounds__(BLOCK) build_tensor_kernel(float *__restrict__ Wc, int L, int method,
                                                            int A, int tail) {
    const int rho = blockIdx.x;
    const int rx = rho % L, ry = rho / L;
    const double dx = (double)sym_reduce(rx, L), dy = (double)sym_reduce(ry, L);
    const double Ld = (double)L;
    double axx = 0.0, axy = 0.0, ayy = 0.0, azz = 0.0;

    if (method == DSMC_W_IMAGE) {
        // W(rho) = sum over images |a|,|b| <= A of (delta - 3 rhat rhat)/r^3  (eq. 1 bracket)
        const int side = 2 * A + 1;
        for (int t = threadIdx.x; t < side * side; t += BLOCK) {
            const int a = t % side - A, b = t / side - A;
            const double x = dx + a * Ld, y = dy + b * Ld;
            const double r2 = x * x + y * y;
            if (r2 == 0.0) continue;  // G = 0 at rho = 0: the self-image term excludes it
            const double inv_r = rsqrt(r2);
            const double inv_r3 = inv_r * inv_r * inv_r;
            const double ux = x * inv_r, uy = y * inv_r;
            axx += (1.0 - 3.0 * ux * ux) * inv_r3;
            axy += (-3.0 * ux * uy) * inv_r3;
            ayy += (1.0 - 3.0 * uy * uy) * inv_r3;
            azz += inv_r3;
        }
    } else {
        // 2-D Ewald (eq. 3-5 at z = 0), alpha = 1/(2 eta)
        const double alpha = kAlphaL / Ld, eta = 0.5 / alpha;
        const double c1 = 2.0 * alpha / sqrt(kPi);
        const double inv_area = 1.0 / (Ld * Ld);
        constexpr int sr = 2 * kNReal + 1, sk = 2 * kNK + 1;
        for (int t = threadIdx.x; t < sr * sr; t += BLOCK) {  // short-range part f_S
            const int a = t % sr - kNReal, b = t / sr - kNReal;
            const double x = dx + a * Ld, y = dy + b * Ld;
            const double r2 = x * x + y * y;
            if (r2 == 0.0) continue;
            const double r = sqrt(r2);
            const double ec = erfc(alpha * r), ex = exp(-alpha * alpha * r2);
            const double B = ec / (r2 * r) + c1 * ex / r2;
            const double C = 3.0 * ec / (r2 * r2 * r) + c1 * (2.0 * alpha * alpha + 3.0 / r2) * ex / r2;
            axx += B - x * x * C;
            axy += -x * y * C;
            ayy += B - y * y * C;
            azz += B;
        }
        for (int t = threadIdx.x; t < sk * sk; t += BLOCK) {  // long-range part f_L
            const int nx = t % sk - kNK, ny = t / sk - kNK;
            if (nx == 0 && ny == 0) {
                azz += (2.0 * sqrt(kPi) / eta) * inv_area;  // k = 0 survives only in zz
                continue;
            }
            const double kx = 2.0 * kPi * nx / Ld, ky = 2.0 * kPi * ny / Ld;
            const double k = sqrt(kx * kx + ky * ky);
            const double cs = cos(kx * dx + ky * dy);
            const double ec = erfc(k * eta);
            const double f = 2.0 * kPi * ec / k * inv_area * cs;
            axx += f * kx * kx;
            axy += f * kx * ky;
            ayy += f * ky * ky;
            azz += ((2.0 * sqrt(kPi) / eta) * exp(-k * k * eta * eta) - 2.0 * kPi * k * ec) * cs * inv_area;
        }
    }

    __shared__ double red[4][BLOCK];
    red[0][threadIdx.x] = axx;
    red[1][threadIdx.x] = axy;
    red[2][threadIdx.x] = ayy;
    red[3][threadIdx.x] = azz;
    __syncthreads();
    for (int s = BLOCK / 2; s > 0; s >>= 1) {
        if (threadIdx.x < s)
            for (int c = 0; c < 4; ++c) red[c][threadIdx.x] += red[c][threadIdx.x + s];
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        double w[4] = {red[0][0], red[1][0], red[2][0], red[3][0]};
        if (method == DSMC_W_IMAGE) {
            if (tail) {  // continuum remainder of the square cutoff (R6)
                const double t = 4.0 * sqrt(2.0) / ((A + 0.5) * Ld * Ld * Ld);
                w[0] -= 0.5 * t;
                w[2] -= 0.5 * t;
                w[3] += t;
            }
        } else if (rho == 0) {  // remove the G = 0 piece of the long-range function
            const double alpha = kAlphaL / Ld;
            const double self = 4.0 * alpha * alpha * alpha / (3.0 * sqrt(kPi));
            w[0] -= self;
            w[2] -= self;
            w[3] -= self;
        }
        const size_t N = (size_t)L * L;
        for (int c = 0; c < 4; ++c) Wc[c * N + rho] = (float)w[c];
    }
}

}  // namespace

cudaError_t launch_build_tensor(double *, float *Wc, int L, int method, int A, int tail, cudaStream_t st,
                                uint64_t *launches) {
    build_tensor_kernel<128><<<L * L, 128, 0, st>>>(Wc, L, method, A, tail);
    ++*launches;
    return cudaGetLastError();
}
