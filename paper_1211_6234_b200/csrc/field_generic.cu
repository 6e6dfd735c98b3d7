// field_generic.cu -- a1, generic shape: dipole field h = W (*) s by direct summation for any
// even L and any R (App. A :331-350).  One thread per (target, replica); source
// rows are staged through shared memory; per-row fp32 partial sums are folded into a running
// total (two-level accumulation).  The register-tiled kernel in
// field_tiled.cu replaces it whenever the shape allows.
#include "dsmc_internal.cuh"

namespace {

constexpr int GT = 128;  // threads per block

// Block = GT consecutive (target a, replica r) pairs of colour `colour` (r fastest).  Which replicas a block
// touches is arbitrary when R is small, so the spins of a source row are read straight from global memory
// (L1/L2 resident: a row is 3*L*R floats) and only W's row is staged in shared memory.
__global__ void __launch_bounds__(GT) field_generic_kernel(const float *__restrict__ S, const float *__restrict__ Wc,
                                                           float *__restrict__ H, int L, int R, int colour) {
    extern __shared__ float wrow[];  // [4][L]: W[c][ry][*] for the current (ys - yt) -- per target row
    const int Lh = L >> 1;
    const size_t Nh = (size_t)L * Lh, N = 2 * Nh, plane = Nh * (size_t)R;
    const size_t t = (size_t)blockIdx.x * GT + threadIdx.x;
    const bool live = t < Nh * (size_t)R;
    const size_t tt = live ? t : Nh * (size_t)R - 1;
    const int r = (int)(tt % (size_t)R);
    const int a = (int)(tt / (size_t)R);
    const int yt = a / Lh, it = a - yt * Lh;
    const int xt = 2 * it + ((yt + colour) & 1);
    // all threads of a block may span several target rows; W rows are therefore indexed per thread
    // from global memory when rows differ, and from the staged copy when the block sits in one row.
    const size_t t_first = (size_t)blockIdx.x * GT;
    const size_t t_last = min(t_first + GT, Nh * (size_t)R) - 1;
    const int y_first = (int)((t_first / (size_t)R) / Lh), y_last = (int)((t_last / (size_t)R) / Lh);
    const bool one_row = (y_first == y_last);

    float hx = 0.f, hy = 0.f, hz = 0.f;
    for (int ys = 0; ys < L; ++ys) {
        const int ry = (ys - yt + L) % L;
        if (one_row) {
            __syncthreads();
            for (int k = threadIdx.x; k < 4 * L; k += GT) wrow[k] = Wc[(size_t)(k / L) * N + (size_t)ry * L + (k % L)];
            __syncthreads();
        }
        float px = 0.f, py = 0.f, pz = 0.f;
        for (int xs = 0; xs < L; ++xs) {
            int rx = xs - xt;
            rx += (rx < 0) ? L : 0;
            const int q = (xs + ys) & 1;
            const float *sp = S + (size_t)q * 3 * plane + ((size_t)ys * Lh + (xs >> 1)) * R + r;
            const float sx = sp[0], sy = sp[plane], sz = sp[2 * plane];
            float wxx, wxy, wyy, wzz;
            if (one_row) {
                wxx = wrow[rx]; wxy = wrow[L + rx]; wyy = wrow[2 * L + rx]; wzz = wrow[3 * L + rx];
            } else {
                const size_t w = (size_t)ry * L + rx;
                wxx = Wc[w]; wxy = Wc[N + w]; wyy = Wc[2 * N + w]; wzz = Wc[3 * N + w];
            }
            px = fmaf(wxx, sx, px); px = fmaf(wxy, sy, px);
            py = fmaf(wxy, sx, py); py = fmaf(wyy, sy, py);
            pz = fmaf(wzz, sz, pz);
        }
        hx += px; hy += py; hz += pz;
    }
    if (live) {
        float *dst = H + (size_t)colour * 3 * plane + (size_t)a * R + r;
        dst[0] = hx;
        dst[plane] = hy;
        dst[2 * plane] = hz;
    }
}

}  // namespace

cudaError_t launch_field_generic(const float *S, const float *Wc, float *H, int L, int R, int colour,
                                 cudaStream_t st, uint64_t *launches) {
    const size_t total = (size_t)L * (L / 2) * R;
    const unsigned grid = (unsigned)((total + GT - 1) / GT);
    field_generic_kernel<<<grid, GT, sizeof(float) * 4 * L, st>>>(S, Wc, H, L, R, colour);
    ++*launches;
    return cudaGetLastError();
}
