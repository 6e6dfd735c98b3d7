// peak_kernels.cu -- measured denominator for the field kernel's roofline: a dependency-free FFMA
// chain microbenchmark (96 independent accumulators per thread, 256 threads per SM, no memory
// traffic in the loop).  bench.py runs it in the same process as the timed path.
#include "dsmc_internal.cuh"

namespace {

constexpr int NACC = 96;

__global__ void __launch_bounds__(256) ffma_peak_kernel(const float *__restrict__ in, float *out, int iters) {
    float acc[NACC], a[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) a[i] = in[threadIdx.x % 7 + i];
    float b = in[threadIdx.x % 5 + 9];
#pragma unroll
    for (int i = 0; i < NACC; ++i) acc[i] = in[i % 13];
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < NACC; ++i) acc[i] = fmaf(a[i & 3], b, acc[i]);
        b += 1e-9f;
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < NACC; ++i) s += acc[i];
    if (s == 123.456f) out[0] = s;  // never true for the inputs used; keeps the chain alive
}

}  // namespace

extern "C" int dsmc_fp32_fma_peak(dsmc_ctx *ctx, double *tflops_out) {
    if (!ctx || !tflops_out) return DSMC_EINVAL;
    if (!ctx->ws) {
        ctx->err = "workspace not bound (call dsmc_bind)";
        return DSMC_ESTATE;
    }
    // scratch: the staging area (>= 3*16*1 floats for every valid shape)
    float *buf = ctx->stage();
    float host[32];
    for (int i = 0; i < 32; ++i) host[i] = 1e-3f * (float)(i % 17 + 1);
    cudaError_t e = cudaMemcpyAsync(buf, host, sizeof(host), cudaMemcpyHostToDevice, ctx->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
    const int iters = 20000, blocks = ctx->sm_count, threads = 256;
    cudaEvent_t e0 = ctx->ev[0], e1 = ctx->ev[1];
    float best = 1e30f;
    for (int rep = 0; rep < 4 && e == cudaSuccess; ++rep) {
        cudaEventRecord(e0, ctx->stream);
        ffma_peak_kernel<<<blocks, threads, 0, ctx->stream>>>(buf, buf + 32, iters);
        ++ctx->launches;
        cudaEventRecord(e1, ctx->stream);
        e = cudaEventSynchronize(e1);
        float ms = 0.f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms < best) best = ms;
    }
    if (e != cudaSuccess) {
        ctx->err = std::string("fp32 peak microbenchmark: ") + cudaGetErrorString(e);
        return DSMC_ECUDA;
    }
    *tflops_out = 2.0 * NACC * (double)iters * threads * blocks / (best * 1e-3) / 1e12;
    return DSMC_OK;
}
