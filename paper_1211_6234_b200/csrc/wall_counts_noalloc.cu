// wall_counts_noalloc.cu -- dsmc_wall_counts_noalloc (include/dsmc.h): the domain-wall counts of eq. 14
// for callers that cannot allocate device memory or lend a workspace.  Same definition and the
// same two-stage reduction as wall_counts_kernel (state_kernels.cu: per-CTA partial sums in scratch memory, the last
// CTA of a replica -- decided by an integer ticket -- adds them in CTA order), but context-free: it reads the
// canonical s[R][3][L][L] directly and its scratch is the file-scope array below instead of workspace memory.
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <mutex>

#include "../../include/dsmc.h"

namespace {

constexpr int kMaxR = DSMC_NOALLOC_MAX_R;
constexpr int kMaxL = DSMC_NOALLOC_MAX_L;
constexpr int kMaxCtasPerReplica = 16;
constexpr int kBlock = 256;
constexpr int kMaxDevices = 64;

struct Scratch {
    unsigned long long part[kMaxR][kMaxCtasPerReplica][8];  // per-CTA partial counts, 6 used (64-byte records)
    unsigned int ticket[kMaxR];                             // CTAs of replica r that have written their partial
};

// The scratch memory: 1 MiB + 4 KiB in every GPU that loads libdsmc.so, until the process exits.  Shared by every call
// (see the header: calls that overlap on one GPU race) and never freed.  In HOST code this name is a stand-in symbol,
// not a device address: the host passes the kernel the address cudaGetSymbolAddress returns for the current device.
static __device__ __align__(256) unsigned char g_scratch[sizeof(Scratch)];

std::mutex g_mu;
Scratch *g_scratch_addr[kMaxDevices];  // per device; null until the first call with that device current

__device__ __forceinline__ int sgnf(float v) { return (v > 0.0f) - (v < 0.0f); }

// grid (P, R): CTA (p, r) walks sites n = p * kBlock + tid, + P * kBlock, ... of replica r (x contiguous: coalesced).
__global__ void __launch_bounds__(kBlock) wall_counts_noalloc_kernel(const float *__restrict__ s, long long *__restrict__ counts,
                                                                     Scratch *__restrict__ scratch, int L) {
    __shared__ unsigned long long warp_sum[kBlock / 32][6];
    __shared__ unsigned int s_last;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int P = gridDim.x, p = blockIdx.x, r = blockIdx.y;
    const size_t N = (size_t)L * L;
    const float *sr = s + (size_t)r * 3 * N;
    unsigned long long acc[6] = {0, 0, 0, 0, 0, 0};
    for (size_t n = (size_t)p * kBlock + tid; n < N; n += (size_t)P * kBlock) {
        const int y = (int)(n / L), x = (int)(n - (size_t)y * L);
        const size_t east = x + 1 == L ? n - x : n + 1;
        const size_t north = y + 1 == L ? (size_t)x : n + L;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const int si = sgnf(sr[c * N + n]);
            acc[2 * c + 0] += (unsigned long long)(1 - si * sgnf(sr[c * N + east]));
            acc[2 * c + 1] += (unsigned long long)(1 - si * sgnf(sr[c * N + north]));
        }
    }
#pragma unroll
    for (int k = 0; k < 6; ++k) {
#pragma unroll
        for (int mask = 16; mask >= 1; mask >>= 1) acc[k] += __shfl_xor_sync(0xFFFFFFFFu, acc[k], mask);
        if (lane == 0) warp_sum[warp][k] = acc[k];
    }
    __syncthreads();
    if (tid < 6) {
        unsigned long long tot = 0;
        for (int w = 0; w < kBlock / 32; ++w) tot += warp_sum[w][tid];
        scratch->part[r][p][tid] = tot;
    }
    __threadfence();
    __syncthreads();
    if (tid == 0) s_last = atomicAdd(&scratch->ticket[r], 1u) == (unsigned)P - 1 ? 1u : 0u;
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    if (tid < 6) {
        unsigned long long tot = 0;
        for (int b = 0; b < P; ++b) tot += __ldcg(&scratch->part[r][b][tid]);
        counts[(size_t)r * 6 + tid] = (long long)tot;
    }
    if (tid == 0) scratch->ticket[r] = 0u;
}

int refuse(char *err, size_t err_len, int code, const char *fmt, long a = 0, long b = 0) {
    if (err && err_len) snprintf(err, err_len, fmt, a, b);
    return code;
}

int refuse_cuda(char *err, size_t err_len, const char *what, cudaError_t e) {
    if (err && err_len) snprintf(err, err_len, "dsmc_wall_counts_noalloc: %s: %s", what, cudaGetErrorString(e));
    return DSMC_ECUDA;
}

}  // namespace

extern "C" int dsmc_wall_counts_noalloc(const float *s_dev, int L, int R, long long *counts_dev, void *cuda_stream, char *err,
                                        size_t err_len) {
    if (err && err_len) err[0] = '\0';
    if (!s_dev || !counts_dev) return refuse(err, err_len, DSMC_EINVAL, "dsmc_wall_counts_noalloc: null argument");
    if (L < 4 || (L & 1))
        return refuse(err, err_len, DSMC_EINVAL, "dsmc_wall_counts_noalloc: L = %ld must be even and >= 4", L);
    if (L > kMaxL)
        return refuse(err, err_len, DSMC_EINVAL, "dsmc_wall_counts_noalloc: L = %ld exceeds DSMC_NOALLOC_MAX_L = %ld", L, kMaxL);
    if (R < 1) return refuse(err, err_len, DSMC_EINVAL, "dsmc_wall_counts_noalloc: R = %ld must be >= 1", R);
    if (R > kMaxR)
        return refuse(err, err_len, DSMC_EINVAL,
                      "dsmc_wall_counts_noalloc: R = %ld exceeds DSMC_NOALLOC_MAX_R = %ld (the static scratch array holds "
                      "partial sums for no more replicas)",
                      R, kMaxR);
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return refuse_cuda(err, err_len, "cudaGetDevice", e);
    if (dev < 0 || dev >= kMaxDevices)
        return refuse(err, err_len, DSMC_EINVAL, "dsmc_wall_counts_noalloc: device %ld beyond the %ld this table holds", dev,
                      kMaxDevices);
    const void *ptrs[2] = {s_dev, counts_dev};
    for (int k = 0; k < 2; ++k) {  // a host pointer here would fault in the kernel: refuse it with a message instead
        cudaPointerAttributes at;
        e = cudaPointerGetAttributes(&at, ptrs[k]);
        if (e != cudaSuccess) return refuse_cuda(err, err_len, "cudaPointerGetAttributes", e);
        const bool on_dev = (at.type == cudaMemoryTypeDevice && at.device == dev) || at.type == cudaMemoryTypeManaged;
        if (!on_dev)
            return refuse(err, err_len, DSMC_EINVAL,
                          k == 0 ? "dsmc_wall_counts_noalloc: s_dev is not device memory of the current device %ld"
                                 : "dsmc_wall_counts_noalloc: counts_dev is not device memory of the current device %ld",
                          dev);
    }
    Scratch *scratch;
    {
        // set-up, once per device, with that device current: the DEVICE address of g_scratch on this GPU
        std::lock_guard<std::mutex> lock(g_mu);
        if (!g_scratch_addr[dev]) {
            void *addr = nullptr;
            e = cudaGetSymbolAddress(&addr, g_scratch);
            if (e != cudaSuccess) return refuse_cuda(err, err_len, "cudaGetSymbolAddress(scratch)", e);
            g_scratch_addr[dev] = static_cast<Scratch *>(addr);
        }
        scratch = g_scratch_addr[dev];
    }
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    // the array keeps the last call's contents: the tickets must start at zero (a call that was aborted, or one that
    // raced with another, may have left them otherwise); the partial sums are all rewritten before they are read
    e = cudaMemsetAsync(scratch->ticket, 0, sizeof(unsigned int) * (size_t)R, st);
    if (e != cudaSuccess) return refuse_cuda(err, err_len, "clearing the tickets", e);
    const size_t N = (size_t)L * L;
    const size_t want = (N + kBlock - 1) / kBlock;
    const unsigned P = (unsigned)(want < (size_t)kMaxCtasPerReplica ? want : (size_t)kMaxCtasPerReplica);
    wall_counts_noalloc_kernel<<<dim3(P, (unsigned)R), kBlock, 0, st>>>(s_dev, counts_dev, scratch, L);
    e = cudaGetLastError();
    if (e != cudaSuccess) return refuse_cuda(err, err_len, "kernel launch", e);
    return DSMC_OK;
}
