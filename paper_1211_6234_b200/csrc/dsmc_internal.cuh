// dsmc_internal.cuh -- context, HBM layout and launcher prototypes shared by the translation
// units of libdsmc.so.  Not part of the public boundary (include/dsmc.h is).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>
#include <string>
#include <vector>

#include "../../include/dsmc.h"

// ---------------------------------------------------------------------------------------------
// Internal HBM layout.  Nh = N/2 sites per colour, Lh = L/2 per row.
//   site (x, y): colour q = (x + y) & 1, in-row index i = x >> 1, colour-site index a = y*Lh + i
//   spins  S[q][c][a][r]   c in {x,y,z}, replica r innermost      (6*Nh*R floats)
//   field  H[q][c][a][r]   same shape
// Replica-innermost makes every per-site access of the Metropolis kernel a contiguous run of R
// floats and lets the field kernel fetch 4 replicas of one source with one 128-bit load; the
// colour split makes the active colour of a half-sweep a dense array and turns the stride-2
// structure of checkerboard targets into a unit-stride sliding window over W (section 5).
// ---------------------------------------------------------------------------------------------

#define DSMC_GRAPH_UNROLL 8  // sweeps (dsmc_run) or passes (dsmc_sublattice_run) per captured CUDA graph
#define DSMC_MAX_BRANCHES 8  // independent chains of replica groups in the sweep graph of the fused FFT path
#define DSMC_KS_MAX 16  // maximum source split (partial-field slabs) of the tiled field kernel
#define DSMC_TILED_MAX_L 1024  // largest lattice the tiled kernel accepts: the size up to which its fp32 accumulation is
                               // tested to meet the field tolerances (include/dsmc.h, dsmc_select_field_kernel)

// ---------------------------------------------------------------------------------------------
// Programmatic dependent launch (sm_90+).  The kernels of a sweep form one dependent chain (x-forward -> y-multiply ->
// x-inverse -> Metropolis -> step counter -> ...) and the small lattices are bound by the ~3 us a kernel-to-kernel edge
// costs.  A kernel launched through launch_pdl calls pdl_wait() before it touches memory an earlier kernel wrote or
// read -- it returns once the predecessor grid has completed and its writes are visible.  INVARIANT the chain relies
// on: every CTA of a launch_pdl grid that touches global memory calls pdl_wait() before its first access, and no
// launch_pdl grid completes without at least one thread having waited (a grid whose every thread returned early
// would let ITS successor start before ITS predecessor has finished, breaking the transitivity of completion along
// the chain).  A CTA calls pdl_trigger() once it is past the bulk of its work:
// when every CTA of the grid has triggered (or exited) the successor's CTAs are scheduled into the room that frees
// up and wait there, so the launch latency of the edge overlaps this grid's tail.  (Triggering at the top instead
// makes the successor resident while this grid still needs the room: measured slower from L = 128 up, DESIGN.md
// section 5.2b.)  A kernel launched with <<<>>> keeps plain stream order on both sides.  DSMC_NO_PDL=1 in the
// environment drops the attribute (A/B timing).
// ---------------------------------------------------------------------------------------------
#ifdef __CUDACC__
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
bool dsmc_pdl_enabled();
template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args &&...args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = dsmc_pdl_enabled() ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kern, static_cast<KArgs>(args)...);
}
#endif

struct DsmcLayout {
    size_t off_Wc;     // canonical W fp32 [4][L][L]
    size_t off_Wk;     // kernel-layout W for the tiled field kernel
    size_t off_S;      // spins, internal layout
    size_t off_H;      // field, internal layout (both colours)
    size_t off_Hpart;  // partial fields [KS][3][Nh][R] of the tiled kernel
    size_t off_M;      // folded spectral tables AB[slot_x < L/2][slot_y][16] of the FFT field (field_fft.cu)
    size_t off_Z;      // line scratch Z[3][L/2][pair blocks][L][lane] complex of the FFT field
    size_t off_C;      // the two half-spectrum caches C[colour][3][L/2][pair blocks][L][lane] complex
    size_t off_stage;  // canonical staging [R][3][L][L] floats
    size_t off_T;      // invT[R], K2[R], K4[R] floats
    size_t off_obs;    // R*8 doubles (raw observable sums)
    size_t off_walls;  // R*8 64-bit wall counts
    size_t off_stats;  // R*8*2 doubles: ensemble sums of x and x^2
    size_t off_opart;  // per-CTA partial sums of the observable walks (state_kernels.cu: deterministic reductions)
    size_t off_ticket; // 4 arrival counters of those walks (zero between launches)
    size_t off_step;   // 64-bit step counters of dsmc_run's graph replay, one per chain (a 256-byte slot: DSMC_MAX_BRANCHES <= 32)
    size_t total;
};

struct dsmc_ctx {
    int L, R;
    float J, g;
    std::vector<float> K2, K4, T;  // host copies
    bool aniso_dirty = true, T_valid = false;
    char *ws = nullptr;
    size_t ws_bytes = 0;
    cudaStream_t stream = nullptr;
    DsmcLayout lay;
    bool tensor_built = false, spins_set = false;
    bool field_valid[2] = {false, false};
    bool spec_valid[2] = {false, false};  // FFT field: the cache holds the half-spectrum of colour c of the CURRENT spins
    int zline = -1;  // FFT field: the colour whose forward-transformed rows (of the CURRENT spins) sit in the scratch Z, or -1
    float w0[4] = {0, 0, 0, 0};  // W(0) components (fp32, as stored)
    uint32_t replica_offset = 0;  // dsmc_set_replica_offset
    int field_kind = -1;  // -1 automatic, 0 generic, 1 tiled, 2 FFT (dsmc_select_field_kernel)
    int timing = 0;
    int no_fuse = 0;  // DSMC_NO_FUSE=1 in the environment at dsmc_create: never fuse the Metropolis decision into the FFT field (A/B)
    int debug = 0;  // dsmc_set_debug: argument checks that cost a kernel (|s| = 1 in dsmc_set_spins)
    cudaEvent_t ev[3] = {nullptr, nullptr, nullptr};
    bool ev_recorded = false;
    uint64_t launches = 0;
    uint64_t ensemble_n = 0;  // snapshots accumulated since dsmc_ensemble_reset
    // one sweep (2 x [field + Metropolis] + step advance) captured as a CUDA graph for dsmc_run
    cudaStream_t capture_stream = nullptr;
    // the fused FFT path replays its sweeps as up to DSMC_MAX_BRANCHES independent chains of line blocks (build_sweep_graph)
    cudaStream_t branch_stream[DSMC_MAX_BRANCHES - 1] = {};
    cudaEvent_t ev_fork = nullptr, ev_join[DSMC_MAX_BRANCHES - 1] = {};
    int fft_pb0 = 0, fft_npb = 0;  // line-block range the next fused half-sweep is enqueued for (0, 0 = all)
    float *fft_SG = nullptr;       // ... on the block-major copy of the spins (null: on S)
    int graph_branches = 1;        // chains the captured sweeps consist of (sweep_graph, branch_graph[])
    int max_branches = DSMC_MAX_BRANCHES;  // DSMC_BRANCHES=n in the environment at dsmc_create (A/B timing; 1 = one chain)
    cudaGraphExec_t sweep_graph = nullptr, branch_graph[DSMC_MAX_BRANCHES - 1] = {};
    uint64_t graph_seed = 0;
    int graph_kind = -1, graph_flags = -1, graph_every = -1;  // graph_every > 0: sweeps + record (dsmc_run_recorded)
    int graph_spec_in = -1, graph_spec_out = -1;  // spec_valid (bit c) the capture started from / ended with
    uint64_t graph_launches = 0;
    // one stride-l pass (field + flip + pass counter += 1) for dsmc_sublattice_run
    cudaGraphExec_t pass_graph = nullptr;
    uint64_t pgraph_seed = 0;
    int pgraph_kind = -1, pgraph_flags = -1, pgraph_l = -1;
    uint64_t pgraph_launches = 0;
    int sm_count = 148;
    int device = 0;  // ordinal of the device the workspace lives on (dsmc_bind); every call runs with it current
    bool tiled_configured = false, fft_configured = false;  // cudaFuncSetAttribute done on this device
    std::string err;

    float *Wc() const { return (float *)(ws + lay.off_Wc); }
    float *Wk() const { return (float *)(ws + lay.off_Wk); }
    float *S() const { return (float *)(ws + lay.off_S); }
    float *H() const { return (float *)(ws + lay.off_H); }
    float *Hpart() const { return (float *)(ws + lay.off_Hpart); }
    float *M() const { return (float *)(ws + lay.off_M); }
    void *Z() const { return (void *)(ws + lay.off_Z); }
    void *C() const { return (void *)(ws + lay.off_C); }
    float *stage() const { return (float *)(ws + lay.off_stage); }
    float *invT() const { return (float *)(ws + lay.off_T); }
    float *K2d() const { return invT() + R; }
    float *K4d() const { return invT() + 2 * R; }
    double *obs() const { return (double *)(ws + lay.off_obs); }
    unsigned long long *walls() const { return (unsigned long long *)(ws + lay.off_walls); }
    double *stats() const { return (double *)(ws + lay.off_stats); }
    double *opart() const { return (double *)(ws + lay.off_opart); }
    unsigned int *ticket(int k) const { return (unsigned int *)(ws + lay.off_ticket) + k; }
    unsigned long long *step_dev() const { return (unsigned long long *)(ws + lay.off_step); }
    size_t Nh() const { return (size_t)L * (L / 2); }
    size_t plane() const { return Nh() * (size_t)R; }  // floats in one [a][r] plane
};

DsmcLayout dsmc_make_layout(int L, int R);

// tiled-kernel W layout size in floats (field_tiled.cu)
size_t dsmc_wk_floats(int L);
bool dsmc_tiled_supported(int L, int R);

// ---- launchers (each returns the cudaError_t of its launch(es); all async on `st`) ----------
cudaError_t launch_build_tensor(double *scratch_unused, float *Wc, int L, int method, int A, int tail,
                                cudaStream_t st, uint64_t *launches);
cudaError_t launch_make_wk(const float *Wc, float *Wk, int L, cudaStream_t st, uint64_t *launches);

cudaError_t launch_canon_to_internal(const float *canon, float *S, int L, int R, cudaStream_t st,
                                     uint64_t *launches);
// colour = -1: both colours; else only that colour's sites are written to canon
cudaError_t launch_internal_to_canon(const float *S, float *canon, int L, int R, int colour,
                                     cudaStream_t st, uint64_t *launches);

cudaError_t launch_field_generic(const float *S, const float *Wc, float *H, int L, int R, int colour,
                                 cudaStream_t st, uint64_t *launches);
// FFT field (field_fft.cu): L in {32, ..., 512}, R even
bool dsmc_fft_supported(int L, int R);
size_t dsmc_fft_m_floats(int L);
size_t dsmc_fft_scratch_bytes(int L, int R);
size_t dsmc_fft_cache_bytes(int L, int R);
cudaError_t launch_make_fft_table(const float *Wc, float *M, void *scratch, int L, cudaStream_t st,
                                  uint64_t *launches);
// colour = -1 writes both colours of H.  valid[2]: which colours' half-spectra in `cache` are those of the current
// spins; updated here (a colour transformed forward becomes valid), cleared by the caller when a colour's spins change
// zline: which colour's forward-transformed rows the scratch Z holds (-1 none).  fuse != null (colour 0 / 1, shape
// dsmc_fft_fused_supported): the last pass also takes the Metropolis decision of the half-sweep and
// transforms the updated rows forward: H is NOT written, the spins of `colour` change
struct MetropolisArgs;
bool dsmc_fft_fused_supported(int L, int R);
cudaError_t launch_field_fft(const float *S, const float *AB, void *scratch, void *cache, float *H, int L, int R, int colour,
                             bool *valid, int *zline, const MetropolisArgs *fuse, int pb0, int npb, float *SG, bool *configured,
                             cudaStream_t st, uint64_t *launches);
// pb0, npb: with fuse, only the line blocks (16 replicas each) pb0 .. pb0 + npb - 1; npb = 0: all of them.  SG (only with a
// proper sub-range): the spins are read and written in the block-major copy SG[pb][q][c][a][16 replicas] instead of S
int dsmc_fft_line_blocks(int L, int R);
// S -> SG (to_blocks) or SG -> S, all line blocks; R % 16 == 0
cudaError_t launch_spin_blocks(float *S, float *SG, int L, int R, bool to_blocks, cudaStream_t st, uint64_t *launches);
// configured: the context's "dynamic shared memory limit raised on this device" flag
cudaError_t launch_field_tiled(const float *S, const float *Wk, float *Hpart, float *H, int L, int R,
                               int colour, int sm_count, bool *configured, cudaStream_t st, uint64_t *launches);

struct MetropolisArgs {
    float *S;
    const float *H;
    const float *invT, *K2, *K4;
    int L, R, colour;
    int rq_shift;  // log2(R/4) when R/4 is a power of two, else -1 (set by the launcher)
    int flip;      // 0: trial uniform on S^2; 1: trial = -s (Ising move of App. B)
    uint32_t r_off;  // index of this context's replica 0 in the whole ladder (Philox counter word 1)
    float J, g, w0xx, w0yy, w0zz, w0xy;
    uint32_t seed_lo, seed_hi, step_lo, step_hi;
    // when non-null the step is *step_dev + step_off instead of (step_lo, step_hi): lets a captured CUDA
    // graph of one sweep be replayed with a step counter that lives on the device (dsmc_run)
    const unsigned long long *step_dev;
    uint32_t step_off;
    uint8_t *accept_out;  // canonical [R][L][L] or null
    float *margin_out;    // canonical [R][L][L] or null
    int pdl_late;  // where the kernel lets its successor be scheduled (set by the launcher): 1 = after its loads and
                   // random numbers (grids of at most one wave), 0 = at its top (larger grids)
};
cudaError_t launch_metropolis(const MetropolisArgs &a, cudaStream_t st, uint64_t *launches);
// the loads and stores of metropolis4_kernel without its arithmetic (R % 4 == 0)
cudaError_t launch_metropolis_stream(const MetropolisArgs &a, cudaStream_t st, uint64_t *launches);
// the paper's stride-l sub-lattice pass: offset (ox, oy) in [0, l)^2, n = (L/l)^2 update sites
void dsmc_sublattice_offset(uint64_t seed, uint64_t pass, int l, int *ox, int *oy);
// scratch: 3 N R floats for the per-slab partial fields (the staging buffer)
// field_in_H: h of the update sites is already in the field array H (FFT route); else it is summed here
cudaError_t launch_sublattice_pass(const MetropolisArgs &a, const float *Wc, float *scratch, int sm_count, int l, int ox,
                                   int oy, bool field_in_H, cudaStream_t st, uint64_t *launches);
// the same schedule with the lattice resident in shared memory: one CTA per replica pair runs all n_passes passes
// (sublattice_kernels.cu); L/l in {1, 2, 4} and 40 L^2 bytes within one CTA's shared memory
bool dsmc_resident_supported(int L, int l);
cudaError_t launch_sublattice_resident(const MetropolisArgs &a, const float *Wc, int l, uint64_t first_pass, uint64_t n_passes,
                                       cudaStream_t st, uint64_t *launches);
// the same schedule with the field of all sites kept in registers and updated by the accepted moves (NEXT-4): H holds the
// field of the current spins at entry and at exit; margin_log: nullable device [n_passes][R][(L/l)^2]
#define DSMC_INCREMENTAL_REFRESH 4096  // passes between two recomputations of the field from scratch (rounding drift)
bool dsmc_incremental_supported(int L, int l);
cudaError_t launch_sublattice_incremental(const MetropolisArgs &a, const float *Wc, float *H, int l, uint64_t first_pass,
                                          uint64_t n_passes, float *margin_log, cudaStream_t st, uint64_t *launches);
// *step = value (add = 0) or *step += value (add = 1): one thread, stream-ordered
cudaError_t launch_step_update(unsigned long long *step, unsigned long long value, int add, cudaStream_t st,
                               uint64_t *launches);
cudaError_t launch_init_spins(float *S, int L, int R, int mode, uint64_t seed, uint32_t r_off, cudaStream_t st,
                              uint64_t *launches);
// Per-replica reductions (state_kernels.cu): deterministic -- warp shuffles / shared memory in index order inside a CTA,
// per-CTA partials in `part` (dsmc_walk_scratch_bytes), summed in CTA order by the last CTA to arrive (`ticket`).  The
// kernels call pdl_wait at their top and are launched as dependent launches (the record chain of dsmc_run_recorded).
size_t dsmc_walk_scratch_bytes(int L, int R);
cudaError_t launch_observables(const float *S, const float *H, const float *K2, const float *K4, double *obs, double *part,
                               unsigned int *ticket, int L, int R, cudaStream_t st, uint64_t *launches);
cudaError_t launch_wall_counts(const float *S, unsigned long long *counts, unsigned long long *part, unsigned int *ticket,
                               int L, int R, cudaStream_t st, uint64_t *launches);
cudaError_t launch_staggered(const float *S, double *sums, double *part, unsigned int *ticket, int L, int R, cudaStream_t st,
                             uint64_t *launches);
cudaError_t launch_ensemble_add(const double *obs, const unsigned long long *walls, double *stats, int L, int R, double J,
                                double g, cudaStream_t st, uint64_t *launches);
// largest |s.s - 1| over all spins -> *out (one float, device): the debug check of dsmc_set_spins
cudaError_t launch_norm_check(const float *S, float *out, int L, int R, cudaStream_t st, uint64_t *launches);
