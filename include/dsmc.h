/*
 * dsmc.h -- C ABI of the B200-native hot path of arXiv 1211.6234 (Stamps & Ambrose):
 * periodic long-range dipole field h = W (*) s on an L x L lattice of Heisenberg
 * spins, batched over R temperature replicas, coupled to a fused checkerboard
 * Metropolis half-sweep that uses the paper's frozen-field approximation.
 *
 * Every step of the path runs in hand-written sm_100a CUDA kernels inside
 * libdsmc.so; there is no CPU fallback.  The library NEVER allocates device
 * memory: the caller (PyTorch in this repo) allocates one workspace and lends
 * it with dsmc_bind().  All calls on one context are ordered on the bound CUDA
 * stream and asynchronous, except the calls that return data to HOST memory.
 *
 * Citations: PAPER.md:<line> = /root/reference/PAPER.md; R<n> = DESIGN.md section 2.
 *
 * Notation: N = L*L; site n = (x, y), n = y*L + x; k_B = 1.
 * External ("canonical") layouts, all fp32, C order:
 *   W[4][L][L]    components xx, xy, yy, zz;  W[c][rho_y][rho_x], rho = (m - n) mod L
 *   s[R][3][L][L] unit spins, component planes x, y, z
 *   h[R][3][L][L] dipole field in lattice units (no factor g)
 * The internal HBM layout (colour-split, replica-innermost) is the library's
 * business; see DESIGN.md section 5.
 *
 * Energy convention (PAPER.md:150 eq. 11, :160 eq. 12, R7, R8):
 *   E = -J sum_bonds s.s - sum_n (K2 s_z^2 + K4 s_z^4) + (g/2) sum_n s_n.h_n
 *
 * Error behaviour: every int-returning call returns DSMC_OK (0) or a negative
 * code; no exceptions, no abort, no global state (the one exception is the static
 * scratch array of the context-free dsmc_wall_counts_noalloc, documented there).
 * dsmc_last_error() returns a message owned by the context (valid until the next
 * call on that context).
 */
#ifndef DSMC_H
#define DSMC_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct dsmc_ctx dsmc_ctx;

enum {
    DSMC_OK = 0,
    DSMC_EINVAL = -1, /* bad L/R/T/colour/flag, null pointer                          */
    DSMC_ESTATE = -2, /* workspace not bound, tensor not built, spins not set         */
    DSMC_ECUDA = -3,  /* CUDA runtime / launch failure (message kept)                 */
    DSMC_ENOMEM = -4  /* workspace lent by the caller is too small / host malloc fail */
};

/* where a caller-supplied buffer lives */
enum { DSMC_HOST = 0, DSMC_DEVICE = 1 };

/* dsmc_build_tensor methods */
enum { DSMC_W_IMAGE = 0, DSMC_W_EWALD = 1 };

/* dsmc_halfsweep_ex flags */
enum {
    DSMC_REUSE_FIELD = 1, /* skip the field step: reuse h kept from the previous field call of
                             the same colour (for timing the Metropolis kernel alone)         */
    DSMC_TRIAL_FLIP = 2,  /* the trial is the reversed spin s' = -s instead of a point uniform on
                             S^2: the Ising move of App. B; u is drawn as usual   */
    DSMC_NO_RESIDENT = 4, /* dsmc_sublattice_pass / _run only: do not use the kernel that keeps the
                             lattice in shared memory (two launches per pass instead)            */
    DSMC_INCREMENTAL = 8  /* dsmc_sublattice_run only: incremental field update (see there)         */
};

/* dsmc_init_spins modes */
enum { DSMC_INIT_RANDOM = 0, DSMC_INIT_UP = 1 };

/* Create a context for an L x L lattice (L even, L >= 4: the checkerboard needs even L and
 * L = 2 makes the +x and -x neighbours coincide) and R >= 1 replicas with couplings J, g = C_D/J,
 * K2, K4 (same for all replicas; see dsmc_set_anisotropy).  Host-only; touches no GPU state.
 * *out is owned by the caller and released with dsmc_destroy.                                 */
int dsmc_create(dsmc_ctx **out, int L, int R, float J, float g, float K2, float K4);

/* Per-replica anisotropy constants (HOST arrays of length R), e.g. BASELINE config 3's two K4
 * values in one R = 16 batch (eq. 12 with K2 = -K(1-a), K4 = -Ka, R7).            */
int dsmc_set_anisotropy(dsmc_ctx *ctx, const float *K2_r, const float *K4_r);

/* Sharding one ladder of replicas over several contexts (one per GPU): this
 * context's replica r is replica first_replica + r of the whole ladder in every Philox counter
 * (trial moves, acceptance, dsmc_init_spins): a sharded run draws the random numbers of the unsharded
 * one, and reproduces it bit for bit when the shards run the same kernels as the whole (FFT field,
 * whose arithmetic per replica pair does not depend on R, and R % 4 == 0 on every shard).  Default 0. */
int dsmc_set_replica_offset(dsmc_ctx *ctx, uint32_t first_replica);

/* Bytes of device workspace a context of this shape needs (0 if the shape is invalid).        */
size_t dsmc_workspace_bytes(int L, int R);

/* Lend `bytes` of DEVICE memory (256-byte aligned) and the CUDA stream (a cudaStream_t passed as
 * void*, NULL = default stream) every later call runs on.  The context borrows both; the caller
 * frees the memory after dsmc_destroy.  DSMC_ENOMEM if bytes < dsmc_workspace_bytes(L, R).      */
int dsmc_bind(dsmc_ctx *ctx, void *dev_workspace, size_t bytes, void *cuda_stream);

/* a0. Build the lattice-summed interaction table once (eq. 1-5):
 *   W^{ab}(rho) = sum_G T^{ab}(rho + G), T = (delta_ab - 3 rhat_a rhat_b)/r^3, G = (aL, bL);
 *   W(0) omits G = 0 (self-image term of eq. 2, coefficient 1/2: R2).
 * method DSMC_W_EWALD: 2-D Ewald split of eq. 3-5 (cutoff_A and tail ignored; converged to fp64
 *   rounding); DSMC_W_IMAGE: square image cutoff |a|,|b| <= cutoff_A centred on rho reduced to
 *   (-L/2, L/2], plus the continuum tail if tail != 0 (R6).  fp64 arithmetic on the device,
 *   rounded once to fp32.                                                                      */
int dsmc_build_tensor(dsmc_ctx *ctx, int method, int cutoff_A, int tail);

/* Copy the table out / in, canonical layout W[4][L][L]; `where` = DSMC_HOST or DSMC_DEVICE.
 * dsmc_set_tensor replaces the built table (tests use it to isolate the field kernel).        */
int dsmc_get_tensor(dsmc_ctx *ctx, float *W_out, int where);
int dsmc_set_tensor(dsmc_ctx *ctx, const float *W_in, int where);

/* Spins in canonical layout s[R][3][L][L].  set does not renormalise: |s| = 1 is the caller's
 * contract.  Host variants copy through a staging area inside the workspace; get to HOST
 * synchronises the stream.  With dsmc_set_debug(ctx, 1) set checks the contract: one reduction
 * kernel takes the largest | |s| - 1 | over all sites and replicas and the call synchronises and
 * returns DSMC_EINVAL (the spins then count as not set) when it exceeds 1e-5 or a spin is NaN;
 * without it the hot path pays nothing.                                                         */
int dsmc_set_spins(dsmc_ctx *ctx, const float *s, int where);
int dsmc_get_spins(dsmc_ctx *ctx, float *s, int where);
/* Debug checks on (1) / off (0, the default): argument checks that cost a kernel launch and a
 * synchronisation (today: |s| = 1 in dsmc_set_spins).  Host-only.                                */
int dsmc_set_debug(dsmc_ctx *ctx, int on);

/* a4. Initial spins on the device: DSMC_INIT_RANDOM = uniform on S^2 from Philox4x32-10 keyed by
 * (seed; site, replica, tag 1) with the same map as the trial move (R9, R10);
 * DSMC_INIT_UP = all +z.                                                                      */
int dsmc_init_spins(dsmc_ctx *ctx, int mode, uint64_t seed);

/* a1. Dipole field of the CURRENT spins (App. A :331-350):
 *   h_n^x = sum_m [W^xx(rho_nm) s_m^x + W^xy(rho_nm) s_m^y],  h_n^y = sum_m [W^xy s_m^x + W^yy s_m^y],
 *   h_n^z = sum_m W^zz(rho_nm) s_m^z,   every m including m = n.
 * colour = 0 / 1: only targets with (x + y) mod 2 == colour; -1: all targets.  The result is
 * kept in the context for the next half-sweep of that colour.  h_out (nullable) receives the
 * canonical h[R][3][L][L]; entries of inactive targets are left untouched.                     */
int dsmc_dipole_field(dsmc_ctx *ctx, int colour, float *h_out, int where);
/* The field array as the context keeps it, canonical h[R][3][L][L], WITHOUT recomputing it: what the last
 * dsmc_dipole_field(colour = -1) left, or the incrementally updated field after a DSMC_INCREMENTAL run.
 * DSMC_ESTATE unless a field of both colours is kept.  To HOST synchronises.                       */
int dsmc_get_field(dsmc_ctx *ctx, float *h_out, int where);

/* a2. One checkerboard Metropolis half-sweep (PAPER.md:60-72 eq. 7; :98; :102-118; R11-R14):
 *   colour c = step & 1.  (i) h <- dipole field of colour c from the state at entry (frozen for
 *   the whole half-sweep).  (ii) for every active site n and replica r, in one fused kernel:
 *   trial s' uniform on S^2 and u in (0,1) from Philox4x32-10(seed; n, r, step); delta = s' - s;
 *     dE = -J delta.(sum of 4 nn) - K2 (s'_z^2 - s_z^2) - K4 (s'_z^4 - s_z^4)
 *          + g [delta.h_n + (1/2) delta.W(0).delta];
 *   accept  <=>  dE / T_r + ln u < 0;  accepted sites take s'.
 * T: HOST array of R temperatures, all > 0 (else DSMC_EINVAL); uploaded only when it changes;
 * NULL reuses the last one.  One sweep (MC step) = steps 2k and 2k+1.            */
int dsmc_halfsweep(dsmc_ctx *ctx, const float *T, uint64_t seed, uint64_t step);

/* Same with flags (DSMC_REUSE_FIELD) and parity hooks, both nullable DEVICE
 * buffers in canonical site order, written at active sites only:
 *   accept_out[R][L][L] bytes (0/1),  margin_out[R][L][L] floats (dE/T + ln u as the kernel saw it). */
int dsmc_halfsweep_ex(dsmc_ctx *ctx, const float *T, uint64_t seed, uint64_t step, int flags,
                      uint8_t *accept_out, float *margin_out);

/* The paper's own update schedule (section 3.1; App. A :307-361).
 * One pass: an offset (S_1, S_2) in [0, l)^2 is drawn from Philox4x32-10(seed; 0xFFFFFFFF, 0xFFFFFFFF,
 * pass) as (x0 mod l, x1 mod l) (R21); the n = (L/l)^2 sites (S_1 + a l, S_2 + b l) are updated
 * simultaneously, each with the trial and u of Philox(seed; site, replica, step = pass), the dipole
 * field of ALL of them taken from the state at entry to the pass (section 3.2), exchange, anisotropy
 * and the self-term exact as in dsmc_halfsweep.  l >= 2 and l | L (DSMC_EINVAL otherwise); l = L is
 * conventional single-spin Metropolis.  One MC step (N attempted updates) = l*l passes.
 * flags: DSMC_TRIAL_FLIP, DSMC_NO_RESIDENT.  accept_out / margin_out: nullable DEVICE buffers
 * [R][L][L], written at the update sites only.  offset_out: nullable HOST int[2] = {S_1, S_2}.                          */
int dsmc_sublattice_pass(dsmc_ctx *ctx, const float *T, uint64_t seed, uint64_t pass, int l, int flags,
                         uint8_t *accept_out, float *margin_out, int *offset_out);
/* n_passes consecutive passes first_pass .. first_pass + n_passes - 1, bit-identical to calling
 * dsmc_sublattice_pass pass by pass with the same flags.  When L/l is 1, 2 or 4 and 40 L^2 bytes fit one
 * CTA's shared memory (L <= 74; the paper's L = 64, l = 32) and the FFT field is not selected, one CTA
 * per replica pair keeps spins and W in shared memory and runs all passes inside one kernel; otherwise
 * (or with DSMC_NO_RESIDENT) long runs are replayed from a captured CUDA graph whose kernels recompute
 * the offset from a pass counter on the device.                                                    */
int dsmc_sublattice_run(dsmc_ctx *ctx, const float *T, uint64_t seed, uint64_t first_pass, uint64_t n_passes, int l,
                        int flags);
/* DSMC_INCREMENTAL (section 3.2, eq. 8 read the other way round): after a pass
 * only the accepted update sites have changed, so the field of EVERY site changes by exactly
 *   h_t += sum over accepted c of W(c - t) . (s'_c - s_c).
 * The run keeps the field of all N sites of a replica pair in the registers of one CTA and applies these rank-n
 * updates instead of summing over all N sources for the n update sites of every pass: work only for accepted moves
 * (the paper's low-temperature regime), no reduction, a pass without acceptance costs two barriers.  Same schedule,
 * same random numbers and the same decisions as the plain run up to the rounding of the field: the field is
 * recomputed from scratch by a field kernel at entry and every 4096 passes, between which it drifts by at most a few
 * 1e-6 relative (tested); it is therefore NOT bit-identical to pass-by-pass calls -- the parity contract is the
 * lock-step one (decisions identical outside |dE/T + ln u| < 1e-4).  On return the field array holds the field of
 * the final state (dsmc_dipole_field semantics).  Needs L / l in {1, 2, 4} and L * L <= 4096 (DSMC_EINVAL otherwise);
 * flags: DSMC_INCREMENTAL | optionally DSMC_TRIAL_FLIP.
 * dsmc_sublattice_run_ex: margin_log (nullable, DEVICE, [n_passes][R][(L/l)^2] floats, only with DSMC_INCREMENTAL)
 * receives dE/T + ln u of every trial, update sites in the order b (rows) outer, a inner: the parity hook of a run
 * that cannot be stopped between passes.                                                              */
int dsmc_sublattice_run_ex(dsmc_ctx *ctx, const float *T, uint64_t seed, uint64_t first_pass, uint64_t n_passes, int l,
                           int flags, float *margin_log);

/* n_half consecutive half-sweeps (steps first_step .. first_step + n_half - 1) without returning
 * to the caller in between.  Long runs are replayed from a CUDA graph of 8 sweeps (each: field +
 * Metropolis of colour 0, of colour 1) whose kernels read the step from a counter in the
 * workspace: one launch per sweep instead of one per kernel; the trajectory is bit-identical to
 * calling dsmc_halfsweep step by step.                                                         */
int dsmc_run(dsmc_ctx *ctx, const float *T, uint64_t seed, uint64_t first_step, uint64_t n_half);
/* Same with flags: DSMC_TRIAL_FLIP (the Ising reversal move of App. B on the checkerboard half-sweeps). */
int dsmc_run_ex(dsmc_ctx *ctx, const float *T, uint64_t seed, uint64_t first_step, uint64_t n_half, int flags);

/* a3. Observables of the current state, out[R][4] doubles in HOST memory:
 *   E/N (eq. 11 with a freshly computed full field), m_z = N^-1 sum s^z,
 *   M_par = (M_x^2 + M_y^2)^(1/2) (eq. 16),
 *   eta = (2/pi) (N^-1 sum_i (arccos s_i^z - pi/2)^2)^(1/2) (eq. 17, R15).
 * Synchronises the stream.                                                                      */
int dsmc_observables(dsmc_ctx *ctx, double *out);

/* Domain-wall observables of the current state (eq. 14-15), HOST outputs:
 *   counts_out[R][6] = n_h^x, n_v^x, n_h^y, n_v^y, n_h^z, n_v^z with
 *     n_h^a = sum_i 1 - sgn(s_i^a s_{i+x}^a),  n_v^a = sum_i 1 - sgn(s_i^a s_{i+y}^a)   (eq. 14),
 *     periodic neighbours, every bond once, sgn(ab) taken as sgn(a) sgn(b), sgn(0) = 0: exact integers;
 *   derived_out[R][4] (nullable) = wall density (n_v^z + n_h^z) / (4N) and the
 *     per-snapshot orientational order O_a = |n_h^a - n_v^a| / (n_h^a + n_v^a), a = x, y, z (eq. 15;
 *     0 when the component has no wall).  The thermal averages of eq. 15 and the variances of
 *     eq. 18 are statistics the caller takes over snapshots.  Needs no field; synchronises.        */
int dsmc_wall_observables(dsmc_ctx *ctx, long long *counts_out, double *derived_out);

/* Staggered magnetisation of App. B (after Binder and Landau) for stripes of width 1, HOST
 * out[R][3] = m_h, m_v, m_st with the sub-lattices of the 2 x 2 plaquette 1 = (x even, y even),
 * 2 = (x odd, y even), 3 = (x odd, y odd), 4 = (x even, y odd), m_lambda = N^-1 sum_{i in lambda} s_i^z (R23),
 *   m_h = m_1 + m_2 - m_3 - m_4,  m_v = m_1 + m_4 - m_3 - m_2,  m_st = (m_h^2 + m_v^2)^(1/2)
 * per snapshot; <m_st> and chi_st = L^2 (<m_st^2> - <m_st>^2) / T are the caller's statistics.  Synchronises. */
int dsmc_staggered_magnetisation(dsmc_ctx *ctx, double *out);

/* Ensemble statistics accumulated on the device (an ensemble of recorded states;
 * eq. 13 standard error, eq. 18 variance).  dsmc_ensemble_add computes, for the CURRENT state and every
 * replica, the eight per-snapshot quantities
 *   0 E/N, 1 m_z, 2 M_par, 3 eta (as dsmc_observables), 4 wall density, 5 O_x, 6 O_y, 7 O_z (as
 *   dsmc_wall_observables)
 * and adds x and x^2 to running fp64 sums; it is asynchronous (no host round trip), so a production run is
 * "sweeps, add, sweeps, add, ..." without synchronisation.  dsmc_ensemble_get returns, as HOST [R][8]
 * arrays, <x>, sigma^2(x) = <x^2> - <x>^2 (eq. 18) and SE = (sigma^2 / n)^(1/2) (eq. 13) over the n
 * snapshots added since dsmc_ensemble_reset (n_out nullable); DSMC_ESTATE if n = 0.  Synchronises.      */
int dsmc_ensemble_reset(dsmc_ctx *ctx);
/* The paper's recording protocol as one call ("the state of the system was recorded every 50 steps"):
 * n_records times [every whole sweeps, then dsmc_ensemble_add], starting at the even step first_step (T as in
 * dsmc_halfsweep: HOST [R] or null to keep the last).  The trajectory and the statistics are those of the
 * equivalent dsmc_run / dsmc_ensemble_add calls; for every <= 16 the sweeps and the record are replayed from one
 * captured CUDA graph per record.  Asynchronous.  DSMC_EINVAL for every < 1, an odd first_step or an unknown flag. */
int dsmc_run_recorded(dsmc_ctx *ctx, const float *T, uint64_t seed, uint64_t first_step, uint64_t n_records, int every,
                      int flags);
int dsmc_ensemble_add(dsmc_ctx *ctx);
int dsmc_ensemble_get(dsmc_ctx *ctx, double *mean, double *var, double *se, uint64_t *n_out);

/* Device time in milliseconds of the last field / Metropolis / reduction launches made by the
 * last dsmc_halfsweep* call, measured with CUDA events on the bound stream when timing was
 * enabled with dsmc_set_timing(ctx, 1); synchronises.  out[3] = {field, metropolis, total}.      */
int dsmc_set_timing(dsmc_ctx *ctx, int on);
int dsmc_last_timing(dsmc_ctx *ctx, float *out_ms);

/* Number of kernels this context has launched since creation (bench.py's gpu_launches).       */
uint64_t dsmc_launch_count(dsmc_ctx *ctx);

/* Which field kernel runs (all three compute the same a1 and meet the same tolerances):
 *   DSMC_FIELD_GENERIC 0  direct sum, any even L, any R;
 *   DSMC_FIELD_TILED   1  direct sum, register-tiled and TMA-staged; needs L % 16 == 0 and R % 4 == 0;
 *   DSMC_FIELD_FFT     2  circular convolution by batched 2-D FFT over replica pairs (PAPER.md:295
 *                         "more efficient parallelization of the dipole sum");
 *                         needs L in {32, 64, 128, 256, 512} and even R.
 * dsmc_select_field_kernel: kind -1 = automatic (the direct sum: tiled when the shape allows, else
 * generic), or one of the three (DSMC_EINVAL if the shape does not support it).                  */
enum { DSMC_FIELD_AUTO = -1, DSMC_FIELD_GENERIC = 0, DSMC_FIELD_TILED = 1, DSMC_FIELD_FFT = 2 };
int dsmc_field_kernel_kind(dsmc_ctx *ctx);
int dsmc_select_field_kernel(dsmc_ctx *ctx, int kind);
/* 1 if this context's shape supports the kernel `kind` (0, 1, 2), else 0.                         */
int dsmc_field_kernel_supported(dsmc_ctx *ctx, int kind);

/* Measured fp32 FMA issue peak of this GPU in TFLOP/s: a dependency-free FFMA-chain microbenchmark
 * (one CTA of 256 threads per SM, 96 independent accumulators per thread), the denominator
 * bench.py reports beside the derived SMs x 128 lanes x 2 x clock figure.  Synchronises.          */
int dsmc_fp32_fma_peak(dsmc_ctx *ctx, double *tflops_out);

/* Measured denominator of the Metropolis kernel's HBM roofline: one launch that moves the bytes of a checkerboard
 * half-sweep of `colour` without its arithmetic -- the grid, the 18 128-bit loads per thread (own spins, h, four
 * neighbours) and the addresses of the 4-replica Metropolis kernel, the thread's own spins always written back
 * (unchanged bits: the state is not modified), no Philox, no trial, no dE.  Reads whatever the field array holds.
 * Asynchronous; the caller times it (bench.py: in the same rotation over three contexts as the Metropolis kernel).
 * Needs R % 4 == 0 (DSMC_EINVAL) and spins (DSMC_ESTATE).                                                    */
int dsmc_stream_footprint(dsmc_ctx *ctx, int colour);

/* The domain-wall counts of eq. 14 (the counts_out of dsmc_wall_observables, bit for bit) for callers
 * that cannot allocate device memory: code under CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc.  Context-free: no dsmc_ctx, no workspace, no cudaMalloc / cudaFree / allocating library call.
 *   s_dev       DEVICE, canonical s[R][3][L][L] fp32 (read only; the caller's)
 *   counts_dev  DEVICE, [R][6] long long = n_h^x, n_v^x, n_h^y, n_v^y, n_h^z, n_v^z (written; the caller's)
 *   cuda_stream a cudaStream_t passed as void* (NULL = default stream); the call is asynchronous on it
 *   err         nullable HOST buffer of err_len bytes that receives the message of a refused call
 * Both pointers must be memory of the CURRENT device (else DSMC_EINVAL).  The per-CTA partial sums of the reduction
 * live in a static device array inside the library (1 MiB + 4 KiB on every GPU that loads it, held until the process
 * exits), which sets the limits: R <= DSMC_NOALLOC_MAX_R, L even, 4 <= L <= DSMC_NOALLOC_MAX_L; anything larger is
 * refused with DSMC_EINVAL and a message, nothing is launched.  Every call on a GPU shares that one array (it keeps the
 * last call's contents; the call clears what must start at zero with a memset node on the stream): calls that OVERLAP on
 * the same GPU -- two streams, two threads -- race and give wrong counts; calls ordered on one stream, or otherwise
 * serialised, are safe.  The first call with a given device current looks the array's device address up
 * (cudaGetSymbolAddress); make that call outside stream capture.                                            */
#define DSMC_NOALLOC_MAX_R 1024
#define DSMC_NOALLOC_MAX_L 4096
int dsmc_wall_counts_noalloc(const float *s_dev, int L, int R, long long *counts_dev, void *cuda_stream, char *err,
                             size_t err_len);

int dsmc_destroy(dsmc_ctx *ctx);
const char *dsmc_last_error(dsmc_ctx *ctx);
const char *dsmc_version(void);

#ifdef __cplusplus
}
#endif
#endif /* DSMC_H */
