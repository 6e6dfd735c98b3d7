// dsmc_api.cu -- the C ABI of include/dsmc.h: argument checks, workspace carving, stream-ordered
// launches.  No device memory is allocated here; no step of the path runs on the host.
#include <cstdio>
#include <cstring>
#include <new>

#include <cstdlib>

#include "dsmc_internal.cuh"

// programmatic dependent launch of the sweep's kernels (dsmc_internal.cuh); DSMC_NO_PDL=1 turns it off
bool dsmc_pdl_enabled() {
    static const bool on = [] {
        const char *v = getenv("DSMC_NO_PDL");
        return !(v && v[0] && v[0] != '0');
    }();
    return on;
}

namespace {

size_t align256(size_t v) { return (v + 255) & ~(size_t)255; }

void drop_sweep_graph(dsmc_ctx *ctx);

bool shape_ok(int L, int R) { return L >= 4 && (L & 1) == 0 && L <= 4096 && R >= 1 && R <= 65535; }

int fail(dsmc_ctx *c, int code, const char *msg) {
    if (c) c->err = msg;
    return code;
}

int cuda_fail(dsmc_ctx *c, cudaError_t e, const char *what) {
    if (c) {
        c->err = std::string(what) + ": " + cudaGetErrorString(e);
    }
    return DSMC_ECUDA;
}

#define CU(call, what)                                       \
    do {                                                     \
        cudaError_t e__ = (call);                            \
        if (e__ != cudaSuccess) return cuda_fail(ctx, e__, what); \
    } while (0)

int need_bound(dsmc_ctx *ctx) {
    if (!ctx) return DSMC_EINVAL;
    if (!ctx->ws) return fail(ctx, DSMC_ESTATE, "workspace not bound (call dsmc_bind)");
    return DSMC_OK;
}

// Every call on a bound context runs with the workspace's device current, whatever the calling thread had
// selected (launches, cudaFuncSetAttribute, graph capture and events all act on the current device), and puts the
// caller's device back on return.
struct DeviceGuard {
    int prev = -1;
    explicit DeviceGuard(int want) {
        int cur = 0;
        if (cudaGetDevice(&cur) == cudaSuccess && cur != want && cudaSetDevice(want) == cudaSuccess) prev = cur;
    }
    ~DeviceGuard() {
        if (prev >= 0) cudaSetDevice(prev);
    }
};
#define ENTER_BOUND(ctx)                         \
    if (int rc__ = need_bound(ctx)) return rc__; \
    DeviceGuard guard__((ctx)->device)

int upload_aniso(dsmc_ctx *ctx);

int upload_params(dsmc_ctx *ctx, const float *T) {
    const int R = ctx->R;
    if (T) {
        for (int r = 0; r < R; ++r)
            if (!(T[r] > 0.0f)) return fail(ctx, DSMC_EINVAL, "temperatures must be > 0");
        if (!ctx->T_valid || std::memcmp(T, ctx->T.data(), sizeof(float) * R) != 0) {
            std::memcpy(ctx->T.data(), T, sizeof(float) * R);
            std::vector<float> inv(R);
            for (int r = 0; r < R; ++r) inv[r] = 1.0f / T[r];
            CU(cudaMemcpyAsync(ctx->invT(), inv.data(), sizeof(float) * R, cudaMemcpyHostToDevice, ctx->stream),
               "upload T");
            CU(cudaStreamSynchronize(ctx->stream), "upload T sync");  // inv is a stack-lifetime buffer
            ctx->T_valid = true;
        }
    } else if (!ctx->T_valid) {
        return fail(ctx, DSMC_EINVAL, "T is NULL and no temperatures were set before");
    }
    return upload_aniso(ctx);
}

// the per-replica anisotropy constants alone (observables need them, but no temperature)
int upload_aniso(dsmc_ctx *ctx) {
    const int R = ctx->R;
    if (ctx->aniso_dirty) {
        CU(cudaMemcpyAsync(ctx->K2d(), ctx->K2.data(), sizeof(float) * R, cudaMemcpyHostToDevice, ctx->stream),
           "upload K2");
        CU(cudaMemcpyAsync(ctx->K4d(), ctx->K4.data(), sizeof(float) * R, cudaMemcpyHostToDevice, ctx->stream),
           "upload K4");
        CU(cudaStreamSynchronize(ctx->stream), "upload K sync");
        ctx->aniso_dirty = false;
    }
    return DSMC_OK;
}

// which field kernel runs: 0 generic, 1 tiled, 2 FFT.  Automatic = the direct sum SURVEY.md section 8
// scopes (tiled when the shape allows, else generic); the FFT route is chosen explicitly.
int field_kind(const dsmc_ctx *ctx) {
    if (ctx->field_kind >= 0) return ctx->field_kind;
    return dsmc_tiled_supported(ctx->L, ctx->R) ? 1 : 0;
}

// colour = -1: both colours; kind_override >= 0 runs that field kernel whatever the selection
int run_field(dsmc_ctx *ctx, int colour, int kind_override = -1) {
    cudaError_t e = cudaSuccess;
    const int kind = kind_override >= 0 ? kind_override : field_kind(ctx);
    if (kind == 2) {
        e = launch_field_fft(ctx->S(), ctx->M(), ctx->Z(), ctx->C(), ctx->H(), ctx->L, ctx->R, colour, ctx->spec_valid,
                             &ctx->zline, nullptr, 0, 0, nullptr, &ctx->fft_configured, ctx->stream, &ctx->launches);
    } else {
        for (int q = 0; q < 2 && e == cudaSuccess; ++q) {
            if (colour >= 0 && colour != q) continue;
            if (kind == 1)
                e = launch_field_tiled(ctx->S(), ctx->Wk(), ctx->Hpart(), ctx->H(), ctx->L, ctx->R, q, ctx->sm_count,
                                       &ctx->tiled_configured, ctx->stream, &ctx->launches);
            else
                e = launch_field_generic(ctx->S(), ctx->Wc(), ctx->H(), ctx->L, ctx->R, q, ctx->stream,
                                         &ctx->launches);
        }
    }
    if (e != cudaSuccess) return cuda_fail(ctx, e, "dipole field launch");
    for (int q = 0; q < 2; ++q)
        if (colour < 0 || colour == q) ctx->field_valid[q] = true;
    return DSMC_OK;
}

int after_tensor_change(dsmc_ctx *ctx) {
    // W(0) for the self term of dE, and the kernel-layout copy for the tiled field kernel
    const size_t N = (size_t)ctx->L * ctx->L;
    for (int c = 0; c < 4; ++c)
        CU(cudaMemcpyAsync(&ctx->w0[c], ctx->Wc() + c * N, sizeof(float), cudaMemcpyDeviceToHost, ctx->stream),
           "read W(0)");
    if (dsmc_tiled_supported(ctx->L, ctx->R))
        CU(launch_make_wk(ctx->Wc(), ctx->Wk(), ctx->L, ctx->stream, &ctx->launches), "W kernel layout");
    if (dsmc_fft_supported(ctx->L, ctx->R))
        CU(launch_make_fft_table(ctx->Wc(), ctx->M(), ctx->Z(), ctx->L, ctx->stream, &ctx->launches),
           "W spectral table");
    CU(cudaStreamSynchronize(ctx->stream), "tensor sync");
    ctx->tensor_built = true;
    ctx->field_valid[0] = ctx->field_valid[1] = false;
    ctx->spec_valid[0] = ctx->spec_valid[1] = false, ctx->zline = -1;
    drop_sweep_graph(ctx);  // W(0) is baked into the captured kernel parameters
    return DSMC_OK;
}

MetropolisArgs metropolis_args(dsmc_ctx *ctx, int colour, uint64_t seed, uint64_t step, int flags, uint8_t *accept_out,
                               float *margin_out) {
    MetropolisArgs a;
    a.S = ctx->S();
    a.H = ctx->H();
    a.invT = ctx->invT();
    a.K2 = ctx->K2d();
    a.K4 = ctx->K4d();
    a.L = ctx->L;
    a.R = ctx->R;
    a.colour = colour;
    a.rq_shift = -1;
    a.flip = (flags & DSMC_TRIAL_FLIP) ? 1 : 0;
    a.r_off = ctx->replica_offset;
    a.J = ctx->J;
    a.g = ctx->g;
    a.w0xx = ctx->w0[0];
    a.w0xy = ctx->w0[1];
    a.w0yy = ctx->w0[2];
    a.w0zz = ctx->w0[3];
    a.seed_lo = (uint32_t)(seed & 0xFFFFFFFFu);
    a.seed_hi = (uint32_t)(seed >> 32);
    a.step_lo = (uint32_t)(step & 0xFFFFFFFFu);
    a.step_hi = (uint32_t)(step >> 32) & 0x7FFFFFFFu;  // bit 31 is the init tag
    a.step_dev = nullptr;
    a.step_off = 0;
    a.accept_out = accept_out;
    a.margin_out = margin_out;
    a.pdl_late = 0;
    return a;
}

// One half-sweep: field of `colour` + Metropolis on it.  With the FFT field on a shape the fused row kernel supports, and no
// parity hooks, timing or field reuse asked for, the Metropolis decision rides in the field's last pass (field_fft.cu:
// two launches per half-sweep, h never written to global memory); otherwise field kernel(s) + metropolis kernel.  Both
// routes take bit-identical decisions (tests/test_gpu_parity.py::test_benchmarked_metropolis_instantiation_is_the_tested_one).
int enqueue_halfsweep(dsmc_ctx *ctx, const MetropolisArgs &a, int flags) {
    const int colour = a.colour;
    const bool fused = field_kind(ctx) == 2 && dsmc_fft_fused_supported(ctx->L, ctx->R) && !a.accept_out && !a.margin_out &&
                       !ctx->timing && !(flags & DSMC_REUSE_FIELD) && !ctx->no_fuse;
    if (fused) {
        const cudaError_t e = launch_field_fft(ctx->S(), ctx->M(), ctx->Z(), ctx->C(), ctx->H(), ctx->L, ctx->R, colour,
                                               ctx->spec_valid, &ctx->zline, &a, ctx->fft_pb0, ctx->fft_npb, ctx->fft_SG,
                                               &ctx->fft_configured, ctx->stream, &ctx->launches);
        if (e != cudaSuccess) return cuda_fail(ctx, e, "fused FFT half-sweep launch");
        ctx->field_valid[colour] = false;                       // h of this half-sweep never reached the field array
        return DSMC_OK;
    }
    if (ctx->timing) CU(cudaEventRecord(ctx->ev[0], ctx->stream), "event");
    if (!(flags & DSMC_REUSE_FIELD)) {
        if (int rc = run_field(ctx, colour)) return rc;
    } else if (!ctx->field_valid[colour]) {
        return fail(ctx, DSMC_ESTATE, "DSMC_REUSE_FIELD without a field of this colour");
    }
    if (ctx->timing) CU(cudaEventRecord(ctx->ev[1], ctx->stream), "event");
    CU(launch_metropolis(a, ctx->stream, &ctx->launches), "metropolis launch");
    if (ctx->timing) {
        CU(cudaEventRecord(ctx->ev[2], ctx->stream), "event");
        ctx->ev_recorded = true;
    }
    ctx->spec_valid[colour] = false;                            // the cached half-spectrum of this colour is stale now
    if (ctx->zline == colour) ctx->zline = -1;
    return DSMC_OK;
}

void drop_sweep_graph(dsmc_ctx *ctx) {
    if (ctx->sweep_graph) cudaGraphExecDestroy(ctx->sweep_graph);
    ctx->sweep_graph = nullptr;
    for (int b = 0; b < DSMC_MAX_BRANCHES - 1; ++b) {
        if (ctx->branch_graph[b]) cudaGraphExecDestroy(ctx->branch_graph[b]);
        ctx->branch_graph[b] = nullptr;
    }
    ctx->graph_branches = 1;
    if (ctx->pass_graph) cudaGraphExecDestroy(ctx->pass_graph);
    ctx->pass_graph = nullptr;
}

// the shared-memory-resident kernel serves the pass unless the FFT field was selected or the caller opts out
bool use_resident(dsmc_ctx *ctx, int l, int flags) {
    return field_kind(ctx) != 2 && !(flags & DSMC_NO_RESIDENT) && dsmc_resident_supported(ctx->L, l);
}

// enqueue one stride-l pass; pass_dev != null: offset and step come from the device counter (graph capture)
int enqueue_pass(dsmc_ctx *ctx, uint64_t seed, uint64_t pass, int l, int flags, uint8_t *accept_out, float *margin_out,
                 int *offset_out, const unsigned long long *pass_dev) {
    int ox = 0, oy = 0;
    if (!pass_dev) dsmc_sublattice_offset(seed, pass, l, &ox, &oy);
    if (offset_out) {
        offset_out[0] = ox;
        offset_out[1] = oy;
    }
    // With the FFT field selected, the whole field costs less than the direct sum over the n update sites
    // once L is large: compute it (for even l all update sites have the colour of the offset, which is
    // only known here when the offset is) and let the flip kernel read it.
    const bool fft = field_kind(ctx) == 2;
    if (use_resident(ctx, l, flags) && !pass_dev) {
        const MetropolisArgs a = metropolis_args(ctx, 0, seed, pass, flags, accept_out, margin_out);
        CU(launch_sublattice_resident(a, ctx->Wc(), l, pass, 1, ctx->stream, &ctx->launches), "resident pass launch");
        ctx->field_valid[0] = ctx->field_valid[1] = false;
        ctx->spec_valid[0] = ctx->spec_valid[1] = false, ctx->zline = -1;
        return DSMC_OK;
    }
    if (fft)
        if (int rc = run_field(ctx, ((l & 1) || pass_dev) ? -1 : ((ox + oy) & 1))) return rc;
    MetropolisArgs a = metropolis_args(ctx, 0, seed, pass, flags, accept_out, margin_out);
    a.step_dev = pass_dev;
    CU(launch_sublattice_pass(a, ctx->Wc(), ctx->stage(), ctx->sm_count, l, ox, oy, fft, ctx->stream, &ctx->launches),
       "sub-lattice pass launch");
    ctx->field_valid[0] = ctx->field_valid[1] = false;
    ctx->spec_valid[0] = ctx->spec_valid[1] = false, ctx->zline = -1;
    return DSMC_OK;
}

int build_pass_graph(dsmc_ctx *ctx, uint64_t seed, int l, int flags) {
    const int kind = field_kind(ctx);
    if (ctx->pass_graph && ctx->pgraph_seed == seed && ctx->pgraph_kind == kind && ctx->pgraph_flags == flags &&
        ctx->pgraph_l == l)
        return DSMC_OK;
    if (ctx->pass_graph) cudaGraphExecDestroy(ctx->pass_graph);
    ctx->pass_graph = nullptr;
    if (!ctx->capture_stream)
        CU(cudaStreamCreateWithFlags(&ctx->capture_stream, cudaStreamNonBlocking), "capture stream");
    cudaStream_t saved = ctx->stream;
    const uint64_t l0 = ctx->launches;
    ctx->stream = ctx->capture_stream;
    cudaGraph_t graph = nullptr;
    cudaError_t e = cudaStreamBeginCapture(ctx->capture_stream, cudaStreamCaptureModeThreadLocal);
    int rc = DSMC_OK;
    if (e == cudaSuccess) {
        for (int rep = 0; rep < DSMC_GRAPH_UNROLL && rc == DSMC_OK && e == cudaSuccess; ++rep) {
            rc = enqueue_pass(ctx, seed, 0, l, flags, nullptr, nullptr, nullptr, ctx->step_dev());
            if (rc == DSMC_OK) e = launch_step_update(ctx->step_dev(), 1, 1, ctx->stream, &ctx->launches);
        }
        cudaError_t e2 = cudaStreamEndCapture(ctx->capture_stream, &graph);
        if (e == cudaSuccess) e = e2;
    }
    ctx->stream = saved;
    ctx->pgraph_launches = ctx->launches - l0;
    ctx->launches = l0;
    if (rc != DSMC_OK || e != cudaSuccess) {
        if (graph) cudaGraphDestroy(graph);
        return rc != DSMC_OK ? rc : cuda_fail(ctx, e, "pass graph capture");
    }
    e = cudaGraphInstantiate(&ctx->pass_graph, graph, 0);
    cudaGraphDestroy(graph);
    if (e != cudaSuccess) {
        ctx->pass_graph = nullptr;
        return cuda_fail(ctx, e, "pass graph instantiate");
    }
    ctx->pgraph_seed = seed;
    ctx->pgraph_kind = kind;
    ctx->pgraph_flags = flags;
    ctx->pgraph_l = l;
    return DSMC_OK;
}

// the kernels of dsmc_ensemble_add: full field of the current state, raw sums, wall counts, running statistics
int enqueue_record(dsmc_ctx *ctx) {
    if (int rc = run_field(ctx, -1)) return rc;
    CU(launch_observables(ctx->S(), ctx->H(), ctx->K2d(), ctx->K4d(), ctx->obs(), ctx->opart(), ctx->ticket(0), ctx->L,
                          ctx->R, ctx->stream, &ctx->launches),
       "observables launch");
    CU(launch_wall_counts(ctx->S(), ctx->walls(), (unsigned long long *)ctx->opart(), ctx->ticket(1), ctx->L, ctx->R,
                          ctx->stream, &ctx->launches),
       "wall counts launch");
    CU(launch_ensemble_add(ctx->obs(), ctx->walls(), ctx->stats(), ctx->L, ctx->R, (double)ctx->J, (double)ctx->g,
                           ctx->stream, &ctx->launches),
       "ensemble launch");
    return DSMC_OK;
}

// Capture n sweeps -- each field + Metropolis of colour 0, of colour 1; then step counter += 2 n -- as a CUDA graph
// whose Metropolis kernels read the step from the device-resident counter, so that dsmc_run replays
// it with one launch per sweep instead of one per kernel (small lattices are launch-bound).
// record_every = 0: n = DSMC_GRAPH_UNROLL (dsmc_run); > 0: n = record_every sweeps followed by the kernels of
// dsmc_ensemble_add (dsmc_run_recorded).
int build_sweep_graph(dsmc_ctx *ctx, uint64_t seed, int flags, int record_every) {
    const int kind = field_kind(ctx);
    // the kernels a field call enqueues depend on which half-spectra are current (FFT field): a graph is only valid
    // from the state it was captured in, and must leave that state behind to be replayed back to back
    const int spec_in = (ctx->spec_valid[0] ? 1 : 0) | (ctx->spec_valid[1] ? 2 : 0) | ((ctx->zline + 1) << 2);
    if (ctx->sweep_graph && ctx->graph_seed == seed && ctx->graph_kind == kind && ctx->graph_flags == flags &&
        ctx->graph_every == record_every && ctx->graph_spec_in == spec_in)
        return DSMC_OK;
    drop_sweep_graph(ctx);
    if (!ctx->capture_stream)
        CU(cudaStreamCreateWithFlags(&ctx->capture_stream, cudaStreamNonBlocking), "capture stream");
    // Fused FFT path in its running state (y pass + fused row kernel per half-sweep): the line blocks of 16 replicas
    // never exchange data, so the sweeps are captured as up to DSMC_MAX_BRANCHES independent chains, one graph each with
    // its own step counter, which dsmc_run replays side by side on streams of the context's own between a fork and a
    // join event.  A chain's y pass (bound by L2 traffic) then overlaps another chain's row kernel (bound by instruction
    // issue) and no launch waits for the tail of a grid it does not depend on.  Same kernels on the same data: the
    // trajectory does not change.  (One graph with parallel branches was measured too and gained a third of what
    // separate graphs on separate streams gain.)
    const int blocks = dsmc_fft_line_blocks(ctx->L, ctx->R);
    int branches = 1;
    // (measured: a gain from L = 64 up -- 10-20 % where the working set fits the L2 -- and a loss of 5 % at L = 32)
    if (kind == 2 && blocks > 1 && ctx->L >= 64 && record_every == 0 && !ctx->no_fuse && !ctx->timing && ctx->zline >= 0 &&
        ctx->spec_valid[1 - ctx->zline] && !ctx->spec_valid[ctx->zline])
        for (int b = 2; b <= ctx->max_branches; ++b)
            if (blocks % b == 0) branches = b;
    for (int b = 0; b + 1 < branches; ++b) {
        if (!ctx->branch_stream[b])
            CU(cudaStreamCreateWithFlags(&ctx->branch_stream[b], cudaStreamNonBlocking), "branch stream");
        if (!ctx->ev_join[b]) CU(cudaEventCreateWithFlags(&ctx->ev_join[b], cudaEventDisableTiming), "join event");
    }
    if (branches > 1 && !ctx->ev_fork) CU(cudaEventCreateWithFlags(&ctx->ev_fork, cudaEventDisableTiming), "fork event");
    cudaStream_t saved = ctx->stream;
    const uint64_t l0 = ctx->launches;
    const int n_sweeps = record_every > 0 ? record_every : DSMC_GRAPH_UNROLL;
    int spec_out = spec_in;
    int rc = DSMC_OK;
    cudaError_t e = cudaSuccess;
    const char *what = "sweep graph capture";
    for (int b = 0; b < branches && rc == DSMC_OK && e == cudaSuccess; ++b) {
        ctx->stream = ctx->capture_stream;
        ctx->spec_valid[0] = spec_in & 1;                       // every chain starts from the state before the capture
        ctx->spec_valid[1] = (spec_in & 2) != 0;
        ctx->zline = (spec_in >> 2) - 1;
        if (branches > 1) {
            ctx->fft_pb0 = b * (blocks / branches);
            ctx->fft_npb = blocks / branches;
            ctx->fft_SG = ctx->stage();                         // the chains work on the block-major copy (replay_sweep_graph)
        }
        cudaGraph_t graph = nullptr;
        e = cudaStreamBeginCapture(ctx->capture_stream, cudaStreamCaptureModeThreadLocal);
        if (e == cudaSuccess) {
            for (int rep = 0; rep < n_sweeps && rc == DSMC_OK; ++rep) {
                for (int colour = 0; colour < 2 && rc == DSMC_OK; ++colour) {
                    MetropolisArgs a = metropolis_args(ctx, colour, seed, 0, flags, nullptr, nullptr);
                    a.step_dev = ctx->step_dev() + b;
                    a.step_off = (uint32_t)(2 * rep + colour);  // the counter moves once per graph, not once per sweep
                    rc = enqueue_halfsweep(ctx, a, flags);
                }
            }
            if (rc == DSMC_OK)
                e = launch_step_update(ctx->step_dev() + b, 2 * (uint64_t)n_sweeps, 1, ctx->stream, &ctx->launches);
            if (e == cudaSuccess && rc == DSMC_OK && record_every > 0) rc = enqueue_record(ctx);
            cudaError_t e2 = cudaStreamEndCapture(ctx->capture_stream, &graph);
            if (e == cudaSuccess) e = e2;
        }
        spec_out = (ctx->spec_valid[0] ? 1 : 0) | (ctx->spec_valid[1] ? 2 : 0) | ((ctx->zline + 1) << 2);
        if (rc == DSMC_OK && e == cudaSuccess) {
            what = "sweep graph instantiate";
            e = cudaGraphInstantiate(b == 0 ? &ctx->sweep_graph : &ctx->branch_graph[b - 1], graph, 0);
        }
        if (graph) cudaGraphDestroy(graph);
    }
    ctx->stream = saved;
    ctx->fft_pb0 = ctx->fft_npb = 0;
    ctx->fft_SG = nullptr;
    ctx->graph_launches = ctx->launches - l0;
    ctx->launches = l0;
    ctx->spec_valid[0] = spec_in & 1;                           // nothing has run: back to the state before the capture
    ctx->spec_valid[1] = (spec_in & 2) != 0;
    ctx->zline = (spec_in >> 2) - 1;
    if (rc == DSMC_OK && e == cudaSuccess && spec_out != spec_in) {
        drop_sweep_graph(ctx);
        return fail(ctx, DSMC_ESTATE, "internal: a captured sweep does not return to the spectrum state it started from");
    }
    if (rc != DSMC_OK) {
        drop_sweep_graph(ctx);
        return rc;
    }
    if (e != cudaSuccess) {
        drop_sweep_graph(ctx);
        return cuda_fail(ctx, e, what);
    }
    ctx->graph_seed = seed;
    ctx->graph_kind = kind;
    ctx->graph_flags = flags;
    ctx->graph_every = record_every;
    ctx->graph_spec_in = spec_in;
    ctx->graph_spec_out = spec_out;
    ctx->graph_branches = branches;
    return DSMC_OK;
}

// replay the captured sweeps `reps` times from step `step`: one chain on the context's stream, or the chains of the fused
// FFT path side by side (build_sweep_graph) -- the others on the context's branch streams, forked from and joined back
// into its stream, so that the call keeps plain stream order towards everything before and after it
int replay_sweep_graph(dsmc_ctx *ctx, uint64_t step, uint64_t reps) {
    const int nb = ctx->graph_branches;
    for (int b = 0; b < nb; ++b)
        CU(launch_step_update(ctx->step_dev() + b, step, 0, ctx->stream, &ctx->launches), "step counter");
    // The chains work on a block-major copy of the spins (in the host-transfer staging area, idle during a run): a chain's
    // 16 replicas are 64 bytes of every 256-byte site record of S, and chains that drift apart would fetch and write back
    // half cache lines at different times; in the copy every chain's spins are dense.  Measured at config 5, four chains:
    // 101.0 us per sweep on S, 91.3 on the copy (one chain: 103.6 either way).
    if (nb > 1) {
        CU(launch_spin_blocks(ctx->S(), ctx->stage(), ctx->L, ctx->R, true, ctx->stream, &ctx->launches), "spins to blocks");
        CU(cudaEventRecord(ctx->ev_fork, ctx->stream), "fork event");
    }
    for (int b = 1; b < nb; ++b) CU(cudaStreamWaitEvent(ctx->branch_stream[b - 1], ctx->ev_fork, 0), "fork wait");
    for (uint64_t j = 0; j < reps; ++j)
        for (int b = 0; b < nb; ++b)
            CU(cudaGraphLaunch(b == 0 ? ctx->sweep_graph : ctx->branch_graph[b - 1], b == 0 ? ctx->stream : ctx->branch_stream[b - 1]),
               "sweep graph launch");
    for (int b = 1; b < nb; ++b) {
        CU(cudaEventRecord(ctx->ev_join[b - 1], ctx->branch_stream[b - 1]), "join event");
        CU(cudaStreamWaitEvent(ctx->stream, ctx->ev_join[b - 1], 0), "join wait");
    }
    if (nb > 1)
        CU(launch_spin_blocks(ctx->S(), ctx->stage(), ctx->L, ctx->R, false, ctx->stream, &ctx->launches), "blocks to spins");
    ctx->launches += reps * ctx->graph_launches;
    return DSMC_OK;
}

}  // namespace

DsmcLayout dsmc_make_layout(int L, int R) {
    DsmcLayout l;
    const size_t N = (size_t)L * L, Nh = N / 2;
    size_t o = 0;
    l.off_Wc = o; o = align256(o + sizeof(float) * 4 * N);
    l.off_Wk = o; o = align256(o + sizeof(float) * dsmc_wk_floats(L));
    l.off_S = o; o = align256(o + sizeof(float) * 6 * Nh * R);
    l.off_H = o; o = align256(o + sizeof(float) * 6 * Nh * R);
    l.off_Hpart = o;
    o = align256(o + (dsmc_tiled_supported(L, R) ? sizeof(float) * DSMC_KS_MAX * 3 * Nh * R : 0));
    const bool fft = dsmc_fft_supported(L, R);
    l.off_M = o; o = align256(o + (fft ? sizeof(float) * dsmc_fft_m_floats(L) : 0));
    l.off_Z = o; o = align256(o + (fft ? dsmc_fft_scratch_bytes(L, R) : 0));
    l.off_C = o; o = align256(o + (fft ? dsmc_fft_cache_bytes(L, R) : 0));
    l.off_stage = o; o = align256(o + sizeof(float) * 3 * N * R);
    l.off_T = o; o = align256(o + sizeof(float) * 3 * R);
    l.off_obs = o; o = align256(o + sizeof(double) * 8 * R);
    l.off_walls = o; o = align256(o + sizeof(unsigned long long) * 8 * R);
    l.off_stats = o; o = align256(o + sizeof(double) * 16 * R);
    l.off_opart = o; o = align256(o + dsmc_walk_scratch_bytes(L, R));
    l.off_ticket = o; o = align256(o + 4 * sizeof(unsigned int));
    l.off_step = o; o = align256(o + sizeof(unsigned long long));
    l.total = o;
    return l;
}

extern "C" {

const char *dsmc_version(void) { return "dsmc 0.1 (sm_100a)"; }

int dsmc_create(dsmc_ctx **out, int L, int R, float J, float g, float K2, float K4) {
    if (!out) return DSMC_EINVAL;
    *out = nullptr;
    if (!shape_ok(L, R)) return DSMC_EINVAL;
    dsmc_ctx *c = new (std::nothrow) dsmc_ctx();
    if (!c) return DSMC_ENOMEM;
    c->L = L;
    c->R = R;
    c->J = J;
    c->g = g;
    c->K2.assign(R, K2);
    c->K4.assign(R, K4);
    c->T.assign(R, 0.0f);
    c->lay = dsmc_make_layout(L, R);
    if (const char *v = getenv("DSMC_NO_FUSE")) c->no_fuse = v[0] && v[0] != '0';
    if (const char *v = getenv("DSMC_BRANCHES")) {
        const int n = atoi(v);
        if (n >= 1 && n <= DSMC_MAX_BRANCHES) c->max_branches = n;
    }
    *out = c;
    return DSMC_OK;
}

int dsmc_set_anisotropy(dsmc_ctx *ctx, const float *K2_r, const float *K4_r) {
    if (!ctx || !K2_r || !K4_r) return fail(ctx, DSMC_EINVAL, "null argument");
    ctx->K2.assign(K2_r, K2_r + ctx->R);
    ctx->K4.assign(K4_r, K4_r + ctx->R);
    ctx->aniso_dirty = true;
    return DSMC_OK;
}

int dsmc_set_replica_offset(dsmc_ctx *ctx, uint32_t first_replica) {
    if (!ctx) return DSMC_EINVAL;
    ctx->replica_offset = first_replica;
    drop_sweep_graph(ctx);  // the offset is baked into the captured kernel parameters
    return DSMC_OK;
}

size_t dsmc_workspace_bytes(int L, int R) {
    if (!shape_ok(L, R)) return 0;
    return dsmc_make_layout(L, R).total;
}

int dsmc_bind(dsmc_ctx *ctx, void *dev_workspace, size_t bytes, void *cuda_stream) {
    if (!ctx || !dev_workspace) return fail(ctx, DSMC_EINVAL, "null argument");
    if (((uintptr_t)dev_workspace & 255) != 0) return fail(ctx, DSMC_EINVAL, "workspace must be 256-byte aligned");
    if (bytes < ctx->lay.total) return fail(ctx, DSMC_ENOMEM, "workspace smaller than dsmc_workspace_bytes");
    cudaPointerAttributes attr;
    CU(cudaPointerGetAttributes(&attr, dev_workspace), "cudaPointerGetAttributes");
    if (attr.type != cudaMemoryTypeDevice && attr.type != cudaMemoryTypeManaged)
        return fail(ctx, DSMC_EINVAL, "workspace is not device memory");
    ctx->device = attr.device;                                  // the workspace's device, not the caller's current one
    DeviceGuard guard__(ctx->device);
    CU(cudaDeviceGetAttribute(&ctx->sm_count, cudaDevAttrMultiProcessorCount, ctx->device), "SM count");
    ctx->tiled_configured = ctx->fft_configured = false;
    drop_sweep_graph(ctx);
    ctx->ws = (char *)dev_workspace;
    ctx->ws_bytes = bytes;
    ctx->stream = (cudaStream_t)cuda_stream;
    ctx->tensor_built = ctx->spins_set = false;
    ctx->field_valid[0] = ctx->field_valid[1] = false;
    ctx->spec_valid[0] = ctx->spec_valid[1] = false, ctx->zline = -1;
    ctx->T_valid = false;
    ctx->aniso_dirty = true;
    for (int i = 0; i < 3; ++i)
        if (!ctx->ev[i]) CU(cudaEventCreate(&ctx->ev[i]), "cudaEventCreate");
    // the ensemble sums start empty; the arrival counters of the observable reductions start (and are left) at zero
    CU(cudaMemsetAsync(ctx->stats(), 0, sizeof(double) * 16 * (size_t)ctx->R, ctx->stream), "ensemble init");
    CU(cudaMemsetAsync(ctx->ticket(0), 0, 4 * sizeof(unsigned int), ctx->stream), "ticket init");
    ctx->ensemble_n = 0;
    return DSMC_OK;
}

int dsmc_build_tensor(dsmc_ctx *ctx, int method, int cutoff_A, int tail) {
    ENTER_BOUND(ctx);
    if (method != DSMC_W_IMAGE && method != DSMC_W_EWALD) return fail(ctx, DSMC_EINVAL, "unknown method");
    if (method == DSMC_W_IMAGE && (cutoff_A < 0 || cutoff_A > 4096)) return fail(ctx, DSMC_EINVAL, "bad cutoff");
    CU(launch_build_tensor(nullptr, ctx->Wc(), ctx->L, method, cutoff_A, tail, ctx->stream, &ctx->launches),
       "build tensor");
    return after_tensor_change(ctx);
}

int dsmc_get_tensor(dsmc_ctx *ctx, float *W_out, int where) {
    ENTER_BOUND(ctx);
    if (!W_out) return fail(ctx, DSMC_EINVAL, "null argument");
    if (!ctx->tensor_built) return fail(ctx, DSMC_ESTATE, "tensor not built");
    const size_t bytes = sizeof(float) * 4 * (size_t)ctx->L * ctx->L;
    CU(cudaMemcpyAsync(W_out, ctx->Wc(), bytes, where == DSMC_HOST ? cudaMemcpyDeviceToHost : cudaMemcpyDeviceToDevice,
                       ctx->stream),
       "get tensor");
    if (where == DSMC_HOST) CU(cudaStreamSynchronize(ctx->stream), "get tensor sync");
    return DSMC_OK;
}

int dsmc_set_tensor(dsmc_ctx *ctx, const float *W_in, int where) {
    ENTER_BOUND(ctx);
    if (!W_in) return fail(ctx, DSMC_EINVAL, "null argument");
    const size_t bytes = sizeof(float) * 4 * (size_t)ctx->L * ctx->L;
    CU(cudaMemcpyAsync(ctx->Wc(), W_in, bytes, where == DSMC_HOST ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice,
                       ctx->stream),
       "set tensor");
    return after_tensor_change(ctx);
}

int dsmc_set_spins(dsmc_ctx *ctx, const float *s, int where) {
    ENTER_BOUND(ctx);
    if (!s) return fail(ctx, DSMC_EINVAL, "null argument");
    const float *src = s;
    if (where == DSMC_HOST) {
        CU(cudaMemcpyAsync(ctx->stage(), s, sizeof(float) * 3 * (size_t)ctx->L * ctx->L * ctx->R,
                           cudaMemcpyHostToDevice, ctx->stream),
           "spins H2D");
        src = ctx->stage();
    }
    CU(launch_canon_to_internal(src, ctx->S(), ctx->L, ctx->R, ctx->stream, &ctx->launches), "set spins");
    ctx->field_valid[0] = ctx->field_valid[1] = false;
    ctx->spec_valid[0] = ctx->spec_valid[1] = false, ctx->zline = -1;
    if (ctx->debug) {
        // |s| = 1 is the caller's contract, checked to 1e-5 when debugging is on (one reduction kernel and
        // one synchronisation; the default path pays nothing)
        float worst = 0.0f;
        float *dev = reinterpret_cast<float *>(ctx->opart());
        CU(launch_norm_check(ctx->S(), dev, ctx->L, ctx->R, ctx->stream, &ctx->launches), "norm check");
        CU(cudaMemcpyAsync(&worst, dev, sizeof(float), cudaMemcpyDeviceToHost, ctx->stream), "norm check D2H");
        CU(cudaStreamSynchronize(ctx->stream), "norm check sync");
        if (!(worst <= 2.0e-5f)) {                             // | |s|^2 - 1 | = 2 | |s| - 1 | to first order
            ctx->spins_set = false;
            char msg[128];
            snprintf(msg, sizeof msg, "dsmc_set_spins: a spin is not a unit vector (max | |s|^2 - 1 | = %.3g)", (double)worst);
            return fail(ctx, DSMC_EINVAL, msg);
        }
    }
    ctx->spins_set = true;
    return DSMC_OK;
}

int dsmc_get_spins(dsmc_ctx *ctx, float *s, int where) {
    ENTER_BOUND(ctx);
    if (!s) return fail(ctx, DSMC_EINVAL, "null argument");
    if (!ctx->spins_set) return fail(ctx, DSMC_ESTATE, "spins not set");
    float *dst = where == DSMC_HOST ? ctx->stage() : s;
    CU(launch_internal_to_canon(ctx->S(), dst, ctx->L, ctx->R, -1, ctx->stream, &ctx->launches), "get spins");
    if (where == DSMC_HOST) {
        CU(cudaMemcpyAsync(s, dst, sizeof(float) * 3 * (size_t)ctx->L * ctx->L * ctx->R, cudaMemcpyDeviceToHost,
                           ctx->stream),
           "spins D2H");
        CU(cudaStreamSynchronize(ctx->stream), "spins D2H sync");
    }
    return DSMC_OK;
}

int dsmc_init_spins(dsmc_ctx *ctx, int mode, uint64_t seed) {
    ENTER_BOUND(ctx);
    if (mode != DSMC_INIT_RANDOM && mode != DSMC_INIT_UP) return fail(ctx, DSMC_EINVAL, "unknown init mode");
    CU(launch_init_spins(ctx->S(), ctx->L, ctx->R, mode, seed, ctx->replica_offset, ctx->stream, &ctx->launches), "init spins");
    ctx->spins_set = true;
    ctx->field_valid[0] = ctx->field_valid[1] = false;
    ctx->spec_valid[0] = ctx->spec_valid[1] = false, ctx->zline = -1;
    return DSMC_OK;
}

int dsmc_dipole_field(dsmc_ctx *ctx, int colour, float *h_out, int where) {
    ENTER_BOUND(ctx);
    if (colour < -1 || colour > 1) return fail(ctx, DSMC_EINVAL, "colour must be -1, 0 or 1");
    if (!ctx->tensor_built) return fail(ctx, DSMC_ESTATE, "tensor not built");
    if (!ctx->spins_set) return fail(ctx, DSMC_ESTATE, "spins not set");
    if (int rc = run_field(ctx, colour)) return rc;
    if (h_out) {
        const size_t bytes = sizeof(float) * 3 * (size_t)ctx->L * ctx->L * ctx->R;
        float *dst = h_out;
        if (where == DSMC_HOST) {
            // inactive entries must stay untouched: bring the caller's buffer in first
            CU(cudaMemcpyAsync(ctx->stage(), h_out, bytes, cudaMemcpyHostToDevice, ctx->stream), "h H2D");
            dst = ctx->stage();
        }
        CU(launch_internal_to_canon(ctx->H(), dst, ctx->L, ctx->R, colour, ctx->stream, &ctx->launches), "get field");
        if (where == DSMC_HOST) {
            CU(cudaMemcpyAsync(h_out, dst, bytes, cudaMemcpyDeviceToHost, ctx->stream), "h D2H");
            CU(cudaStreamSynchronize(ctx->stream), "h D2H sync");
        }
    }
    return DSMC_OK;
}

int dsmc_get_field(dsmc_ctx *ctx, float *h_out, int where) {
    ENTER_BOUND(ctx);
    if (!h_out) return fail(ctx, DSMC_EINVAL, "null argument");
    if (!ctx->field_valid[0] || !ctx->field_valid[1]) return fail(ctx, DSMC_ESTATE, "no field of both colours is kept");
    float *dst = where == DSMC_HOST ? ctx->stage() : h_out;
    CU(launch_internal_to_canon(ctx->H(), dst, ctx->L, ctx->R, -1, ctx->stream, &ctx->launches), "get field");
    if (where == DSMC_HOST) {
        CU(cudaMemcpyAsync(h_out, dst, sizeof(float) * 3 * (size_t)ctx->L * ctx->L * ctx->R, cudaMemcpyDeviceToHost,
                           ctx->stream),
           "h D2H");
        CU(cudaStreamSynchronize(ctx->stream), "h D2H sync");
    }
    return DSMC_OK;
}

int dsmc_halfsweep_ex(dsmc_ctx *ctx, const float *T, uint64_t seed, uint64_t step, int flags, uint8_t *accept_out,
                      float *margin_out) {
    ENTER_BOUND(ctx);
    if (!ctx->tensor_built) return fail(ctx, DSMC_ESTATE, "tensor not built");
    if (!ctx->spins_set) return fail(ctx, DSMC_ESTATE, "spins not set");
    if (flags & ~(DSMC_REUSE_FIELD | DSMC_TRIAL_FLIP)) return fail(ctx, DSMC_EINVAL, "unknown flag");
    if (int rc = upload_params(ctx, T)) return rc;
    const int colour = (int)(step & 1u);
    const MetropolisArgs a = metropolis_args(ctx, colour, seed, step, flags, accept_out, margin_out);
    // field_valid only records that H holds a field of that colour computed since the spins were
    // last set (what DSMC_REUSE_FIELD needs for timing); observables always recompute both colours
    return enqueue_halfsweep(ctx, a, flags);
}

int dsmc_halfsweep(dsmc_ctx *ctx, const float *T, uint64_t seed, uint64_t step) {
    return dsmc_halfsweep_ex(ctx, T, seed, step, 0, nullptr, nullptr);
}

int dsmc_sublattice_pass(dsmc_ctx *ctx, const float *T, uint64_t seed, uint64_t pass, int l, int flags,
                         uint8_t *accept_out, float *margin_out, int *offset_out) {
    ENTER_BOUND(ctx);
    if (!ctx->tensor_built) return fail(ctx, DSMC_ESTATE, "tensor not built");
    if (!ctx->spins_set) return fail(ctx, DSMC_ESTATE, "spins not set");
    if (flags & ~(DSMC_TRIAL_FLIP | DSMC_NO_RESIDENT)) return fail(ctx, DSMC_EINVAL, "unknown flag");
    if (l < 2 || ctx->L % l) return fail(ctx, DSMC_EINVAL, "l must be >= 2 and divide L");
    if (int rc = upload_params(ctx, T)) return rc;
    return enqueue_pass(ctx, seed, pass, l, flags, accept_out, margin_out, offset_out, nullptr);
}

int dsmc_sublattice_run(dsmc_ctx *ctx, const float *T, uint64_t seed, uint64_t first_pass, uint64_t n_passes, int l,
                        int flags) {
    return dsmc_sublattice_run_ex(ctx, T, seed, first_pass, n_passes, l, flags, nullptr);
}

int dsmc_sublattice_run_ex(dsmc_ctx *ctx, const float *T, uint64_t seed, uint64_t first_pass, uint64_t n_passes, int l,
                           int flags, float *margin_log) {
    ENTER_BOUND(ctx);
    if (flags & DSMC_INCREMENTAL) {
        if (flags & ~(DSMC_TRIAL_FLIP | DSMC_INCREMENTAL)) return fail(ctx, DSMC_EINVAL, "unknown flag");
        if (!ctx->tensor_built) return fail(ctx, DSMC_ESTATE, "tensor not built");
        if (!ctx->spins_set) return fail(ctx, DSMC_ESTATE, "spins not set");
        if (l < 2 || ctx->L % l || !dsmc_incremental_supported(ctx->L, l))
            return fail(ctx, DSMC_EINVAL, "DSMC_INCREMENTAL needs L / l in {1, 2, 4} and L * L <= 4096");
        if (int rc = upload_params(ctx, T)) return rc;
        // the field of every site from a field kernel (the FFT one when the shape allows: microseconds), then up to
        // DSMC_INCREMENTAL_REFRESH passes of rank-n updates in registers; the refresh bounds the rounding drift
        const int kind = dsmc_fft_supported(ctx->L, ctx->R) ? 2 : (dsmc_tiled_supported(ctx->L, ctx->R) ? 1 : 0);
        for (uint64_t done = 0; done < n_passes;) {
            const uint64_t chunk = n_passes - done < DSMC_INCREMENTAL_REFRESH ? n_passes - done : DSMC_INCREMENTAL_REFRESH;
            if (int rc = run_field(ctx, -1, kind)) return rc;
            const MetropolisArgs a = metropolis_args(ctx, 0, seed, first_pass + done, flags, nullptr, nullptr);
            CU(launch_sublattice_incremental(a, ctx->Wc(), ctx->H(), l, first_pass + done, chunk,
                                             margin_log ? margin_log + done * (uint64_t)ctx->R * (uint64_t)((ctx->L / l) * (ctx->L / l)) : nullptr,
                                             ctx->stream, &ctx->launches),
               "incremental run launch");
            ctx->spec_valid[0] = ctx->spec_valid[1] = false, ctx->zline = -1;
            done += chunk;
        }
        ctx->field_valid[0] = ctx->field_valid[1] = true;      // H holds the (incrementally updated) field of the final state
        return DSMC_OK;
    }
    if (margin_log) return fail(ctx, DSMC_EINVAL, "margin_log needs DSMC_INCREMENTAL");
    if (n_passes >= 2 && l >= 2 && ctx->L % l == 0 && !(flags & ~(DSMC_TRIAL_FLIP | DSMC_NO_RESIDENT)) &&
        ctx->tensor_built && ctx->spins_set && use_resident(ctx, l, flags)) {
        // every pass of the run inside one kernel (per 65536 passes), the lattice in shared memory
        if (int rc = upload_params(ctx, T)) return rc;
        const MetropolisArgs a = metropolis_args(ctx, 0, seed, first_pass, flags, nullptr, nullptr);
        CU(launch_sublattice_resident(a, ctx->Wc(), l, first_pass, n_passes, ctx->stream, &ctx->launches),
           "resident run launch");
        ctx->field_valid[0] = ctx->field_valid[1] = false;
        ctx->spec_valid[0] = ctx->spec_valid[1] = false, ctx->zline = -1;
        return DSMC_OK;
    }
    uint64_t k = 0;
    auto plain = [&](uint64_t count) -> int {
        for (uint64_t j = 0; j < count; ++j, ++k)
            if (int rc = dsmc_sublattice_pass(ctx, k == 0 ? T : nullptr, seed, first_pass + k, l, flags, nullptr, nullptr,
                                              nullptr))
                return rc;
        return DSMC_OK;
    };
    if (n_passes >= 1 + 2 * DSMC_GRAPH_UNROLL) {
        // the first pass runs launch by launch (argument checks, kernel configuration), the rest is replayed
        // from a captured graph of DSMC_GRAPH_UNROLL passes whose kernels derive offset and step from a device counter
        if (int rc = plain(1)) return rc;
        if (int rc = build_pass_graph(ctx, seed, l, flags)) return rc;
        CU(launch_step_update(ctx->step_dev(), first_pass + k, 0, ctx->stream, &ctx->launches), "pass counter");
        const uint64_t reps = (n_passes - k) / DSMC_GRAPH_UNROLL;
        for (uint64_t j = 0; j < reps; ++j) CU(cudaGraphLaunch(ctx->pass_graph, ctx->stream), "pass graph launch");
        ctx->launches += reps * ctx->pgraph_launches;
        k += reps * DSMC_GRAPH_UNROLL;
    }
    return plain(n_passes - k);
}

int dsmc_run(dsmc_ctx *ctx, const float *T, uint64_t seed, uint64_t first_step, uint64_t n_half) {
    return dsmc_run_ex(ctx, T, seed, first_step, n_half, 0);
}

int dsmc_run_ex(dsmc_ctx *ctx, const float *T, uint64_t seed, uint64_t first_step, uint64_t n_half, int flags) {
    ENTER_BOUND(ctx);
    if (flags & ~DSMC_TRIAL_FLIP) return fail(ctx, DSMC_EINVAL, "unknown flag");
    uint64_t k = 0;
    auto plain = [&](uint64_t count) -> int {
        for (uint64_t j = 0; j < count; ++j, ++k)
            if (int rc = dsmc_halfsweep_ex(ctx, k == 0 ? T : nullptr, seed, first_step + k, flags, nullptr, nullptr)) return rc;
        return DSMC_OK;
    };
    if (n_half >= 4 + 4 * DSMC_GRAPH_UNROLL && !ctx->timing) {
        // an odd first step and one whole sweep run launch by launch (this also configures every kernel
        // before the capture); the bulk is replayed from the captured graph; the tail runs plainly again
        if (int rc = plain((first_step & 1u) + 2)) return rc;
        const uint64_t reps = (n_half - k) / (2 * DSMC_GRAPH_UNROLL);
        if (reps >= 1) {
            if (int rc = build_sweep_graph(ctx, seed, flags, 0)) return rc;
            if (int rc = replay_sweep_graph(ctx, first_step + k, reps)) return rc;
            ctx->field_valid[0] = ctx->field_valid[1] = true;
            ctx->spec_valid[0] = ctx->graph_spec_out & 1;           // (= the state the graph started from)
            ctx->spec_valid[1] = (ctx->graph_spec_out & 2) != 0;
            ctx->zline = (ctx->graph_spec_out >> 2) - 1;
            k += 2 * DSMC_GRAPH_UNROLL * reps;
        }
    }
    return plain(n_half - k);
}

int dsmc_observables(dsmc_ctx *ctx, double *out) {
    ENTER_BOUND(ctx);
    if (!out) return fail(ctx, DSMC_EINVAL, "null argument");
    if (!ctx->tensor_built) return fail(ctx, DSMC_ESTATE, "tensor not built");
    if (!ctx->spins_set) return fail(ctx, DSMC_ESTATE, "spins not set");
    if (int rc = upload_aniso(ctx)) return rc;
    if (int rc = run_field(ctx, -1)) return rc;
    CU(launch_observables(ctx->S(), ctx->H(), ctx->K2d(), ctx->K4d(), ctx->obs(), ctx->opart(), ctx->ticket(0), ctx->L,
                          ctx->R, ctx->stream, &ctx->launches),
       "observables launch");
    std::vector<double> raw(8 * (size_t)ctx->R);
    CU(cudaMemcpyAsync(raw.data(), ctx->obs(), sizeof(double) * raw.size(), cudaMemcpyDeviceToHost, ctx->stream),
       "observables D2H");
    CU(cudaStreamSynchronize(ctx->stream), "observables sync");
    const double N = (double)ctx->L * ctx->L;
    for (int r = 0; r < ctx->R; ++r) {
        const double *s = &raw[8 * (size_t)r];
        const double mx = s[0] / N, my = s[1] / N;
        out[4 * r + 0] = (-(double)ctx->J * s[4] - s[5] + 0.5 * (double)ctx->g * s[6]) / N;
        out[4 * r + 1] = s[2] / N;
        out[4 * r + 2] = sqrt(mx * mx + my * my);
        out[4 * r + 3] = (2.0 / 3.14159265358979323846) * sqrt(s[3] / N);
    }
    return DSMC_OK;
}

int dsmc_wall_observables(dsmc_ctx *ctx, long long *counts_out, double *derived_out) {
    ENTER_BOUND(ctx);
    if (!counts_out) return fail(ctx, DSMC_EINVAL, "null argument");
    if (!ctx->spins_set) return fail(ctx, DSMC_ESTATE, "spins not set");
    unsigned long long *dev = ctx->walls();
    CU(launch_wall_counts(ctx->S(), dev, (unsigned long long *)ctx->opart(), ctx->ticket(1), ctx->L, ctx->R, ctx->stream,
                          &ctx->launches),
       "wall counts launch");
    std::vector<unsigned long long> raw(8 * (size_t)ctx->R);
    CU(cudaMemcpyAsync(raw.data(), dev, sizeof(unsigned long long) * raw.size(), cudaMemcpyDeviceToHost, ctx->stream),
       "wall counts D2H");
    CU(cudaStreamSynchronize(ctx->stream), "wall counts sync");
    const double N = (double)ctx->L * ctx->L;
    for (int r = 0; r < ctx->R; ++r) {
        const unsigned long long *n = &raw[8 * (size_t)r];
        for (int k = 0; k < 6; ++k) counts_out[6 * r + k] = (long long)n[k];
        if (derived_out) {
            derived_out[4 * r] = (double)(n[4] + n[5]) / (4.0 * N);
            for (int c = 0; c < 3; ++c) {
                const unsigned long long nh = n[2 * c], nv = n[2 * c + 1];
                derived_out[4 * r + 1 + c] = nh + nv ? (double)(nh > nv ? nh - nv : nv - nh) / (double)(nh + nv) : 0.0;
            }
        }
    }
    return DSMC_OK;
}

int dsmc_staggered_magnetisation(dsmc_ctx *ctx, double *out) {
    ENTER_BOUND(ctx);
    if (!out) return fail(ctx, DSMC_EINVAL, "null argument");
    if (!ctx->spins_set) return fail(ctx, DSMC_ESTATE, "spins not set");
    CU(launch_staggered(ctx->S(), ctx->obs(), ctx->opart(), ctx->ticket(2), ctx->L, ctx->R, ctx->stream, &ctx->launches),
       "staggered launch");
    std::vector<double> raw(8 * (size_t)ctx->R);
    CU(cudaMemcpyAsync(raw.data(), ctx->obs(), sizeof(double) * raw.size(), cudaMemcpyDeviceToHost, ctx->stream),
       "staggered D2H");
    CU(cudaStreamSynchronize(ctx->stream), "staggered sync");
    const double N = (double)ctx->L * ctx->L;
    for (int r = 0; r < ctx->R; ++r) {
        const double *m = &raw[8 * (size_t)r];
        const double mh = (m[0] + m[1] - m[2] - m[3]) / N, mv = (m[0] + m[3] - m[2] - m[1]) / N;
        out[3 * r + 0] = mh;
        out[3 * r + 1] = mv;
        out[3 * r + 2] = sqrt(mh * mh + mv * mv);
    }
    return DSMC_OK;
}

int dsmc_ensemble_reset(dsmc_ctx *ctx) {
    ENTER_BOUND(ctx);
    CU(cudaMemsetAsync(ctx->stats(), 0, sizeof(double) * 16 * (size_t)ctx->R, ctx->stream), "ensemble reset");
    ctx->ensemble_n = 0;
    return DSMC_OK;
}

int dsmc_ensemble_add(dsmc_ctx *ctx) {
    ENTER_BOUND(ctx);
    if (!ctx->tensor_built) return fail(ctx, DSMC_ESTATE, "tensor not built");
    if (!ctx->spins_set) return fail(ctx, DSMC_ESTATE, "spins not set");
    if (int rc = upload_aniso(ctx)) return rc;
    if (int rc = enqueue_record(ctx)) return rc;
    ++ctx->ensemble_n;
    return DSMC_OK;
}

int dsmc_run_recorded(dsmc_ctx *ctx, const float *T, uint64_t seed, uint64_t first_step, uint64_t n_records, int every,
                      int flags) {
    ENTER_BOUND(ctx);
    if (flags & ~DSMC_TRIAL_FLIP) return fail(ctx, DSMC_EINVAL, "unknown flag");
    if (every < 1) return fail(ctx, DSMC_EINVAL, "every must be >= 1");
    if (first_step & 1u) return fail(ctx, DSMC_EINVAL, "first_step must be even (whole sweeps)");
    uint64_t done = 0;
    auto plain = [&]() -> int {                                  // one record launch by launch
        if (int rc = dsmc_run_ex(ctx, done == 0 ? T : nullptr, seed, first_step + 2 * (uint64_t)every * done,
                                 2 * (uint64_t)every, flags))
            return rc;
        ++done;
        return dsmc_ensemble_add(ctx);
    };
    if (n_records == 0) return T ? upload_params(ctx, T) : DSMC_OK;
    // the first record runs plainly (uploads T, configures every kernel before a capture); short spacings are then
    // replayed from a graph of `every` sweeps + the record; long ones go through dsmc_run's own graph
    if (int rc = plain()) return rc;
    if (every <= 2 * DSMC_GRAPH_UNROLL && n_records - done >= 4 && !ctx->timing) {
        if (int rc = build_sweep_graph(ctx, seed, flags, every)) return rc;
        const uint64_t reps = n_records - done;
        if (int rc = replay_sweep_graph(ctx, first_step + 2 * (uint64_t)every * done, reps)) return rc;
        ctx->field_valid[0] = ctx->field_valid[1] = true;
        ctx->spec_valid[0] = ctx->graph_spec_out & 1;
        ctx->spec_valid[1] = (ctx->graph_spec_out & 2) != 0;
        ctx->zline = (ctx->graph_spec_out >> 2) - 1;
        ctx->ensemble_n += reps;
        done += reps;
    }
    while (done < n_records)
        if (int rc = plain()) return rc;
    return DSMC_OK;
}

int dsmc_ensemble_get(dsmc_ctx *ctx, double *mean, double *var, double *se, uint64_t *n_out) {
    ENTER_BOUND(ctx);
    if (!mean || !var || !se) return fail(ctx, DSMC_EINVAL, "null argument");
    if (n_out) *n_out = ctx->ensemble_n;
    if (ctx->ensemble_n == 0) return fail(ctx, DSMC_ESTATE, "empty ensemble");
    std::vector<double> raw(16 * (size_t)ctx->R);
    CU(cudaMemcpyAsync(raw.data(), ctx->stats(), sizeof(double) * raw.size(), cudaMemcpyDeviceToHost, ctx->stream),
       "ensemble D2H");
    CU(cudaStreamSynchronize(ctx->stream), "ensemble sync");
    const double n = (double)ctx->ensemble_n;
    for (size_t i = 0; i < 8 * (size_t)ctx->R; ++i) {
        const double m = raw[2 * i] / n;
        double v = raw[2 * i + 1] / n - m * m;
        if (v < 0.0) v = 0.0;  // rounding of <x^2> - <x>^2 for a constant series
        mean[i] = m;
        var[i] = v;
        se[i] = sqrt(v / n);
    }
    return DSMC_OK;
}

int dsmc_set_debug(dsmc_ctx *ctx, int on) {
    if (!ctx) return DSMC_EINVAL;
    ctx->debug = on ? 1 : 0;
    return DSMC_OK;
}

int dsmc_stream_footprint(dsmc_ctx *ctx, int colour) {
    ENTER_BOUND(ctx);
    if (colour != 0 && colour != 1) return fail(ctx, DSMC_EINVAL, "colour must be 0 or 1");
    if (!ctx->spins_set) return fail(ctx, DSMC_ESTATE, "spins not set");
    if (ctx->R % 4 != 0) return fail(ctx, DSMC_EINVAL, "needs R % 4 == 0 (the shape of the 4-replica Metropolis kernel)");
    const MetropolisArgs a = metropolis_args(ctx, colour, 0, 0, 0, nullptr, nullptr);
    CU(launch_metropolis_stream(a, ctx->stream, &ctx->launches), "stream footprint launch");
    return DSMC_OK;
}

int dsmc_set_timing(dsmc_ctx *ctx, int on) {
    if (!ctx) return DSMC_EINVAL;
    ctx->timing = on ? 1 : 0;
    ctx->ev_recorded = false;
    return DSMC_OK;
}

int dsmc_last_timing(dsmc_ctx *ctx, float *out_ms) {
    ENTER_BOUND(ctx);
    if (!out_ms) return fail(ctx, DSMC_EINVAL, "null argument");
    if (!ctx->ev_recorded) return fail(ctx, DSMC_ESTATE, "no timed half-sweep yet");
    CU(cudaEventSynchronize(ctx->ev[2]), "event sync");
    CU(cudaEventElapsedTime(&out_ms[0], ctx->ev[0], ctx->ev[1]), "elapsed");
    CU(cudaEventElapsedTime(&out_ms[1], ctx->ev[1], ctx->ev[2]), "elapsed");
    CU(cudaEventElapsedTime(&out_ms[2], ctx->ev[0], ctx->ev[2]), "elapsed");
    return DSMC_OK;
}

uint64_t dsmc_launch_count(dsmc_ctx *ctx) { return ctx ? ctx->launches : 0; }

int dsmc_field_kernel_kind(dsmc_ctx *ctx) { return ctx ? field_kind(ctx) : 0; }

int dsmc_field_kernel_supported(dsmc_ctx *ctx, int kind) {
    if (!ctx) return 0;
    if (kind == 0) return 1;
    if (kind == 1) return dsmc_tiled_supported(ctx->L, ctx->R) ? 1 : 0;
    if (kind == 2) return dsmc_fft_supported(ctx->L, ctx->R) ? 1 : 0;
    return 0;
}

int dsmc_select_field_kernel(dsmc_ctx *ctx, int kind) {
    if (!ctx || kind < -1 || kind > 2) return fail(ctx, DSMC_EINVAL, "kind must be -1, 0, 1 or 2");
    if (kind == 1 && !dsmc_tiled_supported(ctx->L, ctx->R))
        return fail(ctx, DSMC_EINVAL, "tiled kernel needs L % 16 == 0, R % 4 == 0 and L <= 1024 (the largest size its fp32 accumulation is tested to meet the field tolerances at)");
    if (kind == 2 && !dsmc_fft_supported(ctx->L, ctx->R)) return fail(ctx, DSMC_EINVAL, "FFT field needs L in {32, 64, 128, 256, 512} and even R");
    ctx->field_kind = kind;
    ctx->field_valid[0] = ctx->field_valid[1] = false;
    return DSMC_OK;
}

int dsmc_destroy(dsmc_ctx *ctx) {
    if (!ctx) return DSMC_EINVAL;
    for (int i = 0; i < 3; ++i)
        if (ctx->ev[i]) cudaEventDestroy(ctx->ev[i]);
    drop_sweep_graph(ctx);
    if (ctx->capture_stream) cudaStreamDestroy(ctx->capture_stream);
    for (int b = 0; b < DSMC_MAX_BRANCHES - 1; ++b) {
        if (ctx->branch_stream[b]) cudaStreamDestroy(ctx->branch_stream[b]);
        if (ctx->ev_join[b]) cudaEventDestroy(ctx->ev_join[b]);
    }
    if (ctx->ev_fork) cudaEventDestroy(ctx->ev_fork);
    delete ctx;
    return DSMC_OK;
}

const char *dsmc_last_error(dsmc_ctx *ctx) { return ctx ? ctx->err.c_str() : "null context"; }

}  // extern "C"
