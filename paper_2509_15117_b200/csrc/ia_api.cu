/*
 * ia_api.cu -- the C-ABI of include/ia.h: argument checks, parameter preparation (a1), launches.
 * No computation of the method happens on the host beyond deriving the ~30 constants of a cell.
 */
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>

#include "ia_kernels.cuh"

namespace {

/* CODATA 2022 conversion factors (values; the oracle carries its own copy) */
const double ME_PER_U = 1822.888486283;
const double KB_EH_PER_K = 3.1668115634564e-6;
const double PI = 3.14159265358979323846;

} // namespace

struct IaKernelInfo {
    int blocks_per_sm = 0, threads_per_block = 0, regs = 0, local_bytes = 0;
};

#define IA_PIPE_MAX 16

struct IaSlot {
    IaHand *queue = nullptr;
    cudaStream_t tail = nullptr;             /* non-blocking stream of the straggler kernel               */
    cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr}; /* start, bulk end, run end, host copies done */
    bool used = false;                       /* ev[2] has been recorded                                    */
    bool host_used = false;                  /* ev[3] has been recorded                                    */
    void *stage = nullptr;                   /* device staging of the host entry points                    */
    size_t stage_bytes = 0;
};

struct ia_ctx {
    int device = 0;
    IaParams P;
    double derived[16];
    /* per-launch scratch, a ring so that launches queued behind one another on a stream do not share:
     * slot = [work counter of the bulk kernel, number handed over, work counter of the cooperative kernel, pad] */
    unsigned long long *counters = nullptr;
    unsigned counter_next = 0;
    size_t queue_cap = 0; /* entries of one hand-over queue: one per lane of a full bulk grid */
    int handoff_lanes = 16;
    int n_sm = 0;
    IaKernelInfo kinfo[2]; /* 0 bulk, 1 cooperative */
    /* Run slots.  A run occupies slot seq % max(depth, 1): its hand-over queue, the stream its straggler
     * kernel runs on (depth > 0; with depth 0 it follows the bulk kernel on the caller's stream), the
     * events around its kernels and, for the host entry points, its device staging. */
    int depth = 0;
    unsigned long long seq = 0;
    IaSlot slot[IA_PIPE_MAX];
    cudaStream_t host_stream = nullptr; /* ia_submit_host / ia_run_host */
    std::string err;
};

#define IA_COUNTER_RING 256 /* slots of 4 x u64 */

static int fail_cuda(ia_ctx *c, const char *what, cudaError_t e) {
    if (c) c->err = std::string(what) + ": " + cudaGetErrorString(e);
    return IA_ECUDA;
}
static int fail_inval(ia_ctx *c, const char *what) {
    if (c) c->err = what;
    return IA_EINVAL;
}

/* allocates what slot k owns (idempotent) */
static cudaError_t slot_init(ia_ctx *c, int k) {
    IaSlot &s = c->slot[k];
    cudaError_t e = cudaSuccess;
    if (!s.queue) e = cudaMalloc(&s.queue, c->queue_cap * sizeof(IaHand));
    /* default priority, like the caller's stream: the next run's bulk kernel (already queued behind this run's
     * on the caller's stream) takes the SMs first and the straggler kernel fills in as its blocks drain */
    if (e == cudaSuccess && !s.tail) e = cudaStreamCreateWithFlags(&s.tail, cudaStreamNonBlocking);
    for (int j = 0; j < 4 && e == cudaSuccess; ++j)
        if (!s.ev[j]) e = cudaEventCreate(&s.ev[j]);
    return e;
}

extern "C" {

const char *ia_strerror(int code) {
    switch (code) {
    case IA_OK: return "ok";
    case IA_EINVAL: return "invalid argument";
    case IA_ENOMEM: return "out of memory";
    case IA_ECUDA: return "CUDA runtime error";
    case IA_EDEVICE: return "no compute-capability-10.x CUDA device (there is no CPU fallback)";
    default: return "unknown error code";
    }
}

const char *ia_last_error(const ia_ctx *ctx) { return ctx ? ctx->err.c_str() : ""; }

int ia_create(ia_ctx **out, const ia_species *sp, const ia_trap *tr, double De_K, double r0_a0, const ia_tol *tol,
              int cuda_device) {
    if (!out) return IA_EINVAL;
    *out = nullptr;
    if (!sp || !tr) return IA_EINVAL;
    ia_tol T;
    std::memset(&T, 0, sizeof(T));
    if (tol) T = *tol;
    if (T.rtol == 0.0) T.rtol = 1e-10;
    if (T.atol == 0.0) T.atol = 1e-12;
    if (T.t_max_rf == 0.0) T.t_max_rf = 1e4;
    if (T.h_max_rf == 0.0) T.h_max_rf = 0.25;
    if (T.r_coll_a0 == 0.0) T.r_coll_a0 = 500.0;
    if (T.max_steps == 0) T.max_steps = 1ull << 31;
    auto pos = [](double v) { return std::isfinite(v) && v > 0.0; };
    if (!pos(sp->m_ion_u) || !pos(sp->m_atom_u) || !pos(sp->alpha_au) || !pos(De_K) || !pos(r0_a0) ||
        !pos(tr->omega_rf_au))
        return IA_EINVAL;
    for (int k = 0; k < 3; ++k)
        if (!std::isfinite(tr->a[k]) || !std::isfinite(tr->q[k])) return IA_EINVAL;
    if (!(T.rtol >= 1e-13 && T.rtol <= 1e-3) || !pos(T.atol) || !pos(T.t_max_rf) ||
        !(T.h_max_rf > 0.0 && T.h_max_rf <= 0.25) || !pos(T.r_coll_a0) || T.max_steps > (1ull << 32) - 1)
        return IA_EINVAL;

    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || cuda_device < 0 || cuda_device >= ndev) return IA_EDEVICE;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, cuda_device) != cudaSuccess) return IA_EDEVICE;
    if (prop.major != 10) return IA_EDEVICE; /* sm_100a only: no fallback path */

    ia_ctx *c = new (std::nothrow) ia_ctx;
    if (!c) return IA_ENOMEM;
    c->device = cuda_device;

    /* a1: parameter preparation (BASELINE.json north_star) */
    IaParams &P = c->P;
    std::memset(&P, 0, sizeof(P));
    P.m_i = sp->m_ion_u * ME_PER_U;
    P.m_a = sp->m_atom_u * ME_PER_U;
    P.inv_m_a = 1.0 / P.m_a;
    P.neg_inv_m_i = -1.0 / P.m_i;
    P.C4 = sp->alpha_au / 2.0;
    P.De = De_K * KB_EH_PER_K;
    P.C8 = P.C4 * P.C4 / (4.0 * P.De);
    P.r_e = std::pow(2.0 * P.C8 / P.C4, 0.25);
    P.c8x8 = 8.0 * P.C8;
    P.neg_c4x4 = -4.0 * P.C4;
    P.omega = tr->omega_rf_au;
    P.T_rf = 2.0 * PI / P.omega;
    for (int k = 0; k < 3; ++k) {
        P.ka[k] = -tr->a[k] * (P.omega * P.omega / 4.0);
        P.kq[k] = -2.0 * tr->q[k] * (P.omega * P.omega / 4.0);
    }
    P.rtol = T.rtol;
    P.atol = T.atol;
    P.thr = T.atol / T.rtol;
    P.h_max = T.h_max_rf * P.T_rf;
    P.h_min = std::ldexp(P.T_rf, -40);
    P.t_max_rf = T.t_max_rf;
    P.t_max = T.t_max_rf * P.T_rf;
    P.h0_scale = 0.8 * std::pow(T.rtol, 0.2);
    P.r0 = r0_a0;
    P.r0sq = r0_a0 * r0_a0;
    P.r_coll = T.r_coll_a0;
    P.rcsq = T.r_coll_a0 * T.r_coll_a0;
    P.loc_tol = 1e-13 * P.r0sq;
    P.max_steps = T.max_steps;
    const double d[16] = {P.m_i, P.m_a, P.C4, P.C8, P.De, P.r_e, P.omega, P.T_rf,
                          P.thr, P.h_max, P.h_min, P.t_max, P.r0, P.r_coll, P.rtol, P.atol};
    std::memcpy(c->derived, d, sizeof(d));

    c->n_sm = prop.multiProcessorCount;
    cudaError_t e = cudaSetDevice(cuda_device);
    if (e == cudaSuccess) e = cudaMalloc(&c->counters, IA_COUNTER_RING * 4 * sizeof(unsigned long long));
    for (int k = 0; k < 2 && e == cudaSuccess; ++k)
        e = ia_persistent_info(k == 0 ? 1 : 3, &c->kinfo[k].blocks_per_sm, &c->kinfo[k].threads_per_block,
                               &c->kinfo[k].regs, &c->kinfo[k].local_bytes);
    if (e == cudaSuccess) {
        c->queue_cap = (size_t)c->n_sm * c->kinfo[0].blocks_per_sm * c->kinfo[0].threads_per_block;
        e = slot_init(c, 0);
    }
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&c->host_stream, cudaStreamNonBlocking);
    if (e != cudaSuccess) {
        const int rc = e == cudaErrorMemoryAllocation ? IA_ENOMEM : IA_ECUDA;
        ia_destroy(c);
        return rc;
    }
    *out = c;
    return IA_OK;
}

int ia_destroy(ia_ctx *ctx) {
    if (!ctx) return IA_EINVAL;
    cudaSetDevice(ctx->device);
    /* runs still in flight finish first: their kernels use the ctx's scratch */
    if (ctx->host_stream) cudaStreamSynchronize(ctx->host_stream);
    for (int k = 0; k < IA_PIPE_MAX; ++k) {
        IaSlot &s = ctx->slot[k];
        if (s.used) cudaEventSynchronize(s.ev[2]);
        if (s.host_used) cudaEventSynchronize(s.ev[3]);
        if (s.tail) cudaStreamDestroy(s.tail);
        if (s.queue) cudaFree(s.queue);
        if (s.stage) cudaFree(s.stage);
        for (int j = 0; j < 4; ++j)
            if (s.ev[j]) cudaEventDestroy(s.ev[j]);
    }
    if (ctx->host_stream) cudaStreamDestroy(ctx->host_stream);
    if (ctx->counters) cudaFree(ctx->counters);
    delete ctx;
    return IA_OK;
}

int ia_get_derived(const ia_ctx *ctx, double *out16) {
    if (!ctx || !out16) return IA_EINVAL;
    std::memcpy(out16, ctx->derived, sizeof(ctx->derived));
    return IA_OK;
}

int ia_get_kernel_info(const ia_ctx *ctx, int kernel, int *warps_per_sm, int *n_sm, int *regs_per_thread,
                       int *local_bytes_per_thread) {
    if (!ctx || kernel < 0 || kernel > 1) return IA_EINVAL;
    const IaKernelInfo &k = ctx->kinfo[kernel];
    if (warps_per_sm) *warps_per_sm = k.blocks_per_sm * k.threads_per_block / 32;
    if (n_sm) *n_sm = ctx->n_sm;
    if (regs_per_thread) *regs_per_thread = k.regs;
    if (local_bytes_per_thread) *local_bytes_per_thread = k.local_bytes;
    return IA_OK;
}

int ia_set_handoff(ia_ctx *ctx, int lanes) {
    if (!ctx || lanes < 0 || lanes > 32) return IA_EINVAL;
    ctx->handoff_lanes = lanes;
    return IA_OK;
}

int ia_set_pipeline(ia_ctx *ctx, int depth) {
    if (!ctx) return IA_EINVAL;
    if (depth < 0 || depth > IA_PIPE_MAX) return fail_inval(ctx, "ia_set_pipeline: depth must be in [0, 16]");
    cudaError_t e = cudaSetDevice(ctx->device);
    /* runs in flight keep their slots: let them finish before the slot numbering changes */
    for (int k = 0; k < IA_PIPE_MAX && e == cudaSuccess; ++k)
        if (ctx->slot[k].used) e = cudaEventSynchronize(ctx->slot[k].ev[2]);
    for (int k = 0; k < depth && e == cudaSuccess; ++k) e = slot_init(ctx, k);
    if (e == cudaErrorMemoryAllocation) {
        ctx->err = "ia_set_pipeline: hand-over queue allocation failed";
        return IA_ENOMEM;
    }
    if (e != cudaSuccess) return fail_cuda(ctx, "ia_set_pipeline", e);
    ctx->depth = depth;
    return IA_OK;
}

int ia_join(ia_ctx *ctx, void *cuda_stream) {
    if (!ctx) return IA_EINVAL;
    cudaError_t e = cudaSetDevice(ctx->device);
    for (int k = 0; k < IA_PIPE_MAX && e == cudaSuccess; ++k)
        if (ctx->slot[k].used) e = cudaStreamWaitEvent((cudaStream_t)cuda_stream, ctx->slot[k].ev[2], 0);
    if (e != cudaSuccess) return fail_cuda(ctx, "ia_join", e);
    return IA_OK;
}

int ia_get_timing(ia_ctx *ctx, int runs_back, double *bulk_ms, double *coop_ms) {
    if (!ctx || !bulk_ms || !coop_ms) return IA_EINVAL;
    const int ring = ctx->depth > 0 ? ctx->depth : 1;
    if (runs_back < 0 || runs_back >= ring || (unsigned long long)runs_back >= ctx->seq)
        return fail_inval(ctx, "ia_get_timing: that run is no longer (or not yet) on record");
    IaSlot &s = ctx->slot[(ctx->seq - 1 - (unsigned long long)runs_back) % (unsigned long long)ring];
    cudaError_t e = cudaSetDevice(ctx->device);
    if (e == cudaSuccess) e = cudaEventSynchronize(s.ev[2]);
    float a = 0.f, b = 0.f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&a, s.ev[0], s.ev[1]);
    if (e == cudaSuccess) e = cudaEventElapsedTime(&b, s.ev[1], s.ev[2]);
    if (e != cudaSuccess) return fail_cuda(ctx, "ia_get_timing", e);
    *bulk_ms = a;
    *coop_ms = b;
    return IA_OK;
}

int ia_get_last_timing(ia_ctx *ctx, double *bulk_ms, double *coop_ms) {
    return ia_get_timing(ctx, 0, bulk_ms, coop_ms);
}

} // extern "C"

/* validates a launch descriptor and translates it for the device */
static int make_gen(ia_ctx *ctx, const ia_launch *L, IaGen *G, unsigned long long *warn) {
    if (!L) return fail_inval(ctx, "launch is NULL");
    std::memset(G, 0, sizeof(*G));
    *warn = 0;
    if (L->mode != IA_IC_EXPLICIT && L->mode != IA_IC_GRID && L->mode != IA_IC_PHILOX)
        return fail_inval(ctx, "launch.mode is not an ia_ic_mode");
    if (L->path != IA_PATH_AUTO && L->path != IA_PATH_BULK_ONLY && L->path != IA_PATH_COOP_ONLY)
        return fail_inval(ctx, "launch.path is not an ia_path");
    G->mode = L->mode;
    G->n = L->n;
    G->first_index = L->first_index;
    if (L->mode == IA_IC_EXPLICIT) {
        if (L->n > 0 && (!L->y0 || !L->phase)) return fail_inval(ctx, "EXPLICIT launch needs y0 and phase");
        G->y0 = L->y0;
        G->phase = L->phase;
        return IA_OK;
    }
    if (L->domain != 0 && L->domain != 1) return fail_inval(ctx, "launch.domain must be 0 or 1");
    if (L->phase_mode != 0 && L->phase_mode != 1) return fail_inval(ctx, "launch.phase_mode must be 0 or 1");
    if (!std::isfinite(L->phase0)) return fail_inval(ctx, "launch.phase0 is not finite");
    if (!(std::isfinite(L->E_min_uK) && L->E_min_uK > 0.0 && std::isfinite(L->E_max_uK) && L->E_max_uK >= L->E_min_uK))
        return fail_inval(ctx, "need 0 < E_min_uK <= E_max_uK");
    G->domain = L->domain;
    G->phase_mode = L->phase_mode;
    G->phase0 = L->phase0;
    G->seed = L->seed;
    G->cell = L->cell;
    G->theta_span_pi = L->domain == 0 ? 0.5 : 1.0;
    G->phi_span_pi = L->domain == 0 ? 0.5 : 2.0;
    if (L->mode == IA_IC_GRID) {
        if (L->n_theta == 0 || L->n_phi == 0) return fail_inval(ctx, "GRID launch needs n_theta, n_phi > 0");
        if (L->first_index + L->n > (uint64_t)L->n_theta * L->n_phi)
            return fail_inval(ctx, "GRID launch: first_index + n exceeds n_theta * n_phi");
        G->n_theta = L->n_theta;
        G->n_phi = L->n_phi;
    }
    G->E_min_uK = L->E_min_uK;
    if (L->E_max_uK != L->E_min_uK) {
        if (L->mode != IA_IC_PHILOX) return fail_inval(ctx, "an energy range needs the PHILOX generator");
        G->log_E_ratio = std::log(L->E_max_uK / L->E_min_uK);
    } else {
        G->log_E_ratio = 0.0;
        G->E_fixed_au = L->E_min_uK * 1e-6 * KB_EH_PER_K;
        G->v0_fixed = std::sqrt(2.0 * G->E_fixed_au / ctx->P.m_a);
    }
    /* r0 is chosen such that 10 |V(r0)| < E */
    const IaParams &P = ctx->P;
    const double V0 = P.C8 / std::pow(P.r0, 8) - P.C4 / std::pow(P.r0, 4);
    if (10.0 * std::fabs(V0) >= L->E_min_uK * 1e-6 * KB_EH_PER_K) {
        *warn = 1;
        ctx->err = "warning: 10|V(r0)| >= E_min, the start is not in the asymptotic region (PAPER.md:28)";
    }
    return IA_OK;
}

/* blocks of persistent kernel k (0 bulk: 32 trajectories per warp; 1 cooperative: 10) for n trajectories */
static int grid_for(const ia_ctx *ctx, int k, unsigned long long n) {
    const unsigned long long full = (unsigned long long)ctx->n_sm * ctx->kinfo[k].blocks_per_sm;
    const unsigned long long per = k == 0 ? 32ull : 10ull;
    const unsigned long long need = (n + per - 1) / per;
    return (int)(need < full ? need : full);
}

/* ia_run proper; *slot_out receives the run slot (only when something was launched, else -1) */
static int run_impl(ia_ctx *ctx, const ia_launch *launch, const ia_outputs *outputs, cudaStream_t st, int *slot_out) {
    *slot_out = -1;
    ctx->err.clear();
    if (!outputs) return fail_inval(ctx, "outputs is NULL");
    IaGen G;
    unsigned long long warn;
    int rc = make_gen(ctx, launch, &G, &warn);
    if (rc != IA_OK) return rc;
    if (G.n == 0) return IA_OK;
    cudaError_t e = cudaSetDevice(ctx->device);
    if (e != cudaSuccess) return fail_cuda(ctx, "cudaSetDevice", e);
    const int k = ctx->depth > 0 ? (int)(ctx->seq % (unsigned long long)ctx->depth) : 0;
    IaSlot &sl = ctx->slot[k];
    /* the slot's queue and events are free again once the run that used them last has ended; with
     * depth > 0 that run's straggler kernel is on another stream, so the caller's stream waits for it */
    if (ctx->depth > 0 && sl.used) {
        e = cudaStreamWaitEvent(st, sl.ev[2], 0);
        if (e != cudaSuccess) return fail_cuda(ctx, "cudaStreamWaitEvent(slot)", e);
    }
    unsigned long long *scratch = ctx->counters + 4 * (size_t)(ctx->counter_next++ % IA_COUNTER_RING);
    e = cudaMemsetAsync(scratch, 0, 4 * sizeof(unsigned long long), st);
    if (e != cudaSuccess) return fail_cuda(ctx, "cudaMemsetAsync(counter)", e);
    IaOut O;
    O.records = outputs->records;
    O.summary = outputs->summary;
    O.ic_dump = outputs->ic_dump;
    const bool coop_only = launch->path == IA_PATH_COOP_ONLY;
    const bool handoff = launch->path == IA_PATH_AUTO && ctx->handoff_lanes > 0;
    IaSched S;
    std::memset(&S, 0, sizeof(S));
    S.counter = scratch;
    S.warn = warn;
    cudaStream_t end_stream = st;
    e = cudaEventRecord(sl.ev[0], st);
    if (e != cudaSuccess) return fail_cuda(ctx, "cudaEventRecord", e);
    if (coop_only) {
        e = ia_launch_persistent(3, ctx->P, G, O, S, grid_for(ctx, 1, G.n), st);
        if (e == cudaSuccess) e = cudaEventRecord(sl.ev[1], st);
    } else {
        if (handoff) {
            S.q_out = sl.queue;
            S.n_out = scratch + 1;
            S.handoff_lanes = ctx->handoff_lanes;
        }
        const int blocks = grid_for(ctx, 0, G.n);
        e = ia_launch_persistent(1, ctx->P, G, O, S, blocks, st);
        if (e == cudaSuccess) e = cudaEventRecord(sl.ev[1], st);
        if (e == cudaSuccess && handoff) {
            /* the straggler kernel resumes what the bulk kernel queued, with a grid that can hold every lane
             * the bulk grid could have handed over.  depth 0: behind the bulk kernel on the caller's stream.
             * depth > 0: on the slot's own stream, so that the caller's stream is free for the next run's bulk
             * kernel while this run's longest trajectories finish. */
            IaSched S5;
            std::memset(&S5, 0, sizeof(S5));
            S5.counter = scratch + 2;
            S5.q_in = sl.queue;
            S5.n_in = scratch + 1;
            if (ctx->depth > 0) {
                end_stream = sl.tail;
                e = cudaStreamWaitEvent(end_stream, sl.ev[1], 0);
            }
            const unsigned long long most = (unsigned long long)blocks * (unsigned long long)ctx->handoff_lanes;
            if (e == cudaSuccess) e = ia_launch_persistent(3, ctx->P, G, O, S5, grid_for(ctx, 1, most), end_stream);
        }
    }
    if (e == cudaSuccess) e = cudaEventRecord(sl.ev[2], end_stream);
    if (e != cudaSuccess) return fail_cuda(ctx, "persistent kernel launch", e);
    sl.used = true;
    ctx->seq++;
    *slot_out = k;
    return IA_OK;
}

/* enqueues one host-buffer run: H2D, kernels, D2H; nothing here waits for the device */
static int submit_host_impl(ia_ctx *ctx, const ia_launch *launch, const ia_outputs *host_out) {
    ctx->err.clear();
    if (!launch || !host_out) return fail_inval(ctx, "launch or outputs is NULL");
    const uint64_t n = launch->n;
    if (n == 0) return IA_OK;
    if (launch->mode == IA_IC_EXPLICIT && (!launch->y0 || !launch->phase))
        return fail_inval(ctx, "EXPLICIT launch needs y0 and phase");
    cudaError_t e = cudaSetDevice(ctx->device);
    if (e != cudaSuccess) return fail_cuda(ctx, "cudaSetDevice", e);
    const int k = ctx->depth > 0 ? (int)(ctx->seq % (unsigned long long)ctx->depth) : 0;
    IaSlot &sl = ctx->slot[k];
    cudaStream_t st = ctx->host_stream;
    /* staging layout: [summary 512][records n*64][ic_dump n*14*8][y0 n*12*8][phase n*8] */
    const size_t off_rec = sizeof(ia_summary);
    const size_t off_ic = off_rec + (host_out->records ? n * sizeof(ia_record) : 0);
    const size_t off_y0 = off_ic + (host_out->ic_dump ? n * 14 * sizeof(double) : 0);
    const size_t off_ph = off_y0 + (launch->mode == IA_IC_EXPLICIT ? n * 12 * sizeof(double) : 0);
    const size_t total = off_ph + (launch->mode == IA_IC_EXPLICIT ? n * sizeof(double) : 0);
    if (total > sl.stage_bytes) {
        if (sl.host_used) cudaEventSynchronize(sl.ev[3]); /* the slot's previous run still copies from it */
        if (sl.stage) cudaFree(sl.stage);
        sl.stage = nullptr;
        sl.stage_bytes = 0;
        e = cudaMalloc(&sl.stage, total);
        if (e != cudaSuccess) {
            ctx->err = "device staging allocation failed";
            return IA_ENOMEM;
        }
        sl.stage_bytes = total;
    }
    if (sl.host_used) { /* the staging is free again once the slot's previous copies back are done */
        e = cudaStreamWaitEvent(st, sl.ev[3], 0);
        if (e != cudaSuccess) return fail_cuda(ctx, "cudaStreamWaitEvent(staging)", e);
    }
    char *base = (char *)sl.stage;
    ia_launch L = *launch;
    ia_outputs O;
    O.summary = (ia_summary *)base;
    O.records = host_out->records ? (ia_record *)(base + off_rec) : nullptr;
    O.ic_dump = host_out->ic_dump ? (double *)(base + off_ic) : nullptr;
    e = cudaMemsetAsync(base, 0, sizeof(ia_summary), st);
    if (e != cudaSuccess) return fail_cuda(ctx, "cudaMemsetAsync(summary)", e);
    if (launch->mode == IA_IC_EXPLICIT) {
        e = cudaMemcpyAsync(base + off_y0, launch->y0, n * 12 * sizeof(double), cudaMemcpyHostToDevice, st);
        if (e == cudaSuccess)
            e = cudaMemcpyAsync(base + off_ph, launch->phase, n * sizeof(double), cudaMemcpyHostToDevice, st);
        if (e != cudaSuccess) return fail_cuda(ctx, "H2D copy of initial conditions", e);
        L.y0 = (const double *)(base + off_y0);
        L.phase = (const double *)(base + off_ph);
    }
    int used = -1;
    int rc = run_impl(ctx, &L, &O, st, &used);
    if (rc != IA_OK) return rc;
    const std::string warn_text = ctx->err;
    /* the copies back follow the run's last kernel: on the slot's straggler stream when there is one */
    cudaStream_t back = st;
    if (ctx->depth > 0 && launch->path == IA_PATH_AUTO && ctx->handoff_lanes > 0) back = sl.tail;
    if (host_out->records)
        e = cudaMemcpyAsync(host_out->records, O.records, n * sizeof(ia_record), cudaMemcpyDeviceToHost, back);
    if (e == cudaSuccess && host_out->ic_dump)
        e = cudaMemcpyAsync(host_out->ic_dump, O.ic_dump, n * 14 * sizeof(double), cudaMemcpyDeviceToHost, back);
    if (e == cudaSuccess && host_out->summary)
        e = cudaMemcpyAsync(host_out->summary, O.summary, sizeof(ia_summary), cudaMemcpyDeviceToHost, back);
    if (e == cudaSuccess) e = cudaEventRecord(sl.ev[3], back);
    if (e != cudaSuccess) return fail_cuda(ctx, "D2H copy", e);
    sl.host_used = true;
    ctx->err = warn_text;
    return IA_OK;
}

extern "C" {

int ia_run(ia_ctx *ctx, const ia_launch *launch, const ia_outputs *outputs, void *cuda_stream) {
    if (!ctx) return IA_EINVAL;
    int slot;
    return run_impl(ctx, launch, outputs, (cudaStream_t)cuda_stream, &slot);
}

int ia_submit_host(ia_ctx *ctx, const ia_launch *launch, const ia_outputs *host_outputs) {
    if (!ctx) return IA_EINVAL;
    return submit_host_impl(ctx, launch, host_outputs);
}

int ia_wait(ia_ctx *ctx) {
    if (!ctx) return IA_EINVAL;
    cudaError_t e = cudaSetDevice(ctx->device);
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->host_stream);
    for (int k = 0; k < IA_PIPE_MAX && e == cudaSuccess; ++k) {
        if (ctx->slot[k].used) e = cudaEventSynchronize(ctx->slot[k].ev[2]);
        if (e == cudaSuccess && ctx->slot[k].host_used) e = cudaEventSynchronize(ctx->slot[k].ev[3]);
    }
    if (e != cudaSuccess) return fail_cuda(ctx, "ia_wait", e);
    return IA_OK;
}

int ia_run_host(ia_ctx *ctx, const ia_launch *launch, const ia_outputs *host_outputs) {
    if (!ctx) return IA_EINVAL;
    int rc = submit_host_impl(ctx, launch, host_outputs);
    if (rc != IA_OK) return rc;
    const std::string warn_text = ctx->err;
    rc = ia_wait(ctx);
    if (rc == IA_OK) ctx->err = warn_text;
    return rc;
}

int ia_generate(ia_ctx *ctx, const ia_launch *launch, double *ic_dump, void *cuda_stream) {
    if (!ctx) return IA_EINVAL;
    ctx->err.clear();
    IaGen G;
    unsigned long long warn;
    int rc = make_gen(ctx, launch, &G, &warn);
    if (rc != IA_OK) return rc;
    if (G.n == 0) return IA_OK;
    if (!ic_dump) return fail_inval(ctx, "ic_dump is NULL");
    cudaError_t e = cudaSetDevice(ctx->device);
    if (e == cudaSuccess) e = ia_launch_generate(ctx->P, G, ic_dump, (cudaStream_t)cuda_stream);
    if (e != cudaSuccess) return fail_cuda(ctx, "generator launch", e);
    return IA_OK;
}

static bool bad_variant(int v) { return v != IA_ARITH_NOFMA && v != IA_ARITH_FMA && v != IA_ARITH_FMA_COOP; }

int ia_step_map(ia_ctx *ctx, uint64_t n, const double *t_frac, const double *phase, const double *y, const double *h,
                double *ynew, double *err, int variant, void *cuda_stream) {
    if (!ctx) return IA_EINVAL;
    ctx->err.clear();
    if (n == 0) return IA_OK;
    if (!t_frac || !phase || !y || !h || !ynew) return fail_inval(ctx, "ia_step_map: NULL array");
    if (bad_variant(variant)) return fail_inval(ctx, "ia_step_map: variant is not an ia_arith");
    cudaError_t e = cudaSetDevice(ctx->device);
    if (e == cudaSuccess)
        e = ia_launch_step_map(variant, ctx->P, n, t_frac, phase, y, h, ynew, err, (cudaStream_t)cuda_stream);
    if (e != cudaSuccess) return fail_cuda(ctx, "step-map launch", e);
    return IA_OK;
}

int ia_trace(ia_ctx *ctx, const double *y0_host, double phase, double h, uint32_t nsteps, double *states, int variant,
             void *cuda_stream) {
    if (!ctx) return IA_EINVAL;
    ctx->err.clear();
    if (!y0_host || !states) return fail_inval(ctx, "ia_trace: NULL array");
    if (!std::isfinite(phase) || !std::isfinite(h)) return fail_inval(ctx, "ia_trace: non-finite phase or h");
    if (bad_variant(variant)) return fail_inval(ctx, "ia_trace: variant is not an ia_arith");
    IaY12 y0;
    std::memcpy(y0.y, y0_host, sizeof(y0.y));
    cudaError_t e = cudaSetDevice(ctx->device);
    if (e == cudaSuccess) e = ia_launch_trace(variant, ctx->P, y0, phase, h, nsteps, states, (cudaStream_t)cuda_stream);
    if (e != cudaSuccess) return fail_cuda(ctx, "trace launch", e);
    return IA_OK;
}

int ia_fp64_peak(int cuda_device, double target_ms, double *tflops, double *elapsed_ms) {
    if (!tflops || !elapsed_ms) return IA_EINVAL;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || cuda_device < 0 || cuda_device >= ndev) return IA_EDEVICE;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, cuda_device) != cudaSuccess || prop.major != 10) return IA_EDEVICE;
    return ia_run_fp64_peak(cuda_device, target_ms, tflops, elapsed_ms) == cudaSuccess ? IA_OK : IA_ECUDA;
}

} // extern "C"
