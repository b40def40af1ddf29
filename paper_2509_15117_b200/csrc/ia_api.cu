/*
 * ia_api.cu -- the C-ABI of include/ia.h: argument checks, parameter preparation (a1), launches.
 * No computation of the method happens on the host beyond deriving the ~30 constants of a cell.
 */
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

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

#define IA_PIPE_MAX 64      /* runs between two joins (ia_set_pipeline) */
#define IA_RUN_RING 256     /* runs whose kernel events are kept for ia_get_timing */
#define IA_FLUSH_RING 8     /* straggler chains whose events are kept */
#define IA_COUNTER_RING 256 /* work counters of the runs that need no queue */
#define IA_NSTAGE 3         /* device staging buffers of the host entry points */

/* The straggler chain.  What decides the latency of a step is how many warps share an SM
 * sub-partition (measured, profiles/r02_summary.md section 4: bulk layout 2.61 / 1.84 / 1.14 us per step at
 * 3 / 2 / 1 warps, cooperative layout 1.01 us at 1 warp with a third of the trajectories per warp).  The chain
 * therefore moves what is left into ever fewer warps, by COUNT: stage A = the bulk kernel over a full grid until
 * at most 32 x 4 x #SM trajectories run; stage B = the bulk kernel with one warp per sub-partition until at most
 * 10 x 4 x #SM run; stage C = the cooperative kernel, one warp per sub-partition, `levels` launches (the re-packing
 * levels of ia_set_chain: level j passes on what still runs level_budget << j iterations after its queue ran dry;
 * the last keeps everything; one level by default). */
#define IA_BULK_BUDGET 4096u /* the bulk kernel: a warp hands over at the latest this long after the counter ran dry */

/* Device words of the open pipeline cycle (all zeroed when a cycle starts):
 *   cnt[k], k = 0..IA_PIPE_MAX: trajectories handed INTO run k of the cycle (cnt[0] stays 0; run k counts what it
 *                               hands on in cnt[k+1]); cnt[n_open] is what the straggler chain starts from
 *   wc[k]:                      work counter of run k's bulk kernel
 *   chain[3j .. 3j+2]:          stage j of the chain: trajectories queued for it (stage 0 uses cnt[n_open]),
 *                               its work counter, the trajectories it has finished                        */
#define IA_W_CNT 0
#define IA_W_WC (IA_W_CNT + IA_PIPE_MAX + 1)
#define IA_W_CHAIN (IA_W_WC + IA_PIPE_MAX)
#define IA_CHAIN_STAGES (2 + IA_STRAGGLER_LEVELS)
#define IA_W_TOTAL (IA_W_CHAIN + 3 * IA_CHAIN_STAGES + 3)
#define IA_GUARD 4096       /* bytes of guard zone before and after every ctx-owned device buffer (ia_debug_check) */
#define IA_GUARD_BYTE 0xA5

struct IaRunEvents {
    cudaEvent_t ev[2] = {nullptr, nullptr}; /* around the bulk kernel */
    long long flush = -1;                   /* id of the straggler chain that finishes the run; -1: none needed */
};

struct IaFlush {
    cudaEvent_t ev[2] = {nullptr, nullptr}; /* around the chain */
    long long id = -1;
};

struct IaGuarded {
    char *base = nullptr; /* what cudaMalloc returned */
    size_t bytes = 0;     /* payload size */
};

struct IaStage {
    char *buf = nullptr;
    size_t bytes = 0;
    cudaEvent_t ev_free = nullptr; /* after the copies back of the run that used it last */
    bool used = false;
};

/* A host run whose summary (and late records) ia_wait still has to bring back. */
struct IaPending {
    ia_summary *host_summary = nullptr;
    ia_summary *dev_summary = nullptr;
};

struct ia_ctx {
    int device = 0;
    IaParams P;
    double derived[16];
    unsigned long long *counters = nullptr; /* ring of work counters for runs of one kernel (no queue) */
    unsigned counter_next = 0;
    size_t queue_cap = 0; /* hand-over entries one bulk kernel can produce: one per lane of a full grid */
    int handoff_lanes = 16;
    double w_harm = 0.0;                   /* |q_x| Omega / 2^(3/2): the ion's trap frequency in thermal runs */
    int levels = 1;                        /* launches of the cooperative kernel at the end of the chain (ia_set_chain) */
    unsigned level_budget = 8192u;         /* iterations of its first level after the queue ran dry */
    int n_sm = 0;
    IaKernelInfo kinfo[2]; /* 0 bulk, 1 cooperative */
    /* the pipeline (ia_set_pipeline): bulk kernels hand what they leave unfinished to one another through q[0], q[1] */
    int depth = 0;
    IaHand *q[2] = {nullptr, nullptr};
    unsigned long long *words = nullptr; /* IA_W_TOTAL words, see above */
    int n_open = 0;                      /* bulk kernels enqueued since the last chain */
    long long flush_next = 0;            /* id of the chain that will finish them */
    IaFlush flush[IA_FLUSH_RING];
    cudaEvent_t ev_last = nullptr;       /* after the latest kernel of this ctx: the next run waits for it, */
    bool ev_last_valid = false;          /* whatever stream it comes in on (the scratch above is shared)    */
    unsigned long long seq = 0;          /* runs launched so far */
    IaRunEvents run[IA_RUN_RING];
    /* host entry points */
    cudaStream_t host_stream = nullptr, copy_stream = nullptr;
    IaStage stage[IA_NSTAGE];
    unsigned stage_next = 0;
    ia_summary *sum_stage = nullptr;     /* device: one summary per pending host run */
    IaPending pending[IA_PIPE_MAX];
    int n_pending = 0;
    IaLate *late_dev = nullptr, *late_host = nullptr; /* records of late finishers of pipelined host runs */
    unsigned long long *n_late = nullptr;             /* device counter; n_late[1] = the fault word of IaSched */
    unsigned long long late_cap = 0;
    std::vector<IaGuarded> owned; /* every device buffer of the ctx, with its guard zones */
    std::string err;
};

/* device buffer with IA_GUARD bytes of a known pattern on either side (ia_debug_check verifies them) */
static cudaError_t guarded_malloc(ia_ctx *c, void **out, size_t bytes) {
    char *base = nullptr;
    const size_t pay = (bytes + 255) & ~(size_t)255;
    cudaError_t e = cudaMalloc(&base, pay + 2 * IA_GUARD);
    if (e != cudaSuccess) return e;
    e = cudaMemset(base, IA_GUARD_BYTE, IA_GUARD);
    if (e == cudaSuccess) e = cudaMemset(base + IA_GUARD + pay, IA_GUARD_BYTE, IA_GUARD);
    if (e != cudaSuccess) {
        cudaFree(base);
        return e;
    }
    IaGuarded g;
    g.base = base;
    g.bytes = pay;
    c->owned.push_back(g);
    *out = base + IA_GUARD;
    return cudaSuccess;
}
static void guarded_free(ia_ctx *c, void *p) {
    if (!p) return;
    for (size_t k = 0; k < c->owned.size(); ++k)
        if (c->owned[k].base + IA_GUARD == (char *)p) {
            cudaFree(c->owned[k].base);
            c->owned.erase(c->owned.begin() + k);
            return;
        }
}

static int fail_cuda(ia_ctx *c, const char *what, cudaError_t e) {
    if (c) c->err = std::string(what) + ": " + cudaGetErrorString(e);
    return IA_ECUDA;
}
static int fail_inval(ia_ctx *c, const char *what) {
    if (c) c->err = what;
    return IA_EINVAL;
}

/* a1: parameter preparation (BASELINE.json north_star) -- range checks, defaults of the tolerances and
 * the derived constants of one cell (host arithmetic only: no CUDA call).  *w_harm = |q_x| Omega / 2^(3/2), the ion's trap
 * frequency in thermal runs.  Shared by ia_create and ia_run_static. */
static int prepare_cell(IaParams *Pout, double derived[16], double *w_harm, const ia_species *sp, const ia_trap *tr,
                        double De_K, double r0_a0, const ia_tol *tol) {
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
    IaParams &P = *Pout;
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
    P.c8_a = P.c8x8 / P.m_a;
    P.c4_a = P.neg_c4x4 / P.m_a;
    P.c8_i = -P.c8x8 / P.m_i;
    P.c4_i = -P.neg_c4x4 / P.m_i;
    P.omega = tr->omega_rf_au;
    P.T_rf = 2.0 * PI / P.omega;
    for (int k = 0; k < 3; ++k) {
        P.ka[k] = -tr->a[k] * (P.omega * P.omega / 4.0);
        P.kq[k] = -2.0 * tr->q[k] * (P.omega * P.omega / 4.0);
    }
    *w_harm = std::fabs(tr->q[0]) * P.omega / std::pow(2.0, 1.5);
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
    P.n_near = T.t_max_rf > 2.0 ? (unsigned)std::floor(std::fmin(T.t_max_rf - 2.0, 4294967295.0)) : 0u;
    const double d[16] = {P.m_i, P.m_a, P.C4, P.C8, P.De, P.r_e, P.omega, P.T_rf,
                          P.thr, P.h_max, P.h_min, P.t_max, P.r0, P.r_coll, P.rtol, P.atol};
    std::memcpy(derived, d, sizeof(d));
    return IA_OK;
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
    /* a1, and with it the argument checks: they answer before any device is looked at */
    IaParams P0;
    double derived[16], w_harm = 0.0;
    if (prepare_cell(&P0, derived, &w_harm, sp, tr, De_K, r0_a0, tol) != IA_OK) return IA_EINVAL;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || cuda_device < 0 || cuda_device >= ndev) return IA_EDEVICE;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, cuda_device) != cudaSuccess) return IA_EDEVICE;
    if (prop.major != 10) return IA_EDEVICE; /* sm_100a only: no fallback path */

    ia_ctx *c = new (std::nothrow) ia_ctx;
    if (!c) return IA_ENOMEM;
    c->device = cuda_device;
    c->P = P0;
    c->w_harm = w_harm;
    std::memcpy(c->derived, derived, sizeof(derived));
    c->n_sm = prop.multiProcessorCount;
    cudaError_t e = cudaSetDevice(cuda_device);
    if (e == cudaSuccess) e = guarded_malloc(c, (void **)&c->counters, IA_COUNTER_RING * 4 * sizeof(unsigned long long));
    for (int k = 0; k < 2 && e == cudaSuccess; ++k)
        e = ia_persistent_info(k == 0 ? 1 : 3, &c->kinfo[k].blocks_per_sm, &c->kinfo[k].threads_per_block,
                               &c->kinfo[k].regs, &c->kinfo[k].local_bytes);
    if (e == cudaSuccess) {
        /* one entry per lane of a full bulk grid (a full cooperative grid holds fewer) */
        c->queue_cap = (size_t)c->n_sm * c->kinfo[0].blocks_per_sm * c->kinfo[0].threads_per_block;
        for (int j = 0; j < 2 && e == cudaSuccess; ++j) e = guarded_malloc(c, (void **)&c->q[j], c->queue_cap * sizeof(IaHand));
    }
    if (e == cudaSuccess) e = guarded_malloc(c, (void **)&c->words, IA_W_TOTAL * sizeof(unsigned long long));
    if (e == cudaSuccess) e = guarded_malloc(c, (void **)&c->n_late, 2 * sizeof(unsigned long long));
    if (e == cudaSuccess) e = cudaMemset(c->n_late, 0, 2 * sizeof(unsigned long long));
    if (e == cudaSuccess) e = guarded_malloc(c, (void **)&c->sum_stage, IA_PIPE_MAX * sizeof(ia_summary));
    for (int k = 0; k < IA_RUN_RING && e == cudaSuccess; ++k)
        for (int j = 0; j < 2 && e == cudaSuccess; ++j) e = cudaEventCreate(&c->run[k].ev[j]);
    for (int k = 0; k < IA_FLUSH_RING && e == cudaSuccess; ++k)
        for (int j = 0; j < 2 && e == cudaSuccess; ++j) e = cudaEventCreate(&c->flush[k].ev[j]);
    for (int k = 0; k < IA_NSTAGE && e == cudaSuccess; ++k)
        e = cudaEventCreateWithFlags(&c->stage[k].ev_free, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->ev_last, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&c->host_stream, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking);
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
    /* runs still in flight finish first: their kernels use the ctx's scratch (every kernel of the ctx is
     * followed by ev_last on its stream; the host entry points' copies are on the ctx's own streams) */
    if (ctx->ev_last && ctx->ev_last_valid) cudaEventSynchronize(ctx->ev_last);
    if (ctx->host_stream) cudaStreamSynchronize(ctx->host_stream);
    if (ctx->copy_stream) cudaStreamSynchronize(ctx->copy_stream);
    for (size_t k = 0; k < ctx->owned.size(); ++k) cudaFree(ctx->owned[k].base); /* queues, words, staging, ... */
    ctx->owned.clear();
    if (ctx->late_host) cudaFreeHost(ctx->late_host);
    for (int k = 0; k < IA_NSTAGE; ++k)
        if (ctx->stage[k].ev_free) cudaEventDestroy(ctx->stage[k].ev_free);
    for (int k = 0; k < IA_FLUSH_RING; ++k)
        for (int j = 0; j < 2; ++j)
            if (ctx->flush[k].ev[j]) cudaEventDestroy(ctx->flush[k].ev[j]);
    for (int k = 0; k < IA_RUN_RING; ++k)
        for (int j = 0; j < 2; ++j)
            if (ctx->run[k].ev[j]) cudaEventDestroy(ctx->run[k].ev[j]);
    if (ctx->ev_last) cudaEventDestroy(ctx->ev_last);
    if (ctx->host_stream) cudaStreamDestroy(ctx->host_stream);
    if (ctx->copy_stream) cudaStreamDestroy(ctx->copy_stream);
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

int ia_set_chain(ia_ctx *ctx, int levels, uint32_t budget) {
    if (!ctx) return IA_EINVAL;
    if (levels < 1 || levels > IA_STRAGGLER_LEVELS || budget < 64u)
        return fail_inval(ctx, "ia_set_chain: need 1 <= levels <= IA_STRAGGLER_LEVELS and budget >= 64");
    ctx->levels = levels;
    ctx->level_budget = budget;
    return IA_OK;
}

int ia_get_timing(ia_ctx *ctx, int runs_back, double *bulk_ms, double *coop_ms) {
    if (!ctx || !bulk_ms || !coop_ms) return IA_EINVAL;
    if (runs_back < 0 || runs_back >= IA_RUN_RING || (unsigned long long)runs_back >= ctx->seq)
        return fail_inval(ctx, "ia_get_timing: that run is no longer (or not yet) on record");
    const IaRunEvents &R = ctx->run[(ctx->seq - 1 - (unsigned long long)runs_back) % IA_RUN_RING];
    const IaFlush *F = nullptr;
    if (R.flush >= 0) { /* the chain that finished (or will finish) what the run's bulk kernel handed on */
        if (R.flush >= ctx->flush_next)
            return fail_inval(ctx, "ia_get_timing: the run's stragglers are not enqueued yet (ia_join)");
        F = &ctx->flush[R.flush % IA_FLUSH_RING];
        if (F->id != R.flush) return fail_inval(ctx, "ia_get_timing: that run is no longer on record");
    }
    cudaError_t e = cudaSetDevice(ctx->device);
    if (e == cudaSuccess) e = cudaEventSynchronize(F ? F->ev[1] : R.ev[1]);
    float a = 0.f, b = 0.f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&a, R.ev[0], R.ev[1]);
    if (e == cudaSuccess && F) e = cudaEventElapsedTime(&b, F->ev[0], F->ev[1]);
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
    if (L->mode != IA_IC_EXPLICIT && L->mode != IA_IC_GRID && L->mode != IA_IC_PHILOX && L->mode != IA_IC_THERMAL)
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
    if (L->mode == IA_IC_THERMAL) {
        /* a1 for a thermal run: widths of the ion's and the atom's Gaussians */
        if (!(std::isfinite(L->T_atom_uK) && L->T_atom_uK > 0.0 && std::isfinite(L->T_ion_uK) && L->T_ion_uK > 0.0))
            return fail_inval(ctx, "THERMAL launch needs T_atom_uK > 0 and T_ion_uK > 0");
        if (L->domain != 1) return fail_inval(ctx, "THERMAL launch starts on the full sphere: domain must be 1");
        const double w_h = ctx->w_harm;
        if (!(w_h > 0.0)) return fail_inval(ctx, "THERMAL launch needs q_x != 0 (ion trap frequency |q_x| Omega / 2^(3/2))");
        const double kT_i = L->T_ion_uK * 1e-6 * KB_EH_PER_K, kT_a = L->T_atom_uK * 1e-6 * KB_EH_PER_K;
        G->domain = 1;
        G->phase_mode = L->phase_mode;
        G->phase0 = L->phase0;
        G->seed = L->seed;
        G->cell = L->cell;
        G->theta_span_pi = 1.0;
        G->phi_span_pi = 2.0;
        G->sig_v_ion = std::sqrt(kT_i / ctx->P.m_i);
        G->sig_r_ion = G->sig_v_ion / w_h;
        G->sig_v_atom = std::sqrt(kT_a / ctx->P.m_a);
        return IA_OK;
    }
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

/* what every persistent kernel of the ctx is told about the late list (records wanted in host arrays) */
static void sched_late(const ia_ctx *ctx, IaSched *S) {
    S->q_cap = ctx->queue_cap;
    S->fault = ctx->n_late + 1;
    S->late = ctx->late_dev;
    S->n_late = ctx->n_late;
    S->late_cap = ctx->late_dev ? ctx->late_cap : 0ull;
}

/* every kernel of a ctx shares its scratch (queues, counters): a run waits, on the device, for the ctx's latest
 * kernel whatever stream that one is on */
static cudaError_t order_after_last(ia_ctx *ctx, cudaStream_t st) {
    return ctx->ev_last_valid ? cudaStreamWaitEvent(st, ctx->ev_last, 0) : cudaSuccess;
}
static cudaError_t mark_last(ia_ctx *ctx, cudaStream_t st) {
    const cudaError_t e = cudaEventRecord(ctx->ev_last, st);
    if (e == cudaSuccess) ctx->ev_last_valid = true;
    return e;
}

/* Enqueues, on `st`, the straggler chain that finishes what the open runs' bulk kernels left in the queue. */
static int flush_open(ia_ctx *ctx, cudaStream_t st) {
    if (ctx->n_open == 0) return IA_OK;
    cudaError_t e = order_after_last(ctx, st);
    if (e != cudaSuccess) return fail_cuda(ctx, "cudaStreamWaitEvent(chain)", e);
    IaGen G0;
    std::memset(&G0, 0, sizeof(G0));
    IaOut O0 = {nullptr, nullptr, nullptr}; /* every queue entry carries the outputs of its own run */
    int qi = (ctx->n_open - 1) & 1; /* the queue the last bulk kernel wrote */
    unsigned long long *chain = ctx->words + IA_W_CHAIN;
    const int sparse = ctx->n_sm * 4; /* one warp per SM sub-partition */
    const int n_stages = 2 + ctx->levels;
    IaFlush &F = ctx->flush[ctx->flush_next % IA_FLUSH_RING];
    e = cudaEventRecord(F.ev[0], st);
    for (int j = 0; j < n_stages && e == cudaSuccess; ++j) {
        IaSched S5;
        std::memset(&S5, 0, sizeof(S5));
        sched_late(ctx, &S5);
        S5.q_in = ctx->q[qi];
        S5.n_in = j == 0 ? ctx->words + IA_W_CNT + ctx->n_open : chain + 3 * j;
        S5.counter = chain + 3 * j + 1;
        const bool last = j + 1 == n_stages;
        if (!last) {
            S5.q_out = ctx->q[qi ^ 1];
            S5.n_out = chain + 3 * (j + 1);
            S5.handoff_lanes = 0;
            S5.budget = 0xffffffffu;
        }
        if (j < 2) {
            /* stages A, B: bulk layout, leaving by count */
            S5.n_fin = chain + 3 * j + 2;
            S5.run_floor = (unsigned long long)sparse * (j == 0 ? 32ull : 10ull);
            e = ia_launch_persistent(1, ctx->P, G0, O0, S5, j == 0 ? grid_for(ctx, 0, ~0ull >> 8) : sparse, st);
        } else {
            if (!last) {
                const unsigned long long b = (unsigned long long)ctx->level_budget << (j - 2);
                S5.budget = b > 0xffffffffull ? 0xffffffffu : (unsigned)b;
            }
            e = ia_launch_persistent(3, ctx->P, G0, O0, S5, sparse, st);
        }
        qi ^= 1;
    }
    if (e == cudaSuccess) e = cudaEventRecord(F.ev[1], st);
    if (e == cudaSuccess) e = mark_last(ctx, st);
    if (e != cudaSuccess) return fail_cuda(ctx, "straggler chain launch", e);
    F.id = ctx->flush_next++;
    ctx->n_open = 0;
    return IA_OK;
}

/* ia_run proper.  `late_dst` (may be NULL): host array the records of this run are wanted in (a pipelined host
 * run).  *ridx_out receives the run's place in the ring of run events. */
static int run_impl(ia_ctx *ctx, const ia_launch *launch, const ia_outputs *outputs, cudaStream_t st,
                    ia_record *late_dst, int *ridx_out) {
    ctx->err.clear();
    if (ridx_out) *ridx_out = -1;
    if (!outputs) return fail_inval(ctx, "outputs is NULL");
    IaGen Gn;
    unsigned long long warn;
    int rc = make_gen(ctx, launch, &Gn, &warn);
    if (rc != IA_OK) return rc;
    if (Gn.n == 0) return IA_OK;
    cudaError_t e = cudaSetDevice(ctx->device);
    if (e != cudaSuccess) return fail_cuda(ctx, "cudaSetDevice", e);
    const std::string warn_text = ctx->err;
    IaOut O;
    O.records = outputs->records;
    O.summary = outputs->summary;
    O.ic_dump = outputs->ic_dump;
    const bool coop_only = launch->path == IA_PATH_COOP_ONLY;
    const bool handoff = launch->path == IA_PATH_AUTO && ctx->handoff_lanes > 0;
    const bool piped = handoff && ctx->depth > 0;
    if (piped && ctx->n_open >= ctx->depth) { /* the pipeline is full: finish what is open first */
        rc = flush_open(ctx, st);
        if (rc != IA_OK) return rc;
    }
    e = order_after_last(ctx, st);
    if (e != cudaSuccess) return fail_cuda(ctx, "cudaStreamWaitEvent(previous run)", e);
    IaSched S;
    std::memset(&S, 0, sizeof(S));
    sched_late(ctx, &S);
    S.warn = warn;
    const int ridx = (int)(ctx->seq % IA_RUN_RING);
    IaRunEvents &R = ctx->run[ridx];
    if (!handoff) {
        /* one kernel to the end: no queue involved */
        unsigned long long *wc = ctx->counters + 4 * (size_t)(ctx->counter_next++ % IA_COUNTER_RING);
        e = cudaMemsetAsync(wc, 0, 4 * sizeof(unsigned long long), st);
        if (e != cudaSuccess) return fail_cuda(ctx, "cudaMemsetAsync(counter)", e);
        S.counter = wc;
        S.n_in = wc + 1; /* stays 0: nothing to resume */
        e = cudaEventRecord(R.ev[0], st);
        if (e == cudaSuccess)
            e = coop_only ? ia_launch_persistent(3, ctx->P, Gn, O, S, grid_for(ctx, 1, Gn.n), st)
                          : ia_launch_persistent(1, ctx->P, Gn, O, S, grid_for(ctx, 0, Gn.n), st);
        if (e == cudaSuccess) e = cudaEventRecord(R.ev[1], st);
        if (e == cudaSuccess) e = mark_last(ctx, st);
        if (e != cudaSuccess) return fail_cuda(ctx, "persistent kernel launch", e);
        R.flush = -1;
        ctx->seq++;
        if (ridx_out) *ridx_out = ridx;
        ctx->err = warn_text;
        return IA_OK;
    }
    const int k = ctx->n_open; /* place in the open cycle */
    if (k == 0) {
        e = cudaMemsetAsync(ctx->words, 0, IA_W_TOTAL * sizeof(unsigned long long), st);
        if (e != cudaSuccess) return fail_cuda(ctx, "cudaMemsetAsync(pipeline words)", e);
    }
    S.counter = ctx->words + IA_W_WC + k;
    S.q_in = ctx->q[(k & 1) ^ 1];
    S.n_in = ctx->words + IA_W_CNT + k;
    S.q_out = ctx->q[k & 1];
    S.n_out = ctx->words + IA_W_CNT + k + 1;
    /* pipelined: the next bulk kernel takes over everything this one still holds as soon as its counter is empty */
    S.handoff_lanes = piped ? 32 : ctx->handoff_lanes;
    S.budget = IA_BULK_BUDGET;
    S.late_dst = piped ? late_dst : nullptr;
    /* a full grid whenever trajectories may come in through the queue (their number is known on the device only) */
    const int blocks = k > 0 ? grid_for(ctx, 0, ~0ull >> 8) : grid_for(ctx, 0, Gn.n);
    e = cudaEventRecord(R.ev[0], st);
    if (e == cudaSuccess) e = ia_launch_persistent(1, ctx->P, Gn, O, S, blocks, st);
    if (e == cudaSuccess) e = cudaEventRecord(R.ev[1], st);
    if (e == cudaSuccess) e = mark_last(ctx, st);
    if (e != cudaSuccess) return fail_cuda(ctx, "bulk kernel launch", e);
    R.flush = ctx->flush_next;
    ctx->n_open++;
    ctx->seq++;
    if (ridx_out) *ridx_out = ridx;
    if (!piped) {
        rc = flush_open(ctx, st);
        if (rc != IA_OK) return rc;
    }
    ctx->err = warn_text;
    return IA_OK;
}

static int wait_impl(ia_ctx *ctx);

/* enqueues one host-buffer run: H2D, kernels, D2H; nothing here waits for the device unless a buffer has to grow
 * or the pipeline is full */
static int submit_host_impl(ia_ctx *ctx, const ia_launch *launch, const ia_outputs *host_out) {
    ctx->err.clear();
    if (!launch || !host_out) return fail_inval(ctx, "launch or outputs is NULL");
    const uint64_t n = launch->n;
    if (n == 0) return IA_OK;
    if (launch->mode == IA_IC_EXPLICIT && (!launch->y0 || !launch->phase))
        return fail_inval(ctx, "EXPLICIT launch needs y0 and phase");
    cudaError_t e = cudaSetDevice(ctx->device);
    if (e != cudaSuccess) return fail_cuda(ctx, "cudaSetDevice", e);
    cudaStream_t st = ctx->host_stream;
    const bool handoff = launch->path == IA_PATH_AUTO && ctx->handoff_lanes > 0;
    const bool piped = handoff && ctx->depth > 0;
    if (ctx->n_pending >= IA_PIPE_MAX || (piped && ctx->n_open >= ctx->depth)) {
        const int rc = wait_impl(ctx); /* blocks: the summaries and late records of the pending runs come back */
        if (rc != IA_OK) return rc;
    }
    if (piped && host_out->records && !ctx->late_dev) {
        /* late list: at most one entry per lane of a bulk grid and run */
        const unsigned long long cap = (unsigned long long)ctx->queue_cap * IA_PIPE_MAX;
        e = guarded_malloc(ctx, (void **)&ctx->late_dev, cap * sizeof(IaLate));
        if (e == cudaSuccess) e = cudaMallocHost(&ctx->late_host, cap * sizeof(IaLate));
        if (e != cudaSuccess) {
            guarded_free(ctx, ctx->late_dev);
            ctx->late_dev = nullptr;
            ctx->err = "late-record list allocation failed";
            return IA_ENOMEM;
        }
        ctx->late_cap = cap;
    }
    /* staging layout: [records n*64][ic_dump n*14*8][y0 n*12*8][phase n*8]; the summary sits in sum_stage */
    const size_t off_ic = host_out->records ? n * sizeof(ia_record) : 0;
    const size_t off_y0 = off_ic + (host_out->ic_dump ? n * 14 * sizeof(double) : 0);
    const size_t off_ph = off_y0 + (launch->mode == IA_IC_EXPLICIT ? n * 12 * sizeof(double) : 0);
    const size_t total = off_ph + (launch->mode == IA_IC_EXPLICIT ? n * sizeof(double) : 0);
    IaStage &T = ctx->stage[ctx->stage_next++ % IA_NSTAGE];
    if (total > T.bytes) {
        if (T.used) e = cudaEventSynchronize(T.ev_free); /* whatever still reads the old buffer finishes first */
        if (e != cudaSuccess) return fail_cuda(ctx, "synchronise before staging reallocation", e);
        guarded_free(ctx, T.buf);
        T.buf = nullptr;
        T.bytes = 0;
        e = guarded_malloc(ctx, (void **)&T.buf, total);
        if (e != cudaSuccess) {
            ctx->err = "device staging allocation failed";
            return IA_ENOMEM;
        }
        T.bytes = total;
    }
    if (T.used) { /* the copies back of the run that used this staging last */
        e = cudaStreamWaitEvent(st, T.ev_free, 0);
        if (e != cudaSuccess) return fail_cuda(ctx, "cudaStreamWaitEvent(staging)", e);
    }
    char *base = T.buf;
    ia_launch L = *launch;
    ia_outputs dev;
    IaPending &Q = ctx->pending[ctx->n_pending];
    Q.host_summary = host_out->summary;
    Q.dev_summary = ctx->sum_stage + ctx->n_pending;
    dev.summary = Q.dev_summary;
    dev.records = host_out->records ? (ia_record *)base : nullptr;
    dev.ic_dump = host_out->ic_dump ? (double *)(base + off_ic) : nullptr;
    e = cudaMemsetAsync(dev.summary, 0, sizeof(ia_summary), st);
    if (e != cudaSuccess) return fail_cuda(ctx, "cudaMemsetAsync(summary)", e);
    if (launch->mode == IA_IC_EXPLICIT) {
        e = cudaMemcpyAsync(base + off_y0, launch->y0, n * 12 * sizeof(double), cudaMemcpyHostToDevice, st);
        if (e == cudaSuccess)
            e = cudaMemcpyAsync(base + off_ph, launch->phase, n * sizeof(double), cudaMemcpyHostToDevice, st);
        if (e != cudaSuccess) return fail_cuda(ctx, "H2D copy of initial conditions", e);
        L.y0 = (const double *)(base + off_y0);
        L.phase = (const double *)(base + off_ph);
    }
    int ridx = -1;
    int rc = run_impl(ctx, &L, &dev, st, host_out->records, &ridx);
    if (rc != IA_OK) return rc;
    const std::string warn_text = ctx->err;
    ctx->n_pending++;
    /* Records and initial conditions go back as soon as the run's own kernels are done -- for a pipelined run on the
     * copy stream, behind its bulk kernel, while the next run's bulk kernel starts; the trajectories that one carries
     * on report through the late list (ia_wait).  The summary is final only after the chain: ia_wait copies it. */
    cudaStream_t cs = piped ? ctx->copy_stream : st;
    if (piped) e = cudaStreamWaitEvent(cs, ctx->run[ridx].ev[1], 0);
    if (e == cudaSuccess && host_out->records)
        e = cudaMemcpyAsync(host_out->records, dev.records, n * sizeof(ia_record), cudaMemcpyDeviceToHost, cs);
    if (e == cudaSuccess && host_out->ic_dump)
        e = cudaMemcpyAsync(host_out->ic_dump, dev.ic_dump, n * 14 * sizeof(double), cudaMemcpyDeviceToHost, cs);
    if (e == cudaSuccess) e = cudaEventRecord(T.ev_free, cs);
    if (e != cudaSuccess) return fail_cuda(ctx, "D2H copy", e);
    T.used = true;
    ctx->err = warn_text;
    return IA_OK;
}

/* ia_wait proper: chain of the open runs, summaries and late records of the pending host runs, host blocks */
static int wait_impl(ia_ctx *ctx) {
    cudaError_t e = cudaSetDevice(ctx->device);
    if (e != cudaSuccess) return fail_cuda(ctx, "cudaSetDevice", e);
    cudaStream_t st = ctx->host_stream;
    int rc = flush_open(ctx, st);
    if (rc != IA_OK) return rc;
    e = order_after_last(ctx, st);
    for (int k = 0; k < ctx->n_pending && e == cudaSuccess; ++k)
        if (ctx->pending[k].host_summary)
            e = cudaMemcpyAsync(ctx->pending[k].host_summary, ctx->pending[k].dev_summary, sizeof(ia_summary),
                                cudaMemcpyDeviceToHost, st);
    unsigned long long n_late = 0;
    if (e == cudaSuccess && ctx->late_dev) {
        e = cudaMemcpyAsync(&n_late, ctx->n_late, sizeof(n_late), cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        if (n_late > ctx->late_cap) n_late = ctx->late_cap; /* cannot happen: one entry per lane and run */
        if (e == cudaSuccess && n_late > 0)
            e = cudaMemcpyAsync(ctx->late_host, ctx->late_dev, n_late * sizeof(IaLate), cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaMemsetAsync(ctx->n_late, 0, sizeof(unsigned long long), st);
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->copy_stream);
    if (e != cudaSuccess) return fail_cuda(ctx, "ia_wait", e);
    /* the records of the trajectories that outlived their run's bulk kernel: stored over what the early copy left */
    for (unsigned long long k = 0; k < n_late; ++k) *ctx->late_host[k].dst = ctx->late_host[k].rec;
    ctx->n_pending = 0;
    return IA_OK;
}

extern "C" {

int ia_run(ia_ctx *ctx, const ia_launch *launch, const ia_outputs *outputs, void *cuda_stream) {
    if (!ctx) return IA_EINVAL;
    return run_impl(ctx, launch, outputs, (cudaStream_t)cuda_stream, nullptr, nullptr);
}

int ia_join(ia_ctx *ctx, void *cuda_stream) {
    if (!ctx) return IA_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    cudaError_t e = cudaSetDevice(ctx->device);
    if (e != cudaSuccess) return fail_cuda(ctx, "cudaSetDevice", e);
    const int rc = flush_open(ctx, st);
    if (rc != IA_OK) return rc;
    e = order_after_last(ctx, st);
    if (e != cudaSuccess) return fail_cuda(ctx, "ia_join", e);
    return IA_OK;
}

int ia_set_pipeline(ia_ctx *ctx, int depth) {
    if (!ctx) return IA_EINVAL;
    if (depth < 0 || depth > IA_PIPE_MAX) return fail_inval(ctx, "ia_set_pipeline: depth must be in [0, 64]");
    /* runs in flight keep the old setting: finish what is open */
    const int rc = wait_impl(ctx);
    if (rc != IA_OK) return rc;
    ctx->depth = depth;
    return IA_OK;
}

int ia_submit_host(ia_ctx *ctx, const ia_launch *launch, const ia_outputs *host_outputs) {
    if (!ctx) return IA_EINVAL;
    return submit_host_impl(ctx, launch, host_outputs);
}

int ia_sync(ia_ctx *ctx) {
    if (!ctx) return IA_EINVAL;
    cudaError_t e = cudaSetDevice(ctx->device);
    if (e == cudaSuccess && ctx->ev_last_valid) e = cudaEventSynchronize(ctx->ev_last);
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->host_stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->copy_stream);
    if (e != cudaSuccess) return fail_cuda(ctx, "ia_sync", e);
    return IA_OK;
}

int ia_wait(ia_ctx *ctx) {
    if (!ctx) return IA_EINVAL;
    return wait_impl(ctx);
}

int ia_run_host(ia_ctx *ctx, const ia_launch *launch, const ia_outputs *host_outputs) {
    if (!ctx) return IA_EINVAL;
    int rc = submit_host_impl(ctx, launch, host_outputs);
    if (rc != IA_OK) return rc;
    const std::string warn_text = ctx->err;
    rc = wait_impl(ctx);
    if (rc == IA_OK) ctx->err = warn_text;
    return rc;
}

int ia_debug_check(ia_ctx *ctx) {
    if (!ctx) return IA_EINVAL;
    cudaError_t e = cudaSetDevice(ctx->device);
    if (e == cudaSuccess && ctx->ev_last_valid) e = cudaEventSynchronize(ctx->ev_last);
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->host_stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->copy_stream);
    std::vector<unsigned char> g(2 * IA_GUARD);
    for (size_t k = 0; k < ctx->owned.size() && e == cudaSuccess; ++k) {
        const IaGuarded &G = ctx->owned[k];
        e = cudaMemcpy(g.data(), G.base, IA_GUARD, cudaMemcpyDeviceToHost);
        if (e == cudaSuccess) e = cudaMemcpy(g.data() + IA_GUARD, G.base + IA_GUARD + G.bytes, IA_GUARD, cudaMemcpyDeviceToHost);
        for (size_t j = 0; j < g.size() && e == cudaSuccess; ++j)
            if (g[j] != IA_GUARD_BYTE) {
                char msg[160];
                std::snprintf(msg, sizeof(msg), "ia_debug_check: guard zone of ctx buffer %zu (%zu bytes) overwritten at offset %s%zu",
                              k, G.bytes, j < IA_GUARD ? "-" : "+", j < IA_GUARD ? IA_GUARD - j : j - IA_GUARD);
                ctx->err = msg;
                return IA_ECUDA;
            }
    }
    unsigned long long w[2] = {0, 0};
    std::vector<unsigned long long> words(IA_W_TOTAL);
    if (e == cudaSuccess) e = cudaMemcpy(w, ctx->n_late, sizeof(w), cudaMemcpyDeviceToHost);
    if (e == cudaSuccess) e = cudaMemcpy(words.data(), ctx->words, IA_W_TOTAL * sizeof(unsigned long long), cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) return fail_cuda(ctx, "ia_debug_check", e);
    if (w[1] != 0) {
        ctx->err = (w[1] & 1) ? "ia_debug_check: a hand-over queue overflowed" : "ia_debug_check: the late-record list overflowed";
        return IA_ECUDA;
    }
    if (ctx->late_dev && w[0] > ctx->late_cap) return fail_inval(ctx, "ia_debug_check: late-record count beyond capacity");
    for (int k = 0; k <= IA_PIPE_MAX; ++k)
        if (words[IA_W_CNT + k] > ctx->queue_cap) return fail_inval(ctx, "ia_debug_check: hand-over count beyond the queue capacity");
    return IA_OK;
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

int ia_fp64_latency(int cuda_device, double *cycles_dfma, double *cycles_rcp_add) {
    if (!cycles_dfma || !cycles_rcp_add) return IA_EINVAL;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || cuda_device < 0 || cuda_device >= ndev) return IA_EDEVICE;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, cuda_device) != cudaSuccess || prop.major != 10) return IA_EDEVICE;
    return ia_run_fp64_latency(cuda_device, cycles_dfma, cycles_rcp_add) == cudaSuccess ? IA_OK : IA_ECUDA;
}

} // extern "C"

/* ---- ia_run_static: the production kernel pair with every byte of scratch in static device memory ------------------
 *
 * For callers that may not allocate (include/ia.h says who and why).  Nothing below calls cudaMalloc, cudaFree,
 * cudaMallocHost, cudaEventCreate or cudaStreamCreate; the only CUDA calls after the one-time set-up of a device are
 * cudaSetDevice, one cudaMemsetAsync and two kernel launches. */

#include <mutex>

/* The scratch ia_create would have taken from cudaMalloc, for one launch of at most IA_STATIC_MAX_N trajectories:
 *   words[0] work counter of the bulk kernel        words[3] fault word (queue overflow; cannot happen: n <= capacity)
 *   words[1] length of the bulk kernel's input      words[4] late-list length (there is no late list: stays 0)
 *            queue (there is none: stays 0)         words[5] work counter of the cooperative kernel
 *   words[2] trajectories handed over = length of the cooperative kernel's input queue
 *   q[]      the hand-over queue, one entry per trajectory of the launch at most
 * The words are cleared at the start of every call; the queue is not (entries are written before they are read). */
#define IA_STATIC_WORDS 32
struct IaStaticScratch {
    unsigned long long words[IA_STATIC_WORDS]; /* 256 bytes: the queue behind it stays 256-byte aligned */
    IaHand q[IA_STATIC_MAX_N];
};
static_assert(sizeof(IaStaticScratch) == 256 + (size_t)IA_STATIC_MAX_N * 256, "4 MiB + 256 bytes of static scratch");

/* File-scope device array: part of the library's device image on every GPU that loads it, until the process exits.
 * In HOST code this name is only a handle for the runtime -- never a device address: it is handed to nothing but
 * cudaGetSymbolAddress (static_device_setup), and the kernels get the pointer that call returns. */
static __device__ __align__(256) unsigned char ia_static_scratch[sizeof(IaStaticScratch)];

#define IA_STATIC_MAX_DEV 64
struct IaStaticDev {
    bool ready = false;
    IaStaticScratch *scratch = nullptr; /* device address of ia_static_scratch on this device */
    int n_sm = 0;
    IaKernelInfo kinfo[2]; /* 0 bulk, 1 cooperative */
};
static IaStaticDev g_static_dev[IA_STATIC_MAX_DEV];
static std::mutex g_static_mutex;

static int static_fail(char *errbuf, size_t errbuf_len, int code, const char *text) {
    if (errbuf && errbuf_len > 0) std::snprintf(errbuf, errbuf_len, "%s", text);
    return code;
}

/* Once per device, with that device current: the device address of the static array and the launch geometry of
 * the two persistent kernels.  Both are kept for the lifetime of the process. */
static int static_device_setup(int dev, const IaStaticDev **out, char *errbuf, size_t errbuf_len) {
    std::lock_guard<std::mutex> lock(g_static_mutex);
    IaStaticDev &D = g_static_dev[dev];
    if (!D.ready) {
        int major = 0, n_sm = 0;
        cudaError_t e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
        if (e == cudaSuccess) e = cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess || major != 10)
            return static_fail(errbuf, errbuf_len, IA_EDEVICE, "ia_run_static: the device is not compute capability 10.x");
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, ia_static_scratch);
        if (e != cudaSuccess || p == nullptr) {
            char msg[200];
            std::snprintf(msg, sizeof(msg), "ia_run_static: cudaGetSymbolAddress(static scratch): %s",
                          e != cudaSuccess ? cudaGetErrorString(e) : "NULL address");
            return static_fail(errbuf, errbuf_len, IA_ECUDA, msg);
        }
        IaStaticDev T;
        for (int k = 0; k < 2 && e == cudaSuccess; ++k)
            e = ia_persistent_info(k == 0 ? 1 : 3, &T.kinfo[k].blocks_per_sm, &T.kinfo[k].threads_per_block,
                                   &T.kinfo[k].regs, &T.kinfo[k].local_bytes);
        if (e != cudaSuccess || T.kinfo[0].blocks_per_sm < 1 || T.kinfo[1].blocks_per_sm < 1) {
            char msg[200];
            std::snprintf(msg, sizeof(msg), "ia_run_static: kernel attributes: %s", cudaGetErrorString(e));
            return static_fail(errbuf, errbuf_len, IA_ECUDA, msg);
        }
        T.scratch = (IaStaticScratch *)p;
        T.n_sm = n_sm;
        T.ready = true;
        D = T;
    }
    *out = &D;
    return IA_OK;
}

extern "C" int ia_run_static(const ia_species *species, const ia_trap *trap, double De_K, double r0_a0,
                             const ia_tol *tol, int cuda_device, const ia_launch *launch, const ia_outputs *outputs,
                             void *cuda_stream, char *errbuf, size_t errbuf_len) {
    if (errbuf && errbuf_len > 0) errbuf[0] = '\0';
    if (!species || !trap || !launch || !outputs)
        return static_fail(errbuf, errbuf_len, IA_EINVAL, "ia_run_static: species, trap, launch or outputs is NULL");
    /* the size limit first: it depends on nothing but the argument */
    if (launch->n > (uint64_t)IA_STATIC_MAX_N) {
        char msg[256];
        std::snprintf(msg, sizeof(msg),
                      "ia_run_static: launch.n = %llu exceeds IA_STATIC_MAX_N = %d, the capacity of the hand-over queue in "
                      "static device memory; cut the launch into several calls on one stream or use ia_create / ia_run",
                      (unsigned long long)launch->n, IA_STATIC_MAX_N);
        return static_fail(errbuf, errbuf_len, IA_EINVAL, msg);
    }
    if (launch->path != IA_PATH_AUTO)
        return static_fail(errbuf, errbuf_len, IA_EINVAL, "ia_run_static: launch.path must be IA_PATH_AUTO (it runs the production pair)");
    ia_ctx cell; /* host-only: parameters and error text; owns no stream, event or device memory */
    int rc = prepare_cell(&cell.P, cell.derived, &cell.w_harm, species, trap, De_K, r0_a0, tol);
    if (rc != IA_OK)
        return static_fail(errbuf, errbuf_len, rc, "ia_run_static: a species, trap, well-depth, r0 or tolerance value is out of range");
    IaGen Gn;
    unsigned long long warn = 0;
    rc = make_gen(&cell, launch, &Gn, &warn);
    if (rc != IA_OK) return static_fail(errbuf, errbuf_len, rc, cell.err.c_str());
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || cuda_device < 0 || cuda_device >= ndev || cuda_device >= IA_STATIC_MAX_DEV)
        return static_fail(errbuf, errbuf_len, IA_EDEVICE, "ia_run_static: no such CUDA device (there is no CPU fallback)");
    cudaError_t e = cudaSetDevice(cuda_device);
    if (e != cudaSuccess) return static_fail(errbuf, errbuf_len, IA_ECUDA, cudaGetErrorString(e));
    const IaStaticDev *D = nullptr;
    rc = static_device_setup(cuda_device, &D, errbuf, errbuf_len);
    if (rc != IA_OK) return rc;
    if (Gn.n == 0) return IA_OK;

    cudaStream_t st = (cudaStream_t)cuda_stream;
    unsigned long long *w = D->scratch->words; /* device addresses: arithmetic only, never dereferenced on the host */
    IaHand *queue = D->scratch->q;
    e = cudaMemsetAsync(w, 0, IA_STATIC_WORDS * sizeof(unsigned long long), st);
    if (e != cudaSuccess) return static_fail(errbuf, errbuf_len, IA_ECUDA, cudaGetErrorString(e));
    IaOut O;
    O.records = outputs->records;
    O.summary = outputs->summary;
    O.ic_dump = outputs->ic_dump;
    /* bulk kernel: generates and propagates; a drained warp with at most 16 running lanes -- or any drained warp 4096
     * iterations on -- hands them to the queue (ia_create's defaults) */
    IaSched S;
    std::memset(&S, 0, sizeof(S));
    S.counter = w + 0;
    S.n_in = w + 1;
    S.q_out = queue;
    S.n_out = w + 2;
    S.handoff_lanes = 16;
    S.budget = IA_BULK_BUDGET;
    S.q_cap = IA_STATIC_MAX_N;
    S.fault = w + 3;
    S.n_late = w + 4;
    S.warn = warn;
    const unsigned long long full0 = (unsigned long long)D->n_sm * D->kinfo[0].blocks_per_sm;
    const unsigned long long need0 = (Gn.n + 31ull) / 32ull;
    e = ia_launch_persistent(1, cell.P, Gn, O, S, (int)(need0 < full0 ? need0 : full0), st);
    /* cooperative kernel: finishes whatever the queue holds (possibly nothing), one warp per SM sub-partition at most */
    if (e == cudaSuccess) {
        IaGen G0;
        std::memset(&G0, 0, sizeof(G0));
        IaOut O0 = {nullptr, nullptr, nullptr}; /* every queue entry carries its own output pointers */
        IaSched C5;
        std::memset(&C5, 0, sizeof(C5));
        C5.q_in = queue;
        C5.n_in = w + 2;
        C5.counter = w + 5;
        C5.q_cap = IA_STATIC_MAX_N;
        C5.fault = w + 3;
        C5.n_late = w + 4;
        const unsigned long long sparse = (unsigned long long)D->n_sm * 4ull;
        const unsigned long long need1 = (Gn.n + 9ull) / 10ull;
        e = ia_launch_persistent(3, cell.P, G0, O0, C5, (int)(need1 < sparse ? need1 : sparse), st);
    }
    if (e != cudaSuccess) {
        char msg[200];
        std::snprintf(msg, sizeof(msg), "ia_run_static: kernel launch: %s", cudaGetErrorString(e));
        return static_fail(errbuf, errbuf_len, IA_ECUDA, msg);
    }
    if (!cell.err.empty()) static_fail(errbuf, errbuf_len, IA_OK, cell.err.c_str()); /* the PAPER.md:28 warning */
    return IA_OK;
}
