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

#define IA_PIPE_MAX 64     /* runs per generation */
#define IA_RUN_RING 128    /* runs whose kernel events are kept for ia_get_timing */
#define IA_COUNTER_RING 256 /* slots of 4 x u64 */
#define IA_SCRATCH_WORDS 32

/* The straggler chain: the cooperative kernel is launched IA_STRAGGLER_LEVELS times in a
 * row.  Level j runs until its queue is empty and then for level_budget << j more iterations per warp; what
 * still runs then is passed on to level j+1, which packs it ten trajectories to a warp again, in the
 * lowest-numbered blocks.  The survivors -- the longest trajectories -- so end up in a few dense warps, each
 * with an SM sub-partition to itself, where the latency of a step is lowest, instead of in thousands of
 * thinned-out warps that share sub-partitions.  A level lasts twice as long as the one before, so a
 * trajectory of N steps passes ~log2(N / budget) hand-overs of 256 bytes.  The last level keeps everything. */
#define IA_BULK_BUDGET 4096u /* the bulk kernel: a warp hands over at the latest this long after the counter ran dry */

/* One run of a generation: what the host entry points have to copy back once its stragglers are done. */
struct IaPending {
    ia_outputs host = {nullptr, nullptr, nullptr}; /* host destinations (all NULL for a device-resident run) */
    ia_outputs dev = {nullptr, nullptr, nullptr};  /* where they sit in the staging */
    uint64_t n = 0;
};

/* A generation = the runs whose stragglers ONE launch of the cooperative kernel finishes (ia_set_pipeline).
 * With depth 0 every run is a generation of its own and everything stays on the caller's stream. */
struct IaGeneration {
    IaHand *queue = nullptr;        /* hand-over queue shared by the generation's bulk kernels          */
    size_t queue_cap = 0;           /* in entries                                                       */
    IaHand *queue2 = nullptr;       /* second queue of the straggler chain (the levels ping-pong)       */
    unsigned long long *scratch = nullptr; /* per level j: [2j] entries queued for it, [2j+1] its work counter */
    cudaStream_t tail = nullptr;    /* stream of the cooperative kernel when depth > 0                  */
    cudaEvent_t ev_coop[2] = {nullptr, nullptr}; /* around the cooperative kernel                        */
    cudaEvent_t ev_end = nullptr;   /* after it and after the copies back of the host entry points      */
    bool used = false;              /* ev_end has been recorded                                         */
    int n_pending = 0;              /* bulk kernels enqueued, cooperative kernel not yet                */
    unsigned long long serial = 0;  /* counts the generations this buffer has served                    */
    IaPending pending[IA_PIPE_MAX];
    int run_idx[IA_PIPE_MAX] = {};  /* their places in the ring of run events                           */
    cudaStream_t last_stream = nullptr; /* stream of the generation's latest bulk kernel                */
    void *stage[IA_PIPE_MAX] = {};  /* device staging of the host entry points, per run of the generation */
    size_t stage_bytes[IA_PIPE_MAX] = {};
};

struct IaRunEvents {
    cudaEvent_t ev[2] = {nullptr, nullptr}; /* around the bulk kernel */
    int gen = 0;                            /* generation buffer and its serial at the time: where the  */
    unsigned long long gen_serial = 0;      /* cooperative-kernel time of this run is found             */
};

struct ia_ctx {
    int device = 0;
    IaParams P;
    double derived[16];
    /* per-launch scratch, a ring so that launches queued behind one another on a stream do not share:
     * slot = [work counter of the bulk kernel, pad, pad, pad] */
    unsigned long long *counters = nullptr;
    unsigned counter_next = 0;
    size_t queue_cap = 0; /* hand-over entries ONE run can produce: one per lane of a full bulk grid */
    int handoff_lanes = 16;
    double w_harm = 0.0;                   /* |q_x| Omega / 2^(3/2): the ion's trap frequency in thermal runs */
    int levels = IA_STRAGGLER_LEVELS;      /* launches of the straggler chain (ia_set_chain) */
    unsigned level_budget = 8192u;         /* iterations of its first level after the queue ran dry */
    int n_sm = 0;
    IaKernelInfo kinfo[2]; /* 0 bulk, 1 cooperative */
    int depth = 0;          /* runs per generation - 1 ... 0 = every run on its own (see ia_set_pipeline) */
    int cur = 0;            /* generation buffer the next run joins */
    IaGeneration gen[2];    /* two, so that the bulk kernels of one generation overlap the stragglers of the last */
    unsigned long long seq = 0; /* runs launched so far */
    IaRunEvents run[IA_RUN_RING];
    cudaStream_t host_stream = nullptr; /* ia_submit_host / ia_run_host */
    std::string err;
};

static int fail_cuda(ia_ctx *c, const char *what, cudaError_t e) {
    if (c) c->err = std::string(what) + ": " + cudaGetErrorString(e);
    return IA_ECUDA;
}
static int fail_inval(ia_ctx *c, const char *what) {
    if (c) c->err = what;
    return IA_EINVAL;
}

/* (re)allocates what generation buffer g owns for `runs` runs per generation */
static cudaError_t gen_init(ia_ctx *c, int g, int runs) {
    IaGeneration &G = c->gen[g];
    cudaError_t e = cudaSuccess;
    const size_t cap = c->queue_cap * (size_t)runs;
    if (cap > G.queue_cap) {
        if (G.queue) cudaFree(G.queue);
        G.queue = nullptr;
        G.queue_cap = 0;
        e = cudaMalloc(&G.queue, cap * sizeof(IaHand));
        if (e == cudaSuccess) G.queue_cap = cap;
    }
    if (e == cudaSuccess && !G.queue2)
        e = cudaMalloc(&G.queue2, (size_t)c->n_sm * c->kinfo[1].blocks_per_sm * 10 * sizeof(IaHand));
    if (e == cudaSuccess && !G.scratch) e = cudaMalloc(&G.scratch, IA_SCRATCH_WORDS * sizeof(unsigned long long));
    if (e == cudaSuccess && !G.tail) e = cudaStreamCreateWithFlags(&G.tail, cudaStreamNonBlocking);
    for (int j = 0; j < 2 && e == cudaSuccess; ++j)
        if (!G.ev_coop[j]) e = cudaEventCreate(&G.ev_coop[j]);
    if (e == cudaSuccess && !G.ev_end) e = cudaEventCreate(&G.ev_end);
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
    c->w_harm = std::fabs(tr->q[0]) * P.omega / std::pow(2.0, 1.5);
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
        e = gen_init(c, 0, 1);
    }
    for (int k = 0; k < IA_RUN_RING && e == cudaSuccess; ++k)
        for (int j = 0; j < 2 && e == cudaSuccess; ++j) e = cudaEventCreate(&c->run[k].ev[j]);
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
    /* runs still in flight finish first: their kernels use the ctx's scratch.  (Bulk kernels whose generation
     * was never joined are on the caller's stream: the caller synchronises that one.) */
    if (ctx->host_stream) cudaStreamSynchronize(ctx->host_stream);
    for (int g = 0; g < 2; ++g) {
        IaGeneration &G = ctx->gen[g];
        if (G.used) cudaEventSynchronize(G.ev_end);
        if (G.tail) cudaStreamDestroy(G.tail);
        if (G.queue) cudaFree(G.queue);
        if (G.queue2) cudaFree(G.queue2);
        if (G.scratch) cudaFree(G.scratch);
        for (int k = 0; k < IA_PIPE_MAX; ++k)
            if (G.stage[k]) cudaFree(G.stage[k]);
        for (int j = 0; j < 2; ++j)
            if (G.ev_coop[j]) cudaEventDestroy(G.ev_coop[j]);
        if (G.ev_end) cudaEventDestroy(G.ev_end);
    }
    for (int k = 0; k < IA_RUN_RING; ++k)
        for (int j = 0; j < 2; ++j)
            if (ctx->run[k].ev[j]) cudaEventDestroy(ctx->run[k].ev[j]);
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
    if (R.gen < 0) { /* one kernel to the end (IA_PATH_BULK_ONLY / IA_PATH_COOP_ONLY / hand-over off) */
        cudaError_t e0 = cudaSetDevice(ctx->device);
        if (e0 == cudaSuccess) e0 = cudaEventSynchronize(R.ev[1]);
        float a0 = 0.f;
        if (e0 == cudaSuccess) e0 = cudaEventElapsedTime(&a0, R.ev[0], R.ev[1]);
        if (e0 != cudaSuccess) return fail_cuda(ctx, "ia_get_timing", e0);
        *bulk_ms = a0;
        *coop_ms = 0.0;
        return IA_OK;
    }
    const IaGeneration &G = ctx->gen[R.gen];
    if (G.serial != R.gen_serial + 1 || !G.used)
        return fail_inval(ctx, G.serial == R.gen_serial ? "ia_get_timing: the run's stragglers are not enqueued yet (ia_join)"
                                                        : "ia_get_timing: that run is no longer on record");
    cudaError_t e = cudaSetDevice(ctx->device);
    if (e == cudaSuccess) e = cudaEventSynchronize(G.ev_end);
    float a = 0.f, b = 0.f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&a, R.ev[0], R.ev[1]);
    if (e == cudaSuccess) e = cudaEventElapsedTime(&b, G.ev_coop[0], G.ev_coop[1]);
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

/* Enqueues the cooperative kernel that finishes the hand-overs of generation buffer g, and the copies back
 * of its host runs.  `st` is the stream the call came in on; with depth 0 everything stays on it. */
static int flush_generation(ia_ctx *ctx, int g, cudaStream_t st) {
    IaGeneration &G = ctx->gen[g];
    if (G.n_pending == 0) return IA_OK;
    cudaError_t e = cudaSuccess;
    cudaStream_t ts = st;
    if (ctx->depth > 0) {
        /* on the generation's own stream, behind the bulk kernels of all its runs: the caller's stream is free
         * for the next generation's bulk kernels while this one's longest trajectories finish */
        ts = G.tail;
        for (int k = 0; k < G.n_pending && e == cudaSuccess; ++k)
            e = cudaStreamWaitEvent(ts, ctx->run[G.run_idx[k]].ev[1], 0);
        if (e != cudaSuccess) return fail_cuda(ctx, "cudaStreamWaitEvent(generation)", e);
    }
    IaGen G0;
    std::memset(&G0, 0, sizeof(G0));
    IaOut O0 = {nullptr, nullptr, nullptr}; /* every queue entry carries the outputs of its own run */
    unsigned long long most = (unsigned long long)G.n_pending * ctx->queue_cap / 32ull *
                              (unsigned long long)(ctx->handoff_lanes > 0 ? ctx->handoff_lanes : 32);
    IaHand *q_in = G.queue, *q_out = G.queue2;
    e = cudaEventRecord(G.ev_coop[0], ts);
    for (int j = 0; j < ctx->levels && e == cudaSuccess; ++j) {
        IaSched S5;
        std::memset(&S5, 0, sizeof(S5));
        S5.q_in = q_in;
        S5.n_in = G.scratch + 2 * j;
        S5.counter = G.scratch + 2 * j + 1;
        if (j + 1 < ctx->levels) {
            S5.q_out = q_out;
            S5.n_out = G.scratch + 2 * (j + 1);
            S5.handoff_lanes = 0;
            const unsigned long long b = (unsigned long long)ctx->level_budget << j;
            S5.budget = b > 0xffffffffull ? 0xffffffffu : (unsigned)b;
        }
        const int blocks = grid_for(ctx, 1, most);
        e = ia_launch_persistent(3, ctx->P, G0, O0, S5, blocks, ts);
        most = (unsigned long long)blocks * 10ull; /* what level j can pass on at most: all it holds */
        IaHand *t = q_in;
        q_in = q_out;
        q_out = t;
    }
    if (e == cudaSuccess) e = cudaEventRecord(G.ev_coop[1], ts);
    for (int k = 0; k < G.n_pending && e == cudaSuccess; ++k) {
        const IaPending &Q = G.pending[k];
        if (Q.host.records)
            e = cudaMemcpyAsync(Q.host.records, Q.dev.records, Q.n * sizeof(ia_record), cudaMemcpyDeviceToHost, ts);
        if (e == cudaSuccess && Q.host.ic_dump)
            e = cudaMemcpyAsync(Q.host.ic_dump, Q.dev.ic_dump, Q.n * 14 * sizeof(double), cudaMemcpyDeviceToHost, ts);
        if (e == cudaSuccess && Q.host.summary)
            e = cudaMemcpyAsync(Q.host.summary, Q.dev.summary, sizeof(ia_summary), cudaMemcpyDeviceToHost, ts);
    }
    if (e == cudaSuccess) e = cudaEventRecord(G.ev_end, ts);
    if (e != cudaSuccess) return fail_cuda(ctx, "cooperative kernel launch", e);
    G.used = true;
    G.serial++;
    G.n_pending = 0;
    if (ctx->depth > 0) ctx->cur ^= 1;
    return IA_OK;
}

/* ia_run proper.  `pend` (may be NULL) describes the copies back a host entry point wants once the run's
 * last kernel is done; *deferred says whether they were left to the generation's flush. */
static int run_impl(ia_ctx *ctx, const ia_launch *launch, const ia_outputs *outputs, cudaStream_t st,
                    const IaPending *pend, bool *deferred) {
    if (deferred) *deferred = false;
    ctx->err.clear();
    if (!outputs) return fail_inval(ctx, "outputs is NULL");
    IaGen Gn;
    unsigned long long warn;
    int rc = make_gen(ctx, launch, &Gn, &warn);
    if (rc != IA_OK) return rc;
    if (Gn.n == 0) return IA_OK;
    cudaError_t e = cudaSetDevice(ctx->device);
    if (e != cudaSuccess) return fail_cuda(ctx, "cudaSetDevice", e);
    const std::string warn_text = ctx->err;
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
    const int ridx = (int)(ctx->seq % IA_RUN_RING);
    IaRunEvents &R = ctx->run[ridx];
    if (!handoff) {
        /* one kernel to the end, on the caller's stream: no generation involved */
        e = cudaEventRecord(R.ev[0], st);
        if (e == cudaSuccess)
            e = coop_only ? ia_launch_persistent(3, ctx->P, Gn, O, S, grid_for(ctx, 1, Gn.n), st)
                          : ia_launch_persistent(1, ctx->P, Gn, O, S, grid_for(ctx, 0, Gn.n), st);
        if (e == cudaSuccess) e = cudaEventRecord(R.ev[1], st);
        if (e != cudaSuccess) return fail_cuda(ctx, "persistent kernel launch", e);
        R.gen = -1;
        ctx->seq++;
        ctx->err = warn_text;
        return IA_OK;
    }
    const int g = ctx->depth > 0 ? ctx->cur : 0;
    IaGeneration &G = ctx->gen[g];
    /* the generation buffer is free again once the cooperative kernel that read it last has ended */
    if (G.used) {
        e = cudaStreamWaitEvent(st, G.ev_end, 0);
        if (e != cudaSuccess) return fail_cuda(ctx, "cudaStreamWaitEvent(generation buffer)", e);
    }
    if (G.n_pending == 0) {
        e = cudaMemsetAsync(G.scratch, 0, IA_SCRATCH_WORDS * sizeof(unsigned long long), st);
        if (e != cudaSuccess) return fail_cuda(ctx, "cudaMemsetAsync(generation)", e);
    }
    S.q_out = G.queue;
    S.n_out = G.scratch;
    S.handoff_lanes = ctx->handoff_lanes;
    S.budget = IA_BULK_BUDGET;
    e = cudaEventRecord(R.ev[0], st);
    if (e == cudaSuccess) e = ia_launch_persistent(1, ctx->P, Gn, O, S, grid_for(ctx, 0, Gn.n), st);
    if (e == cudaSuccess) e = cudaEventRecord(R.ev[1], st);
    if (e != cudaSuccess) return fail_cuda(ctx, "bulk kernel launch", e);
    R.gen = g;
    R.gen_serial = G.serial;
    G.pending[G.n_pending] = pend ? *pend : IaPending();
    G.run_idx[G.n_pending] = ridx;
    G.last_stream = st;
    G.n_pending++;
    ctx->seq++;
    if (deferred) *deferred = true;
    if (G.n_pending >= (ctx->depth > 0 ? ctx->depth : 1)) {
        rc = flush_generation(ctx, g, st);
        if (rc != IA_OK) return rc;
    }
    ctx->err = warn_text;
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
    cudaStream_t st = ctx->host_stream;
    /* the staging belongs to the place the run will take in its generation (runs without a hand-over use the
     * first place of buffer 0, strictly in stream order) */
    const bool handoff = launch->path == IA_PATH_AUTO && ctx->handoff_lanes > 0;
    const int g = (handoff && ctx->depth > 0) ? ctx->cur : 0;
    IaGeneration &G = ctx->gen[g];
    const int k = handoff ? G.n_pending : 0;
    /* staging layout: [summary 1024][records n*64][ic_dump n*14*8][y0 n*12*8][phase n*8] */
    const size_t off_rec = sizeof(ia_summary);
    const size_t off_ic = off_rec + (host_out->records ? n * sizeof(ia_record) : 0);
    const size_t off_y0 = off_ic + (host_out->ic_dump ? n * 14 * sizeof(double) : 0);
    const size_t off_ph = off_y0 + (launch->mode == IA_IC_EXPLICIT ? n * 12 * sizeof(double) : 0);
    const size_t total = off_ph + (launch->mode == IA_IC_EXPLICIT ? n * sizeof(double) : 0);
    if (total > G.stage_bytes[k]) {
        /* whatever still reads the old staging finishes first */
        e = cudaStreamSynchronize(st);
        if (e == cudaSuccess && G.used) e = cudaEventSynchronize(G.ev_end);
        if (e != cudaSuccess) return fail_cuda(ctx, "synchronise before staging reallocation", e);
        if (G.stage[k]) cudaFree(G.stage[k]);
        G.stage[k] = nullptr;
        G.stage_bytes[k] = 0;
        e = cudaMalloc(&G.stage[k], total);
        if (e != cudaSuccess) {
            ctx->err = "device staging allocation failed";
            return IA_ENOMEM;
        }
        G.stage_bytes[k] = total;
    }
    if (G.used) { /* the copies back of the generation that used this staging last are behind ev_end */
        e = cudaStreamWaitEvent(st, G.ev_end, 0);
        if (e != cudaSuccess) return fail_cuda(ctx, "cudaStreamWaitEvent(staging)", e);
    }
    char *base = (char *)G.stage[k];
    ia_launch L = *launch;
    IaPending Q;
    Q.host = *host_out;
    Q.n = n;
    Q.dev.summary = (ia_summary *)base;
    Q.dev.records = host_out->records ? (ia_record *)(base + off_rec) : nullptr;
    Q.dev.ic_dump = host_out->ic_dump ? (double *)(base + off_ic) : nullptr;
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
    bool deferred = false;
    int rc = run_impl(ctx, &L, &Q.dev, st, &Q, &deferred);
    if (rc != IA_OK || deferred) return rc;
    /* no hand-over: the run ended on st, the copies back follow it there */
    const std::string warn_text = ctx->err;
    if (Q.host.records)
        e = cudaMemcpyAsync(Q.host.records, Q.dev.records, n * sizeof(ia_record), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess && Q.host.ic_dump)
        e = cudaMemcpyAsync(Q.host.ic_dump, Q.dev.ic_dump, n * 14 * sizeof(double), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess && Q.host.summary)
        e = cudaMemcpyAsync(Q.host.summary, Q.dev.summary, sizeof(ia_summary), cudaMemcpyDeviceToHost, st);
    if (e != cudaSuccess) return fail_cuda(ctx, "D2H copy", e);
    ctx->err = warn_text;
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
    for (int g = 0; g < 2; ++g) {
        const int rc = flush_generation(ctx, g, st);
        if (rc != IA_OK) return rc;
    }
    for (int g = 0; g < 2 && e == cudaSuccess; ++g)
        if (ctx->gen[g].used) e = cudaStreamWaitEvent(st, ctx->gen[g].ev_end, 0);
    if (e != cudaSuccess) return fail_cuda(ctx, "ia_join", e);
    return IA_OK;
}

int ia_set_pipeline(ia_ctx *ctx, int depth) {
    if (!ctx) return IA_EINVAL;
    if (depth < 0 || depth > IA_PIPE_MAX) return fail_inval(ctx, "ia_set_pipeline: depth must be in [0, 64]");
    cudaError_t e = cudaSetDevice(ctx->device);
    if (e != cudaSuccess) return fail_cuda(ctx, "cudaSetDevice", e);
    /* runs in flight keep the old layout: enqueue what is pending and let everything finish */
    for (int g = 0; g < 2; ++g) {
        const int rc = flush_generation(ctx, g, ctx->gen[g].last_stream);
        if (rc != IA_OK) return rc;
    }
    for (int g = 0; g < 2 && e == cudaSuccess; ++g)
        if (ctx->gen[g].used) e = cudaEventSynchronize(ctx->gen[g].ev_end);
    if (e == cudaSuccess) e = gen_init(ctx, 0, depth > 0 ? depth : 1);
    if (e == cudaSuccess && depth > 0) e = gen_init(ctx, 1, depth);
    if (e == cudaErrorMemoryAllocation) {
        ctx->err = "ia_set_pipeline: hand-over queue allocation failed";
        return IA_ENOMEM;
    }
    if (e != cudaSuccess) return fail_cuda(ctx, "ia_set_pipeline", e);
    ctx->depth = depth;
    ctx->cur = 0;
    return IA_OK;
}

int ia_submit_host(ia_ctx *ctx, const ia_launch *launch, const ia_outputs *host_outputs) {
    if (!ctx) return IA_EINVAL;
    return submit_host_impl(ctx, launch, host_outputs);
}

int ia_wait(ia_ctx *ctx) {
    if (!ctx) return IA_EINVAL;
    int rc = ia_join(ctx, ctx->host_stream);
    if (rc != IA_OK) return rc;
    cudaError_t e = cudaStreamSynchronize(ctx->host_stream);
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
