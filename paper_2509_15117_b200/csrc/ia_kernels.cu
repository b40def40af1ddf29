/*
 * ia_kernels.cu -- the persistent propagation kernels (K1 bulk, K5 straggler), the initial-condition
 * generator (K2) and the verification kernels (K3).  Compiled with -fmad=false: see ia_dev.cuh.
 *
 * ia_persistent_kernel<LPT, SRC>: state, accelerations of all seven stages and step size live in
 * registers, what is touched only when a trajectory starts, bounces or ends in one shared-memory struct;
 * nothing per step touches global memory.  A group of LPT lanes owns one trajectory.  A group whose
 * trajectory has terminated writes its 64-byte record, adds to the ensemble summary and takes the next
 * index from a global work counter (one atomicAdd per warp-refill), so warps stay full although
 * trajectory lengths span 10^3..10^7 steps.  Exit localisation
 * (reading R7) re-uses the same step body with the group in mode LOC, so the warp never diverges on it.
 * The step loop proper is an inner loop of up to IA_INNER attempts that is left when a trajectory of the
 * warp terminates; counter, queue and budget logic sit outside it and out of its registers.
 *
 *   K1 = <1, IA_SRC_BOTH>: one lane per trajectory, the throughput layout.  Its work counter first deals out
 *        the trajectories an earlier bulk kernel left unfinished (a hand-over queue; empty for a run on its
 *        own), then the indices of its own launch, which it generates.  Once the counter is empty and a warp
 *        is down to `handoff_lanes` running lanes (or `budget` attempts later at the latest) it writes their
 *        states to a queue and exits.  With ia_set_pipeline that queue feeds the bulk kernel of the NEXT run
 *        (handoff_lanes = 32: at once), so a trajectory of 10^7 steps lives in full warps across many runs
 *        and only the last run of a stream is followed by a straggler chain.
 *   K5 = <3, IA_SRC_QUEUE>: three lanes per trajectory (x/y/z split); resumes trajectories from a queue.  A
 *        third of the FP64 instructions per lane and step: what counts for the longest trajectories is the
 *        latency of one step.  Launched as a chain of levels (ia_api.cu): each level passes what still runs
 *        after its budget to the next, which deals it out ten to a warp again.
 *   <3, IA_SRC_GEN>: the cooperative layout from the first step (IA_PATH_COOP_ONLY, verification).
 * All run the same arithmetic (ia_dev.cuh) and give bit-identical trajectories, so where a trajectory is
 * handed over does not show in its result.
 */
#include "ia_kernels.cuh"

#define IA_THREADS 32
#define IA_INNER 64u /* step attempts between two looks at the work counter / hand-over rules */

enum { MODE_IDLE = 0, MODE_RUN = 1, MODE_LOC = 2 };

/* ---- generator (readings R1-R3) ------------------------------------------------------------ */

/* Philox4x32-10 (Salmon et al., SC'11), from the published round function. */
__device__ __forceinline__ void ia_philox(unsigned c0, unsigned c1, unsigned c2, unsigned c3, unsigned k0, unsigned k1,
                                          unsigned (&out)[4]) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const unsigned lo0 = 0xD2511F53u * c0, hi0 = __umulhi(0xD2511F53u, c0);
        const unsigned lo1 = 0xCD9E8D57u * c2, hi1 = __umulhi(0xCD9E8D57u, c2);
        const unsigned n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* 53-bit uniform from two words (reading R2): (k + 1/2) 2^-53 for k < 2^52; from 2^52 on the sum k + 1/2 ties to even, so
 * the map is onto (0, 1] -- u = 1 for the one word pair with all 53 bits set (pinned on the oracle side) */
__device__ __forceinline__ double ia_u53(unsigned we, unsigned wo) {
    return ((double)(we >> 5) * 67108864.0 + (double)(wo >> 6) + 0.5) * (1.0 / 9007199254740992.0);
}

struct IaIC {
    double x[6], v[6]; /* r_i, r_a | v_i, v_a */
    double phase, E_au;
};

/* THERMAL runs (reading R18) draw fourteen numbers per trajectory from seven Philox blocks; block b
 * is one task: b = 0 -> (u1, u2), the direction of the atom's position; b = 1 -> (u3, u4), the rf phase;
 * b = 2..6 -> a Box-Muller pair
 * (z_2k, z_2k+1) = sqrt(-2 ln u_a) (cos 2 pi u_b, sin 2 pi u_b), k = b - 2.  The bulk kernel spreads the tasks of
 * the lanes that start a trajectory over the whole warp (seven lanes work for one idle lane instead of the idle lane
 * working seven times as long while 31 wait); ia_generate_ic runs them one after the other.  Same function, same
 * inputs: the two give identical initial conditions. */
__device__ __forceinline__ void ia_thermal_task(const IaGen &G, unsigned long long gi, unsigned b, double &a0, double &a1) {
    unsigned w[4];
    ia_philox((unsigned)gi, (unsigned)(gi >> 32), G.cell, b, (unsigned)G.seed, (unsigned)(G.seed >> 32), w);
    const double ua = ia_u53(w[0], w[1]), ub = ia_u53(w[2], w[3]);
    if (b < 2u) {
        a0 = ua;
        a1 = ub;
    } else {
        const double R = sqrt(-2.0 * log(ua));
        double sb, cb;
        sincospi(2.0 * ub, &sb, &cb);
        a0 = R * cb;
        a1 = R * sb;
    }
}

/* the thermal initial condition from its fourteen numbers t[2b], t[2b+1] (see ia_thermal_task) */
__device__ __forceinline__ void ia_thermal_assemble(const IaParams &P, const IaGen &G, const double *t, IaIC *ic) {
    const double ct = 2.0 * t[0] - 1.0;
    const double st = sqrt(1.0 - ct * ct);
    double sp, cp;
    sincospi(2.0 * t[1], &sp, &cp);
    const double *z = t + 4;
    const double n0 = st * cp, n1 = st * sp, n2 = ct;
    double va0 = G.sig_v_atom * z[6], va1 = G.sig_v_atom * z[7], va2 = G.sig_v_atom * z[8];
    const double vr = va0 * n0 + va1 * n1 + va2 * n2;
    const double sign = (vr > 0.0) ? -1.0 : 1.0;
    ic->E_au = 0.5 * P.m_a * (va0 * va0 + va1 * va1 + va2 * va2);
    ic->x[0] = G.sig_r_ion * z[0]; ic->x[1] = G.sig_r_ion * z[1]; ic->x[2] = G.sig_r_ion * z[2];
    ic->v[0] = G.sig_v_ion * z[3]; ic->v[1] = G.sig_v_ion * z[4]; ic->v[2] = G.sig_v_ion * z[5];
    ic->x[3] = P.r0 * n0; ic->x[4] = P.r0 * n1; ic->x[5] = P.r0 * n2;
    ic->v[3] = sign * va0; ic->v[4] = sign * va1; ic->v[5] = sign * va2;
    ic->phase = (G.phase_mode == 1) ? 6.28318530717958647692 * t[2] : G.phase0;
}

/* Initial condition of local trajectory j.  Out of line and writing through a pointer on purpose:
 * the struct lives in the stack frame for the duration of a refill only, and the persistent state
 * of the caller stays in registers. */
template <bool WITH_THERMAL = true> /* false: the caller generates thermal initial conditions itself (bulk kernel) */
__device__ __forceinline__ void ia_generate_ic(const IaParams &P, const IaGen &G, unsigned long long j, IaIC *ic) {
    if (G.mode == IA_IC_EXPLICIT) {
#pragma unroll
        for (int i = 0; i < 6; ++i) {
            ic->x[i] = G.y0[j * 12 + i];
            ic->v[i] = G.y0[j * 12 + 6 + i];
        }
        ic->phase = G.phase[j];
        ic->E_au = 0.5 * P.m_a * (ic->v[3] * ic->v[3] + ic->v[4] * ic->v[4] + ic->v[5] * ic->v[5]);
        return;
    }
    const unsigned long long gi = G.first_index + j;
    if (WITH_THERMAL && G.mode == IA_IC_THERMAL) {
        /* thermal run (reading R18): atom uniform on the r0 sphere, Maxwell-Boltzmann velocity
         * negated if needed so that v_r < 0; ion Gaussian in position and velocity */
        double t[14];
#pragma unroll
        for (unsigned b = 0; b < 7u; ++b) ia_thermal_task(G, gi, b, t[2 * b], t[2 * b + 1]);
        ia_thermal_assemble(P, G, t, ic);
        return;
    }
    unsigned w0[4], w1[4];
    ia_philox((unsigned)gi, (unsigned)(gi >> 32), G.cell, 0u, (unsigned)G.seed, (unsigned)(G.seed >> 32), w0);
    ia_philox((unsigned)gi, (unsigned)(gi >> 32), G.cell, 1u, (unsigned)G.seed, (unsigned)(G.seed >> 32), w1);
    const double u1 = ia_u53(w0[0], w0[1]), u2 = ia_u53(w0[2], w0[3]);
    const double u3 = ia_u53(w1[0], w1[1]), u4 = ia_u53(w1[2], w1[3]);
    double ct, st, sp, cp;
    if (G.mode == IA_IC_GRID) {
        const unsigned long long ii = gi / G.n_phi, jj = gi % G.n_phi;
        /* theta = (i + 1/2) span / n_theta, evaluated as sincospi(theta/pi) */
        sincospi(((double)ii + 0.5) * G.theta_span_pi / (double)G.n_theta, &st, &ct);
        sincospi(((double)jj + 0.5) * G.phi_span_pi / (double)G.n_phi, &sp, &cp);
    } else {
        ct = (G.domain == 0) ? u1 : 2.0 * u1 - 1.0;
        st = sqrt(1.0 - ct * ct);
        sincospi(G.phi_span_pi * u2, &sp, &cp);
    }
    ic->phase = (G.phase_mode == 1) ? 6.28318530717958647692 * u3 : G.phase0;
    double v0;
    if (G.log_E_ratio != 0.0) {
        const double E_uK = G.E_min_uK * exp(u4 * G.log_E_ratio);
        ic->E_au = E_uK * 1e-6 * 3.1668115634564e-6; /* k_B in E_h/K (CODATA 2022) */
        v0 = sqrt(2.0 * ic->E_au / P.m_a);
    } else {
        ic->E_au = G.E_fixed_au;
        v0 = G.v0_fixed;
    }
    const double n0 = st * cp, n1 = st * sp, n2 = ct;
    ic->x[0] = 0.0; ic->x[1] = 0.0; ic->x[2] = 0.0;   /* ion at the trap centre, at rest */
    ic->v[0] = 0.0; ic->v[1] = 0.0; ic->v[2] = 0.0;
    ic->x[3] = P.r0 * n0; ic->x[4] = P.r0 * n1; ic->x[5] = P.r0 * n2;   /* atom on the r0 sphere ...   */
    ic->v[3] = -v0 * n0; ic->v[4] = -v0 * n1; ic->v[5] = -v0 * n2;      /* ... aimed at the ion        */
}

__global__ void ia_generate_kernel(const __grid_constant__ IaParams P, const __grid_constant__ IaGen G,
                                   double *ic_dump) {
    const unsigned long long j = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= G.n) return;
    IaIC ic;
    ia_generate_ic(P, G, j, &ic);
    double *o = ic_dump + j * 14;
#pragma unroll
    for (int i = 0; i < 6; ++i) {
        o[i] = ic.x[i];
        o[6 + i] = ic.v[i];
    }
    o[12] = ic.phase;
    o[13] = ic.E_au;
}

/* ---- helpers ---------------------------------------------------------------------------------- */

__device__ __forceinline__ bool ia_isfinite(double a) { return fabs(a) <= 1.79769313486231570815e308; }

__device__ __forceinline__ unsigned long long ia_globaltimer() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t));
    return t;
}

/* element `axis` (0..2) of a 3-array held in registers, without dynamic indexing */
__device__ __forceinline__ double ia_sel3(double a0, double a1, double a2, unsigned axis) {
    return axis == 0u ? a0 : (axis == 1u ? a1 : a2);
}

template <int LPT>
__device__ __forceinline__ void ia_park(const IaLane<LPT> &L, IaVec<LPT> &Y) {
    /* harmless finite state for idle lanes: ion at the origin, atom at (4,5,6) */
#pragma unroll
    for (int a = 0; a < 3 / LPT; ++a) {
        Y.xi[a] = 0.0;
        Y.xa[a] = 4.0 + (double)(L.axis0 + a);
        Y.vi[a] = 0.0; Y.va[a] = 0.0; Y.Ai[a] = 0.0; Y.Aa[a] = 0.0;
    }
}

/* ---- K1 / K5 ---------------------------------------------------------------------------------- */

/* SRC says where the kernel's trajectories come from (ia_kernels.cuh): IA_SRC_QUEUE = a level of the straggler
 * chain, which only resumes what a queue holds -- a compile-time switch, so that the chain's kernel carries neither
 * the generator nor its registers: the latency of its step loop is what the longest trajectories of a launch wait
 * for.  IA_SRC_BOTH = the bulk kernel: it first resumes what the bulk kernel of the run before left unfinished
 * (ia_set_pipeline: long trajectories keep living in full warps while fresh ones keep arriving), then generates. */
template <int LPT, int SRC>
__global__ void __launch_bounds__(IA_THREADS, LPT == 1 ? 12 : 16)
ia_persistent_kernel(const __grid_constant__ IaParams P, const __grid_constant__ IaGen G, const IaOut O,
                     const IaSched S) {
    constexpr int NA = 3 / LPT;
    const unsigned lane = threadIdx.x & 31u;
    const IaLane<LPT> L = ia_make_lane<LPT>(P, lane);
    /* group state (replicated in the LPT lanes of a group) */
    IaVec<LPT> Y;
    double tf = 0.0, h = 0.0;
    unsigned n_per = 0, steps_acc = 0;
    /* rarely touched per-group state lives in shared memory, not in registers: one struct of arrays, so that
     * a lane reaches all of it from two address registers (8-byte and 4-byte members) */
    __shared__ struct {
        double t_first[IA_THREADS], t_last[IA_THREADS], phase[IA_THREADS], s_old[IA_THREADS];
        unsigned long long slot[IA_THREADS];
        ia_record *rec[IA_THREADS];   /* outputs of the run the group's trajectory belongs to */
        ia_summary *sum[IA_THREADS];
        unsigned steps_in[IA_THREADS], n_coll[IA_THREADS], n_tp[IA_THREADS], n_loc[IA_THREADS], att0[IA_THREADS],
            cnt[IA_THREADS], wexh[IA_THREADS], iters[IA_THREADS];
        unsigned per_fin[IA_THREADS];     /* warp-uniform: 16 x running mean of the iterations per finished trajectory */
        unsigned last_fin[IA_THREADS];    /* warp-uniform: iteration count at the last finish */
        unsigned flags[IA_THREADS];       /* IA_HAND_LATE | IA_CARRIED */
        unsigned steps_entry[IA_THREADS]; /* attempted steps the trajectory had taken when this kernel got it */
        double loc_lo[IA_THREADS], loc_hi[IA_THREADS]; /* bracket of the exit localisation (R7) */
        double t_fin[IA_THREADS];                      /* time at which the trajectory ended */
    } sh;
    /* the fourteen numbers of a thermal initial condition per lane (bulk kernel only) */
    __shared__ double sh_gen[(LPT == 1 && SRC != IA_SRC_QUEUE) ? IA_THREADS : 1][14];
    double &t_first = sh.t_first[threadIdx.x], &t_last = sh.t_last[threadIdx.x], &phase = sh.phase[threadIdx.x],
           &s_old = sh.s_old[threadIdx.x];
    phase = 0.0; s_old = 0.0;
    unsigned long long &slot = sh.slot[threadIdx.x];
    ia_record *&out_rec = sh.rec[threadIdx.x];
    ia_summary *&out_sum = sh.sum[threadIdx.x];
    out_rec = O.records; out_sum = O.summary;
    unsigned &steps_in = sh.steps_in[threadIdx.x], &n_coll = sh.n_coll[threadIdx.x], &n_tp = sh.n_tp[threadIdx.x],
             &n_loc = sh.n_loc[threadIdx.x];
    /* attempts are not counted step by step: a running trajectory makes one per iteration of its warp, so the number
     * it has made is att0 + iters (att0 = attempts before it got here minus the warp's iteration count then) */
    unsigned &att0 = sh.att0[threadIdx.x];
    bool s_neg = false;   /* sign of s = d.w at the current state (the value s_old is needed at a bounce only) */
    bool outside = false; /* |d| >= r0 at the current state: such a trajectory has no exit crossing to localise (R7) */
    unsigned &cnt = sh.cnt[threadIdx.x]; /* warp-uniform: step attempts since the queue ran dry */
    cnt = 0;
    unsigned &iters = sh.iters[threadIdx.x]; /* warp-uniform: step attempts of this warp so far */
    iters = 0;
    unsigned &flags = sh.flags[threadIdx.x], &steps_entry = sh.steps_entry[threadIdx.x];
    flags = 0; steps_entry = 0;
    sh.per_fin[threadIdx.x] = 16u * 1024u; /* start from "long trajectories": no waiting until finishes say otherwise */
    sh.last_fin[threadIdx.x] = 0u;
    t_first = 0.0; t_last = 0.0; slot = 0; steps_in = 0; n_coll = 0; n_tp = 0; n_loc = 0; att0 = 0;
    int mode = MODE_IDLE;
    bool failed = false;
    unsigned &wexh = sh.wexh[threadIdx.x]; /* warp-uniform flag: the work counter is empty */
    wexh = 0u;
    ia_park<LPT>(L, Y);
    if (SRC != IA_SRC_QUEUE && O.summary != nullptr && threadIdx.x == 0) {
        const unsigned long long t0 = ia_globaltimer();
        if (blockIdx.x == 0) {
            atomicCAS((unsigned long long *)&O.summary->t_start_ns, 0ull, t0);
            if (S.warn) atomicOr((unsigned long long *)&O.summary->warn, S.warn);
        }
    }

    constexpr unsigned long long PER_WARP = (LPT == 1) ? 32ull : 10ull; /* trajectories a warp holds */
    /* A kernel that resumes from a queue deals the first gridDim.x * PER_WARP entries out by block index, so that
     * when the queue is short the work sits in the lowest-numbered blocks -- which the hardware spreads over the
     * SMs -- instead of wherever the race for the counter ends; the counter serves the rest of the queue. */
    constexpr bool resume = (SRC == IA_SRC_QUEUE);
#define IA_CARRIED 2u /* flags: the trajectory came out of a hand-over queue */
#define IA_DEALT (resume ? (unsigned long long)gridDim.x * PER_WARP : 0ull)
#define IA_N_IN (SRC == IA_SRC_GEN ? 0ull : *S.n_in) /* final: the producer kernel has ended */
#define IA_N_TOTAL (resume ? IA_N_IN : IA_N_IN + G.n)
    bool first_refill = resume;

    for (;;) {
        const bool was_exh = wexh != 0u;
        /* ---- refill idle groups from the global work counter (a12) ----
         * Starting a trajectory costs the whole warp ~1e3 instructions (generator, first acceleration, first step
         * size), an idle lane ~27 per step it sits out.  When trajectories are short (thermal bars: 100-400 steps, one
         * of the warp's 32 ends every few steps) it pays to let a few lanes idle and start several together: with I
         * the warp's iterations per finished trajectory (running mean), B = floor(sqrt(K / I)) lanes are collected,
         * K = 111 for the thermal generator, 59 otherwise -- B = 1 (no waiting) from ~900 resp. ~1900 steps per
         * trajectory on.  Which lane runs which index changes, no trajectory does. */
        const bool want = L.valid && (mode == MODE_IDLE) && !wexh;
        unsigned wm = __ballot_sync(IA_FULL, want && L.leader);
        if (!resume && wm != 0u) {
            const unsigned I = max(sh.per_fin[threadIdx.x] >> 4, 1u); /* 1/16 iterations, warp-uniform */
            const unsigned K = (G.mode == IA_IC_THERMAL) ? 111u : 59u;
            unsigned B = 1u;
            while (B < 8u && (B + 1u) * (B + 1u) * I <= K) ++B;
            /* ... but not for longer than collecting B lanes should take (the rest of the warp may be long-lived) */
            const bool overdue = iters - sh.last_fin[threadIdx.x] > 2u * B * I + IA_INNER;
            if ((unsigned)__popc(wm) < B && !overdue && __any_sync(IA_FULL, mode != MODE_IDLE)) wm = 0u;
        }
        if (wm) {
            const int first = __ffs(wm) - 1;
            unsigned long long base = 0;
            if (first_refill) {
                base = (unsigned long long)blockIdx.x * PER_WARP;
                first_refill = false;
            } else {
                if ((int)lane == first) base = IA_DEALT + atomicAdd(S.counter, (unsigned long long)__popc(wm));
                base = __shfl_sync(IA_FULL, base, first);
            }
            const unsigned long long j = base + __popc(wm & ((1u << L.gbase) - 1u));
            const unsigned long long n_in = IA_N_IN;
            const bool got = want && (j < (resume ? n_in : n_in + G.n));
            if (__any_sync(IA_FULL, want && !got)) {
                if (!wexh && O.summary != nullptr && !resume && lane == 0)
                    atomicCAS((unsigned long long *)&O.summary->t_first_idle_ns, 0ull, ia_globaltimer());
                wexh = 1u;
            }
            /* thermal runs: the seven Philox / Box-Muller tasks of every lane that starts a trajectory, spread over
             * the warp (ia_thermal_task) */
            constexpr bool coop_gen = (LPT == 1 && SRC != IA_SRC_QUEUE);
            if (coop_gen && G.mode == IA_IC_THERMAL) {
                const bool fresh = got && j >= n_in;
                const unsigned fm = __ballot_sync(IA_FULL, fresh);
                const unsigned long long gi_mine = G.first_index + (j - n_in);
                const unsigned n_tasks = 7u * (unsigned)__popc(fm);
                for (unsigned t0 = 0; t0 < n_tasks; t0 += 32u) {
                    const unsigned t = t0 + lane;
                    const bool act = t < n_tasks;
                    const unsigned rank = act ? t / 7u : 0u;
                    const unsigned blk = act ? t - 7u * rank : 0u;
                    const unsigned owner = __fns(fm, 0u, (int)rank + 1);
                    const unsigned long long gi_o = __shfl_sync(IA_FULL, gi_mine, (int)(owner & 31u));
                    if (act) ia_thermal_task(G, gi_o, blk, sh_gen[owner][2u * blk], sh_gen[owner][2u * blk + 1u]);
                }
                __syncwarp();
            }
            if (got) {
                if (resume || (SRC == IA_SRC_BOTH && j < n_in)) {
                    /* resume a trajectory an earlier kernel handed over */
                    const IaHand *H = S.q_in + j;
#pragma unroll
                    for (int a = 0; a < NA; ++a) {
                        const unsigned ax = L.axis0 + a;
                        Y.xi[a] = H->x[ax];  Y.xa[a] = H->x[3 + ax];
                        Y.vi[a] = H->v[ax];  Y.va[a] = H->v[3 + ax];
                        Y.Ai[a] = H->A1[ax]; Y.Aa[a] = H->A1[3 + ax];
                    }
                    tf = H->tf; h = H->h; phase = H->phase; s_old = H->s_old;
                    s_neg = H->s_old < 0.0;
                    outside = H->r2_cur >= P.r0sq;
                    t_first = H->t_first; t_last = H->t_last; slot = H->slot;
                    out_rec = H->records; out_sum = H->summary;
                    n_per = H->n_per; n_coll = H->n_coll; n_tp = H->n_tp;
                    steps_acc = H->steps_acc; failed = H->failed != 0u;
                    att0 = H->steps_acc + H->steps_rej - iters;
                    steps_in = H->steps_in;
                    flags = (H->flags & IA_HAND_LATE) | IA_CARRIED;
                    steps_entry = H->steps_acc + H->steps_rej;
                    n_loc = 0;
                    mode = MODE_RUN;
                } else if (SRC != IA_SRC_QUEUE) {
                    const unsigned long long jf = j - n_in; /* index within this launch */
                    IaIC ic;
                    if (coop_gen && G.mode == IA_IC_THERMAL)
                        ia_thermal_assemble(P, G, sh_gen[coop_gen ? threadIdx.x : 0], &ic);
                    else
                        ia_generate_ic<!coop_gen>(P, G, jf, &ic);
                    if (O.ic_dump != nullptr && L.leader) {
                        double *o = O.ic_dump + jf * 14;
#pragma unroll
                        for (int i = 0; i < 6; ++i) {
                            o[i] = ic.x[i];
                            o[6 + i] = ic.v[i];
                        }
                        o[12] = ic.phase;
                        o[13] = ic.E_au;
                    }
                    slot = jf;
                    out_rec = O.records; out_sum = O.summary;
                    flags = 0; steps_entry = 0;
                    tf = 0.0; n_per = 0; n_coll = 0; n_tp = 0; steps_acc = 0; n_loc = 0; steps_in = 0;
                    att0 = 0u - iters;
                    t_first = 0.0; t_last = 0.0; failed = false;
                    phase = ic.phase;
                    bool ok = ia_isfinite(phase);
#pragma unroll
                    for (int i = 0; i < 6; ++i) ok = ok && ia_isfinite(ic.x[i]) && ia_isfinite(ic.v[i]);
                    if (!ok) {
                        /* status 3: non-finite initial state; record it and stay idle */
                        if (L.leader) {
                            if (O.records != nullptr) {
                                ia_record r;
                                r.ke_ion = 0.5 * P.m_i * (ic.v[0] * ic.v[0] + ic.v[1] * ic.v[1] + ic.v[2] * ic.v[2]);
                                r.t_dwell = 0.0; r.t_life = 0.0;
                                r.va_f[0] = ic.v[3]; r.va_f[1] = ic.v[4]; r.va_f[2] = ic.v[5];
                                r.n_coll = 0; r.n_tp = 0; r.steps_acc = 0; r.steps_rej = 0; r.status = 3; r.n_loc = 0;
                                O.records[jf] = r;
                            }
                            if (O.summary != nullptr) {
                                atomicAdd((unsigned long long *)&O.summary->n_done, 1ull);
                                atomicAdd((unsigned long long *)&O.summary->n_status[3], 1ull);
                                atomicAdd((unsigned long long *)&O.summary->hist_ncoll[0], 1ull);
                            }
                        }
                        phase = 0.0;
                    } else {
                        /* keep the cosine argument in the folded range for any caller-supplied phase */
                        if (fabs(phase) > 6.5) phase -= 6.28318530717958647692 * rint(phase * 0.15915494309189533577);
                        /* A(0, x0) for all six components in the one-lane layout (same arithmetic per
                         * component as the group layout), then the ode45 first step (R5):
                         * h = min(h_max, t_max); rho = ||f0 / max(|y0|, thr)||_inf / (0.8 rtol^(1/5)) */
                        const IaLane<1> L1 = ia_make_lane<1>(P, lane);
                        const double xi3[3] = {ic.x[0], ic.x[1], ic.x[2]}, xa3[3] = {ic.x[3], ic.x[4], ic.x[5]};
                        double ai3[3], aa3[3], D[3], r2, s;
                        ia_accel<1, true>(P, L1, xi3, xa3, ia_cos_folded(phase), ai3, aa3, D, r2, s);
                        /* the largest of the twelve ratios |f_i| / max(|y_i|, thr), found by cross-multiplication
                         * and divided once (a correctly rounded quotient is monotone, so this is the maximum of the
                         * twelve quotients; twelve inline FP64 divisions are 500 instructions of code and of time
                         * per started trajectory) */
                        double rn = 0.0, rd = 1.0;
#pragma unroll
                        for (int i = 0; i < 3; ++i) {
                            ia_ratio_max(rn, rd, ic.v[i], ia_absmax_raw(ic.x[i], P.thr));
                            ia_ratio_max(rn, rd, ic.v[3 + i], ia_absmax_raw(ic.x[3 + i], P.thr));
                            ia_ratio_max(rn, rd, ai3[i], ia_absmax_raw(ic.v[i], P.thr));
                            ia_ratio_max(rn, rd, aa3[i], ia_absmax_raw(ic.v[3 + i], P.thr));
                        }
                        double rho = fabs(rn) / fabs(rd);
                        rho = rho / P.h0_scale;
                        h = fmin(P.h_max, P.t_max);
                        if (h * rho > 1.0) h = 1.0 / rho;
                        if (h < P.h_min) h = P.h_min;
                        const double W[3] = {ic.v[3] - ic.v[0], ic.v[4] - ic.v[1], ic.v[5] - ic.v[2]};
                        s_old = ia_dot3<true>(D, W);
                        s_neg = s_old < 0.0;
                        outside = r2 >= P.r0sq;
#pragma unroll
                        for (int a = 0; a < NA; ++a) {
                            const unsigned ax = L.axis0 + a;
                            Y.xi[a] = (LPT == 1) ? ic.x[a] : ia_sel3(ic.x[0], ic.x[1], ic.x[2], ax);
                            Y.xa[a] = (LPT == 1) ? ic.x[3 + a] : ia_sel3(ic.x[3], ic.x[4], ic.x[5], ax);
                            Y.vi[a] = (LPT == 1) ? ic.v[a] : ia_sel3(ic.v[0], ic.v[1], ic.v[2], ax);
                            Y.va[a] = (LPT == 1) ? ic.v[3 + a] : ia_sel3(ic.v[3], ic.v[4], ic.v[5], ax);
                            Y.Ai[a] = (LPT == 1) ? ai3[a] : ia_sel3(ai3[0], ai3[1], ai3[2], ax);
                            Y.Aa[a] = (LPT == 1) ? aa3[a] : ia_sel3(aa3[0], aa3[1], aa3[2], ax);
                        }
                        mode = MODE_RUN;
                    }
                }
            }
        }

        /* a warp whose groups are all busy never asks the counter: let it notice an empty queue anyway */
        if (!wexh) {
            unsigned long long c = 0;
            if (lane == 0) c = IA_DEALT + *(volatile unsigned long long *)S.counter;
            c = __shfl_sync(IA_FULL, c, 0);
            if (c >= IA_N_TOTAL) wexh = 1u;
        }
        if (wexh && !was_exh) cnt = 0u;

        /* ---- hand what still runs in a drained warp over to the next kernel of the chain: when few
         * trajectories are left in the warp (handoff_lanes), or when the warp has gone on for `budget`
         * iterations since the queue ran dry (so that no warp holds a level of the chain up) ---- */
        if (S.q_out != nullptr && wexh) {
            const unsigned am = __ballot_sync(IA_FULL, mode == MODE_RUN && L.leader); /* one bit per trajectory */
            const unsigned lm = __ballot_sync(IA_FULL, mode == MODE_LOC);
            /* a stage of the straggler chain also leaves when few of its trajectories are left altogether: the
             * next stage runs them in fewer warps per SM sub-partition, i.e. at a lower latency per step */
            bool few = false;
            if (S.n_fin != nullptr) {
                unsigned long long f = 0;
                if (lane == 0) f = *(volatile unsigned long long *)S.n_fin;
                f = __shfl_sync(IA_FULL, f, 0);
                few = IA_N_IN - f <= S.run_floor;
            }
            if (am != 0u && lm == 0u && (__popc(am) <= S.handoff_lanes || cnt >= S.budget || few)) {
                const int first = __ffs(am) - 1;
                unsigned long long base = 0;
                if ((int)lane == first) base = atomicAdd(S.n_out, (unsigned long long)__popc(am));
                base = __shfl_sync(IA_FULL, base, first);
                const unsigned long long qidx = base + __popc(am & ((1u << L.gbase) - 1u));
                if (mode == MODE_RUN && L.valid && qidx >= S.q_cap) {
                    /* cannot happen (the host sizes the queues for a full grid); never write out of bounds */
                    if (L.leader) atomicOr(S.fault, 1ull);
                    mode = MODE_IDLE;
                }
                if (mode == MODE_RUN && L.valid) {
                    /* every lane of the group writes the axes it holds, the leader the rest */
                    IaHand *H = S.q_out + qidx;
#pragma unroll
                    for (int a = 0; a < NA; ++a) {
                        const unsigned ax = L.axis0 + a;
                        H->x[ax] = Y.xi[a];  H->x[3 + ax] = Y.xa[a];
                        H->v[ax] = Y.vi[a];  H->v[3 + ax] = Y.va[a];
                        H->A1[ax] = Y.Ai[a]; H->A1[3 + ax] = Y.Aa[a];
                    }
                    if (L.leader) {
                        const bool carried = (flags & IA_CARRIED) != 0u;
                        const unsigned attempts = att0 + iters;
                        H->tf = tf; H->h = h; H->phase = phase; H->s_old = s_old;
                        H->r2_cur = outside ? P.r0sq : 0.0; /* only whether it is beyond r0 matters (R7) */
                        H->t_first = t_first; H->t_last = t_last; H->slot = slot;
                        /* a trajectory of a pipelined host run leaves with the HOST address of its record array */
                        const bool to_host = !carried && S.late_dst != nullptr;
                        H->records = to_host ? S.late_dst : out_rec;
                        H->flags = to_host ? IA_HAND_LATE : (flags & IA_HAND_LATE);
                        H->summary = out_sum;
                        H->n_per = n_per; H->n_coll = n_coll; H->n_tp = n_tp;
                        H->steps_acc = steps_acc; H->steps_rej = attempts - steps_acc; H->failed = failed ? 1u : 0u;
                        /* steps taken before the first hand-over */
                        H->steps_in = carried ? steps_in : attempts;
                        if (SRC != IA_SRC_QUEUE && O.summary != nullptr)
                            atomicAdd((unsigned long long *)&O.summary->steps_kernel,
                                      (unsigned long long)(attempts - steps_entry));
                    }
                    mode = MODE_IDLE;
                }
            }
        }
        if (!__any_sync(IA_FULL, mode != MODE_IDLE)) {
            if (wexh) break;
            continue;
        }

        /* ---- the step loop proper: up to IA_INNER attempts without looking at the counter, the queues or the
         * budget; it is left as soon as a trajectory of the warp terminates.  Everything that is only needed
         * between two visits here stays out of its registers. ---- */
        int fin;          /* >= 0: terminate with this status (0: at the localised exit, i.e. at state N) */
        double &t_fin = sh.t_fin[threadIdx.x]; /* written when a trajectory ends: kept out of the loop's registers */
        IaVec<LPT> N;
        unsigned it = 0;
        /* R5, status 4: the loop never takes a trajectory past max_steps attempts.  Attempts are not counted per
         * step: a running trajectory makes one per iteration of its warp, so their number is att0 + iters. */
        unsigned inner = IA_INNER;
        {
            unsigned long long left = ~0ull;
            if (mode == MODE_RUN) {
                const unsigned long long done = (unsigned long long)(att0 + iters);
                left = P.max_steps > done ? P.max_steps - done : 1ull;
            }
            inner = __reduce_min_sync(IA_FULL, (unsigned)(left < (unsigned long long)IA_INNER ? left : IA_INNER));
        }
        do {
        /* one DP5(4) attempt for every lane (idle lanes step a harmless dummy state) */
        const bool run = (mode == MODE_RUN), loc = (mode == MODE_LOC);
        /* clip the last step to land on t_max (R5/R8): only within the last two rf periods */
        bool last = false;
        if (run && n_per >= P.n_near) {
            const double rem = (P.t_max_rf - (double)n_per) * P.T_rf - tf;
            last = h >= rem;
            h = last ? rem : h;
        }
        IaStepOut so;
        ia_dp5_attempt<LPT, true>(P, L, Y, tf, phase, h, N, so);

        /* ---- controller (R5): straight-line selects; everything that happens once per bounce or per trajectory
         * (turning points, exit, localisation, termination) sits in one branch ---- */
        const double hs = h; /* the step just attempted */
        const double denr = P.rtol * so.err.den;
        const bool accept = so.finite && (so.err.num <= denr);
        /* 0.8 (rtol/err)^(1/5).  err = 0 (or below 2^-126 rtol) gives a huge factor and err = NaN or inf gives NaN or 0:
         * ia_min / ia_max below cap the former at 5 and return their second operand for NaN, i.e. growth by 5 and
         * shrinkage by 10 as the step law says.  A step that is not finite shrinks by 10 whatever its error norm reads
         * (a NaN in a component the norm's maxima drop must not let the step grow). */
        const double fac0 = 0.8 * ia_inv_fifth_root(so.err.num * ia_rcp(denr));
        const double fac = so.finite ? fac0 : 0.1;
        const bool acc = run && accept, rej = run && !accept;
        steps_acc += acc ? 1u : 0u;
        const bool neg_new = so.s_new < 0.0;
        const bool flip = acc && (neg_new != s_neg); /* events (R6): sign changes of s = d.w at accepted-step ends */
        /* exit (R7): first upward crossing of |d| = r0 */
        const bool exitc = acc && (so.r2n > P.r0sq) && (so.s_new > 0.0);
        const bool commit = acc && !exitc;
        fin = -1;
        if (flip || exitc || loc || (commit && last) || (rej && hs <= P.h_min)) {
            const double now = (double)n_per * P.T_rf + tf; /* t_n: nothing is committed yet */
            if (flip) {
                ++n_tp;
                if (s_neg && so.r2n < P.rcsq) { /* a minimum of r(t) at short range: a bounce */
                    const double s_prev = s_old;
                    const double tc = now + (hs * s_prev) * ia_rcp(s_prev - so.s_new);
                    if (n_coll == 0u) t_first = tc;
                    t_last = tc;
                    ++n_coll;
                }
            }
            if (exitc || loc) {
                /* localisation by bracketed Newton on g(hk) = |d(t_n + hk)|^2 - r0^2 over uncontrolled steps from
                 * (t_n, y_n).  A trajectory that was already outside at t_n (a thermal start beyond r0 that never
                 * came in) has no crossing to localise: it ends with the detecting step */
                const double g = so.r2n - P.r0sq;
                const bool g_small = fabs(g) <= P.loc_tol;
                bool fin_exit;
                if (loc) {
                    ++n_loc;
                    fin_exit = g_small || n_loc >= 60u;
                } else {
                    fin_exit = g_small || outside;
                }
                if (!fin_exit) {
                    /* Newton kept inside the bracket [lo, hi] of step sizes: g(hi) > 0 is known, lo = 0 where the
                     * trajectory was still inside.  A proposal that leaves the bracket (near-tangential exit,
                     * d.w ~ 0) is replaced by the midpoint -- one uncontrolled step of many rf periods would blow
                     * the ion's state up.  NaN compares false and ends in the midpoint too. */
                    double lo = 0.0, hi = hs;
                    if (exitc) {
                        n_loc = 0u;
                    } else {
                        lo = sh.loc_lo[threadIdx.x];
                        hi = sh.loc_hi[threadIdx.x];
                        if (g > 0.0) hi = hs; else lo = hs;
                    }
                    double hn = hs - g * ia_rcp(2.0 * so.s_new);
                    if (!(so.s_new > 0.0 && hn > lo && hn < hi)) hn = 0.5 * (lo + hi);
                    h = hn; /* neither accepted-and-committed nor rejected: the step law below leaves it alone */
                    sh.loc_lo[threadIdx.x] = lo;
                    sh.loc_hi[threadIdx.x] = hi;
                    mode = MODE_LOC;
                } else {
                    /* a localisation step that is not finite (unreachable from a finite accepted step, since it only
                     * shortens it) must not leave as an escape with a non-finite energy: status 3 at the last state */
                    fin = so.finite ? 0 : 3;
                    t_fin = so.finite ? now + hs : now;
                }
            }
            if (fin == 0 || fin == 3) {
                /* ended at the localised exit (or with a localisation step that is not finite) */
            } else if (commit && last) {
                fin = 1;
                t_fin = P.t_max;
            } else if (rej && hs <= P.h_min) {
                fin = 2;
                t_fin = now;
            }
        }
        /* commit the accepted step: y <- ynew, k1 <- k7 (FSAL), t <- t + h with the time kept folded (R9) */
        {
            const double tfn = tf + hs;
            tf = commit ? tfn : tf;
            if (commit && tfn >= P.T_rf) {
                tf = tfn - P.T_rf;
                ++n_per;
            }
#pragma unroll
            for (int a = 0; a < NA; ++a) {
                Y.xi[a] = commit ? N.xi[a] : Y.xi[a];
                Y.xa[a] = commit ? N.xa[a] : Y.xa[a];
                Y.vi[a] = commit ? N.vi[a] : Y.vi[a];
                Y.va[a] = commit ? N.va[a] : Y.va[a];
                Y.Ai[a] = commit ? N.Ai[a] : Y.Ai[a];
                Y.Aa[a] = commit ? N.Aa[a] : Y.Aa[a];
            }
            if (commit) s_old = so.s_new; /* its value is read at the next bounce only; its sign is s_neg */
            s_neg = commit ? neg_new : s_neg;
            outside = commit ? (so.r2n >= P.r0sq) : outside;
        }
        /* step size of the next attempt (R5) */
        {
            const double h_acc = ia_min(failed ? hs : hs * ia_min(fac, 5.0), P.h_max);
            const double h_rej = ia_max(failed ? 0.5 * hs : hs * ia_max(fac, 0.1), P.h_min);
            h = commit ? h_acc : (rej ? h_rej : h);
            failed = commit ? false : (rej ? true : failed);
        }
        ++it;
        } while (!__any_sync(IA_FULL, fin >= 0) && it < inner);
        cnt += it;
        iters += it;
        if (fin < 0 && mode == MODE_RUN && (unsigned long long)(att0 + iters) >= P.max_steps) {
            fin = 4;
            t_fin = (double)n_per * P.T_rf + tf;
        }

        if (__any_sync(IA_FULL, fin >= 0)) {
            {   /* iterations per finished trajectory, running mean with weight 1/4 (for the refill rule above) */
                const unsigned nf = (unsigned)__popc(__ballot_sync(IA_FULL, fin >= 0 && L.leader));
                const unsigned per = 16u * min(iters - sh.last_fin[threadIdx.x], 4096u) / max(nf, 1u);
                sh.per_fin[threadIdx.x] = (3u * sh.per_fin[threadIdx.x] + per) >> 2;
                sh.last_fin[threadIdx.x] = iters;
            }
            /* observables (R10) + record (a10) + ensemble reduction (a11); the velocity vectors of the
             * terminating state are gathered by the whole warp, the group leader writes */
            double wi[NA], wa[NA], VI[3], VA[3];
#pragma unroll
            for (int a = 0; a < NA; ++a) {
                wi[a] = (fin == 0) ? N.vi[a] : Y.vi[a];
                wa[a] = (fin == 0) ? N.va[a] : Y.va[a];
            }
            ia_gather3<LPT>(L, wi, VI);
            ia_gather3<LPT>(L, wa, VA);
            if (fin >= 0) {
                if (L.leader) {
                    const double ke = (0.5 * P.m_i) * ia_dot3<true>(VI, VI);
                    const bool carried = (flags & IA_CARRIED) != 0u;
                    const unsigned steps_rej = att0 + iters - n_loc - steps_acc; /* attempts that were not accepted */
                    if (out_rec != nullptr) {
                        ia_record r;
                        r.ke_ion = ke;
                        r.t_dwell = t_fin;
                        r.t_life = (n_coll >= 2u) ? (t_last - t_first) : 0.0;
                        r.va_f[0] = VA[0]; r.va_f[1] = VA[1]; r.va_f[2] = VA[2];
                        r.n_coll = n_coll;
                        r.n_tp = n_tp;
                        r.steps_acc = steps_acc;
                        r.steps_rej = (uint16_t)min(steps_rej, 65535u);
                        r.status = (uint8_t)fin;
                        r.n_loc = (uint8_t)n_loc;
                        if (flags & IA_HAND_LATE) {
                            const unsigned long long k = atomicAdd(S.n_late, 1ull);
                            if (k < S.late_cap) {
                                S.late[k].rec = r;
                                S.late[k].dst = out_rec + slot;
                            } else {
                                atomicOr(S.fault, 2ull);
                            }
                        } else {
                            out_rec[slot] = r;
                        }
                    }
                    if (SRC != IA_SRC_QUEUE && O.summary != nullptr)
                        atomicAdd((unsigned long long *)&O.summary->steps_kernel,
                                  (unsigned long long)(steps_acc + steps_rej + n_loc - steps_entry));
                    if (S.n_fin != nullptr) atomicAdd(S.n_fin, 1ull);
                    if (out_sum != nullptr) {
                        ia_summary *Sm = out_sum;
                        atomicAdd((unsigned long long *)&Sm->n_done, 1ull);
                        atomicAdd((unsigned long long *)&Sm->n_status[fin], 1ull);
                        if (n_coll >= 2u) atomicAdd((unsigned long long *)&Sm->n_complex, 1ull);
                        atomicAdd((unsigned long long *)&Sm->steps_acc, (unsigned long long)steps_acc);
                        atomicAdd((unsigned long long *)&Sm->steps_rej, (unsigned long long)steps_rej);
                        atomicAdd((unsigned long long *)&Sm->steps_loc, (unsigned long long)n_loc);
                        if (carried) {
                            atomicMax((unsigned long long *)&Sm->t_end_ns, ia_globaltimer());
                            atomicAdd((unsigned long long *)&Sm->n_handoff, 1ull);
                            atomicAdd((unsigned long long *)&Sm->steps_coop,
                                      (unsigned long long)(steps_acc + steps_rej - steps_in + n_loc));
                        }
                        if (fin == 0) {
                            atomicAdd(&Sm->sum_ke, ke);
                            atomicAdd(&Sm->sum_ke2, ke * ke);
                        }
                        const int bin = (n_coll == 0u) ? 0 : min(32 - __clz(n_coll), IA_HIST_BINS - 1);
                        atomicAdd((unsigned long long *)&Sm->hist_ncoll[bin], 1ull);
                        if (n_coll >= 2u) { /* lifetime of the complex, quarter-octave bins of t_life / T_rf (R17) */
                            const double q = (t_last - t_first) / P.T_rf;
                            const double q2 = q * q;
                            const double q4 = q2 * q2;
                            const int e = ((__double2hiint(q4) >> 20) & 0x7ff) - 1023;
                            atomicAdd((unsigned long long *)&Sm->hist_tlife[max(0, min(e + 8, IA_LIFE_BINS - 1))], 1ull);
                        }
                    }
                }
                mode = MODE_IDLE;
            }
        }
    }
    if (O.summary != nullptr && lane == 0) {
        const unsigned long long t1 = ia_globaltimer();
        atomicMax((unsigned long long *)&O.summary->t_end_ns, t1);
        if (!resume) atomicMax((unsigned long long *)&O.summary->t_bulk_end_ns, t1);
        if (!resume && LPT == 1)
            atomicAdd((unsigned long long *)&O.summary->slots_bulk, (unsigned long long)iters * PER_WARP);
    }
}

/* ---- K3: verification kernels (BASELINE.json north_star: fixed-step mode, fmad off) ------------ */

/* n independent uncontrolled steps: the one-step map of reading R12(i).  With LPT = 3 a warp takes ten
 * states; every lane runs the step (shuffles) and lanes without a state of their own recompute one. */
template <int LPT, bool FUSED>
__global__ void ia_step_map_kernel(const __grid_constant__ IaParams P, unsigned long long n, const double *t_frac,
                                   const double *phase, const double *y, const double *h, double *ynew,
                                   double *err_out) {
    constexpr int NA = 3 / LPT;
    const unsigned lane = threadIdx.x & 31u;
    const IaLane<LPT> L = ia_make_lane<LPT>(P, lane);
    const unsigned long long warp = ((unsigned long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const unsigned per_warp = (LPT == 1) ? 32u : 10u;
    unsigned long long j = warp * per_warp + (LPT == 1 ? lane : L.gbase / 3u);
    const bool mine = L.valid && (j < n);
    if (j >= n) j = n - 1;
    IaVec<LPT> Y, N;
#pragma unroll
    for (int a = 0; a < NA; ++a) {
        const unsigned ax = L.axis0 + a;
        Y.xi[a] = y[j * 12 + ax];     Y.xa[a] = y[j * 12 + 3 + ax];
        Y.vi[a] = y[j * 12 + 6 + ax]; Y.va[a] = y[j * 12 + 9 + ax];
    }
    const double tf = t_frac[j], ph = phase[j];
    double D[3], r2, s;
    ia_accel<LPT, FUSED>(P, L, Y.xi, Y.xa, ia_cos_folded(ia_fma<FUSED>(P.omega, tf, ph)), Y.Ai, Y.Aa, D, r2, s);
    IaStepOut so;
    ia_dp5_attempt<LPT, FUSED>(P, L, Y, tf, ph, h[j], N, so);
    if (!mine) return;
#pragma unroll
    for (int a = 0; a < NA; ++a) {
        const unsigned ax = L.axis0 + a;
        ynew[j * 12 + ax] = N.xi[a];     ynew[j * 12 + 3 + ax] = N.xa[a];
        ynew[j * 12 + 6 + ax] = N.vi[a]; ynew[j * 12 + 9 + ax] = N.va[a];
    }
    if (err_out != nullptr && L.leader)
        err_out[j] = so.finite ? so.err.num / so.err.den : __longlong_as_double(0x7ff8000000000000ll);
}

/* nsteps uncontrolled steps of one trajectory, every state written out (reading R12(ii)); one warp,
 * every group integrates the same trajectory and group 0 writes */
template <int LPT, bool FUSED>
__global__ void ia_trace_kernel(const __grid_constant__ IaParams P, IaY12 y0, double phase, double h,
                                unsigned nsteps, double *states) {
    constexpr int NA = 3 / LPT;
    const unsigned lane = threadIdx.x & 31u;
    const IaLane<LPT> L = ia_make_lane<LPT>(P, lane);
    const bool writer = (lane < (unsigned)LPT);
    IaVec<LPT> Y, N;
#pragma unroll
    for (int a = 0; a < NA; ++a) {
        const unsigned ax = L.axis0 + a;
        Y.xi[a] = ia_sel3(y0.y[0], y0.y[1], y0.y[2], ax);  Y.xa[a] = ia_sel3(y0.y[3], y0.y[4], y0.y[5], ax);
        Y.vi[a] = ia_sel3(y0.y[6], y0.y[7], y0.y[8], ax);  Y.va[a] = ia_sel3(y0.y[9], y0.y[10], y0.y[11], ax);
    }
    double tf = 0.0;
    unsigned n_per = 0;
    auto store = [&](unsigned row, double t) {
        if (!writer) return;
        double *o = states + (unsigned long long)row * 13;
        if (L.leader) o[0] = t;
#pragma unroll
        for (int a = 0; a < NA; ++a) {
            const unsigned ax = L.axis0 + a;
            o[1 + ax] = Y.xi[a]; o[4 + ax] = Y.xa[a]; o[7 + ax] = Y.vi[a]; o[10 + ax] = Y.va[a];
        }
    };
    store(0, 0.0);
    double D[3], r2, s;
    ia_accel<LPT, FUSED>(P, L, Y.xi, Y.xa, ia_cos_folded(phase), Y.Ai, Y.Aa, D, r2, s);
    for (unsigned n = 0; n < nsteps; ++n) {
        IaStepOut so;
        ia_dp5_attempt<LPT, FUSED>(P, L, Y, tf, phase, h, N, so);
        tf += h;
        if (tf >= P.T_rf) {
            tf -= P.T_rf;
            ++n_per;
        }
        Y = N;
        store(n + 1, (double)n_per * P.T_rf + tf);
    }
}

/* ---- host launchers ------------------------------------------------------------------------ */

cudaError_t ia_launch_persistent(int lanes_per_traj, const IaParams &P, const IaGen &G, const IaOut &O,
                                 const IaSched &S, int grid_blocks, cudaStream_t st) {
    if (lanes_per_traj == 1) {
        if (S.n_in == nullptr) return cudaErrorInvalidValue; /* the bulk kernel always looks at a queue length */
        ia_persistent_kernel<1, IA_SRC_BOTH><<<grid_blocks, IA_THREADS, 0, st>>>(P, G, O, S);
    } else if (S.q_in != nullptr) {
        ia_persistent_kernel<3, IA_SRC_QUEUE><<<grid_blocks, IA_THREADS, 0, st>>>(P, G, O, S);
    } else {
        ia_persistent_kernel<3, IA_SRC_GEN><<<grid_blocks, IA_THREADS, 0, st>>>(P, G, O, S);
    }
    return cudaGetLastError();
}

cudaError_t ia_persistent_info(int lanes_per_traj, int *blocks_per_sm, int *threads_per_block, int *regs,
                               int *local_bytes) {
    const void *fn = lanes_per_traj == 1 ? (const void *)ia_persistent_kernel<1, IA_SRC_BOTH>
                                         : (const void *)ia_persistent_kernel<3, IA_SRC_QUEUE>;
    cudaFuncAttributes fa;
    cudaError_t e = cudaFuncGetAttributes(&fa, fn);
    if (e != cudaSuccess) return e;
    int nb = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, fn, IA_THREADS, 0);
    if (e != cudaSuccess) return e;
    *blocks_per_sm = nb;
    *threads_per_block = IA_THREADS;
    *regs = fa.numRegs;
    *local_bytes = (int)fa.localSizeBytes;
    return cudaSuccess;
}

cudaError_t ia_launch_generate(const IaParams &P, const IaGen &G, double *ic_dump, cudaStream_t st) {
    const unsigned threads = 128;
    const unsigned long long blocks = (G.n + threads - 1) / threads;
    ia_generate_kernel<<<(unsigned)blocks, threads, 0, st>>>(P, G, ic_dump);
    return cudaGetLastError();
}

cudaError_t ia_launch_step_map(int variant, const IaParams &P, unsigned long long n, const double *t_frac,
                               const double *phase, const double *y, const double *h, double *ynew, double *err,
                               cudaStream_t st) {
    if (n == 0) return cudaSuccess;
    const unsigned threads = 64;
    const unsigned long long per_block = (variant == IA_ARITH_FMA_COOP) ? 20ull : 64ull;
    const unsigned blocks = (unsigned)((n + per_block - 1) / per_block);
    if (variant == IA_ARITH_NOFMA)
        ia_step_map_kernel<1, false><<<blocks, threads, 0, st>>>(P, n, t_frac, phase, y, h, ynew, err);
    else if (variant == IA_ARITH_FMA)
        ia_step_map_kernel<1, true><<<blocks, threads, 0, st>>>(P, n, t_frac, phase, y, h, ynew, err);
    else
        ia_step_map_kernel<3, true><<<blocks, threads, 0, st>>>(P, n, t_frac, phase, y, h, ynew, err);
    return cudaGetLastError();
}

cudaError_t ia_launch_trace(int variant, const IaParams &P, IaY12 y0, double phase, double h, unsigned nsteps,
                            double *states, cudaStream_t st) {
    if (variant == IA_ARITH_NOFMA)
        ia_trace_kernel<1, false><<<1, 32, 0, st>>>(P, y0, phase, h, nsteps, states);
    else if (variant == IA_ARITH_FMA)
        ia_trace_kernel<1, true><<<1, 32, 0, st>>>(P, y0, phase, h, nsteps, states);
    else
        ia_trace_kernel<3, true><<<1, 32, 0, st>>>(P, y0, phase, h, nsteps, states);
    return cudaGetLastError();
}
