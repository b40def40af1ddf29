/*
 * ia.h -- C-ABI boundary of the B200-native batched ion+atom trajectory propagator
 * (the data-parallel hot path of arXiv 2509.15117, Chowdhury & Perez-Rios).
 *
 * What the library computes (citations are /root/reference/PAPER.md lines and DESIGN.md readings):
 *   For each of n independent trajectories it integrates Newton's equations of the Hamiltonian of
 *   Eq. 1-2 -- a Paul-trapped ion and a neutral atom interacting through
 *   V(r) = C8/r^8 - C4/r^4, C4 = alpha/2, C8 = C4^2/(4 De) (BASELINE.json north_star) --
 *   for the twelve variables (r_i, r_a, v_i, v_a) in FP64 atomic units with the adaptive fourth/fifth
 *   order embedded Runge-Kutta pair of refs [22,23] (Dormand-Prince 5(4) with
 *   the ode45 controller, reading R5), from "head-on" initial conditions to
 *   the termination test (R7/R8), and reduces every trajectory on the device to its
 *   scattering observables: final ion kinetic energy, number of short-range
 *   collisions ("bounces") and of r(t) turning points, dwell time, complex lifetime, final atom
 *   velocity (-> outgoing direction, scattering angle, momentum transfer).
 *
 * All of it runs in hand-written sm_100a CUDA kernels.  There is NO CPU fallback: on a machine
 * without a compute-capability-10.x device ia_create fails with IA_EDEVICE.
 *
 * Conventions
 *   - "device" pointers are CUDA device pointers valid on the ctx's device; "host" pointers are
 *     ordinary process memory.  Each argument says which it is.
 *   - The library never allocates, frees or keeps caller memory.  A ctx owns only its own scratch
 *     (work counters, hand-over queues, host-call staging buffers).  Which calls block the host or
 *     allocate is listed at ia_submit_host below.
 *   - Every function returns IA_OK (0) or a negative ia_status; on failure nothing was launched.
 *     A failed *trajectory* is not a call error: see ia_record.status.
 *   - A ctx is not thread-safe.  Two ctxs may run concurrently on different streams.
 *   - ia_destroy waits for the runs still in flight on the ctx.
 */
#ifndef IA_H
#define IA_H
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ia_ctx ia_ctx; /* opaque, owned by the library */

typedef enum {
    IA_OK = 0,
    IA_EINVAL = -1,  /* NULL / non-finite / out-of-range argument                          */
    IA_ENOMEM = -2,  /* host or device allocation of ctx scratch failed                    */
    IA_ECUDA = -3,   /* a CUDA runtime call failed; text in ia_last_error                  */
    IA_EDEVICE = -4  /* no CUDA device, or the device is not compute capability 10.x       */
} ia_status;

/* Species: masses in unified atomic mass units, static dipole polarisability of the
 * atom in atomic units.  C4 = alpha/2. */
typedef struct {
    double m_ion_u, m_atom_u, alpha_au;
} ia_species;

/* Paul trap (Eq. 2): Mathieu parameters a_k, q_k per Cartesian axis k = x,y,z of
 * the ION's coordinates (trap centre = origin) and the rf angular frequency in atomic units.
 * Force on the ion: -(a_k + 2 q_k cos(Omega_rf t + phase)) m_ion Omega_rf^2/4 * r_k. */
typedef struct {
    double a[3], q[3], omega_rf_au;
} ia_trap;

/* Integration controls (readings R4, R5, R6, R8).  Zero in a field selects the default. */
typedef struct {
    double rtol;        /* relative tolerance, in [1e-13, 1e-3]; default 1e-10                       */
    double atol;        /* absolute tolerance (a.u., one scalar for all 12 components); default 1e-12 */
    double t_max_rf;    /* time limit in rf periods; default 1e4                                      */
    double h_max_rf;    /* step-size cap in rf periods, in (0, 0.25]; default 0.25                    */
    double r_coll_a0;   /* a minimum of r(t) counts as a bounce if r < r_coll; default 500 a0         */
    uint64_t max_steps; /* cap on attempted steps per trajectory; default 2^31                        */
} ia_tol;

/* Creates a context for one (species, trap, De, r0, tolerances) cell on CUDA device `cuda_device`.
 * All pointers are host pointers; *out receives the handle.  De_K is the well depth in kelvin
 * (C8 = C4^2/(4 De)), r0_a0 the radius of the start/exit sphere in Bohr radii. */
int ia_create(ia_ctx **out, const ia_species *species, const ia_trap *trap, double De_K, double r0_a0,
              const ia_tol *tol, int cuda_device);

typedef enum {
    IA_IC_EXPLICIT = 0, /* caller supplies y0[n][12] and phase[n]                                  */
    IA_IC_GRID = 1,     /* cell-centred uniform (theta,phi) grid, head-on (R1)      */
    IA_IC_PHILOX = 2,   /* Philox4x32-10(seed; index, cell) directions / phases / energies (R2)     */
    IA_IC_THERMAL = 3   /* thermal run (R18): atom uniform on the r0 sphere with a
                           Maxwell-Boltzmann velocity at T_atom_uK, negated if needed so that v_r < 0; ion
                           position and velocity Gaussian at T_ion_uK in a harmonic trap of frequency
                           |q_x| Omega_rf / 2^(3/2); normal deviates by Box-Muller on Philox blocks 2..6;
                           rf phase as phase_mode says                                              */
} ia_ic_mode;

/* Most launches of the cooperative kernel at the end of a straggler chain (ia_set_chain). */
#define IA_STRAGGLER_LEVELS 12

/* Which kernels propagate a launch.  The bulk kernel runs one lane per trajectory; once the work
 * counter is empty and a warp is down to a few running lanes (ia_set_handoff) it hands them to the
 * cooperative kernel (three lanes per trajectory, a third of the FP64 instructions per lane and
 * step), which finishes the long stragglers at a lower latency per step.  Both run the same
 * arithmetic and give bit-identical records. */
typedef enum {
    IA_PATH_AUTO = 0,      /* bulk kernel, stragglers handed to the cooperative kernel             */
    IA_PATH_BULK_ONLY = 1, /* bulk kernel to the end                                                */
    IA_PATH_COOP_ONLY = 2  /* cooperative kernel from the first step (verification)                */
} ia_path;

/* Initial conditions of one launch.  Trajectory j of the launch (0 <= j < n) has global index
 * first_index + j; its outputs go to slot j. */
typedef struct {
    int32_t mode;          /* ia_ic_mode                                                            */
    int32_t domain;        /* GRID/PHILOX: 0 = one octant, 1 = full sphere            */
    int32_t phase_mode;    /* GRID/PHILOX: 0 = fixed phase0, 1 = uniform in [0,2pi) from Philox      */
    uint32_t n_theta, n_phi; /* GRID: theta_i = (i+1/2) span/n_theta, i = j / n_phi; phi likewise   */
    int32_t path;          /* ia_path: which kernels propagate (0 = the production pair)            */
    uint64_t n;            /* number of trajectories in this launch                                 */
    const double *y0;      /* EXPLICIT: [n][12] = r_i, r_a, v_i, v_a (a.u.); device for ia_run,
                              host for ia_run_host                                                  */
    const double *phase;   /* EXPLICIT: [n] rf phase at t = 0 (rad); same residency as y0           */
    double phase0;         /* fixed rf phase (rad)                                                  */
    double E_min_uK, E_max_uK; /* collision energy E/k_B in microkelvin; equal -> fixed, else
                              log-uniform from Philox (BASELINE.json configs[4])                   */
    uint64_t seed;         /* PHILOX key                                                            */
    uint32_t cell;         /* PHILOX counter word 2 (BASELINE.json configs[2]: Philox(seed,cell,index)) */
    uint64_t first_index;  /* global index of trajectory 0 (GRID: must be 0 <= first_index, the
                              grid position is first_index + j)                                     */
    double T_atom_uK, T_ion_uK; /* THERMAL: bath and ion temperatures in microkelvin (> 0)         */
} ia_launch;

/* Per-trajectory outcome, 64 bytes, little-endian (R6, R7, R10). */
typedef struct {
    double ke_ion;      /* 1/2 m_i |v_i|^2 at termination (E_h)                                     */
    double t_dwell;     /* time from start to termination (a.u.)                                    */
    double t_life;      /* t(last bounce) - t(first bounce) if n_coll >= 2, else 0 (a.u.)           */
    double va_f[3];     /* atom velocity at termination (a.u.)                                      */
    uint32_t n_coll;    /* short-range collisions: minima of r(t) with r < r_coll                   */
    uint32_t n_tp;      /* all turning points of r(t) (sign changes of d.w at accepted steps)       */
    uint32_t steps_acc; /* accepted RK steps                                                        */
    uint16_t steps_rej; /* rejected RK steps, saturating at 65535                                   */
    uint8_t status;     /* 0 escaped (|d| > r0 after closest approach), 1 t_max reached,
                           2 step size underflow, 3 non-finite initial state (or exit-localisation
                           step), 4 max_steps                                                      */
    uint8_t n_loc;      /* exit-localisation iterations used (R7)                                   */
} ia_record;

#define IA_HIST_BINS 32
#define IA_LIFE_BINS 64
/* Ensemble reduction of one launch (R16, R17), 1024 bytes.  The library
 * ACCUMULATES into it: the caller zeroes it before the first launch it should cover -- on the stream the
 * launch is enqueued on, or ordered before it (a zero-fill on another stream races with the kernels). */
typedef struct {
    uint64_t n_done;            /* trajectories finished                                            */
    uint64_t n_status[5];       /* by ia_record.status                                              */
    uint64_t n_complex;         /* n_coll >= 2 (more than a single bounce)             */
    uint64_t steps_acc, steps_rej; /* totals (exact, not saturated); rejected excludes localisation */
    uint64_t steps_loc;         /* extra uncontrolled steps spent localising exits                  */
    double sum_ke, sum_ke2;     /* sum of ke_ion and ke_ion^2 over status == 0 trajectories (R16)    */
    uint64_t hist_ncoll[IA_HIST_BINS]; /* bin 0: n_coll = 0; bin b >= 1: 2^(b-1) <= n_coll < 2^b    */
    uint64_t t_first_idle_ns;   /* %globaltimer when the first lane found the work counter empty    */
    uint64_t t_start_ns, t_end_ns; /* first / last %globaltimer over the warps of both kernels       */
    uint64_t warn;              /* bit 0: 10|V(r0)| >= E_min (PAPER.md:28 asymptotic-start rule)     */
    uint64_t n_handoff;         /* trajectories finished by the cooperative kernel after a hand-over */
    uint64_t steps_coop;        /* attempted steps (incl. localisation) they took there              */
    uint64_t t_bulk_end_ns;     /* last %globaltimer over the warps of the bulk kernel               */
    uint64_t slots_bulk;        /* 32 x (step attempts of every warp of the bulk kernel): attempted steps there /
                                   slots_bulk = the share of lane-steps that advanced a trajectory            */
    uint64_t steps_kernel;      /* attempted steps (incl. localisation) the bulk kernel of THIS run executed,
                                   whichever run their trajectories belong to (ia_set_pipeline: it also advances
                                   what earlier runs left unfinished)                                          */
    uint64_t reserved[11];
    /* Lifetimes of the complexes (n_coll >= 2), quarter-octave bins of q = t_life / T_rf (PAPER.md:34,40,
     * Fig. 2: the fraction of complexes still alive after t is 1 - cumulative sum / n_complex; R17):
     * bin b = clamp(ilogb(((q q) (q q))) + 8, 0, 63), products rounded separately, i.e. bin b holds
     * 2^((b-8)/4) <= q < 2^((b-7)/4): from T_rf/4 in bin 0 to 13 777 T_rf and beyond in bin 63. */
    uint64_t hist_tlife[IA_LIFE_BINS];
} ia_summary;

typedef struct {
    ia_record *records;  /* [n] or NULL                                                            */
    ia_summary *summary; /* one ia_summary or NULL                                                 */
    double *ic_dump;     /* [n][14] = y0[12], phase, E (E_h) as generated, or NULL                 */
} ia_outputs;

/* Enqueues the propagation of one launch on `cuda_stream` (a cudaStream_t; NULL = legacy default
 * stream) and returns without synchronising.  Every pointer inside `launch` and `outputs` is a
 * DEVICE pointer; outputs are valid once the stream has been synchronised by the caller.
 * n = 0 is valid and launches nothing. */
int ia_run(ia_ctx *ctx, const ia_launch *launch, const ia_outputs *outputs, void *cuda_stream);

/* Same computation with HOST buffers: copies launch->y0/phase (EXPLICIT mode) to ctx-owned device
 * staging, runs, copies records / summary / ic_dump back and synchronises.  The host summary is
 * overwritten (not accumulated).  This is the end-to-end entry bench.py times. */
int ia_run_host(ia_ctx *ctx, const ia_launch *launch, const ia_outputs *host_outputs);

/* Pipelining of successive runs.  Trajectory lengths are power-law distributed
 * (PAPER.md:40): the last few trajectories of a launch take 10^3 times longer than the median, and a
 * trajectory is a serial chain of dependent steps.  With depth 0 (the default) every run finishes on its
 * own: bulk kernel, then the straggler chain for what it left, both on the caller's stream.  With depth
 * d > 0 (at most 64) successive runs of the ctx form a pipeline: the bulk kernel of a run hands everything
 * it still holds when its work counter is empty to the bulk kernel of the NEXT run, which resumes those
 * trajectories first and then generates its own -- long trajectories keep living in full warps while new
 * ones keep arriving, and the machine never idles between runs.  Every trajectory in flight carries the
 * output pointers of the run it belongs to.  Only ia_join ends the pipeline: it enqueues ONE straggler
 * chain on `cuda_stream` for what the last bulk kernel left (after d runs without a join the next ia_run
 * does that itself, on its own stream).  The outputs of a pipelined ia_run are therefore complete -- and
 * its buffers may be released -- only after ia_join; the host does not block in either call.  Runs on
 * different streams of one ctx are ordered on the device one after the other (they share the ctx's
 * queues).  ia_set_pipeline blocks until everything in flight on the ctx has finished. */
int ia_set_pipeline(ia_ctx *ctx, int depth);
int ia_join(ia_ctx *ctx, void *cuda_stream);

/* Asynchronous form of ia_run_host: enqueues the copies in, the kernels and the copies back on
 * ctx-owned streams and returns; host buffers must be page-locked for the copies to overlap and stay
 * untouched until ia_wait.  With ia_set_pipeline(d) the submitted runs form a pipeline as above: the
 * records of a run are copied back right behind its bulk kernel, while the next run's bulk kernel works;
 * the few trajectories (at most one per lane of the grid) that outlive their run's bulk kernel report
 * through a ctx-owned list which ia_wait copies back and stores into the host arrays.
 *   ia_sync blocks the host until every kernel and copy enqueued so far has finished, without ending
 *           the pipeline (trajectories in flight stay in flight; their records and the summaries are not
 *           final yet).
 *   ia_wait ends the pipeline (the straggler chain), brings back summaries and late records, and blocks
 *           until every run submitted on this ctx (either way) has finished.
 * Blocking and allocation: ia_create, ia_set_pipeline, ia_wait, ia_sync, ia_run_host, ia_get_timing and
 * ia_destroy block the host.  ia_submit_host blocks only when it has to grow a staging buffer, when
 * d runs are open or when 64 summaries are pending (it then does an ia_wait first); it allocates
 * ctx-owned device staging (three buffers of the largest run's size) and, pipelined, a late-record list
 * in device and page-locked host memory (IA_ENOMEM).  ia_run, ia_join, ia_generate, ia_step_map and
 * ia_trace never block, allocate or synchronise.  The library reads no environment variables. */
int ia_submit_host(ia_ctx *ctx, const ia_launch *launch, const ia_outputs *host_outputs);
int ia_sync(ia_ctx *ctx);
int ia_wait(ia_ctx *ctx);

/* Generator only (R1-R3): ic_dump is a DEVICE buffer [n][14]. */
int ia_generate(ia_ctx *ctx, const ia_launch *launch, double *ic_dump, void *cuda_stream);

/* Arithmetic variants of the verification entry points. */
typedef enum {
    IA_ARITH_NOFMA = 0,   /* every product and sum rounded separately ("fmad off")                  */
    IA_ARITH_FMA = 1,     /* production arithmetic, one lane per trajectory (bulk kernel layout)     */
    IA_ARITH_FMA_COOP = 2 /* production arithmetic, three lanes per trajectory (cooperative layout) */
} ia_arith;

/* Verification entry points (BASELINE.json north_star: "fixed-step mode built with fmad off").
 * variant is an ia_arith; IA_ARITH_FMA and IA_ARITH_FMA_COOP give bit-identical results.
 *
 * ia_step_map: n independent single uncontrolled DP5(4) steps.  DEVICE arrays t_frac[n] (time folded
 * into [0,T_rf), R9), phase[n], y[n][12], h[n] in; ynew[n][12] and err[n] (the ode45 error norm of the
 * step, R5) out.  err may be NULL.
 * ia_trace: nsteps uncontrolled steps of size h from y0[12] (HOST pointer) with rf phase `phase`;
 * states is a DEVICE buffer [nsteps+1][13] = (t, y) rows, row 0 the start. */
int ia_step_map(ia_ctx *ctx, uint64_t n, const double *t_frac, const double *phase, const double *y,
                const double *h, double *ynew, double *err, int variant, void *cuda_stream);
int ia_trace(ia_ctx *ctx, const double *y0_host, double phase, double h, uint32_t nsteps, double *states,
             int variant, void *cuda_stream);

/* Derived constants as the device sees them (host pointer, 16 doubles):
 * m_i, m_a, C4, C8, De, r_e, Omega, T_rf, thr, h_max, h_min, t_max, r0, r_coll, rtol, atol. */
int ia_get_derived(const ia_ctx *ctx, double *out16);

/* Launch geometry of ia_run on this ctx (host pointers): resident warps per SM, SM count,
 * registers per thread and local-memory bytes per thread (0: no stack frame, no spills) of persistent
 * kernel `kernel`: 0 bulk (one lane per trajectory), 1 cooperative (the straggler chain's instance). */
int ia_get_kernel_info(const ia_ctx *ctx, int kernel, int *warps_per_sm, int *n_sm, int *regs_per_thread,
                       int *local_bytes_per_thread);

/* Hand-over threshold of IA_PATH_AUTO: a warp of the bulk kernel hands its running lanes over once
 * the work counter is empty and at most `lanes` of them (0..32) still run -- or, whatever their number,
 * 4096 step attempts after the counter ran dry; 0 = never hand over (the default is 16: the cooperative
 * kernel with ten trajectories per warp does the work of ~18 bulk lanes). */
int ia_set_handoff(ia_ctx *ctx, int lanes);

/* The straggler chain moves what a bulk kernel left unfinished into ever fewer warps, because
 * the latency of a step falls with the number of warps that share an SM sub-partition: the bulk kernel over a
 * full grid until at most 128 x #SM trajectories run, the bulk kernel with one warp per sub-partition until at
 * most 40 x #SM run, then the cooperative kernel with one warp per sub-partition, `levels` times in a row
 * (1..IA_STRAGGLER_LEVELS; default 1: one launch finishes everything).  With levels > 1, cooperative level
 * j = 0, 1, ... runs until its queue is empty and then for budget << j further iterations per warp (default
 * 8192, at least 64); what still runs then goes to the next level, which packs it ten trajectories to a warp
 * again; the last level keeps everything.  Applies to the chains enqueued afterwards. */
int ia_set_chain(ia_ctx *ctx, int levels, uint32_t budget);

/* Device times of a run of this ctx, from CUDA events the library records around its kernels: the run's
 * bulk kernel, and the straggler chain that ended the pipeline the run was part of (shared by all runs
 * since the join before; 0 for a run that needed none), in ms.  runs_back = 0 is the most recent run, 1
 * the one before ...; the last 256 runs and 8 chains are on record, a pipelined run only once its chain
 * has been enqueued (IA_EINVAL otherwise).  Synchronises with the end of that run.  Host pointers.
 * ia_get_last_timing(ctx, ...) = ia_get_timing(ctx, 0, ...). */
int ia_get_timing(ia_ctx *ctx, int runs_back, double *bulk_ms, double *coop_ms);
int ia_get_last_timing(ia_ctx *ctx, double *bulk_ms, double *coop_ms);

/* FP64 FMA peak microbenchmark (the roofline denominator): runs independent DFMA chains on every SM
 * of `cuda_device` for about `target_ms` and reports the sustained rate.  Host pointers.
 * tflops = 2 * DFMA/s / 1e12; elapsed_ms = CUDA-event time of the timed launch. */
int ia_fp64_peak(int cuda_device, double target_ms, double *tflops, double *elapsed_ms);

/* Latency microbenchmark behind the numbers DESIGN.md "Tail" argues from (measured on B200: 8 cycles per dependent DFMA,
 * 39 per reciprocal + DADD; profiles/r02_summary.md section 4 -- the lone warp of the straggler chain is bound by its
 * in-order instruction stream, not by the step's arithmetic chain): one warp, one dependent chain.
 * cycles_dfma = SM cycles per dependent DFMA; cycles_rcp_add = SM cycles per reciprocal as the right-hand side
 * computes it (MUFU.RCP64H and three dependent DFMA) followed by one dependent DADD.  Host pointers. */
int ia_fp64_latency(int cuda_device, double *cycles_dfma, double *cycles_rcp_add);

/* Debugging aid (compute-sanitizer is not available on every machine): every device buffer a ctx owns -- hand-over
 * queues, counters, summaries and records staged for the host entry points, the late-record list -- is allocated
 * with 4 KiB guard zones of a known byte pattern on either side, and the kernels refuse to write a queue or list
 * entry beyond the capacity they were given, setting a fault word instead.  ia_debug_check blocks until the ctx's
 * work in flight has finished, then verifies every guard zone, the fault word and the device-side counts
 * (IA_ECUDA / IA_EINVAL with the finding in ia_last_error). */
int ia_debug_check(ia_ctx *ctx);

/* ia_run_static -- one launch of the production kernel pair for callers that must not allocate device memory.
 *
 * Who needs it.  Every other way into this library goes through ia_create, which takes its work counters and
 * hand-over queues from cudaMalloc.  Some hosts of this code cannot do that: a plug-in running inside an application
 * whose own pool allocator has already claimed the GPU's memory (a cudaMalloc next to it fails, or fragments the
 * pool), and a control loop that launches between other streams' work and cannot afford the device-wide
 * synchronisation cudaMalloc / cudaFree imply.  For them this call needs no ctx and calls no cudaMalloc, cudaFree,
 * cudaMallocHost or any other allocating routine, on any call: its scratch (six counter words and a hand-over queue
 * of IA_STATIC_MAX_N entries of 256 bytes, 4 MiB + 256 bytes in all) is a static array inside the library's device
 * image.  Every GPU the process loads the library on carries those 4 MiB from the moment the module is loaded until
 * the process exits, used or not; that is the price, and why the limit is modest.
 *
 * What it computes.  Exactly what ia_create + ia_run(IA_PATH_AUTO, no pipeline) compute for the same cell and
 * launch: the bulk kernel (one lane per trajectory) propagates, hands what still runs in a drained warp to the
 * queue, and one launch of the cooperative kernel (three lanes per trajectory) finishes it.  Records are
 * bit-identical to ia_run's; the summary is accumulated into, as there (zero it first, on `cuda_stream`).
 * species / trap / De_K / r0_a0 / tol are ia_create's arguments (HOST pointers, tol may be NULL), launch and
 * outputs are ia_run's (the structs are HOST memory, every pointer inside them a DEVICE pointer on `cuda_device`:
 * the caller still owns and passes all inputs and outputs).  launch->path must be IA_PATH_AUTO.  Enqueues a
 * 256-byte memset and two kernels on `cuda_stream` and returns without synchronising; makes `cuda_device` the
 * calling thread's current device.  n = 0 is valid and launches nothing.
 *
 * Limit.  launch->n <= IA_STATIC_MAX_N (the queue holds one entry per trajectory of the launch).  A larger launch
 * is refused with IA_EINVAL before anything is enqueued, and the text says so; cut it into several calls on one
 * stream (first_index advances), or use ia_create / ia_run.
 *
 * First call on a device.  It looks up the device address of the static array and the launch geometry of the two
 * kernels (which makes the CUDA runtime load the library's kernels onto that device) and keeps both for the
 * process's lifetime; later calls on that device only launch.  Make that first call during start-up, outside any
 * stream capture and before the phase in which allocation is forbidden.
 *
 * Sharing.  All calls on a device use the same array.  The call clears the counter words it needs on
 * `cuda_stream` before its kernels; the queue keeps whatever the previous call left and is never read beyond what
 * the current call wrote.  Two calls whose kernels can overlap on the GPU -- different streams without an event
 * between them, or two host threads -- race on the counters and corrupt each other's results: keep all calls of a
 * device on one stream, or order them with events.  The host side of the call is thread-safe.
 *
 * Errors.  IA_EINVAL / IA_EDEVICE / IA_ECUDA as elsewhere; errbuf (HOST, may be NULL) receives at most
 * errbuf_len - 1 characters of explanation and a terminating NUL -- "" on plain success, the PAPER.md:28
 * asymptotic-start warning when that applies.  On failure nothing was enqueued. */
#define IA_STATIC_MAX_N 16384
int ia_run_static(const ia_species *species, const ia_trap *trap, double De_K, double r0_a0, const ia_tol *tol,
                  int cuda_device, const ia_launch *launch, const ia_outputs *outputs, void *cuda_stream,
                  char *errbuf, size_t errbuf_len);

int ia_destroy(ia_ctx *ctx);
const char *ia_strerror(int code);
const char *ia_last_error(const ia_ctx *ctx); /* "" if none; valid until the next call on ctx */

#ifdef __cplusplus
}
#endif
#endif /* IA_H */
