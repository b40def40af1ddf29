/*
 * ia_kernels.cuh -- declarations shared by the translation units of libia_b200.so (host side).
 */
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/ia.h"
#include "ia_dev.cuh"

/* generator description as the device sees it (readings R1-R3) */
struct IaGen {
    int mode, domain, phase_mode;
    unsigned n_theta, n_phi;
    unsigned long long n, first_index, seed;
    unsigned cell;
    const double *y0, *phase;
    double phase0;
    double E_min_uK, log_E_ratio; /* E_uK = E_min exp(u4 log(E_max/E_min)); log_E_ratio = 0 -> fixed */
    double E_fixed_au, v0_fixed;  /* fixed-energy case, computed on the host                        */
    double theta_span_pi, phi_span_pi; /* angular spans in units of pi: 0.5/0.5 octant, 1/2 sphere   */
    double sig_r_ion, sig_v_ion, sig_v_atom; /* THERMAL: sqrt(kT_i/m_i)/w_h, sqrt(kT_i/m_i), sqrt(kT_a/m_a) */
};

struct IaOut {
    ia_record *records;
    ia_summary *summary;
    double *ic_dump;
};

/* A finished trajectory whose home record array is HOST memory (a pipelined host run, ia_submit_host): the kernel
 * appends the record and its destination to a ctx-owned list, ia_wait copies the list back and stores every record. */
struct IaLate {
    ia_record rec;
    ia_record *dst; /* host address */
};
static_assert(sizeof(IaLate) == 72, "IaLate is 72 bytes");

#define IA_HAND_LATE 1u /* IaHand.flags: `records` is a host array, the record goes to the late list */

/* A trajectory in flight, as a kernel hands it to the next one (256 bytes). */
struct IaHand {
    double x[6], v[6], A1[6]; /* r_i, r_a | v_i, v_a | FSAL accelerations */
    double tf, h, phase, s_old, t_first, t_last;
    unsigned long long slot;
    unsigned n_per, n_coll, n_tp, steps_acc, steps_rej, failed;
    ia_record *records;  /* where its outcome goes: the outputs of the run it came from, so that one straggler */
    ia_summary *summary; /* kernel can finish the hand-overs of several runs (ia_set_pipeline)                */
    unsigned steps_in;   /* attempted steps before the first hand-over */
    unsigned flags;      /* IA_HAND_LATE */
    double r2_cur;       /* |d|^2 at the current state (decides whether an exit can be localised, R7) */
};
static_assert(sizeof(IaHand) == 256, "IaHand is 256 bytes");

/* where a persistent kernel takes its work from and where unfinished work goes */
struct IaSched {
    unsigned long long *counter;     /* work counter of this launch (zeroed by the host)                 */
    const IaHand *q_in;              /* non-NULL: resume the trajectories of this queue (a level of the straggler
                                        chain: only those; the bulk kernel: those first, then it generates its own) */
    const unsigned long long *n_in;  /* ... their number (device memory, written by the producing kernel) */
    IaHand *q_out;                   /* non-NULL: hand unfinished trajectories over to this queue ...     */
    unsigned long long *n_out;       /* ... counting them here                                           */
    int handoff_lanes;               /* ... once the counter is empty and <= this many trajectories of a warp run */
    unsigned budget;                 /* ... or once it has run this many iterations since the counter ran dry */
    unsigned long long q_cap;        /* capacity of q_out in entries; an entry beyond it is dropped and ...    */
    unsigned long long *fault;       /* ... bit 0 of this word set (bit 1: late list full); checked by ia_debug_check */
    unsigned long long *n_fin;       /* non-NULL: counts the trajectories this kernel finishes; a warp hands over  */
    unsigned long long run_floor;    /* ... also once at most this many of the n_in it resumed are still running   */
    unsigned long long warn;
    IaLate *late;                    /* list of finished trajectories whose records live on the host ...  */
    unsigned long long *n_late;      /* ... its length ...                                                */
    unsigned long long late_cap;     /* ... and capacity                                                  */
    ia_record *late_dst;             /* non-NULL: the records of THIS run's trajectories are wanted in this host
                                        array: a trajectory handed over carries it instead of O.records   */
};

/* where a persistent kernel's trajectories come from */
enum { IA_SRC_GEN = 0,   /* the generator (a2)                                                            */
       IA_SRC_QUEUE = 1, /* a hand-over queue, dealt out by block index (a level of the straggler chain)  */
       IA_SRC_BOTH = 2 };/* a hand-over queue first, then the generator (the bulk kernel)                 */

/* persistent propagation kernels: lanes_per_traj = 1 (bulk) or 3 (straggler / cooperative layout) */
cudaError_t ia_launch_persistent(int lanes_per_traj, const IaParams &P, const IaGen &G, const IaOut &O,
                                 const IaSched &S, int grid_blocks, cudaStream_t st);
cudaError_t ia_persistent_info(int lanes_per_traj, int *blocks_per_sm, int *threads_per_block, int *regs,
                               int *local_bytes);
cudaError_t ia_launch_generate(const IaParams &P, const IaGen &G, double *ic_dump, cudaStream_t st);

/* verification kernels; variant = ia_arith (include/ia.h) */
cudaError_t ia_launch_step_map(int variant, const IaParams &P, unsigned long long n, const double *t_frac,
                               const double *phase, const double *y, const double *h, double *ynew, double *err,
                               cudaStream_t st);
struct IaY12 {
    double y[12];
};
cudaError_t ia_launch_trace(int variant, const IaParams &P, IaY12 y0, double phase, double h, unsigned nsteps,
                            double *states, cudaStream_t st);

/* DFMA peak microbenchmark */
cudaError_t ia_run_fp64_peak(int device, double target_ms, double *tflops, double *elapsed_ms);
/* latency of a dependent DFMA, and of the reciprocal (MUFU.RCP64H + 3 DFMA) plus one DADD, in SM cycles */
cudaError_t ia_run_fp64_latency(int device, double *cycles_dfma, double *cycles_rcp_add);
