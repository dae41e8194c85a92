/* heget-b200: C-ABI of the hot path of arxiv 0909.5257 ("Calculation of QCD processes on GPU"), built for NVIDIA B200.
 *
 * What the path computes (eq. 4; eqs. 7-12): for each phase-space point the helicity-summed,
 * colour-summed and averaged tree-level squared matrix element of a massless-QCD n-jet subprocess
 *
 *      me2 = S * 1/4 * 1/(n_a n_b) * sum_lambda  sum_{alpha,beta} J_alpha^* C_{alpha beta} J_beta ,
 *      J_alpha = sum_l c_{alpha l} A_l(lambda)                       (eqs. 8-10)
 *
 * where A_l are the HELAS-style diagram amplitudes built from ixxxxx/oxxxxx/vxxxxx wavefunctions and the qqg, ggg, gggg
 * vertex functions of the paper's section 4, C is the real symmetric colour matrix of eq. 9, S the
 * identical-particle factor, 1/4 the spin average (eq. 12) and 1/(n_a n_b) the colour average (eq. 9).
 *
 * Conventions shared by every entry point
 *   - plain C, no exceptions cross the boundary; every function that can fail returns heget_status_t and leaves a
 *     message retrievable with heget_last_error() (thread-local);
 *   - pointers named d_* are DEVICE pointers owned by the caller (e.g. torch tensors), pointers named h_* are HOST
 *     pointers owned by the caller; the library never frees or reallocates them;
 *   - work is enqueued asynchronously on `cuda_stream` (a cudaStream_t passed as void*; NULL = the legacy default
 *     stream); the d_* entry points do not synchronise.  The h_* ("host buffer") entry points copy in/out on that
 *     stream and synchronise it before returning;
 *   - momenta are always FP64, laid out structure-of-arrays  mom[(leg*4 + mu)*n_events + e],  mu = (E, px, py, pz) in GeV,
 *     legs = the two initial partons followed by the finals in process-string order;
 *   - there is no CPU fallback: without a CUDA device the compute entry points return HEGET_ECUDA.
 */
#ifndef HEGET_H
#define HEGET_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct heget_process heget_process_t;      /* opaque; created by heget_process_create, freed by heget_destroy */

typedef enum {
    HEGET_OK = 0,
    HEGET_EINVAL = 1,        /* NULL handle / NULL required pointer / malformed argument                       */
    HEGET_EUNSUPPORTED = 2,  /* a syntactically valid process outside massless QCD {g, u, u~}, or too large     */
    HEGET_ECUDA = 3,         /* a CUDA runtime call failed (message holds cudaGetErrorString)                   */
    HEGET_ENOMEM = 4,
    HEGET_ECOMPILE = 5       /* no pre-built kernel for the process and run-time generation/compilation failed  */
} heget_status_t;

/* HEGET_FP32X2: the FP32 arithmetic of HEGET_FP32 (same rounding, same tolerances, float output), executed two helicity
 * configurations per thread on Blackwell's packed f32x2 instructions (FFMA2/FMUL2/FADD2): half the instructions per event.
 * Needs at least one external gluon (the two configurations differ in its helicity), else HEGET_EUNSUPPORTED. */
typedef enum { HEGET_FP64 = 0, HEGET_FP32 = 1, HEGET_FP32X2 = 2 } heget_precision_t;

/* Kernel back end of steps a3-a8.  STRAIGHT: one specialised kernel per process whose helicity body is
 * straight-line code written by the generator and compiled by nvcc (pre-built for the configured processes, else compiled
 * at heget_process_create).  TABLE: generic kernels that interpret the process's table program -- merged sub-currents,
 * closings at the centroid vertex, every sub-current computed once per helicity assignment of its own legs and reused by
 * all configurations (no compiler needed).  AUTO: TABLE for processes with >= 6 external legs, STRAIGHT below. */
typedef enum { HEGET_KERNEL_AUTO = 0, HEGET_KERNEL_STRAIGHT = 1, HEGET_KERNEL_TABLE = 2 } heget_kernel_t;

/* Colour stage of the TABLE back end (step a7, eq. 10): how J^+ C J is formed on the accumulated basis.
 * SYMMETRIC: t_a = C_aa J_a + sum_{b>a} 2 C_ab J_b in register tiles, coefficients streamed as numbers (default).
 * DISTINCT:  the paper's own scheme (Table 4): only the distinct values of the matrix are stored,
 *            an index map (one byte per element) says which value sits where.
 * CHOLESKY:  C = L L^T (rank-revealing: null directions of a semi-definite C drop out), form = |L^T J|^2.
 * TENSOR:    the J vectors of every (event, configuration) go to HBM as rows of X and a second kernel contracts Y = X C on the
 *            tensor cores (FP32: TF32 mma with a 3-term error-compensated split; FP64: DMMA), then sum_a X_a Y_a per row;
 *            at most 128 colour elements; HEL_SUM only; the library keeps the J buffer (<= 1 GiB, events go through it in chunks). */
typedef enum { HEGET_COLOUR_SYMMETRIC = 0, HEGET_COLOUR_DISTINCT = 1, HEGET_COLOUR_CHOLESKY = 2, HEGET_COLOUR_TENSOR = 3 } heget_colour_stage_t;

/* helicity treatment of eq. 12.  SUM: all 2^n_ext configurations (the graded mode, reading A8).
 * SAMPLE: one configuration per event drawn from Philox(seed, global event index), weighted by 2^n_ext -- what the paper
 * itself ran.  FIXED: the single configuration given in `hel` (no weight). */
typedef enum { HEGET_HEL_SUM = 0, HEGET_HEL_SAMPLE = 1, HEGET_HEL_FIXED = 2 } heget_hel_mode_t;

/* jet cuts in the partonic centre-of-mass frame (eqs. 14a, 14b, 15b; reading A9): pT > pt_min [GeV],
 * |eta| < eta_max, Delta R_ij > dr_min for every final pair; a value <= 0 disables that cut. */
typedef struct { double pt_min, eta_max, dr_min; } heget_cuts_t;

typedef struct {
    int n_ext;                 /* external legs                                                                  */
    int n_hel;                 /* 2^n_ext helicity configurations of eq. 12                                       */
    int n_hel_eval;            /* of which not identically zero (massless quark lines conserve chirality)         */
    int n_diagrams;            /* Table 1 convention: a four-gluon vertex counts three times    */
    int n_topologies;          /* plain Feynman-diagram topologies                                                */
    int n_color;               /* colour-basis size in the paper's convention (Table 1)                           */
    int n_color_eval;          /* size of the basis the kernel accumulates J on                                   */
    int n_color_reduced;       /* after merging elements whose J are proportional for every phase-space point     */
    int n_color_accum;         /* dimension J is accumulated on: the span of the diagrams' colour vectors (TABLE), else = n_color_reduced */
    int color_rank;            /* rank of the n_color x n_color colour matrix of eq. 9 (A13: 12 of 40 for u u -> u u g g); -1 if not computed */
    double avg_spin;           /* 1/4                       (eq. 12)                                              */
    double avg_color;          /* 1/(n_a n_b)               (eq. 9)                                               */
    double sym_factor;         /* 1/prod k!                                         */
    double flops_per_event;    /* counted by the generator from the code it emitted, HEL_SUM, FMA = 2             */
    double flops_per_helicity;
    int regs_per_thread;       /* of the kernel variant heget_set_lanes currently selects, this precision         */
    int local_bytes_per_thread;/* stack frame (spills) of the same kernel; 0 = everything stays in registers      */
    int threads_per_block;
    int lanes_wide;            /* helicity lanes per event of the wide kernel variant (see heget_set_lanes)        */
    int lanes;                 /* lanes per event of the variant currently selected                               */
    int kernel;                /* back end the next heget_eval_me2 takes: HEGET_KERNEL_STRAIGHT or HEGET_KERNEL_TABLE */
    int events_per_block;
    int n_hel_computed;        /* configurations the kernel actually evaluates: n_hel_eval, or half of it when the TABLE back end folds the sum by parity (|M|^2 is invariant under flipping every helicity; each evaluated configuration counts twice) */
    int colour_stage;          /* heget_colour_stage_t in use (TABLE back end) */
    int n_color_distinct;      /* distinct non-zero values of the n_color_accum x n_color_accum matrix the kernel contracts */
    int packed_pairs;          /* TABLE back end, FP32: 1 if two events share a warp on packed f32x2 instructions (FFMA2) */
    int j_in_tmem;             /* TABLE back end: 1 if the warps keep their J in tensor memory (TMEM), 0 = shared memory */
    double flops_per_event_tensor; /* flops of the colour stage executed on the tensor pipe (0: vector pipes)        */
    int warps_per_j;           /* TABLE back end: warps that serve one block of J (32 configurations of one event, or of an event pair): 1 = one warp walks the
                                  closing list and updates J; n > 1 = n warps walk the list in turn (colour groups dealt out two at a time) and each applies
                                  its J_k += x_gk S_g when its turn comes, i.e. in the original group order -- the result is bit-identical for every n
                                  (heget_tab.cuh) */
} heget_info_t;

/* Build (or look up) the specialised kernels of one process.
 *   process     "u u~ > g g", "g g > g g g", ...: two initial and >= 2 final partons out of {g, u, u~}   (eq. 3/13)
 *   sqrt_s_hat  partonic centre-of-mass energy in GeV (> 0)                                              (eq. 2)
 *   alpha_s     fixed strong coupling (> 0); g_s = sqrt(4 pi alpha_s)
 *   cuts        may be NULL (no cuts)
 *   out         receives the handle on HEGET_OK; untouched otherwise
 * The kernels of a process come from the pre-built plug-in paper_0909_5257_b200/kernels/heget_<tag>.so if it exists;
 * otherwise the generator runs in-process, nvcc compiles its output for sm_100a and the result is cached there
 * (HEGET_ECOMPILE if nvcc is missing or fails).  Synchronous. */
heget_status_t heget_process_create(const char* process, double sqrt_s_hat, double alpha_s, const heget_cuts_t* cuts,
                                    heget_precision_t prec, heget_process_t** out);

heget_status_t heget_process_info(const heget_process_t* proc, heget_info_t* out);

/* Colour matrix C of eq. 9 WITHOUT the 1/(n_a n_b) average, row-major.
 *   which = 0: n_color x n_color in the paper's basis (Tables 1 and 4);  which = 1: the reduced (merged-basis) matrix;
 *   which = 2: the n_color_accum x n_color_accum congruence B^T C B the TABLE kernels contract (STRAIGHT: same as 1).
 * h_out may be NULL to query the dimension only; *n receives the dimension. */
heget_status_t heget_color_matrix(const heget_process_t* proc, int which, double* h_out, int* n);

/* Steps a1-a2: Philox4x32-10 uniforms -> massless RAMBO momenta in the partonic CM frame -> cuts, re-drawing a failed
 * event with attempt = 0, 1, 2, ... (cap 65536; then weight 0) (readings A7, A9, A17, A18).
 * Event e of this call is global event first_event + e: the result does not depend on how events are sharded.
 *   d_mom     double[n_ext*4*n_events]   required
 *   d_weight  double[n_events] or NULL   flat phase-space weight of the accepted point (0 if the cap was hit)
 *   d_tries   uint32[n_events] or NULL   attempts used
 * n_events == 0 is a no-op returning HEGET_OK. */
heget_status_t heget_sample_momenta(heget_process_t* proc, uint64_t seed, uint64_t first_event, uint64_t n_events,
                                    double* d_mom, double* d_weight, uint32_t* d_tries, void* cuda_stream);

/* Steps a3-a8: me2[e] of eq. 4 for every event.
 *   d_mom   double[n_ext*4*n_events] as written by heget_sample_momenta (any on-shell massless momenta with
 *           p_a + p_b = sum p_final are accepted)
 *   mode    see heget_hel_mode_t;  hel = n_ext entries of +-1 (host pointer) for FIXED, else ignored;
 *           seed/first_event only matter for SAMPLE
 *   d_me2   double[n_events] (HEGET_FP64 handle) or float[n_events] (HEGET_FP32 / HEGET_FP32X2 handle)
 * n_events == 0 is a no-op returning HEGET_OK. */
heget_status_t heget_eval_me2(heget_process_t* proc, const double* d_mom, uint64_t n_events, heget_hel_mode_t mode,
                              const int8_t* hel, uint64_t seed, uint64_t first_event, void* d_me2, void* cuda_stream);

/* The same two steps with HOST buffers: the library stages through a device scratch it owns (grown on demand, freed by
 * heget_destroy), copies on `cuda_stream` and synchronises it before returning; calls on ONE handle from several host
 * threads are serialised by the library (the scratch belongs to the handle).  h_me2 is double[] or float[] per the
 * handle's precision.  Either of h_mom_in / h_mom_out may be NULL:
 *   heget_run_host(.., h_mom_in = NULL, ..)  samples (seed, first_event) on the device, evaluates, returns me2 (and the
 *                                            momenta / weights if h_mom_out / h_weight are non-NULL);
 *   heget_run_host(.., h_mom_in != NULL, ..) uploads the given momenta and evaluates them. */
heget_status_t heget_run_host(heget_process_t* proc, uint64_t seed, uint64_t first_event, uint64_t n_events,
                              const double* h_mom_in, double* h_mom_out, double* h_weight, heget_hel_mode_t mode,
                              const int8_t* hel, void* h_me2, void* cuda_stream);

/* Choose the kernel back end (see heget_kernel_t).  Builds or loads what the choice needs (HEGET_ECOMPILE /
 * HEGET_EUNSUPPORTED as for heget_process_create; the previous choice stays on failure).  HEGET_FP32X2 handles are STRAIGHT only. */
heget_status_t heget_set_kernel(heget_process_t* proc, heget_kernel_t kernel);

/* TABLE back end only: choose the colour stage (see heget_colour_stage_t); takes effect at the next heget_eval_me2. */
heget_status_t heget_set_colour_stage(heget_process_t* proc, heget_colour_stage_t stage);

/* STRAIGHT back end only (TABLE accepts 0 and nothing else).  Choose the kernel variant: `lanes` threads share one event and split its helicity configurations among them.
 * 0 = automatic (FP64: the wide variant, FP32: one event per thread where built, else wide; wide = info.lanes_wide = the largest power of two <= 32 dividing n_hel_eval, so a warp works
 * on 32/lanes events, event-cache reads are broadcasts and the per-event prologue is spread over the lanes);
 * 1 = one event per thread (not built for processes with >= 6 legs); lanes_wide = the wide variant. Else HEGET_EINVAL. */
heget_status_t heget_set_lanes(heget_process_t* proc, int lanes);

void heget_destroy(heget_process_t* proc);          /* NULL is allowed */

const char* heget_last_error(void);                 /* thread-local, valid until the next call on this thread */

/* Measurement aid for the ALU roofline: n_threads threads (a multiple of 256) each run 8 independent
 * register-resident chains of `iters` dependent FMAs in the given precision; *flops receives the flops enqueued
 * (16 * iters * n_threads).  d_out: device array of n_threads elements of that precision.  Not part of the hot path and
 * not counted by heget_launch_count. */
heget_status_t heget_fma_probe(heget_precision_t prec, uint64_t iters, void* d_out, uint64_t n_threads, double* flops,
                               void* cuda_stream);

/* number of kernel launches this library has enqueued since it was loaded (bench.py's gpu_launches) */
uint64_t heget_launch_count(void);

/* ---- An entry point that allocates nothing -------------------------------------------------------------------------------------
 * For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it).
 * heget_eval_me2_static computes what heget_eval_me2(.., HEGET_HEL_SUM, ..) computes with the tensor-core colour stage (eqs. 8-12,
 * the table kernel writes the rows of J, the tensor-core kernel contracts them with the colour matrix, a third kernel
 * sums over helicities), but the scratch between the kernels -- the rows of J and the row forms -- lives in ONE file-scope device array
 * of HEGET_STATIC_SCRATCH_BYTES inside the library instead of in cudaMalloc'ed memory.  Every GPU that loads the library holds that
 * array until the process exits.  The call itself performs no cudaMalloc, cudaFree or allocating library routine: three kernel launches.
 *
 * Set-up (this part allocates, once):  TABLE back end (heget_set_kernel or automatic), heget_set_colour_stage(HEGET_COLOUR_TENSOR),
 * then heget_static_prepare(proc) with the device current -- it uploads the process tables and asks the runtime for the device
 * address of the array (once per device).  A later heget_set_kernel / heget_set_colour_stage that changes the selection undoes it.
 *
 *   d_mom     DEVICE, [n_ext][4][n_events] float64 as for heget_eval_me2 (stride n_events), caller-owned
 *   n_events  at most heget_static_max_events(proc) (C5 FP64: 1083, FP32: 2166; C4 FP64: 5242); more -> HEGET_EINVAL with the limit
 *             in heget_last_error(), nothing launched.  0 is a no-op.
 *   d_me2     DEVICE, [n_events] float64 (FP64 handle) or float32 (FP32 handle), caller-owned
 * Asynchronous on cuda_stream.  All handles and all calls on a device SHARE the array, which keeps the contents of the last call;
 * nothing in it has to start at zero (every element a call reads it has written before), so no clearing is done.  Calls that overlap
 * on the GPU (different streams, or graphs replayed concurrently) race on it: serialise them on one stream.
 * Errors: HEGET_EINVAL (not prepared, size, NULL pointer), HEGET_ECUDA. */
#define HEGET_STATIC_SCRATCH_BYTES (64u << 20)
heget_status_t heget_static_prepare(heget_process_t* proc);
uint64_t heget_static_max_events(const heget_process_t* proc);      /* 0 if the handle is not prepared */
heget_status_t heget_eval_me2_static(heget_process_t* proc, const double* d_mom, uint64_t n_events, void* d_me2, void* cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* HEGET_H */
