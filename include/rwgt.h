/* include/rwgt.h — C ABI of the B200-native LO event-reweighting hot path.
 *
 * What it computes (arXiv 2312.07440; citations are /root/reference/PAPER.md lines):
 *   for every stored event, the tree-level squared matrix element |M|^2 under the
 *   original parameter set and |M'|^2 under the modified one, and the new weight
 *        W' = W * |M'|^2 / |M|^2                      (§2.2 eq. 3)
 *   i.e. steps 3-6 of the reweighting procedure of PAPER.md:87 (§3.2), fused into ONE
 *   kernel launch per call.  |M|^2 is a helicity-amplitude evaluation (PAPER.md:66,
 *   §3.1): external wavefunctions, vertex/propagator recursion, colour-flow amplitudes,
 *   colour quadratic form J^dagger C J, helicity sum.  The paper prints none of those
 *   formulas; the conventions are the readings listed in DESIGN.md ("Readings", from
 *   SURVEY.md §8(c) C1-C8), and they are binding because the modified model of the
 *   configs (ggg/gggg couplings rescaled, qqg not) is not gauge invariant (reading Q1).
 *
 * Plain C: no exceptions, no C++/torch types cross this boundary.  All event buffers
 * are DEVICE pointers unless a function says HOST.
 */
#ifndef RWGT_H
#define RWGT_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct rwgt_handle rwgt_handle; /* opaque; owned by the library */

/* One physics parameter set (PAPER.md:87 steps 1 and 4: "Input reweight parameters",
 * "Overwrite physics parameters with new values").  POD, copied by value at create. */
typedef struct {
  double alpha_em;    /* electromagnetic coupling, e = sqrt(4 pi alpha_em)               */
  double alpha_s;     /* strong coupling, g_s = sqrt(4 pi alpha_s)                       */
  double mZ;          /* Z mass, GeV                                                     */
  double GammaZ;      /* Z width, GeV (fixed-width Breit-Wigner s - mZ^2 + i mZ GammaZ)  */
  double sin2_thetaW; /* direct input; cos^2 = 1 - sin^2                                 */
  double mt;          /* top mass, GeV (used in spinors and propagators)                 */
  double Gamma_t;     /* top width, GeV; must be 0 (no config uses it; reading Q7)       */
  double ggg_scale;   /* multiplies the 3-gluon coupling: g_3 = g_s * ggg_scale          */
  double gggg_scale;  /* multiplies the 4-gluon coupling: g_4 = g_s^2 * gggg_scale       */
} rwgt_params;

/* Precision modes of rwgt_set_precision. I/O buffers are FP64 in every mode. */
#define RWGT_FP64 0  /* all arithmetic in double (default)                               */
#define RWGT_FP32 1  /* all per-event arithmetic in float                                */
#define RWGT_MIXED 2 /* float vertex algebra; momentum sums, propagator denominators,
                        helicity/colour accumulation in double                           */

/* Create a handle for one process and one (old, new) pair of parameter sets.
 *   process: "epem_mupmum" | "gg_ttx" | "gg_ttxg" | "gg_ttxgg" | "gg_ttxggg"
 *            | "qqx_ttx" | "qqx_ttxg"   (q qbar -> t tbar (+ g), massless quark, leg order [q,qbar,t,tbar,(g)]: a structurally
 *              different amplitude for the final states of gg_ttx / gg_ttxg; FP64 only)
 *            | "epem_aa" | "epem_aaa" | "epem_aaaa" | "epem_aaaaa"   (e+ e- -> 2..5 photons, leg order [e+, e-, gamma...];
 *              "epem_aaaaa" is the process the paper measured, Table 1; only alpha_em enters; FP64 only)
 *            leg order in `momenta`: [e+,e-,mu+,mu-] resp. [g,g,t,tbar,(g,(g,(g)))];
 *            legs 0,1 incoming, all momenta physical (E>0).
 * Builds the per-process tables (ordered-current schedule, colour matrix) on the host and
 * copies them and the couplings to the CURRENT device; every later call on the handle makes that device current for its
 * duration (and restores the caller's), so streams passed to it must belong to that device.  Returns NULL on error (unknown
 * process, non-positive alpha, sin2_thetaW outside (0,1), Gamma_t != 0, no CUDA device);
 * rwgt_last_error() then describes it.  PAPER.md:87 restricts reweighting to parameters
 * "that can be modified at runtime": old and new share the process. */
rwgt_handle* rwgt_create(const char* process, const rwgt_params* params_old, const rwgt_params* params_new);

/* Several new parameter sets for the same events in one pass (PAPER.md:87 step 7, "Repeat steps 4 - 6 for all parameter
 * sets"; PAPER.md:91 and Fig. 3: run time against the number of parameter sets).  `params_new` points to n_new sets,
 * 1 <= n_new <= RWGT_MAX_SETS.  The event is loaded and its external wavefunctions, momentum sums and propagator
 * denominators are formed ONCE; each set then costs at most one more evaluation of the currents and one more colour form
 * (gg_ttxg: one evaluation serves all sets of equal mass; gg_ttxgg / gg_ttxggg: coupling-only sets beyond the rank of their
 * coupling polynomials cost a colour-form combination each; epem_a...: a multiplication; gg_ttx: two multiply-adds per helicity).
 * Sets may differ in any field; a differing top mass makes the externals of that set be recomputed.
 * rwgt_create(p, old, new) is rwgt_create_multi(p, old, new, 1).  Same error behaviour as rwgt_create. */
#define RWGT_MAX_SETS 16
rwgt_handle* rwgt_create_multi(const char* process, const rwgt_params* params_old, const rwgt_params* params_new, int n_new);

/* Number K of new parameter sets of the handle (1 for rwgt_create); -1 on NULL. */
int rwgt_n_sets(const rwgt_handle* h);

/* 0 on success, -1 on bad handle/mode or a mode the process does not support
 * (epem_mupmum and gg_ttx are FP64 only). */
int rwgt_set_precision(rwgt_handle* h, int mode);

/* Number of external legs (4..7), so callers can size `momenta`; -1 on bad handle. */
int rwgt_n_external(const rwgt_handle* h);

/* Algorithmic floating-point operations per event that the kernel of this handle executes on
 * the FP64 (FP32 in the FP32/mixed modes) FMA pipe: FMA = 2, MUL = ADD = 1, both parameter
 * sets, all helicities.  It is an operation count of the algorithm the kernel runs (for gg -> ttbar g with
 * sets of equal mass the one-pass form, for coupling-only sets of the larger processes the node evaluations of the polynomial mode).
 * In FP64 it is checked against the executed 2 DFMA + DMUL + DADD count of an ncu capture (profiles/counts.json; bench.py prints the
 * ratio); in the FP32 / mixed modes it is the model alone (ncu's FFMA counters do not see the packed FFMA2).  Roofline use.
 * Multiprocess handle: the unweighted mean over the member processes (the mix of an event list is not known before run time);
 * weight the members' own counts (one handle per process) with the list's composition for a roofline figure. */
double rwgt_flops_per_event(const rwgt_handle* h);

/* Algorithmic flops per event of the colour form |L^T J|^2 (step a5), which the engine evaluates with FP64 mma.m8n8k4
 * in every precision mode (0 for the 2->2 kernels, whose colour form is part of rwgt_flops_per_event).  DFMA and DMMA
 * share one pipe on B200, so in FP64 mode the roofline numerator is the sum of the two counts. */
double rwgt_tensor_flops_per_event(const rwgt_handle* h);

/* The hot path: a1-a7 of SURVEY.md §8(a) in one kernel launch on `stream`.
 *   momenta   DEVICE, SoA double [n_ext][4][n_events]: momenta[(ip*4+mu)*n_events + ievt],
 *             mu = (E,px,py,pz), GeV
 *   weights   DEVICE double [n_events]              original weights W
 *   out_me_old, out_me_new  DEVICE double [n_events] |M|^2, |M'|^2, summed over helicities
 *             and colours, averaged over initial helicities/colours and divided by the
 *             identical-particle factor (reading Q3)
 *   out_w_new DEVICE double [n_events]              W' of eq. 3
 *   stream    a cudaStream_t (NULL = default stream).  Work is enqueued; the call does not
 *             synchronise, allocate, or copy between host and device.
 * Outputs must not alias inputs or each other.  Caller owns all buffers.
 * If |M|^2 == 0 (outside the validity condition of PAPER.md:46) the IEEE result of
 * W * (|M'|^2 / |M|^2) is written (inf/nan); no error is raised.
 * Returns 0 on success (n_events == 0 is a no-op), -1 on bad argument (NULL pointer,
 * n_events < 0), otherwise the positive cudaError_t of the launch. */
int rwgt_run(rwgt_handle* h, const double* momenta, const double* weights, double* out_me_old,
             double* out_me_new, double* out_w_new, long long n_events, void* stream);

/* The same launch for a handle with K = rwgt_n_sets(h) new parameter sets:
 *   out_me_new, out_w_new  DEVICE double [K][n_events]: set k at offset k * n_events
 * (out_me_old stays [n_events]).  rwgt_run is this call restricted to K == 1 (it returns -1 for K > 1, so that a
 * caller who sized the outputs for one set cannot be overrun).
 * Ordering: a handle of gg_ttxgg / gg_ttxggg created with three or more coupling-only sets runs in the polynomial mode, whose
 * kernel keeps intermediate colour vectors in device scratch that belongs to the HANDLE (one slice per CTA, allocated at create).
 * Two launches of one such handle that can overlap on the GPU (different streams with no event between them, or two host
 * threads) overwrite each other's scratch and return wrong weights without an error.  Rule for every handle: enqueue the run
 * calls of ONE handle on one stream, or order them with events; use one handle per stream for concurrent launches (handles are
 * independent).  Handles outside the polynomial mode hold no mutable device state in rwgt_run / rwgt_run_multi. */
int rwgt_run_multi(rwgt_handle* h, const double* momenta, const double* weights, double* out_me_old,
                   double* out_me_new, double* out_w_new, long long n_events, void* stream);

/* Same computation with HOST buffers (pageable or pinned): copies the inputs to device
 * scratch owned by the handle (grown on demand), runs the kernel, copies the three outputs
 * back and synchronises `stream`.  The events are processed in up to 8 chunks so that the host->device copy of one
 * chunk, the kernel of the previous one and the device->host copy of the one before overlap (two internal copy
 * streams; the overlap needs pinned host buffers, pageable ones still work).  This is the end-to-end path of
 * bench.py's `e2e` key (host<->device transfer is part of what a user pays).  Same return codes. */
int rwgt_run_host(rwgt_handle* h, const double* momenta, const double* weights, double* out_me_old,
                  double* out_me_new, double* out_w_new, long long n_events, void* stream);

/* rwgt_run_host for K >= 1 new sets: out_me_new, out_w_new are HOST double [K][n_events]. */
int rwgt_run_multi_host(rwgt_handle* h, const double* momenta, const double* weights, double* out_me_old,
                        double* out_me_new, double* out_w_new, long long n_events, void* stream);

/* LO multiprocess (real-emission contributions "can be treated as LO multiprocesses", last sentence:
 * "reweighting between structurally different amplitude routines"): ONE event list whose events belong to different processes with
 * the same number of external legs, e.g. "gg_ttxg,qqx_ttxg".  `processes`: comma-separated names, at most RWGT_MAX_PROCESSES;
 * QCD processes only: the epem_* kernels take no event index list, and an e+ e- sample never shares an event list with a hadronic
 * one, so such a member is refused.  Parameter sets as in rwgt_create_multi, shared by all members.  NULL on error.
 * rwgt_set_precision on such a handle sets the mode of the members that have FP32 / mixed kernels (gg_ttxg, gg_ttxgg, gg_ttxggg);
 * the other members stay FP64, and a mode other than RWGT_FP64 is refused (-1) when no member has one. */
#define RWGT_MAX_PROCESSES 4
rwgt_handle* rwgt_create_multiprocess(const char* processes, const rwgt_params* params_old, const rwgt_params* params_new, int n_new);

/* Number of member processes (1 for a handle of rwgt_create / rwgt_create_multi); -1 on NULL. */
int rwgt_n_processes(const rwgt_handle* h);

/* rwgt_run_multi for a multiprocess handle.  Buffers as in rwgt_run_multi (DEVICE, K = rwgt_n_sets(h)); in addition
 *   process_id  HOST int [n_events]: index of event i's process in the list given at create.
 * The library partitions the event indices by process on the host (stable), copies the index lists to the device on `stream`
 * (4 bytes per event; pinned staging and device list belong to the handle and grow on demand, which allocates and waits for
 * `stream`) and launches one kernel per member process that has events; each kernel reads its events through its index list and
 * writes the outputs at the events' own positions.  Returns 0, -1 (bad argument, id outside the list), or a cudaError_t. */
int rwgt_run_multiprocess(rwgt_handle* h, const double* momenta, const double* weights, const int* process_id, double* out_me_old,
                          double* out_me_new, double* out_w_new, long long n_events, void* stream);

/* eq. 2 (§2.1): "the total cross section is the sum of all event weights", sigma ~ sum_k W_k.  Writes the sum of each
 * of n_rows weight rows to out_sums:
 *   w         DEVICE double [n_rows][n_events], row r at offset r * n_events: the original weights (n_rows = 1) or the
 *             out_w_new of rwgt_run_multi (n_rows = K), i.e. the reweighted cross section of every parameter set
 *   out_sums  DEVICE double [n_rows]
 * 1 <= n_rows <= 1 + RWGT_MAX_SETS.  One kernel launch on `stream`, no atomics in the arithmetic: a fixed block partition and fixed
 * summation trees, so the result depends on the values and n_events only (bitwise reproducible); the relative error against the
 * exact sum is bounded by ~(n_events / 16384 + 30) * 2^-53 * sum|W| / |sum W|.  Uses scratch of the handle: calls on one handle must be
 * stream-ordered.  No allocation, no synchronisation.  Returns 0, -1 on a bad argument, or the cudaError_t of the launch. */
int rwgt_sum_weights(rwgt_handle* h, const double* w, int n_rows, long long n_events, double* out_sums, void* stream);

/* rwgt_sum_weights for callers that are not allowed to allocate device memory.
 *
 * Who that is: a host program that has given all of the GPU's memory to an arena of its own (an event generator or an analysis
 * framework that hands out every device buffer itself: a cudaMalloc from a plug-in library then fails, or takes memory behind the
 * arena's back), and a loop that must not stall (cudaMalloc and cudaFree wait for the whole device, so one call in a side thread
 * stops every stream of the process).  Every other entry point of this library needs a handle, and rwgt_create allocates; this
 * one needs no handle and calls neither cudaMalloc, cudaFree nor any routine that allocates.
 *
 * Same arithmetic as rwgt_sum_weights (eq. 2: sigma ~ sum_k W_k per row; same block partition, same summation trees,
 * so the two return bitwise the same sums).  The caller still owns input and output:
 *   w         DEVICE double [n_rows][n_events], row r at offset r * n_events
 *   out_sums  DEVICE double [n_rows]
 * on the device that is current at the call.  What differs is where the per-block partial sums and the per-row arrival counters
 * live: in a fixed array inside the library image (RWGT_STATIC_SCRATCH_BYTES = 9,216 bytes of global memory on every GPU that has
 * loaded librwgt.so, held until the process exits) instead of a handle's buffers.  That fixes the limit:
 *   1 <= n_rows <= RWGT_STATIC_SUM_MAX_ROWS (17 = 1 + RWGT_MAX_SETS: the old weights and every parameter set in one call);
 * more rows are refused with -1 and a message in rwgt_last_error() (split the rows over several calls).  n_events is not limited.
 *
 * First call on a device: the library looks up the array's device address (once per device, kept afterwards).  That lookup may
 * load the library's device code; make this first call during set-up, before any stream capture is open on the thread.
 * Shared state: every call on a device, from any thread or stream, uses the same array, and the array keeps what the last call
 * left in it.  The call clears the counters it needs on `stream` before its kernel (one cudaMemsetAsync of 68 bytes), so stale
 * contents never reach a result; but two calls that can run on the GPU at the same time (different streams without an event
 * between them, or two host threads) race on the array and return wrong sums.  Keep calls on one device stream-ordered.
 * No synchronisation.  Returns 0, -1 on a bad argument (NULL buffer, n_events < 0, n_rows outside the limit, more than
 * RWGT_STATIC_MAX_DEVICES = 64 devices), or the cudaError_t of the address lookup, the clear or the launch. */
#define RWGT_STATIC_SUM_MAX_ROWS 17
#define RWGT_STATIC_SCRATCH_BYTES 9216
#define RWGT_STATIC_MAX_DEVICES 64
int rwgt_sum_weights_static(const double* w, int n_rows, long long n_events, double* out_sums, void* stream);

/* Binary event files: the stand-in for the LHE event files the paper's library parses (PAPER.md:87 step 2), which do
 * not exist here.  Little endian, structure of arrays, the layout rwgt_run takes:
 *   event file  = rwgt_event_file_header, double momenta[n_ext][4][n_events], double weights[n_events]
 *   result file = rwgt_result_file_header, double me_old[n_events], me_new[K][n_events], w_new[K][n_events],
 *                 double sum_w_old, sum_w_new[K]       (eq. 2 of the processed range, old weights and every parameter set) */
typedef struct {
  char magic[8];               /* "RWGTEVT1"                                        */
  unsigned int version;        /* 1                                                 */
  unsigned int n_ext;          /* external legs per event                           */
  unsigned long long n_events;
  char process[32];            /* process name as given to rwgt_create, NUL padded  */
  unsigned long long reserved;
} rwgt_event_file_header;
typedef struct {
  char magic[8];               /* "RWGTRES1"                                        */
  unsigned int version;        /* 1                                                 */
  unsigned int n_sets;         /* K new parameter sets                              */
  unsigned long long n_events; /* events in this file                               */
  char process[32];
  unsigned long long first_event; /* index in the event file of this file's event 0 */
} rwgt_result_file_header;

/* The whole procedure of PAPER.md:87 (steps 2-8) for events [first_event, first_event + n_events) of the event file `in_path`
 * (n_events < 0: to the end of the file): parse, copy to the device, evaluate |M|^2 and every |M'_k|^2, eq. 3, copy back, write the
 * result file `out_path`, including the eq. 2 sums (the file is written as "<out_path>.tmp" and renamed when complete, so a failed
 * call leaves no result file of this call behind and an existing `out_path` as it was; `out_path` must not be the event file).  The range is cut into chunks; a reader thread fills one
 * pinned buffer from the file while the previous chunk goes through the overlapped H2D / kernel / D2H pipeline of
 * rwgt_run_multi_host and a writer thread stores the chunk before.  Pinned buffers and device scratch belong to the handle and are
 * grown on first use.  Synchronises `stream`.  A rank of a multi-GPU job passes its own contiguous range and result path
 * (events are independent: no exchange).
 * Returns 0, -1 (bad argument, unreadable / foreign / truncated event file, range outside the file, write error; see
 * rwgt_last_error()) or a positive cudaError_t. */
int rwgt_run_file(rwgt_handle* h, const char* in_path, const char* out_path, long long first_event, long long n_events, void* stream);

/* Frees device tables and scratch. 0 on success, -1 on NULL. */
int rwgt_destroy(rwgt_handle* h);

/* Thread-local, static storage; never NULL. */
const char* rwgt_last_error(void);

/* Identity of the build: the first 12 hex digits of the SHA-256 over the library's sources (csrc/*.cu, csrc/*.cuh, include/rwgt.h, in
 * name order), baked in by paper_2312_07440_b200/build.py; "unknown" for a build made otherwise.  Static storage.  bench.py compares it
 * with the build id stored beside the ncu counts in profiles/counts.json and drops those figures when the library is another build. */
const char* rwgt_build_id(void);

/* HOST: writes the n! x n! colour matrix C (row-major, permutations of the gluon labels in
 * lexicographic order) the library uses for a process with n_gluons in 2..5; computed with
 * the SU(3) Fierz identity in exact integer arithmetic.  Returns n! or -1. */
int rwgt_colour_matrix(int n_gluons, double* out);

#ifdef __cplusplus
}
#endif
#endif /* RWGT_H */
