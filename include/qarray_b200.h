/*
 * qarray_b200.h -- C ABI of the B200-native constant-capacitance-model ground-state search.
 *
 * The library implements ONE thing: the per-pixel ground-state charge search of arXiv 2404.04994 ("QArray") --
 * continuous minimum -> integer candidates -> free energy -> argmin -- for open and closed quantum-dot arrays with the
 * default, thresholded and brute-force candidate sets, as hand-written CUDA kernels for sm_100a.  "Lnnn" = line nnn of
 * the paper text; R1..R12 = the readings listed in DESIGN.md.
 *
 * Notation (paper's): n_dot dots, n_gate gates, P gate-voltage vectors ("pixels"), c_dd the dot-dot Maxwell
 * capacitance matrix (L35-L39 Eq. (2)), M = c_dd^-1 (L41), c_gd the positive gate->dot couplings, N_c = c_gd V_g
 * (Eq. (6)), F the free energy (Eq. (4)), |e| = 1 (L486).
 *
 * Conventions
 *   - "host" pointers are ordinary CPU memory; "device" pointers are CUDA global memory of the model's device.
 *   - All matrices are row-major fp64.  V_g is [P, n_gate]; N is [P, n_dot] int32; E is [P] fp64 (L454 output shape).
 *   - Output and workspace buffers are allocated and owned by the caller; the library never frees them.
 *   - qa_ground_state_open / _closed are ASYNCHRONOUS on `cuda_stream` (a cudaStream_t passed as void*; NULL = the
 *     legacy default stream): they only enqueue kernels, never synchronise and never allocate.
 *   - A qa_model is immutable after qa_model_set_sensor_dots and may be used by concurrent calls on different streams
 *     (each call needs its own workspace).  It belongs to the CUDA device that was current at qa_model_create: every
 *     call that takes the model (or a batch of models) returns QA_ERR_INVALID_ARG when another device is current.
 *   - Errors are returned as qa_status; nothing throws or aborts.  There is no CPU fallback: without a CUDA device every
 *     entry point that needs one returns QA_ERR_CUDA.
 */
#ifndef QARRAY_B200_H
#define QARRAY_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define QA_API __attribute__((visibility("default")))
#else
#define QA_API
#endif

typedef struct qa_model qa_model; /* opaque, library-owned */

typedef enum {
    QA_OK = 0,
    QA_ERR_INVALID_ARG = 1,      /* NULL pointer, P < 0, t outside [0,1], n_max < 0, workspace too small, ...          */
    QA_ERR_NOT_SYMMETRIC = 2,    /* |C_ij - C_ji| > 1e-12 max|C|                                              (L204)   */
    QA_ERR_NOT_POSDEF = 3,       /* Cholesky of c_dd fails                                                    (L204)   */
    QA_ERR_UNSUPPORTED_SIZE = 4, /* n_dot > 16 or n_gate > 64                                                          */
    QA_ERR_INFEASIBLE = 5,       /* closed array: N_hat < 0, or brute force with n_dot * n_max < N_hat                 */
    QA_ERR_OVERFLOW = 6,         /* brute force: (n_max + 1)^n_dot >= 2^62                                             */
    QA_ERR_CUDA = 7,             /* a CUDA runtime call failed; see qa_last_cuda_error()                               */
    QA_ERR_UNSUPPORTED = 8,      /* reserved (earlier versions refused a c_dd with a positive off-diagonal entry)      */
    QA_ERR_STATIC_WORKSPACE = 9  /* qa_ground_state_open_static: the sweep needs more scratch than the static array     */
} qa_status;

/* The three candidate sets of the paper (Table I). */
typedef enum {
    QA_ALG_DEFAULT = 0,     /* all 2^n_dot floor/ceil roundings of the continuous minimum           (L123-L127)        */
    QA_ALG_THRESHOLDED = 1, /* both roundings only where |frac - 1/2| <= t/2, Eq. (9)               (L131-L141)        */
    QA_ALG_BRUTE_FORCE = 2  /* every N in {0..n_max}^n_dot                                          (L13)              */
} qa_algorithm;

/* Optional per-call counters, accumulated on the device with atomics (zero the struct before the call). */
typedef struct {
    int64_t n_pixels;
    int64_t n_qp_pixels;             /* pixels whose analytic minimum had a negative component (L82-L84, L106)         */
    int64_t n_qp_rounds;             /* total active-set rounds over those pixels                                      */
    int64_t n_candidates_enumerated; /* sum over pixels of the size of the enumerated set                              */
    int64_t n_candidates_scored;     /* ... of those whose energy entered the argmin (closed: sum N = N_hat); with the
                                        pruned walk (qa_model_set_walk_variant(m, 2)) it still counts the whole set:
                                        the pruned candidates are covered by a bound                                   */
    int64_t n_threshold_doublings;   /* closed + thresholded: times t was doubled (L141, reading R5)                   */
    int64_t n_widened_pixels;        /* always 0 (kept for layout): the closed floor/ceil set is never empty at t = 1, so
                                        the widened set of an earlier reading R5 does not exist (R5)         */
    int64_t n_qp_failed;             /* pixels whose QP did not reach a KKT point (must be 0)                          */
} qa_stats;

/* ---- model ------------------------------------------------------------------------------------------------------- */

/* Problem statement: the constructor of the paper's DotArray (L185-L201) with Maxwell-format inputs.
 * C_dd : host, [n_dot*n_dot], symmetric positive definite; a Maxwell matrix has off-diagonals <= 0 (L35, Eq. (B1)).
 *        Validated as in L204: finite, symmetric (QA_ERR_NOT_SYMMETRIC), positive definite (QA_ERR_NOT_POSDEF).  A
 *        positive off-diagonal entry is legal input: the continuous QP then runs its general active-set phase and the
 *        open default search of n_dot >= 13 uses the exact-compare walk (reading R3).
 * C_gd : host, [n_dot*n_gate], gate->dot couplings (positive convention, reading on L35 vs L90).
 * Computes M = c_dd^-1, c_dd 1, 1^T c_dd 1 (Eq. (7)) and the pixel-independent pair-energy tables on the host, and
 * uploads them to the CURRENT CUDA device.  *out is owned by the library until qa_model_destroy. */
QA_API qa_status qa_model_create(const double *C_dd, const double *C_gd, int n_dot, int n_gate, qa_model **out);

/* Charge-sensor dots (L149, reading R8): the search runs on the sub-blocks C_dd[D,D], C_gd[D,:] of the non-sensor dots
 * D; then each sensor dot's carrier number and potential V_s = [M (N - N_c)]_s (Eq. (3)) are computed in the full
 * model.  dot_idx: host, n_sensor distinct indices in [0, n_dot); n_sensor = 0 clears.  Must be called before the model
 * is used by any ground-state call still in flight. */
QA_API qa_status qa_model_set_sensor_dots(qa_model *model, const int *dot_idx, int n_sensor);

QA_API qa_status qa_model_destroy(qa_model *model);

QA_API int qa_model_n_dot(const qa_model *model);    /* dots of the full model                                   */
QA_API int qa_model_n_gate(const qa_model *model);
QA_API int qa_model_n_sensor(const qa_model *model);
QA_API int qa_model_n_search(const qa_model *model); /* n_dot - n_sensor: columns of d_xcont                     */
/* M = c_dd^-1 of the full model as the library computed it (host, [n_dot*n_dot]) and E_C = 1/2 min_i M_ii. */
QA_API qa_status qa_model_get_inverse(const qa_model *model, double *M_host, double *E_C);

/* ---- ground state ------------------------------------------------------------------------------------------------ */

/* Bytes of device scratch a call on P pixels needs (0 on invalid arguments).  The buffer must be 256-byte aligned. */
QA_API size_t qa_workspace_bytes(const qa_model *model, int64_t P);

/* Open array: constraints (i) integer, (ii) N_i >= 0 (L49-L52).  Paper API: ground_state_open(vg) (L454-L458).
 *   d_Vg        device [P*n_gate]      gate voltages
 *   alg, t      candidate set; t in [0,1] is read for QA_ALG_THRESHOLDED only (Eq. (9))
 *   n_max       read for QA_ALG_BRUTE_FORCE only (L13)
 *   d_N         device [P*n_dot] int32 ground-state charges N* (Eq. (5)); sensor dots in their own columns
 *   d_E         device [P]             E(N*) = 1/2 (N*-N_c)^T M (N*-N_c) of the searched (sub-)model, recomputed from
 *                                      the definition (Eq. (C1)); equals Eq. (4) + 1/2 N_c^T M N_c (reading R2)
 *   d_xcont     device [P*n_search] or NULL   continuous minimum (Eq. (6)/(7)/(8))
 *   d_Vsensor   device [P*n_sensor] or NULL   sensor-dot potentials (only for models with sensor dots)
 *   d_stats     device qa_stats or NULL
 *   d_workspace device, >= qa_workspace_bytes(model, P) bytes, 256-byte aligned; contents undefined afterwards
 * Returns QA_OK once the work is enqueued. */
QA_API qa_status qa_ground_state_open(const qa_model *model, const double *d_Vg, int64_t P, qa_algorithm alg, double t,
                               int n_max, int32_t *d_N, double *d_E, double *d_xcont, double *d_Vsensor,
                               qa_stats *d_stats, void *d_workspace, size_t workspace_bytes, void *cuda_stream);

/* ---- the same search without any allocation on the caller's side ---------------------------------------------------- */

/* qa_ground_state_open for callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid allocation): identical arguments, kernels and results, but the workspace is a file-scope
 * `static __device__` array inside the library of QA_STATIC_WORKSPACE_BYTES (16 MiB; every GPU that loads the library holds
 * it until the process exits) instead of a buffer the caller allocates.
 *   - Limit: qa_workspace_bytes(model, P) <= QA_STATIC_WORKSPACE_BYTES, i.e. P <= 25 000 pixels at 16 dots (664 bytes per
 *     pixel; a 100x100 diagram needs 6.7 MB), more for smaller arrays.  A larger sweep is rejected with
 *     QA_ERR_STATIC_WORKSPACE before anything is enqueued; qa_static_workspace_last_error() says how much was needed.
 *   - Every call on a device shares the one array, which keeps the previous call's contents.  Nothing in it has to start at
 *     zero except the work counter of the pruned walk, which the first kernel of every call zeroes itself.  Calls that
 *     OVERLAP on the GPU (different streams or host threads, same device) race on the array: the caller serialises them
 *     (same stream, or an event between them).
 *   - The device address of the array is fetched once per device (cudaGetSymbolAddress, with that device current) at the
 *     first call on that device, or ahead of time by qa_static_workspace_init() -- call it once, with the device current,
 *     before a stream capture begins.  The call itself calls no cudaMalloc / cudaFree / allocating library routine (with
 *     the kernel-timing aid of qarray_b200_aids.h off).
 * Other arguments, stream semantics and errors as qa_ground_state_open. */
#define QA_STATIC_WORKSPACE_BYTES ((size_t)16 << 20)
QA_API size_t qa_static_workspace_bytes(void); /* = QA_STATIC_WORKSPACE_BYTES */
QA_API qa_status qa_static_workspace_init(void);
QA_API const char *qa_static_workspace_last_error(void); /* text of this host thread's last failure of the calls above/below */
QA_API qa_status qa_ground_state_open_static(const qa_model *model, const double *d_Vg, int64_t P, qa_algorithm alg, double t,
                                             int n_max, int32_t *d_N, double *d_E, double *d_xcont, double *d_Vsensor,
                                             qa_stats *d_stats, void *cuda_stream);

/* Closed array: additionally (iii) sum_i N_i = N_hat (L54-L56).  Paper API: ground_state_closed(vg, n_charges) (L454).
 * Candidates with the wrong total are eliminated (L127, L159); thresholded: per-pixel threshold doubling (L141, R5). */
QA_API qa_status qa_ground_state_closed(const qa_model *model, const double *d_Vg, int64_t P, int N_hat, qa_algorithm alg,
                                 double t, int n_max, int32_t *d_N, double *d_E, double *d_xcont, double *d_Vsensor,
                                 qa_stats *d_stats, void *d_workspace, size_t workspace_bytes, void *cuda_stream);

/* Host-buffer convenience (the end-to-end path): same semantics with HOST pointers.  Copies V_g to the device, runs the
 * search, copies the results back and synchronises before returning.  The model keeps a private stream and a grow-only
 * device staging buffer for these calls (released by qa_model_destroy); concurrent host calls on one model serialise.
 * closed = 0/1; N_hat is ignored for open arrays.  h_stats may be NULL; it is overwritten, not accumulated.  Pinned
 * host buffers make the copies asynchronous DMA transfers; pageable ones work too. */
QA_API qa_status qa_ground_state_host(const qa_model *model, const double *h_Vg, int64_t P, int closed, int N_hat,
                               qa_algorithm alg, double t, int n_max, int32_t *h_N, double *h_E, double *h_xcont,
                               double *h_Vsensor, qa_stats *h_stats);

/* ---- thermal broadening (section IV.B, Eq. (10)) ------------------------------------------------------- */

/* The arg min of Eq. (5) replaced by the soft arg min of Eq. (10): the Boltzmann-weighted mean of the charge states of the
 * SAME candidate set the chosen algorithm enumerates (closed: only sum N = N_hat, L159),
 *     <N> = sum_N N exp(-E(N)/kT) / sum_N exp(-E(N)/kT).
 * kT > 0 (finite) is k_B T in the energy units of E (|e| = 1; reading R13); QA_ERR_INVALID_ARG otherwise.
 *   d_Nmean  device [P*n_search] fp64   mean occupation of the searched dots (-1 where the candidate set is empty)
 *   d_Emin   device [P] or NULL         smallest energy of the candidate set (= E(N*) of the ground-state search, evaluated
 *                                       incrementally: not bit-identical to qa_ground_state's d_E)
 * Other arguments, workspace, stream semantics and errors as qa_ground_state_open / _closed.  Sensor dots are not part of
 * the average (the search model of qa_model_set_sensor_dots is used). */
QA_API qa_status qa_thermal_open(const qa_model *model, const double *d_Vg, int64_t P, qa_algorithm alg, double t, int n_max,
                                 double kT, double *d_Nmean, double *d_Emin, qa_stats *d_stats, void *d_workspace,
                                 size_t workspace_bytes, void *cuda_stream);
QA_API qa_status qa_thermal_closed(const qa_model *model, const double *d_Vg, int64_t P, int N_hat, qa_algorithm alg, double t,
                                   int n_max, double kT, double *d_Nmean, double *d_Emin, qa_stats *d_stats,
                                   void *d_workspace, size_t workspace_bytes, void *cuda_stream);

/* ---- charge-sensor response and noise (section IV.A, Fig. 3; reading R14) ------------------ */

/* L149: "we compute the charge sensor's response based on Lorentzian or an approximately Gaussian profile in the weak and
 * strong coupling regimes ... whilst white, 1/f, and sensor jump noise can be added on top"; L464: the figures show the
 * derivative of the sensor signal along the swept gate, and a qpc is modelled by "a linear function" instead.  The paper
 * gives no formula or parameter; reading R14 fixes them and every parameter is the caller's.  With x = (V_s - v0) / width:
 *   QA_PROFILE_LORENTZIAN  S = amplitude / (1 + x^2)            width = half width at half maximum
 *   QA_PROFILE_GAUSSIAN    S = amplitude exp(-x^2 / 2)          width = standard deviation
 *   QA_PROFILE_LINEAR      S = amplitude x
 * plus, in pixel order p (the raster is the time axis): white noise white_sigma z; 1/f noise pink_sigma / sqrt(K) times
 * the sum of K = pink_octaves sources, source j redrawn every 2^j pixels (Voss-McCartney); jump noise: at every pixel,
 * with probability jump_rate, the baseline shifts by jump_sigma z and keeps the shift.  The random numbers are counter
 * based (SplitMix64 finaliser of seed, stream and index; Box-Muller), so the result depends on `seed` only. */
typedef enum { QA_PROFILE_LORENTZIAN = 0, QA_PROFILE_GAUSSIAN = 1, QA_PROFILE_LINEAR = 2 } qa_sensor_profile;
typedef struct {
    int32_t profile;      /* qa_sensor_profile                                  */
    int32_t pink_octaves; /* K in [0, 30]                                       */
    double v0;            /* peak position, in the units of V_s                 */
    double width;         /* > 0                                                */
    double amplitude;
    double white_sigma;   /* >= 0; 0 switches the term off                      */
    double pink_sigma;    /* >= 0                                               */
    double jump_rate;     /* probability per pixel, in [0, 1]                   */
    double jump_sigma;    /* >= 0                                               */
    uint64_t seed;
} qa_sensor_params;

/* Device scratch for qa_sensor_response on P pixels and n_sensor sensors (256-byte aligned buffer). */
QA_API size_t qa_sensor_response_workspace_bytes(int64_t P, int n_sensor);

/*   d_Vsensor  device [P*n_sensor]   sensor potentials (the d_Vsensor output of a ground-state call)
 *   W          length of the fast axis of the sweep (P must be a multiple of W); only the gradient reads it
 *   params     HOST, n_sensor entries (1 <= n_sensor <= 16)
 *   d_signal   device [P*n_sensor]   response + noise
 *   d_gradient device [P*n_sensor] or NULL: along the fast axis, central differences inside a row, one-sided at its
 *              ends, in signal units per pixel, of the noisy signal
 * Asynchronous on cuda_stream; never allocates.  QA_ERR_INVALID_ARG for a parameter outside its range. */
QA_API qa_status qa_sensor_response(const double *d_Vsensor, int64_t P, int n_sensor, int64_t W, const qa_sensor_params *params,
                                    double *d_signal, double *d_gradient, void *d_workspace, size_t workspace_bytes,
                                    void *cuda_stream);

/* ---- dataset batch (BASELINE.json configs[4]) ------------------------------------------------------------------------ */

/* A list of models that share n_dot (<= 8) and n_gate, have no sensor dots and live on the same device.  A batch call
 * is semantically a loop over the single-model call -- array b reads V_g[b] and writes N[b], E[b] -- but runs as ONE
 * launch of the one-kernel path (every step S1-S7 in registers, one thread per pixel).  The models must outlive the batch.
 * models: host array of n_models handles.  Errors: QA_ERR_UNSUPPORTED_SIZE (n_dot > 8 or sensor dots),
 * QA_ERR_INVALID_ARG (mixed shapes or devices, NULL). */
typedef struct qa_batch qa_batch;
QA_API qa_status qa_batch_create(const qa_model *const *models, int n_models, qa_batch **out);
QA_API qa_status qa_batch_destroy(qa_batch *batch);
QA_API int qa_batch_size(const qa_batch *batch);
/* d_Vg device [n_models*P*n_gate], d_N device [n_models*P*n_dot] int32, d_E device [n_models*P], d_xcont device
 * [n_models*P*n_dot] or NULL, d_stats device or NULL (summed over the batch).  closed = 0/1 (N_hat read when closed).
 * Asynchronous on cuda_stream; needs no workspace.  Argument errors as for the single-model calls. */
QA_API qa_status qa_ground_state_batch(const qa_batch *batch, const double *d_Vg, int64_t P, int closed, int N_hat,
                                       qa_algorithm alg, double t, int n_max, int32_t *d_N, double *d_E, double *d_xcont,
                                       qa_stats *d_stats, void *cuda_stream);

/* Several algorithms on the SAME sweep in one launch: a dataset run searches every diagram with the default algorithm and
 * with one or more thresholds (datasets for training; section IV.A: thresholds trade accuracy for speed).
 * Semantically a loop over qa_ground_state_batch(batch, d_Vg, P, open, algs[a], ts[a]) -> d_N[a], d_E[a] for a = 0 ..
 * n_alg - 1, with bit-identical results; V_g is read once and N_c and the continuous minimum (S1-S3, the QP) are computed
 * once per pixel instead of once per algorithm.  Open arrays only; algs[a] is QA_ALG_DEFAULT or QA_ALG_THRESHOLDED (ts[a]
 * in [0, 1], ignored for the default algorithm); 1 <= n_alg <= 4.  algs, ts, d_N, d_E: HOST arrays of n_alg entries, d_N[a] /
 * d_E[a] device buffers shaped as in qa_ground_state_batch; d_xcont device or NULL (the same for every algorithm);
 * d_stats device or NULL (summed over the algorithms).  Asynchronous on cuda_stream; needs no workspace; never allocates. */
QA_API qa_status qa_ground_state_batch_multi(const qa_batch *batch, const double *d_Vg, int64_t P, int n_alg,
                                             const qa_algorithm *algs, const double *ts, int32_t *const *d_N,
                                             double *const *d_E, double *d_xcont, qa_stats *d_stats, void *cuda_stream);

/* ---- diagnostics ------------------------------------------------------------------------------------------------- */
/* (Measurement and cross-check aids -- FP64 issue-rate probe, per-kernel event timing, launch plan, kernel selection --
 * are declared in qarray_b200_aids.h; they are not part of the product surface.) */

QA_API const char *qa_status_string(qa_status s);
QA_API const char *qa_last_cuda_error(void);
QA_API const char *qa_version(void);

#ifdef __cplusplus
}
#endif
#endif /* QARRAY_B200_H */
