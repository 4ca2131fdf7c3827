// qa_internal.cuh -- structures shared by the host API (qa_api.cu) and the kernels.  Not part of the C ABI.
#pragma once
#include <cstddef>
#include <cstdint>
#include <cuda_runtime.h>

#include "../../include/qarray_b200.h"

constexpr int QA_MAXN = 16;  // dots
constexpr int QA_MAXG = 64;  // gates
constexpr int QA_WALK_NL = 8;  // low bits walked per thread by the static Gray walk (2^8 candidates per thread)
constexpr int QA_FUSED_MAXN = 8; // largest n of the one-kernel path (qa_kernels_fused.cu)
constexpr int QA_CLOSED_MAXB = 16; // most blocks of high patterns per pixel in the closed walk (qa_kernels_closed.cu)
constexpr int QA_PAIR_NL = 10; // low bits covered by the model's pair-energy table QL (min-plus walk: NL <= 10)

// Pixel-independent model constants in device global memory (one per qa_model).
// "search" model = the model the candidate search runs on: the full model, or (sensor dots set) the sub-blocks of the
// non-sensor dots (reading R8).  Matrices use fixed strides so that kernels index them without knowing n at compile time.
struct QaDevModel {
    int n;       // dots of the search model
    int g;       // gates
    int nf;      // dots of the full model
    int ns;      // sensor dots (nf = n + ns)
    double C[QA_MAXN * QA_MAXN];    // search c_dd, stride QA_MAXN
    double M[QA_MAXN * QA_MAXN];    // search c_dd^-1, stride QA_MAXN
    double Cgd[QA_MAXN * QA_MAXG];  // search c_gd, stride QA_MAXG
    double C1[QA_MAXN];             // c_dd 1        (Eq. (7))
    double oneC1;                   // 1^T c_dd 1
    double EC;                      // 1/2 min_i M_ii
    double qsum;                    // sum_{i<j} |M_ij| of the search model (>= the pair energy of any bit pattern)
    double pad16;                   // (keeps the 16-byte alignment of the tables below: they are read as double2)
    double Mf[QA_MAXN * QA_MAXN];   // full c_dd^-1, stride QA_MAXN
    double Cgdf[QA_MAXN * QA_MAXG]; // full c_gd
    int arr_idx[QA_MAXN];           // search dot a -> dot index in the full model
    int sens_idx[QA_MAXN];          // sensor s -> dot index in the full model
    // QL[b] = sum_{j<j', both set in b} M[n-1-j][n-1-j']: pair energy of the low-bit pattern b (low bit j <-> search dot
    // n-1-j), j ascending then j' ascending; entries with a bit >= n set are 0.  The table of NL < QA_PAIR_NL bits is
    // its prefix.
    double QL[1 << QA_PAIR_NL];
    // Min-plus walk (n >= 13; NL = QA_WALK_NL low bits per thread, NH = n - NL high bits = one thread per pattern t):
    //   VT[t][j] = sum over the high bits jh of t (ascending) of M[n-1-j][n-1-NL-jh]      cross term of t with low bit j
    //   QHT[t]   = E_C + sum_{jh<jh' in t} M[n-1-NL-jh][n-1-NL-jh']                       pair energy of t, plus E_C
    double VT[(1 << QA_WALK_NL) * QA_WALK_NL];
    double QHT[1 << QA_WALK_NL];
    double VTt[QA_WALK_NL * (1 << QA_WALK_NL)];  // VT transposed, [j][t]: coalesced when the lanes hold consecutive t
    // One-kernel path of n <= 8 (qa_kernels_fused_open.cu): its shared-memory tables as ONE contiguous block, so that a CTA
    // stages them with 16-byte copies and no index arithmetic:  MT[j*n + i] = M[i][j] (n^2) | C compact row-major (n^2) |
    // T[b] = QL[b] (2^n) | CgT[k*n + i] = Cgd[i][k] (g n, zero padded to an even count).  Zero for n > 8.
    alignas(16) double fo_pack[2 * 64 + 256 + QA_MAXG * 8 + 2];
};

// (kernels read these tables 16 bytes at a time)
static_assert(offsetof(QaDevModel, QL) % 16 == 0 && offsetof(QaDevModel, VT) % 16 == 0 && offsetof(QaDevModel, QHT) % 16 == 0 &&
                  offsetof(QaDevModel, VTt) % 16 == 0 && offsetof(QaDevModel, fo_pack) % 16 == 0 &&
                  offsetof(QaDevModel, M) % 16 == 0 && offsetof(QaDevModel, C) % 16 == 0,
              "QaDevModel: tables read as double2 must stay 16-byte aligned");

// Per-call scratch, structure-of-arrays over pixels ([i][P] so that thread-per-pixel accesses coalesce).
struct QaWorkspace {
    double *h;        // [n][P]  g0_i + 1/2 M_ii at the base point: energy increment of raising dot i by one
    double *nc;       // [n][P]  N_c of the search model
    int32_t *base;    // [n][P]  smallest candidate value of dot i
    int32_t *cnt;     // [n][P]  number of candidate values of dot i (1, 2, n_max + 1, or up to 4 when widened)
    uint64_t *total;  // [P]     product of cnt = size of the enumerated set
    uint64_t *best;   // [P]     mixed-radix index (dot 0 most significant) of the argmin, ~0 if the set is empty
    double *e0;       // [P]     E(base) = 1/2 (base - N_c)^T M (base - N_c) >= 0, the energy of the base point
    unsigned long long *counter;  // work counter of the pruned min-plus walk (zeroed by the prologue kernel)
    uint2 *rec;       // [P][2^(n-13)]  min-plus walk: per warp of the pixel (min of L over its lanes, ballot of lanes near it)
    double2 *rec2;    // [nb][P]        closed walk (same storage as rec): per block of high patterns (best energy, its index)
    // [3][P] (n >= 13, behind the walk's records in the same region): thread-independent per-pixel constants of the min-plus
    // walk, written by the lanes prologue: offW = E_C + sum |h| of the 4 lowest bits' dots, offU = sum |h| of the next 4,
    // C' = the fixed-point constant of the keys (qa_kernels_minplus.cu)
    double *ext;
    int64_t P;
};

struct QaCallArgs {
    int closed;
    int N_hat;
    int alg;
    double t;
    int n_max;
    int general_qp;  // c_dd has a positive off-diagonal: the QP continues with the primal active-set phase (R3)
    int walk_ext;    // 1: the min-plus walk follows (open, default, n >= 13, Maxwell): the lanes prologue also writes ws.ext
};

// Several algorithms on one sweep in one launch (qa_ground_state_batch_multi): per pass the threshold and the outputs.
constexpr int QA_MULTI_MAX = 4;
// thresholded algorithm in the one-kernel path of n <= 8: at or below this t the pixels are not bucket-sorted by their number
// of free dots (measured on config 5: crossover between 0.5 and 0.7); the multi-algorithm kernel has only that form
constexpr double QA_FO_NOSORT_T = 0.6;
struct QaMultiArgs {
    int n_alg;
    int thr[QA_MULTI_MAX];      // 1: thresholded (Eq. (9)), 0: default
    double t[QA_MULTI_MAX];
    int32_t *N[QA_MULTI_MAX];   // device [n_models * P * n]
    double *E[QA_MULTI_MAX];    // device [n_models * P]
};

// Pair-energy table of the low QA_WALK_NL bits for the static walk: QL[b] = sum_{j<j', both set in b} M[a_j][a_j'],
// a_j = n-1-j the dot of low bit j.  Passed by value (constant bank) so the unrolled walk reads it with static offsets.
struct QaWalkTable {
    double QL[1 << QA_WALK_NL];
};

// launch-plan log (host, thread-local; filled by the launchers)
void qa_plan_reset();
void qa_plan_add(const char *kernel_name);
void qa_timing_mark(cudaStream_t stream);  // measurement aid: event between two kernels of a call (no-op unless enabled)

// launchers (each enqueues exactly one kernel on `stream` and logs it)
cudaError_t qa_launch_prologue(const QaDevModel *d_model, int n, int g, const double *d_Vg, QaWorkspace ws,
                               QaCallArgs args, double *d_xcont, qa_stats *d_stats, cudaStream_t stream, bool lanes = false);
cudaError_t qa_launch_enumerate(const QaDevModel *d_model, int n, QaWorkspace ws, QaCallArgs args, double expect_cand,
                                qa_stats *d_stats, cudaStream_t stream);
cudaError_t qa_launch_walk(const QaDevModel *d_model, int n, const QaWalkTable &tab, QaWorkspace ws, qa_stats *d_stats,
                           int sm_count, cudaStream_t stream);
cudaError_t qa_launch_closed_walk(const QaDevModel *d_model, int n, const QaWalkTable &tab, QaWorkspace ws, QaCallArgs args,
                                  int sm_count, cudaStream_t stream, int *nb_out);
cudaError_t qa_launch_minplus_walk(const QaDevModel *d_model, int n, const double *QLhost, QaWorkspace ws, int32_t *d_N,
                                   double *d_E, int sm_count, int pruned, cudaStream_t stream);
cudaError_t qa_launch_minplus_finish(const QaDevModel *d_model, int n, QaWorkspace ws, int32_t *d_N, double *d_E, unsigned slack,
                                     int sm_count, cudaStream_t stream);
cudaError_t qa_launch_minplus_fused(const QaDevModel *d_model, const double *QLhost, const double *d_Vg, int64_t P, QaCallArgs args,
                                    int32_t *d_N, double *d_E, double *d_xcont, qa_stats *d_stats, int sm_count,
                                    cudaStream_t stream);
cudaError_t qa_launch_minplus_walk32(const QaDevModel *d_model, int n, const double *QLhost, QaWorkspace ws, int32_t *d_N,
                                     double *d_E, int sm_count, cudaStream_t stream);
cudaError_t qa_launch_fused_mid(const QaDevModel *d_model, int n, const QaWalkTable &tab, const double *d_Vg, int64_t P,
                                QaCallArgs args, int32_t *d_N, double *d_E, double *d_xcont, qa_stats *d_stats,
                                cudaStream_t stream);
cudaError_t qa_launch_fused_small(const QaDevModel *const *d_models, int n_models, int n, const double *d_Vg, int64_t P,
                                  QaCallArgs args, int32_t *d_N, double *d_E, double *d_xcont, double *d_Vs,
                                  qa_stats *d_stats, cudaStream_t stream);
cudaError_t qa_launch_fused_open(const QaDevModel *const *d_models, int n_models, int n, int g, const double *d_Vg,
                                 int64_t P, QaCallArgs args, int32_t *d_N, double *d_E, double *d_xcont, double *d_Vs,
                                 qa_stats *d_stats, cudaStream_t stream);
cudaError_t qa_launch_fused_open_multi(const QaDevModel *const *d_models, int n_models, int n, int g, const double *d_Vg,
                                       int64_t P, int general_qp, const QaMultiArgs &ma, double *d_xcont, qa_stats *d_stats,
                                       cudaStream_t stream);
cudaError_t qa_launch_thermal(const QaDevModel *d_model, int n, QaWorkspace ws, QaCallArgs args, double kT,
                              double expect_cand, double *d_Nmean, double *d_Emin, qa_stats *d_stats, cudaStream_t stream);
cudaError_t qa_launch_thermal_sp(const QaDevModel *d_model, int n, const double *QLhost, QaWorkspace ws, double kT,
                                 double *d_Nmean, double *d_Emin, int sm_count, cudaStream_t stream);
// closed_nb > 0: the winner of a pixel is the lexicographic minimum of its closed_nb records ws.rec2 (closed walk); N_hat is
// then read for the scored-candidate counter
cudaError_t qa_launch_finalize(const QaDevModel *d_model, const double *d_Vg, QaWorkspace ws, int32_t *d_N, double *d_E,
                               double *d_Vsensor, qa_stats *d_stats, cudaStream_t stream, int closed_nb = 0, int N_hat = 0,
                               int n_lanes = 0);  // n_lanes = n_dot when the sixteen-lanes-per-pixel kernel may be used, else 0
cudaError_t qa_launch_sensor_response(const qa_sensor_params *params, int ns, const double *d_Vs, int64_t P, int64_t W,
                                      double *d_S, double *d_G, double *d_partial, cudaStream_t stream);
size_t qa_sensor_workspace_bytes_impl(int64_t P, int ns);
cudaError_t qa_launch_fp64_probe(double *d_sink, int blocks, int threads, int iters, cudaStream_t stream);

// ---- small device helpers ------------------------------------------------------------------------------------------
#ifdef __CUDACC__
// Programmatic dependent launch (sm_90+): a kernel launched with cudaLaunchAttributeProgrammaticStreamSerialization may
// become resident while its predecessor in the stream is still running; it must call qa_pdl_wait() before it touches
// anything the predecessor wrote (the wait returns once that grid has completed and its writes are visible).
// qa_pdl_launch_dependents() lets the successor's CTAs be scheduled as soon as resources free up.
__device__ __forceinline__ void qa_pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void qa_pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

// Launch `kernel` as a programmatic dependent of the previous kernel in `stream`.
template <typename... KArgs, typename... Args>
inline cudaError_t qa_launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, cudaStream_t stream, Args... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = 0;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

__device__ __forceinline__ void qa_atomic_add64(int64_t *addr, int64_t v)
{
    atomicAdd(reinterpret_cast<unsigned long long *>(addr), static_cast<unsigned long long>(v));
}

// warp-aggregated counter add (all 32 lanes must call)
__device__ __forceinline__ void qa_warp_count(int64_t *addr, int64_t v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if ((threadIdx.x & 31) == 0 && v != 0) qa_atomic_add64(addr, v);
}

// lexicographic (energy, index) minimum: deterministic regardless of thread scheduling
__device__ __forceinline__ void qa_lexmin(double &e, uint64_t &i, double e2, uint64_t i2)
{
    if (e2 < e || (e2 == e && i2 < i)) {
        e = e2;
        i = i2;
    }
}
// S8 for one pixel: with the array charges Ns[0..n-1] fixed, every sensor dot's carrier number (lower energy of
// max(0, floor s) and that + 1, s = N_c,s - M_sD d_D / M_ss) in the full model, the full charge row and the sensor
// potentials V_s = [M (N - N_c)]_s (L149, Eq. (3), reading R8).
__device__ __forceinline__ void qa_sensor_pixel(const QaDevModel *__restrict__ mdl, const double *__restrict__ Vg, int64_t p,
                                                const int32_t *Ns, int32_t *__restrict__ outN, double *__restrict__ outVs)
{
    const int n = mdl->n, nf = mdl->nf, ns = mdl->ns, g = mdl->g;
    // full model: N_c of every dot (same fma order), array dots fixed, then each sensor independently
    double ncf[QA_MAXN], df[QA_MAXN];
    int32_t Nf[QA_MAXN];
    for (int i = 0; i < nf; ++i) {
        double acc = 0.0;
        for (int k = 0; k < g; ++k) acc = fma(mdl->Cgdf[i * QA_MAXG + k], __ldg(Vg + p * g + k), acc);
        ncf[i] = acc;
        df[i] = 0.0;
        Nf[i] = 0;
    }
    for (int a = 0; a < n; ++a) {
        const int i = mdl->arr_idx[a];
        Nf[i] = Ns[a];
        df[i] = (double)Ns[a] - ncf[i];
    }
    for (int a = 0; a < ns; ++a) {
        const int s = mdl->sens_idx[a];
        double y = 0.0;
        for (int b = 0; b < n; ++b) {
            const int j = mdl->arr_idx[b];
            y += mdl->Mf[s * QA_MAXN + j] * df[j];
        }
        const double Mss = mdl->Mf[s * QA_MAXN + s];
        const double sstar = ncf[s] - y / Mss;
        const double fl = floor(sstar);
        const int32_t c0 = fl > 0.0 ? (int32_t)fl : 0;
        const double d0 = (double)c0 - ncf[s], d1 = (double)(c0 + 1) - ncf[s];
        const double e0 = d0 * y + 0.5 * Mss * d0 * d0;
        const double e1 = d1 * y + 0.5 * Mss * d1 * d1;
        Nf[s] = e1 < e0 ? c0 + 1 : c0;
    }
    for (int a = 0; a < ns; ++a) {
        const int s = mdl->sens_idx[a];
        df[s] = (double)Nf[s] - ncf[s];
    }
    for (int i = 0; i < nf; ++i) outN[p * nf + i] = Nf[i];
    if (outVs) {
        for (int a = 0; a < ns; ++a) {
            const int s = mdl->sens_idx[a];
            double vsum = 0.0;
            for (int j = 0; j < nf; ++j) vsum += mdl->Mf[s * QA_MAXN + j] * df[j];
            outVs[p * ns + a] = vsum;
        }
    }
}

// S7 + S8 for one pixel, one thread: N* = base + digits of the winning mixed-radix index `idx`; E(N*) recomputed from the
// definition (Eq. (C1)); sensor dots (L149 + Eq. (3), reading R8).  idx = ~0: empty candidate set.
__device__ __forceinline__ void qa_finalize_pixel(const QaDevModel *__restrict__ mdl, const double *__restrict__ Vg,
                                                  const QaWorkspace &ws, int64_t p, uint64_t idx,
                                                  int32_t *__restrict__ outN, double *__restrict__ outE,
                                                  double *__restrict__ outVs)
{
    const int64_t P = ws.P;
    const int n = mdl->n, nf = mdl->nf, ns = mdl->ns, g = mdl->g;
    int32_t Ns[QA_MAXN];
    double d[QA_MAXN];
    const bool empty = idx == ~0ull;
    for (int i = n - 1; i >= 0; --i) {
        const uint64_t c = (uint64_t)ws.cnt[i * P + p];
        const int32_t dgt = (int32_t)(idx % c);
        idx /= c;
        Ns[i] = empty ? -1 : ws.base[i * P + p] + dgt;
        d[i] = (double)Ns[i] - ws.nc[i * P + p];
    }
    double E = 0.0;
    for (int i = 0; i < n; ++i) {
        double row = 0.0;
        for (int j = 0; j < n; ++j) row = fma(mdl->M[i * QA_MAXN + j], d[j], row);
        E = fma(d[i], row, E);
    }
    outE[p] = empty ? INFINITY : 0.5 * E;
    if (ns == 0) {
        for (int i = 0; i < n; ++i) outN[p * n + i] = Ns[i];
        return;
    }
    qa_sensor_pixel(mdl, Vg, p, Ns, outN, outVs);
}
#endif
