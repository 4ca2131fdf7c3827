// qa_internal.cuh -- structures shared by the host API (qa_api.cu) and the kernels.  Not part of the C ABI.
#pragma once
#include <cstddef>
#include <cstdint>
#include <cuda_runtime.h>

#include "../../include/qarray_b200.h"

constexpr int QA_MAXN = 16;  // dots
constexpr int QA_MAXG = 64;  // gates
constexpr int QA_WALK_NL = 8;  // low bits walked per thread by the static Gray walk (2^8 candidates per thread)

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
    double Mf[QA_MAXN * QA_MAXN];   // full c_dd^-1, stride QA_MAXN
    double Cgdf[QA_MAXN * QA_MAXG]; // full c_gd
    int arr_idx[QA_MAXN];           // search dot a -> dot index in the full model
    int sens_idx[QA_MAXN];          // sensor s -> dot index in the full model
};

// Per-call scratch, structure-of-arrays over pixels ([i][P] so that thread-per-pixel accesses coalesce).
struct QaWorkspace {
    double *h;        // [n][P]  g0_i + 1/2 M_ii at the base point: energy increment of raising dot i by one
    double *nc;       // [n][P]  N_c of the search model
    int32_t *base;    // [n][P]  smallest candidate value of dot i
    int32_t *cnt;     // [n][P]  number of candidate values of dot i (1, 2, n_max + 1, or up to 4 when widened)
    uint64_t *total;  // [P]     product of cnt = size of the enumerated set
    uint64_t *best;   // [P]     mixed-radix index (dot 0 most significant) of the argmin, ~0 if the set is empty
    int64_t P;
};

struct QaCallArgs {
    int closed;
    int N_hat;
    int alg;
    double t;
    int n_max;
};

// Pair-energy table of the low QA_WALK_NL bits for the static walk: QL[b] = sum_{j<j', both set in b} M[a_j][a_j'],
// a_j = n-1-j the dot of low bit j.  Passed by value (constant bank) so the unrolled walk reads it with static offsets.
struct QaWalkTable {
    double QL[1 << QA_WALK_NL];
};

// launch-plan log (host, thread-local; filled by the launchers)
void qa_plan_reset();
void qa_plan_add(const char *kernel_name);

// launchers (each enqueues exactly one kernel on `stream` and logs it)
cudaError_t qa_launch_prologue(const QaDevModel *d_model, int n, int g, const double *d_Vg, QaWorkspace ws,
                               QaCallArgs args, double *d_xcont, qa_stats *d_stats, cudaStream_t stream);
cudaError_t qa_launch_enumerate(const QaDevModel *d_model, int n, QaWorkspace ws, QaCallArgs args, double expect_cand,
                                qa_stats *d_stats, cudaStream_t stream);
cudaError_t qa_launch_walk(const QaDevModel *d_model, int n, const QaWalkTable &tab, QaWorkspace ws, qa_stats *d_stats,
                           int sm_count, cudaStream_t stream);
cudaError_t qa_launch_finalize(const QaDevModel *d_model, const double *d_Vg, QaWorkspace ws, int32_t *d_N, double *d_E,
                               double *d_Vsensor, qa_stats *d_stats, cudaStream_t stream);
cudaError_t qa_launch_fp64_probe(double *d_sink, int blocks, int threads, int iters, cudaStream_t stream);

// ---- small device helpers ------------------------------------------------------------------------------------------
#ifdef __CUDACC__
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
#endif
