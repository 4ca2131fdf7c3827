// qa_kernels_fused.cu -- the whole path S1-S7 of SURVEY.md section 8(a) in ONE kernel, one thread per pixel, for small
// arrays (n <= 8) whose candidate sets are small (default: 2^n <= 256, thresholded: ~(1+t)^n): nothing but V_g is read
// from HBM and nothing but N*, E(N*) [, x] is written -- the bound of the dataset-batch workload (BASELINE.json
// configs[4]: 8 g + 4 n + 8 bytes per pixel).  blockIdx.y selects the model, so a batch of
// independently seeded arrays is one launch (qa_ground_state_batch); the single-model entry points use it with one model.
//
// The arithmetic is that of the three-kernel path (qa_prologue_kernel, qa_enumerate_kernel<N,1>, qa_finalize_kernel): the
// same functions for S1-S4 (qa_prologue.cuh), the same mixed-radix odometer with rank-1 energy updates
//     E(d + delta e_i) = E(d) + delta grad_i + 1/2 delta^2 M_ii,   grad += delta M[:, i]                  (from (C1) L607)
// in lexicographic order (dot 0 most significant; strict '<' keeps the lexicographically first of equal energies, R6),
// and E(N*) recomputed from the definition.  The open default set (every dot has exactly two values) is scored with the
// static Gray walk of qa_kernels_walk.cu instead (3 FP64 instructions per candidate; pair table staged in shared memory).
// Closed arrays score only candidates with sum N = N_hat (L127, L159).  A single model with charge-sensor dots (L149,
// reading R8) also gets its sensor step S8 here (qa_sensor_pixel).
#include "qa_internal.cuh"
#include "qa_prologue.cuh"

namespace {

constexpr int FS_THREADS = 128;

__host__ __device__ constexpr int fs_ctz(int k)
{
    int j = 0;
    while (((k >> j) & 1) == 0) ++j;
    return j;
}

// GRAY: the open default set (compiled separately: the two scoring loops have very different register needs)
template <int N, bool GRAY>
__global__ void __launch_bounds__(FS_THREADS, GRAY ? 2 : 4) qa_fused_small_kernel(const QaDevModel *const *__restrict__ models,
                                                                    const double *__restrict__ Vg, int64_t P,
                                                                    QaCallArgs args, int32_t *__restrict__ outN,
                                                                    double *__restrict__ outE, double *__restrict__ xcont,
                                                                    double *__restrict__ outVs, qa_stats *stats)
{
    __shared__ double sM[N * N], sC[N * N], sCgd[N * QA_MAXG], sC1[N];
    __shared__ __align__(16) double sT[1 << N];  // pair table of the low-bit patterns: sT[k] = QL[k]
    const QaDevModel *__restrict__ mdl = models[blockIdx.y];
    const int g = mdl->g;
    for (int e = threadIdx.x; e < N * N; e += FS_THREADS) {
        sM[e] = mdl->M[(e / N) * QA_MAXN + (e % N)];
        sC[e] = mdl->C[(e / N) * QA_MAXN + (e % N)];
    }
    for (int e = threadIdx.x; e < N * g; e += FS_THREADS) sCgd[e] = mdl->Cgd[(e / g) * QA_MAXG + (e % g)];
    if (threadIdx.x < N) sC1[threadIdx.x] = mdl->C1[threadIdx.x];
    for (int k = threadIdx.x; k < (1 << N); k += FS_THREADS) sT[k] = mdl->QL[k];
    const double oneC1 = mdl->oneC1;
    __syncthreads();

    const int64_t p = blockIdx.x * (int64_t)FS_THREADS + threadIdx.x;  // pixel within the array
    const bool live = p < P;
    const int64_t gp = (int64_t)blockIdx.y * P + (live ? p : P - 1);   // pixel within the batch
    const bool closed = args.closed != 0;

    // S1-S4
    double nc[N], x[N];
    int32_t base[N], cnt[N];
    QaPixelFlags fl;
    qa_prologue_pixel<N>(sCgd, sC, sC1, oneC1, g, Vg + gp * g, args, nc, x, base, cnt, fl);
    uint64_t total = 1;
#pragma unroll
    for (int i = 0; i < N; ++i) total *= (uint64_t)cnt[i];

    // S5-S6: first candidate from the definition, then the odometer
    int32_t dg[N];
    double d[N], grad[N];
    int64_t sumN = 0;
#pragma unroll
    for (int i = 0; i < N; ++i) {
        dg[i] = 0;
        d[i] = (double)base[i] - nc[i];
        sumN += base[i];
    }
    double E = 0.0;
#pragma unroll
    for (int i = 0; i < N; ++i) {
        double gi = 0.0;
#pragma unroll
        for (int j = 0; j < N; ++j) gi = fma(sM[i * N + j], d[j], gi);
        grad[i] = gi;
        E = fma(d[i], gi, E);
    }
    E *= 0.5;
    double best = INFINITY;
    uint64_t bidx = ~0ull;
    int64_t scored = 0;
    constexpr bool gray = GRAY;  // every cnt_i = 2: the static Gray walk of qa_kernels_walk.cu
    if constexpr (GRAY) {
        // E(base + b) - E(base) = sum_i b_i h_i + QL[b], h_i = grad_i + 1/2 M_ii; low bit j <-> dot N-1-j; 3 FP64
        // instructions per candidate, every index static.  The winning pattern IS the mixed-radix index (cnt_i = 2).
        double hp[N];
#pragma unroll
        for (int j = 0; j < N; ++j) hp[j] = grad[N - 1 - j] + 0.5 * sM[(N - 1 - j) * N + (N - 1 - j)];
        // counting order (qa_kernels_walk.cu): step k-1 -> k moves the linear part by c_ctz(k); ascending k + strict '<'
        // keeps the smallest index among bitwise-equal energies (reading R6)
        double cj[N];
        {
            double pre = 0.0;
#pragma unroll
            for (int j = 0; j < N; ++j) {
                cj[j] = hp[j] - pre;
                pre += hp[j];
            }
        }
        double s = 0.0, m = 0.0;
        unsigned idx = 0;
#pragma unroll
        for (int k = 1; k < (1 << N); ++k) {
            s += cj[fs_ctz(k)];
            const double e = s + sT[k];
            if (e < m) {
                m = e;
                idx = k;
            }
        }
        bidx = idx;
        scored = (int64_t)total;
    }
    // Thresholded set of an open array: every dot has one or two values, i.e. base + a subset of the k free dots.  Walked in
    // Gray order over the free dots (one rank-1 update per candidate instead of the odometer's ~two); the running key
    // holds the digits with dot 0 most significant, so equal energies fall to the lexicographically smallest N (R6).
    const bool subset = !GRAY && !closed && args.alg == QA_ALG_THRESHOLDED;
    if (!GRAY && subset && live) {
        unsigned flist = 0;  // 4-bit dot indices of the free dots, highest dot first
        int k = 0;
#pragma unroll
        for (int i = N - 1; i >= 0; --i)
            if (cnt[i] == 2) flist |= (unsigned)i << (4 * k++);
        unsigned key = 0, bkey = 0;
        best = E;
        for (unsigned st = 1; st < (1u << k); ++st) {
            const int i = (int)((flist >> (4 * (__ffs(st) - 1))) & 15u);
            const unsigned bit = 1u << (N - 1 - i);
            const double dl = (key & bit) ? -1.0 : 1.0;
            double gi = 0.0;
#pragma unroll
            for (int j = 0; j < N; ++j)
                if (j == i) gi = grad[j];
            E += dl * (gi + 0.5 * dl * sM[i * N + i]);
#pragma unroll
            for (int j = 0; j < N; ++j) grad[j] = fma(dl, sM[j * N + i], grad[j]);
            key ^= bit;
            if (E < best || (E == best && key < bkey)) {
                best = E;
                bkey = key;
            }
        }
        bidx = bkey;  // binary digits, dot 0 most significant (decoded without division below)
        scored = (int64_t)total;
    }
    const uint64_t len = (live && !gray && !subset) ? total : 0;
    for (uint64_t it = 0; it < len; ++it) {
        if (!closed || sumN == args.N_hat) {
            ++scored;
            if (E < best) {
                best = E;
                bidx = it;
            }
        }
        if (it + 1 == len) break;
        bool carry = true;  // odometer step, least significant digit = dot N-1
#pragma unroll
        for (int i = N - 1; i >= 0; --i) {
            if (carry) {
                int delta;
                if (dg[i] == cnt[i] - 1) {
                    delta = -dg[i];
                    dg[i] = 0;
                } else {
                    delta = 1;
                    ++dg[i];
                    carry = false;
                }
                if (delta != 0) {
                    const double dl = (double)delta;
                    E += dl * (grad[i] + 0.5 * dl * sM[i * N + i]);
#pragma unroll
                    for (int j = 0; j < N; ++j) grad[j] = fma(dl, sM[j * N + i], grad[j]);
                    sumN += delta;
                }
            }
        }
    }

    // S7: N* = base + digits of the winner; E(N*) = 1/2 d^T M d from the definition (Eq. (C1))
    if (live) {
        const bool empty = bidx == ~0ull;
        int32_t Ns[N];
        if (gray || subset) {  // the winner's digits are the bits of bidx (64-bit division is ~100 instructions a digit)
#pragma unroll
            for (int i = 0; i < N; ++i) Ns[i] = base[i] + (int32_t)((bidx >> (N - 1 - i)) & 1ull);
        } else {
            uint64_t idx = bidx;
#pragma unroll
            for (int i = N - 1; i >= 0; --i) {
                const uint64_t c = (uint64_t)cnt[i];
                const int32_t dgt = (int32_t)(idx % c);
                idx /= c;
                Ns[i] = empty ? -1 : base[i] + dgt;
            }
        }
#pragma unroll
        for (int i = 0; i < N; ++i) d[i] = (double)Ns[i] - nc[i];
        double Ed = 0.0;
#pragma unroll
        for (int i = 0; i < N; ++i) {
            double row = 0.0;
#pragma unroll
            for (int j = 0; j < N; ++j) row = fma(sM[i * N + j], d[j], row);
            Ed = fma(d[i], row, Ed);
        }
        outE[gp] = empty ? INFINITY : 0.5 * Ed;
        if (mdl->ns == 0) {
#pragma unroll
            for (int i = 0; i < N; ++i) outN[gp * N + i] = Ns[i];
        } else {  // S8: sensor dots in the full model (single-model calls only: gp = p)
            qa_sensor_pixel(mdl, Vg, gp, Ns, outN, outVs);
        }
        if (xcont) {
#pragma unroll
            for (int i = 0; i < N; ++i) xcont[gp * N + i] = x[i];
        }
    }
    if (stats) {
        qa_warp_count(&stats->n_pixels, live ? 1 : 0);
        qa_warp_count(&stats->n_qp_pixels, (live && fl.neg) ? 1 : 0);
        qa_warp_count(&stats->n_qp_rounds, live ? fl.rounds : 0);
        qa_warp_count(&stats->n_qp_failed, (live && fl.failed) ? 1 : 0);
        qa_warp_count(&stats->n_threshold_doublings, live ? fl.doublings : 0);
        qa_warp_count(&stats->n_candidates_enumerated, live ? (int64_t)total : 0);
        qa_warp_count(&stats->n_candidates_scored, live ? scored : 0);
    }
}

template <int N>
cudaError_t launch_fused_n(const QaDevModel *const *d_models, int n_models, const double *d_Vg, int64_t P, QaCallArgs args,
                           int32_t *d_N, double *d_E, double *d_xcont, double *d_Vs, qa_stats *d_stats, cudaStream_t stream)
{
    const dim3 grid((unsigned)((P + FS_THREADS - 1) / FS_THREADS), (unsigned)n_models);
    if (args.alg == QA_ALG_DEFAULT && !args.closed)
        qa_fused_small_kernel<N, true><<<grid, FS_THREADS, 0, stream>>>(d_models, d_Vg, P, args, d_N, d_E, d_xcont, d_Vs, d_stats);
    else
        qa_fused_small_kernel<N, false><<<grid, FS_THREADS, 0, stream>>>(d_models, d_Vg, P, args, d_N, d_E, d_xcont, d_Vs, d_stats);
    return cudaGetLastError();
}

}  // namespace

// d_models: device array of n_models device model pointers (all with the same n <= QA_FUSED_MAXN dots and g gates, no
// sensor dots for n_models > 1); V_g is [n_models][P][g], N is [n_models][P][n], E is [n_models][P].  A single model with
// sensor dots writes N as [P][n_full] and the sensor potentials d_Vs [P][n_sensor] (may be NULL).
cudaError_t qa_launch_fused_small(const QaDevModel *const *d_models, int n_models, int n, const double *d_Vg, int64_t P,
                                  QaCallArgs args, int32_t *d_N, double *d_E, double *d_xcont, double *d_Vs,
                                  qa_stats *d_stats, cudaStream_t stream)
{
    qa_plan_add("qa_fused_small_kernel");
    if (n_models > 65535) return cudaErrorInvalidValue;
#define CALL(NN) launch_fused_n<NN>(d_models, n_models, d_Vg, P, args, d_N, d_E, d_xcont, d_Vs, d_stats, stream)
    switch (n) {
        case 1: return CALL(1);
        case 2: return CALL(2);
        case 3: return CALL(3);
        case 4: return CALL(4);
        case 5: return CALL(5);
        case 6: return CALL(6);
        case 7: return CALL(7);
        case 8: return CALL(8);
        default: return cudaErrorInvalidValue;
    }
#undef CALL
}
