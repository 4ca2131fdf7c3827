// qa_kernels_walk.cu -- the hot kernel: default algorithm, open array (S5 + S6 of SURVEY.md section 8(a)).
//
// Every pixel scores all 2^n floor/ceil candidates N = base + b, b in {0,1}^n (L123-L127).  With d0 = base - N_c,
//     E(base + b) = E(base) + sum_i b_i h_i + sum_{i<j} b_i b_j M_ij,     h_i = [M d0]_i + 1/2 M_ii          (from (C1) L607)
// so the pixel enters only through the n numbers h_i (written by the prologue); the pair term is pixel-independent.
//
// Decomposition (B200: FP64 pipe bound, 64 lanes/SM): the n bits are split into NH high bits, one thread per high
// pattern t (2^NH threads share a pixel), and NL <= 8 low bits walked by each thread in counting order (each step moves
// the linear part by a per-pixel constant c_ctz(k), like a Gray step, and ascending order makes the tie-break of
// reading R6 free), fully unrolled so that every index is static:
//     per thread, once:   v_j  = sum_{hi bit j' in t} M[a_j][a_j']          (cross term hi x lo, pixel-independent)
//                         QH   = sum_{hi pairs in t} M                      (pixel-independent)
//     per thread x pixel: h'_j = h[a_j] + v_j   (NL adds),   base_t = QH + sum_{hi bits in t} h   (<= NH adds)
//     per candidate:      s += c_ctz(k), c_j = h'_j - sum_{i<j} h'_i   1 DADD   (running linear part of pattern k)
//                         e  = s + QL[k]                        1 DADD   (pair table of the low bits, constant bank)
//                         (e < m) ? (m, idx) = (e, k)           1 DSETP + selects
// i.e. 3 FP64-pipe instructions per candidate, independent of n (the definition costs n^2 + n FMAs, the lazy Gray update
// of SURVEY.md section 8(d) about 5.5).  The winner over the 2^NH threads is taken by a lexicographic (E, index) min over
// shuffles / shared memory, so the result does not depend on scheduling.  E(N*) itself is recomputed from the definition
// by the finalize kernel; the incremental energies only decide the argmin (drift << the 1e-9 E_C near-tie rule).
//
// Index convention: candidate index = sum_i b_i 2^(n-1-i) (dot 0 most significant) = the mixed-radix index the generic
// enumeration and the finalize kernel use for cnt_i = 2.  Low bit j <-> dot n-1-j; high bit j' of t <-> dot n-1-NL-j'.
#include "qa_internal.cuh"

namespace {

constexpr int WALK_THREADS = 256;

__host__ __device__ constexpr int qa_ctz(int k)
{
    int j = 0;
    while (((k >> j) & 1) == 0) ++j;
    return j;
}

template <int NL, int NH>
__global__ void __launch_bounds__(WALK_THREADS) qa_walk_kernel(const QaDevModel *__restrict__ mdl,
                                                               const __grid_constant__ QaWalkTable tab, QaWorkspace ws)
{
    constexpr int N = NL + NH;
    constexpr int TPP = 1 << NH;               // threads per pixel
    constexpr int PPC = WALK_THREADS / TPP;    // pixels per CTA iteration
    constexpr int WPP = TPP > 32 ? TPP / 32 : 1;  // warps per pixel
    __shared__ double sE[2][WALK_THREADS / 32];
    __shared__ unsigned sI[2][WALK_THREADS / 32];

    const unsigned t = threadIdx.x & (TPP - 1);
    const int slot = threadIdx.x >> NH;
    const int64_t P = ws.P;

    // pixel-independent per-thread constants
    double v[NL];
    double QH = 0.0;
#pragma unroll
    for (int j = 0; j < NL; ++j) {
        double s = 0.0;
#pragma unroll
        for (int jh = 0; jh < NH; ++jh)
            if ((t >> jh) & 1u) s += mdl->M[(N - 1 - j) * QA_MAXN + (N - 1 - NL - jh)];
        v[j] = s;
    }
#pragma unroll
    for (int jh = 0; jh < NH; ++jh)
#pragma unroll
        for (int jh2 = jh + 1; jh2 < NH; ++jh2)
            if (((t >> jh) & 1u) && ((t >> jh2) & 1u)) QH += mdl->M[(N - 1 - NL - jh) * QA_MAXN + (N - 1 - NL - jh2)];

    qa_pdl_launch_dependents();
    qa_pdl_wait();  // the constants above are model data; h comes from the prologue kernel
    const int64_t groups = (P + PPC - 1) / PPC;
    int buf = 0;
    for (int64_t grp = blockIdx.x; grp < groups; grp += gridDim.x, buf ^= 1) {
        const int64_t p = grp * PPC + slot;
        const bool live = p < P;
        const int64_t pp = live ? p : P - 1;
        double hp[NL];
#pragma unroll
        for (int j = 0; j < NL; ++j) hp[j] = ws.h[(int64_t)(N - 1 - j) * P + pp] + v[j];
        double baseE = QH;
#pragma unroll
        for (int jh = 0; jh < NH; ++jh)
            if ((t >> jh) & 1u) baseE += ws.h[(int64_t)(N - 1 - NL - jh) * P + pp];

        // Walk over the 2^NL low patterns in counting order k = 0, 1, 2, ...: the step k-1 -> k sets bit j = ctz(k) and clears
        // the bits below it, so the linear part moves by c_j = h'_j - sum_{i<j} h'_i whatever k is (one DADD, like a Gray
        // step), and because k ascends the strict '<' keeps the smallest index among bitwise-equal energies (reading R6).
        // k = 0 is the all-zero pattern with e = 0.
        double cj[NL];
        {
            double pre = 0.0;
#pragma unroll
            for (int j = 0; j < NL; ++j) {
                cj[j] = hp[j] - pre;
                pre += hp[j];
            }
        }
        double s = 0.0, m = 0.0;
        unsigned idx = 0;
#pragma unroll
        for (int k = 1; k < (1 << NL); ++k) {
            s += cj[qa_ctz(k)];
            const double e = s + tab.QL[k];
            if (e < m) {
                m = e;
                idx = k;
            }
        }
        double tot = m + baseE;
        unsigned full = (t << NL) | idx;

        if (NH > 0) {
            constexpr int W = TPP < 32 ? TPP : 32;
#pragma unroll
            for (int o = W / 2; o > 0; o >>= 1) {
                const double e2 = __shfl_xor_sync(0xffffffffu, tot, o);
                const unsigned i2 = __shfl_xor_sync(0xffffffffu, full, o);
                if (e2 < tot || (e2 == tot && i2 < full)) {
                    tot = e2;
                    full = i2;
                }
            }
            if (WPP > 1) {
                const int w = threadIdx.x >> 5;
                if ((threadIdx.x & 31) == 0) {
                    sE[buf][w] = tot;
                    sI[buf][w] = full;
                }
                __syncthreads();
                if (t == 0) {
#pragma unroll
                    for (int q = 1; q < WPP; ++q) {
                        const double e2 = sE[buf][w + q];
                        const unsigned i2 = sI[buf][w + q];
                        if (e2 < tot || (e2 == tot && i2 < full)) {
                            tot = e2;
                            full = i2;
                        }
                    }
                }
            }
        }
        if (live && t == 0) ws.best[p] = (uint64_t)full;
    }
}

template <int NL, int NH>
cudaError_t launch_walk(const QaDevModel *d_model, const QaWalkTable &tab, QaWorkspace ws, int sm_count,
                        cudaStream_t stream)
{
    constexpr int PPC = WALK_THREADS >> NH;
    const int64_t groups = (ws.P + PPC - 1) / PPC;
    int per_sm = 0;
    cudaError_t err =
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, qa_walk_kernel<NL, NH>, WALK_THREADS, 0);
    if (err != cudaSuccess) return err;
    if (per_sm < 1) per_sm = 1;
    int64_t grid = (int64_t)sm_count * per_sm;
    if (grid > groups) grid = groups;
    return qa_launch_pdl(qa_walk_kernel<NL, NH>, dim3((unsigned)grid), dim3(WALK_THREADS), stream, d_model, tab, ws);
}

}  // namespace

cudaError_t qa_launch_walk(const QaDevModel *d_model, int n, const QaWalkTable &tab, QaWorkspace ws, qa_stats *d_stats,
                           int sm_count, cudaStream_t stream)
{
    (void)d_stats;
    qa_plan_add("qa_walk_kernel");
    switch (n) {
        case 1: return launch_walk<1, 0>(d_model, tab, ws, sm_count, stream);
        case 2: return launch_walk<2, 0>(d_model, tab, ws, sm_count, stream);
        case 3: return launch_walk<3, 0>(d_model, tab, ws, sm_count, stream);
        case 4: return launch_walk<4, 0>(d_model, tab, ws, sm_count, stream);
        case 5: return launch_walk<5, 0>(d_model, tab, ws, sm_count, stream);
        case 6: return launch_walk<6, 0>(d_model, tab, ws, sm_count, stream);
        case 7: return launch_walk<7, 0>(d_model, tab, ws, sm_count, stream);
        case 8: return launch_walk<8, 0>(d_model, tab, ws, sm_count, stream);
        case 9: return launch_walk<8, 1>(d_model, tab, ws, sm_count, stream);
        case 10: return launch_walk<8, 2>(d_model, tab, ws, sm_count, stream);
        case 11: return launch_walk<8, 3>(d_model, tab, ws, sm_count, stream);
        case 12: return launch_walk<8, 4>(d_model, tab, ws, sm_count, stream);
        case 13: return launch_walk<8, 5>(d_model, tab, ws, sm_count, stream);
        case 14: return launch_walk<8, 6>(d_model, tab, ws, sm_count, stream);
        case 15: return launch_walk<8, 7>(d_model, tab, ws, sm_count, stream);
        case 16: return launch_walk<8, 8>(d_model, tab, ws, sm_count, stream);
        default: return cudaErrorInvalidValue;
    }
}
