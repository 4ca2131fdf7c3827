// qa_kernels_fused_mid.cu -- the whole path S1-S7 in ONE kernel for OPEN arrays of 9..12 dots with the default algorithm
// (2^9 .. 2^12 candidates per pixel).  With three launches (prologue, walk, finalize) a 100x100 diagram of such an array
// is bound by launch gaps and cold starts (0.04 - 0.065 ms for 5*10^6 .. 4*10^7 candidates); here a warp carries TWO pixels
// through the whole path and nothing goes through global memory in between:
//   S1-S4   sixteen lanes per pixel (qa_prologue_lanes.cuh: lane i <-> dot i, fixed fma chain of N_c, QP in registers),
//   S5-S6   the two pixels one after the other, all 32 lanes: lane t owns the pattern t of the five high bits and walks the
//           2^(N-5) low patterns in counting order (the static walk of qa_kernels_walk.cu: 3 FP64 instructions per
//           candidate, exact compare, ascending index: reading R6); the h_i of the pixel travel by shuffles; the warp's
//           winner is a lexicographic (energy, index) minimum (three warp reductions on a monotone integer key),
//   S7      sixteen lanes per pixel again: N*_i, d_i, row i of M d by shuffles, E(N*) from the definition (Eq. (C1)).
// V_g is the only global read, N*, E(N*) (and x) the only writes.  Models with sensor dots, thresholded and brute-force
// sets and closed arrays keep the three-kernel path.
#include "qa_internal.cuh"
#include "qa_prologue_lanes.cuh"

namespace {

constexpr int FM_THREADS = 256;
constexpr int FM_PPB = FM_THREADS / 16;  // pixels per CTA

__host__ __device__ constexpr int fm_ctz(int k)
{
    int j = 0;
    while (((k >> j) & 1) == 0) ++j;
    return j;
}

// monotone map double -> uint64 (orders like the values, negative ones included)
__device__ __forceinline__ unsigned long long fm_key(double e)
{
    const unsigned long long b = (unsigned long long)__double_as_longlong(e);
    return (b >> 63) ? ~b : (b | 0x8000000000000000ull);
}

template <int N>
__global__ void __launch_bounds__(FM_THREADS) qa_fused_mid_kernel(const QaDevModel *__restrict__ mdl,
                                                                  const __grid_constant__ QaWalkTable tab,
                                                                  const double *__restrict__ Vg, int64_t P, QaCallArgs args,
                                                                  int32_t *__restrict__ outN, double *__restrict__ outE,
                                                                  double *__restrict__ xcont, qa_stats *stats)
{
    constexpr int NH = 5, NL = N - NH;
    static_assert(N >= 9 && N <= 12, "five high bits = one lane each, 4..7 low bits per lane");
    __shared__ double sCgT[QA_MAXG * N], sC[N * N], sMT[N * N], sV[FM_PPB][QA_MAXG], sX[FM_PPB][2 * N], sC1[N];
    const int g = mdl->g;
    const int tid = threadIdx.x;
    for (int e = tid; e < N * N; e += FM_THREADS) {
        sMT[e] = mdl->M[(e % N) * QA_MAXN + (e / N)];
        sC[e] = mdl->C[(e / N) * QA_MAXN + (e % N)];
    }
    for (int e = tid; e < N * g; e += FM_THREADS) sCgT[e] = mdl->Cgd[(e % N) * QA_MAXG + (e / N)];
    if (tid < N) sC1[tid] = mdl->C1[tid];
    const int64_t p0 = (int64_t)blockIdx.x * FM_PPB;
    for (int e = tid; e < FM_PPB * g; e += FM_THREADS) {
        const int64_t pe = p0 + e / g;
        sV[e / g][e % g] = pe < P ? __ldg(Vg + p0 * g + e) : 0.0;
    }
    __syncthreads();

    const unsigned lane = tid & 31u;
    const unsigned t = lane;                 // high pattern of this lane in the walk
    const int i = tid & 15;                  // dot of this lane in the per-pixel phases
    const int s = tid >> 4;                  // pixel slot
    const int gb = (int)(lane & 16u);
    const int64_t p = p0 + s;
    const bool live = p < P;
    const bool dot = i < N;

    // pixel-independent constants of the walk: cross terms of t with the low bits, pair energy of t (M is symmetric)
    double v[NL], QH = 0.0;
#pragma unroll
    for (int j = 0; j < NL; ++j) {
        double sv = 0.0;
#pragma unroll
        for (int jh = 0; jh < NH; ++jh)
            if ((t >> jh) & 1u) sv += sMT[(N - 1 - j) * N + (N - 1 - NL - jh)];
        v[j] = sv;
    }
#pragma unroll
    for (int jh = 0; jh < NH; ++jh)
#pragma unroll
        for (int jh2 = jh + 1; jh2 < NH; ++jh2)
            if (((t >> jh) & 1u) && ((t >> jh2) & 1u)) QH += sMT[(N - 1 - NL - jh) * N + (N - 1 - NL - jh2)];

    // ---- S1-S4 + base-point gradient, sixteen lanes per pixel
    QaLaneOut lo;
    qa_lanes_pixel<N>(sCgT, sC, sMT, sC1, 1.0, sV[s], sX[s], g, i, gb, dot, args, lo);  // (open: 1^T C 1 is not read)
    const double h = dot ? lo.gi + 0.5 * sMT[i * N + i] : 0.0;  // E(base + e_i) - E(base)

    // ---- S5-S6: the warp's two pixels, one after the other
    unsigned win = 0;
#pragma unroll 1
    for (int q = 0; q < 2; ++q) {
        const int src = q << 4;
        double hp[NL];
#pragma unroll
        for (int j = 0; j < NL; ++j) hp[j] = __shfl_sync(0xffffffffu, h, src + N - 1 - j) + v[j];
        double baseE = QH;
#pragma unroll
        for (int jh = 0; jh < NH; ++jh) {
            const double hv = __shfl_sync(0xffffffffu, h, src + N - 1 - NL - jh);
            if ((t >> jh) & 1u) baseE += hv;
        }
        // counting-order walk over the 2^NL low patterns (qa_kernels_walk.cu): step k-1 -> k sets bit ctz(k) and clears the
        // bits below it, the linear part moves by c_j = h'_j - sum_{i<j} h'_i; k = 0 is the all-zero pattern with e = 0
        double cj[NL];
        {
            double pre = 0.0;
#pragma unroll
            for (int j = 0; j < NL; ++j) {
                cj[j] = hp[j] - pre;
                pre += hp[j];
            }
        }
        double sl = 0.0, m = 0.0;
        unsigned idx = 0;
#pragma unroll
        for (int k = 1; k < (1 << NL); ++k) {
            sl += cj[fm_ctz(k)];
            const double e = sl + tab.QL[k];
            if (e < m) {
                m = e;
                idx = k;
            }
        }
        const double tot = m + baseE;
        const unsigned full = (t << NL) | idx;
        const unsigned long long key = fm_key(tot);
        const unsigned khi = (unsigned)(key >> 32), klo = (unsigned)key;
        const unsigned mhi = __reduce_min_sync(0xffffffffu, khi);
        const unsigned mlo = __reduce_min_sync(0xffffffffu, khi == mhi ? klo : 0xffffffffu);
        const unsigned mi = __reduce_min_sync(0xffffffffu, (khi == mhi && klo == mlo) ? full : 0xffffffffu);
        if (gb == src) win = mi;
    }

    // ---- S7: N* = base + bits of the winner, E(N*) = 1/2 d^T M d from the definition; sixteen lanes per pixel
    const int32_t Ni = lo.base + (int32_t)((win >> (N - 1 - (dot ? i : 0))) & 1u);
    const double d = dot ? (double)Ni - lo.nc : 0.0;
    double row = 0.0;
    const int ii = dot ? i : 0;
#pragma unroll
    for (int j = 0; j < N; ++j) row = fma(sMT[j * N + ii], __shfl_sync(0xffffffffu, d, gb + j), row);
    double E = dot ? d * row : 0.0;
#pragma unroll
    for (int o = 8; o > 0; o >>= 1) E += __shfl_xor_sync(0xffffffffu, E, o);
    if (live && dot) {
        outN[p * N + i] = Ni;
        if (xcont) xcont[p * N + i] = lo.x;
    }
    if (live && i == 0) outE[p] = 0.5 * E;
    if (stats) {
        const bool one = live && i == 0;
        qa_warp_count(&stats->n_pixels, one ? 1 : 0);
        qa_warp_count(&stats->n_qp_pixels, (one && lo.neg0 != 0u) ? 1 : 0);
        qa_warp_count(&stats->n_qp_rounds, one ? lo.rounds : 0);
        qa_warp_count(&stats->n_qp_failed, (one && lo.failed) ? 1 : 0);
        qa_warp_count(&stats->n_candidates_enumerated, one ? (int64_t)lo.total : 0);
        qa_warp_count(&stats->n_candidates_scored, one ? (int64_t)lo.total : 0);
    }
}

template <int N>
cudaError_t launch_fm(const QaDevModel *d_model, const QaWalkTable &tab, const double *d_Vg, int64_t P, QaCallArgs args,
                      int32_t *d_N, double *d_E, double *d_xcont, qa_stats *d_stats, cudaStream_t stream)
{
    const unsigned blocks = (unsigned)((P + FM_PPB - 1) / FM_PPB);
    qa_fused_mid_kernel<N><<<blocks, FM_THREADS, 0, stream>>>(d_model, tab, d_Vg, P, args, d_N, d_E, d_xcont, d_stats);
    return cudaGetLastError();
}

}  // namespace

// Open array, default algorithm, 9 <= n <= 12, no sensor dots.
cudaError_t qa_launch_fused_mid(const QaDevModel *d_model, int n, const QaWalkTable &tab, const double *d_Vg, int64_t P,
                                QaCallArgs args, int32_t *d_N, double *d_E, double *d_xcont, qa_stats *d_stats,
                                cudaStream_t stream)
{
    qa_plan_add("qa_fused_mid_kernel");
    switch (n) {
        case 9: return launch_fm<9>(d_model, tab, d_Vg, P, args, d_N, d_E, d_xcont, d_stats, stream);
        case 10: return launch_fm<10>(d_model, tab, d_Vg, P, args, d_N, d_E, d_xcont, d_stats, stream);
        case 11: return launch_fm<11>(d_model, tab, d_Vg, P, args, d_N, d_E, d_xcont, d_stats, stream);
        case 12: return launch_fm<12>(d_model, tab, d_Vg, P, args, d_N, d_E, d_xcont, d_stats, stream);
        default: return cudaErrorInvalidValue;
    }
}
