// qa_kernels_closed.cu -- closed arrays at scale (Fig. 4(b)):
// default algorithm, closed array, 9 <= n <= 16.  Of the 2^n floor/ceil candidates N = base + b only those with
// sum_i N_i = N_hat are admissible, i.e. popcount(b) = k := N_hat - sum_i base_i -- C(n, k) states (12 870 of 65 536 at
// n = 16, k = 8).  This kernel visits ONLY those: no state with the wrong total is ever formed.
//
// Same separation of (C1) L607 as the min-plus walk (qa_kernels_minplus.cu): bits w = [0,4), u = [4,8), t = [8,n) (low bit
// j <-> dot n-1-j), one thread per high pattern t of a pixel,
//     e(t,u,w) = A[u] + ( B[w] + QL[u,w] ),   B[w] = sum_{j in w} h'_j,   A[u] = be + sum_{j in u} h'_j,
//     h'_j = h_j + VT[t][j],   be = E(base) + QHT[t] + sum_{jh in t} h_jh,   QL = pair energies of the low 8 bits
// and the admissible (u, w) of a thread are those with popcount(u) + popcount(w) = kr := k - popcount(t): for every u the
// popcount class kr - popcount(u) of the 4-bit patterns w (1, 4, 6, 4, 1 members).  The loop over u and the members of each
// class are unrolled, so every register and table index is static (the table is a kernel parameter: constant bank); what is
// dynamic is only WHICH class a thread walks for a given u.  To keep that choice uniform inside a warp the 2^NH patterns
// t are handed to the threads sorted by popcount (colex rank inside a class), so at most two or three classes meet in a warp.
// Per candidate: 2 DADD + 1 DSETP (the energy itself is compared, exactly; ascending index order + strict '<' gives the
// lexicographically smallest N among bitwise ties, reading R6); the winner over the threads of the pixel is a
// lexicographic (e, index) minimum.  E(N*) is recomputed from the definition by qa_finalize_kernel.
//
// Works for any SPD c_dd (no positivity offsets are used).  Index convention as in qa_kernels_walk.cu.
#include "qa_internal.cuh"

namespace {

constexpr int CW_THREADS = 256;

__host__ __device__ constexpr int cw_popc4(int x) { return (x & 1) + ((x >> 1) & 1) + ((x >> 2) & 1) + ((x >> 3) & 1); }
// number of 4-bit patterns of popcount c, and the i-th of them in ascending order
__host__ __device__ constexpr int cw_cls_n(int c) { return c == 0 || c == 4 ? 1 : (c == 2 ? 6 : 4); }
__host__ __device__ constexpr int cw_cls_w(int c, int i)
{
    int seen = 0;
    for (int w = 0; w < 16; ++w)
        if (cw_popc4(w) == c) {
            if (seen == i) return w;
            ++seen;
        }
    return 0;
}
__host__ __device__ constexpr int cw_binom(int n, int k)
{
    if (k < 0 || k > n) return 0;
    long long r = 1;
    for (int i = 1; i <= k; ++i) r = r * (n - k + i) / i;
    return (int)r;
}
__host__ __device__ constexpr int cw_ctz(int k)
{
    int j = 0;
    while (((k >> j) & 1) == 0) ++j;
    return j;
}

// the members I, I+1, ... of class C for a given u, in ascending w (static recursion: every index is a constant)
template <int U, int C, int I>
__device__ __forceinline__ void cw_class(const QaWalkTable &tab, const double (&B)[16], double a, double &best, unsigned &bi)
{
    if constexpr (I < cw_cls_n(C)) {
        constexpr int w = cw_cls_w(C, I);
        const double e = a + (B[w] + tab.QL[(U << 4) | w]);
        if (e < best) {
            best = e;
            bi = (unsigned)((U << 4) | w);
        }
        cw_class<U, C, I + 1>(tab, B, a, best, bi);
    }
}

template <int U>
__device__ __forceinline__ void cw_u(const QaWalkTable &tab, const double (&B)[16], double a, int kr, double &best,
                                     unsigned &bi)
{
    const int c = kr - cw_popc4(U);
    if (c == 0) cw_class<U, 0, 0>(tab, B, a, best, bi);
    else if (c == 1) cw_class<U, 1, 0>(tab, B, a, best, bi);
    else if (c == 2) cw_class<U, 2, 0>(tab, B, a, best, bi);
    else if (c == 3) cw_class<U, 3, 0>(tab, B, a, best, bi);
    else if (c == 4) cw_class<U, 4, 0>(tab, B, a, best, bi);
}

template <int U>
struct CwLoop {
    static __device__ __forceinline__ void run(const QaWalkTable &tab, const double (&B)[16], const double (&A)[16], int kr,
                                               double &best, unsigned &bi)
    {
        cw_u<U>(tab, B, A[U], kr, best, bi);
        CwLoop<U + 1>::run(tab, B, A, kr, best, bi);
    }
};
template <>
struct CwLoop<16> {
    static __device__ __forceinline__ void run(const QaWalkTable &, const double (&)[16], const double (&)[16], int, double &,
                                               unsigned &)
    {
    }
};

template <int NH>
__global__ void __launch_bounds__(CW_THREADS) qa_closed_walk_kernel(const QaDevModel *__restrict__ mdl,
                                                                    const __grid_constant__ QaWalkTable tab, QaWorkspace ws,
                                                                    QaCallArgs args, qa_stats *stats)
{
    constexpr int NL = QA_WALK_NL;
    constexpr int N = NL + NH;
    constexpr int TPP = 1 << NH;            // threads per pixel
    constexpr int PPB = CW_THREADS / TPP;   // pixels per CTA
    constexpr int WPP = TPP > 32 ? TPP / 32 : 1;
    static_assert(NL == 8 && NH >= 1 && NH <= 8, "low bits = two groups of four");
    __shared__ double sIn[PPB][N + 1];
    __shared__ int sK[PPB];
    __shared__ unsigned char sPerm[TPP];
    __shared__ double sE[CW_THREADS / 32];
    __shared__ unsigned sI[CW_THREADS / 32];

    const unsigned r = threadIdx.x & (TPP - 1);
    const int slot = threadIdx.x >> NH;
    const int64_t P = ws.P;
    // patterns sorted by popcount, colex rank inside a class: rank(x) = #(popcount < pc) + sum_i C(p_i, i), p_1 < p_2 < ...
    if (threadIdx.x < TPP) {
        const unsigned x = threadIdx.x;
        const int pc = __popc(x);
        int rank = 0;
        for (int c = 0; c < pc; ++c) rank += cw_binom(NH, c);
        int i = 0;
        for (int b = 0; b < NH; ++b)
            if ((x >> b) & 1u) rank += cw_binom(b, ++i);
        sPerm[rank] = (unsigned char)x;
    }
    __syncthreads();
    const unsigned t = sPerm[r];
    double v[NL];
#pragma unroll
    for (int j = 0; j < NL; ++j) v[j] = mdl->VT[t * NL + j];
    const double QH = mdl->QHT[t];
    qa_pdl_launch_dependents();
    qa_pdl_wait();  // model constants above; h, e0, base come from the prologue kernel

    // persistent: a CTA walks pixel groups blockIdx.x, blockIdx.x + gridDim.x, ... (the per-thread tables above are loaded once)
    const int64_t groups = (P + PPB - 1) / PPB;
    for (int64_t grp = blockIdx.x; grp < groups; grp += gridDim.x) {
        const int64_t p0 = grp * PPB;
        if (threadIdx.x < PPB) sK[threadIdx.x] = 0;
        __syncthreads();  // also: the previous group's sIn / sE / sI have been read
        for (int e = threadIdx.x; e < PPB * (N + 1); e += CW_THREADS) {
            const int s = e / (N + 1), i = e % (N + 1);
            int64_t p = p0 + s;
            if (p >= P) p = P - 1;
            if (i < N) {
                sIn[s][i] = __ldg(ws.h + (int64_t)i * P + p);
                atomicAdd(&sK[s], ws.base[(int64_t)i * P + p]);
            } else {
                sIn[s][N] = __ldg(ws.e0 + p);
            }
        }
        __syncthreads();
        const int64_t p = p0 + slot;
        const bool live = p < P;
        const int k = args.N_hat - sK[slot];  // ones to place
        const int kr = k - __popc(t);

        double best = INFINITY;
        unsigned bi = 0xffffffffu;
        if (kr >= 0 && kr <= NL) {
            double hp[NL];
#pragma unroll
            for (int j = 0; j < NL; ++j) hp[j] = sIn[slot][N - 1 - j] + v[j];
            double be = sIn[slot][N] + QH;
#pragma unroll
            for (int jh = 0; jh < NH; ++jh)
                if ((t >> jh) & 1u) be += sIn[slot][N - 1 - NL - jh];
            double B[16], A[16];
            B[0] = 0.0;
            A[0] = be;
#pragma unroll
            for (int w = 1; w < 16; ++w) {
                B[w] = B[w & (w - 1)] + hp[cw_ctz(w)];
                A[w] = A[w & (w - 1)] + hp[4 + cw_ctz(w)];
            }
            CwLoop<0>::run(tab, B, A, kr, best, bi);
            if (bi != 0xffffffffu) bi |= t << NL;
        }

        // lexicographic (e, index) minimum over the threads of the pixel
        constexpr int W = TPP < 32 ? TPP : 32;
#pragma unroll
        for (int o = W / 2; o > 0; o >>= 1) {
            const double e2 = __shfl_xor_sync(0xffffffffu, best, o);
            const unsigned i2 = __shfl_xor_sync(0xffffffffu, bi, o);
            if (e2 < best || (e2 == best && i2 < bi)) {
                best = e2;
                bi = i2;
            }
        }
        if (WPP > 1) {
            const int wq = threadIdx.x >> 5;
            if ((threadIdx.x & 31) == 0) {
                sE[wq] = best;
                sI[wq] = bi;
            }
            __syncthreads();
            if (r == 0) {
#pragma unroll
                for (int q = 1; q < WPP; ++q) {
                    const double e2 = sE[wq + q];
                    const unsigned i2 = sI[wq + q];
                    if (e2 < best || (e2 == best && i2 < bi)) {
                        best = e2;
                        bi = i2;
                    }
                }
            }
        }
        if (live && r == 0) {
            ws.best[p] = bi == 0xffffffffu ? ~0ull : (uint64_t)bi;
            if (stats) qa_atomic_add64(&stats->n_candidates_scored, (int64_t)cw_binom(N, k));
        }
    }
}

template <int NH>
cudaError_t launch_cw(const QaDevModel *d_model, const QaWalkTable &tab, QaWorkspace ws, QaCallArgs args, qa_stats *d_stats,
                      int sm_count, cudaStream_t stream)
{
    constexpr int PPB = CW_THREADS >> NH;
    const int64_t groups = (ws.P + PPB - 1) / PPB;
    int per_sm = 0;
    cudaError_t err = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, qa_closed_walk_kernel<NH>, CW_THREADS, 0);
    if (err != cudaSuccess) return err;
    if (per_sm < 1) per_sm = 1;
    int64_t grid = (int64_t)sm_count * per_sm;
    if (grid > groups) grid = groups;
    return qa_launch_pdl(qa_closed_walk_kernel<NH>, dim3((unsigned)grid), dim3(CW_THREADS), stream, d_model, tab, ws, args,
                         d_stats);
}

}  // namespace

cudaError_t qa_launch_closed_walk(const QaDevModel *d_model, int n, const QaWalkTable &tab, QaWorkspace ws, QaCallArgs args,
                                  qa_stats *d_stats, int sm_count, cudaStream_t stream)
{
    qa_plan_add("qa_closed_walk_kernel");
    switch (n) {
        case 9: return launch_cw<1>(d_model, tab, ws, args, d_stats, sm_count, stream);
        case 10: return launch_cw<2>(d_model, tab, ws, args, d_stats, sm_count, stream);
        case 11: return launch_cw<3>(d_model, tab, ws, args, d_stats, sm_count, stream);
        case 12: return launch_cw<4>(d_model, tab, ws, args, d_stats, sm_count, stream);
        case 13: return launch_cw<5>(d_model, tab, ws, args, d_stats, sm_count, stream);
        case 14: return launch_cw<6>(d_model, tab, ws, args, d_stats, sm_count, stream);
        case 15: return launch_cw<7>(d_model, tab, ws, args, d_stats, sm_count, stream);
        case 16: return launch_cw<8>(d_model, tab, ws, args, d_stats, sm_count, stream);
        default: return cudaErrorInvalidValue;
    }
}
