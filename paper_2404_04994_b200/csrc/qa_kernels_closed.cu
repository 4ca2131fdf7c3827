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
// dynamic is only WHICH class a thread walks for a given u.  The work of a pattern follows C(8, k - popcount(t)) (70 states
// for the middle class, 1 for the outer ones), so the patterns are cut into BLOCKS of up to 32 of (nearly) one popcount
// (host table CwBlocks) and a WORK ITEM is (pixel, block): every warp is an independent worker over the items
// gw, gw + #warps, ... -- no CTA barrier, lanes of a warp walk the same class, light and heavy blocks mix over the grid.
// Per candidate: 2 DADD + 1 DSETP (the energy itself is compared, exactly; ascending index order + strict '<' gives the
// lexicographically smallest N among bitwise ties, reading R6); the warp's winner (lexicographic (e, index) minimum, three
// warp reductions on a monotone integer key of the energy) is one 16-byte record per item, and qa_finalize_kernel takes the
// lexicographic minimum of a pixel's records before it decodes N* and recomputes E(N*) from the definition.
//
// Works for any SPD c_dd (no positivity offsets are used).  Index convention as in qa_kernels_walk.cu.
#include <cstring>

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

// blocks of high patterns: up to 32 patterns per block, a class of >= 16 patterns starts its own block
struct CwBlocks {
    int nb;
    unsigned mask[QA_CLOSED_MAXB];
    unsigned char t[QA_CLOSED_MAXB][32];
};

// monotone map double -> uint64 (orders like the values, negative ones included)
__device__ __forceinline__ unsigned long long cw_key(double e)
{
    const unsigned long long b = (unsigned long long)__double_as_longlong(e);
    return (b >> 63) ? ~b : (b | 0x8000000000000000ull);
}
__device__ __forceinline__ double cw_unkey(unsigned long long k)
{
    const unsigned long long b = (k >> 63) ? (k & 0x7fffffffffffffffull) : ~k;
    return __longlong_as_double((long long)b);
}

template <int NH>
__global__ void __launch_bounds__(CW_THREADS, 3) qa_closed_walk_kernel(const QaDevModel *__restrict__ mdl,
                                                                       const __grid_constant__ QaWalkTable tab,
                                                                       const __grid_constant__ CwBlocks blk, QaWorkspace ws,
                                                                       QaCallArgs args)
{
    constexpr int NL = QA_WALK_NL;
    constexpr int N = NL + NH;
    constexpr int WARPS = CW_THREADS / 32;
    static_assert(NL == 8 && NH >= 1 && NH <= 8, "low bits = two groups of four");
    __shared__ double sIn[WARPS][N + 1];
    const unsigned lane = threadIdx.x & 31u;
    const int wid = threadIdx.x >> 5;
    const int64_t P = ws.P;
    const int NB = blk.nb;
    const int64_t items = P * NB;
    const bool small = items < 0x7fffffff;  // 32-bit division of the item index (a 64-bit one costs ~100 instructions)
    auto pixel_of = [&](int64_t item) -> int64_t {
        return small ? (int64_t)((unsigned)item / (unsigned)NB) : item / NB;
    };
    const int64_t gw = (int64_t)wid * gridDim.x + blockIdx.x;  // consecutive warps sit in different CTAs
    const int64_t tw = (int64_t)gridDim.x * WARPS;
    qa_pdl_launch_dependents();
    qa_pdl_wait();  // h, e0, base come from the prologue kernel

    // inputs of an item's pixel, one value per lane, requested one item ahead
    double in_v = 0.0;
    int in_base = 0;
    auto request = [&](int64_t item) {
        if (item >= items) return;
        const int64_t p = pixel_of(item);
        if (lane <= (unsigned)N) in_v = lane < (unsigned)N ? __ldg(ws.h + (int64_t)lane * P + p) : __ldg(ws.e0 + p);
        in_base = lane < (unsigned)N ? ws.base[(int64_t)lane * P + p] : 0;
    };
    request(gw);
    for (int64_t item = gw; item < items; item += tw) {
        const int64_t p = pixel_of(item);
        const int b = (int)(item - p * NB);
        const int k = args.N_hat - __reduce_add_sync(0xffffffffu, in_base);  // ones to place
        if (lane <= (unsigned)N) sIn[wid][lane] = in_v;
        __syncwarp();
        request(item + tw);
        const bool active = (blk.mask[b] >> lane) & 1u;
        const unsigned t = blk.t[b][lane];
        const int kr = k - __popc(t);
        double best = INFINITY;
        unsigned bi = 0xffffffffu;
        if (active && kr >= 0 && kr <= NL) {
            const double *__restrict__ h = sIn[wid];
            double hp[NL];
#pragma unroll
            for (int j = 0; j < NL; ++j) hp[j] = h[N - 1 - j] + __ldg(mdl->VT + t * NL + j);
            double be = h[N] + __ldg(mdl->QHT + t);
#pragma unroll
            for (int jh = 0; jh < NH; ++jh)
                if ((t >> jh) & 1u) be += h[N - 1 - NL - jh];
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
        // lexicographic (e, index) minimum over the lanes: minimum of the key's high word, then of its low word among the
        // lanes that hold it, then of the index among those
        const unsigned long long key = bi != 0xffffffffu ? cw_key(best) : ~0ull;
        const unsigned khi = (unsigned)(key >> 32), klo = (unsigned)key;
        const unsigned mhi = __reduce_min_sync(0xffffffffu, khi);
        const unsigned mlo = __reduce_min_sync(0xffffffffu, khi == mhi ? klo : 0xffffffffu);
        const unsigned mi = __reduce_min_sync(0xffffffffu, (khi == mhi && klo == mlo) ? bi : 0xffffffffu);
        if (lane == 0) {
            const double e = mi != 0xffffffffu ? cw_unkey(((unsigned long long)mhi << 32) | mlo) : INFINITY;
            ws.rec2[(int64_t)b * P + p] = make_double2(e, __longlong_as_double((long long)(unsigned long long)mi));
        }
        __syncwarp();  // sIn is rewritten by the next iteration
    }
}

template <int NH>
cudaError_t launch_cw(const QaDevModel *d_model, const QaWalkTable &tab, QaWorkspace ws, QaCallArgs args, int sm_count,
                      cudaStream_t stream, int *nb_out)
{
    // patterns by popcount (ascending value inside a class); a class of >= 16 patterns starts a new block
    CwBlocks blk;
    std::memset(&blk, 0, sizeof(blk));
    int nb = 0, fill = 0;
    for (int c = 0; c <= NH; ++c) {
        if (cw_binom(NH, c) >= 16 && fill > 0) {
            ++nb;
            fill = 0;
        }
        for (int t = 0; t < (1 << NH); ++t) {
            if (__builtin_popcount((unsigned)t) != c) continue;
            if (fill == 32) {
                ++nb;
                fill = 0;
            }
            blk.t[nb][fill] = (unsigned char)t;
            blk.mask[nb] |= 1u << fill;
            ++fill;
        }
        if (cw_binom(NH, c) >= 16) {
            ++nb;
            fill = 0;
        }
    }
    if (fill > 0) ++nb;
    blk.nb = nb;
    *nb_out = nb;
    int per_sm = 0;
    cudaError_t err = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, qa_closed_walk_kernel<NH>, CW_THREADS, 0);
    if (err != cudaSuccess) return err;
    if (per_sm < 1) per_sm = 1;
    int64_t grid = (int64_t)sm_count * per_sm;
    const int64_t need = (ws.P * nb + CW_THREADS / 32 - 1) / (CW_THREADS / 32);
    if (grid > need) grid = need;
    return qa_launch_pdl(qa_closed_walk_kernel<NH>, dim3((unsigned)grid), dim3(CW_THREADS), stream, d_model, tab, blk, ws, args);
}

}  // namespace

// *nb_out = records per pixel (ws.rec2[b * P + p]) for qa_launch_finalize
cudaError_t qa_launch_closed_walk(const QaDevModel *d_model, int n, const QaWalkTable &tab, QaWorkspace ws, QaCallArgs args,
                                  int sm_count, cudaStream_t stream, int *nb_out)
{
    qa_plan_add("qa_closed_walk_kernel");
    switch (n) {
        case 9: return launch_cw<1>(d_model, tab, ws, args, sm_count, stream, nb_out);
        case 10: return launch_cw<2>(d_model, tab, ws, args, sm_count, stream, nb_out);
        case 11: return launch_cw<3>(d_model, tab, ws, args, sm_count, stream, nb_out);
        case 12: return launch_cw<4>(d_model, tab, ws, args, sm_count, stream, nb_out);
        case 13: return launch_cw<5>(d_model, tab, ws, args, sm_count, stream, nb_out);
        case 14: return launch_cw<6>(d_model, tab, ws, args, sm_count, stream, nb_out);
        case 15: return launch_cw<7>(d_model, tab, ws, args, sm_count, stream, nb_out);
        case 16: return launch_cw<8>(d_model, tab, ws, args, sm_count, stream, nb_out);
        default: return cudaErrorInvalidValue;
    }
}
