// qa_kernels_filter.cu -- the hot path for n >= 13: default algorithm, open array (S5 + S6 [+ S7] of SURVEY.md section
// 8(a)) as a "filtered" static Gray walk: 2 FP64-pipe instructions per candidate and no synchronisation between warps.
//
// Same decomposition as qa_kernels_walk.cu (NH high bits = one thread per high pattern t, NL = 8 low bits walked per
// thread in binary-reflected Gray order, fully unrolled; E(base + b) = E(base) + sum_i b_i h_i + sum_{i<j} b_i b_j M_ij
// from (C1) L607), but the running minimum no longer sits on the FP64 pipe, and the work is split into two kernels:
//
//   qa_filter_walk_kernel (pass 1; every thread, every candidate):
//         s +-= h'_ctz(k)              1 DADD
//         e   = s + T[k]               1 DADD   (T[k] = QL[gray(k)]: pair table in walk order, shared memory, LDS.128)
//         mh  = min(mh, hi32(e))       1/2 integer min3 (ALU pipe)
//     e is the FULL energy of the candidate plus a fixed positive offset E_C (s starts at E(base) + E_C + the high
//     pattern's terms), so e > 0 and the high 32 bits of the fp64 pattern order like the values themselves.  Every
//     thread walks TWO pixels at once (two independent DADD chains; each T[k] load serves both).  Each warp then stores
//     (min of mh over its lanes, ballot of the lanes attaining it) for its 32 high patterns of the pixel: 8 bytes.
//     Warps never wait for one another (no barrier, no atomics in the loop).  The steps are pinned with asm volatile:
//     left to itself the compiler schedules the whole s-chain first and spills every intermediate.
//   qa_filter_finish_kernel (pass 2 + S7/S8; one thread per pixel):
//     H = min over the pixel's warp records; every thread t_s with mh == H (normally ONE per pixel) is a survivor; its
//     2^NL candidates are walked again with pass 1's arithmetic and an exact lexicographic (energy, index) compare.
//     A candidate outside the survivors has hi32(e) > H, i.e. is strictly worse than the best survivor, so the result is
//     exactly the argmin of the pass-1 energies (which carry <= ~300 ulp of rounding, eleven orders of magnitude below
//     the 1e-9 E_C near-tie rule).  The same thread then runs the finalize step (S7/S8:
//     qa_finalize_pixel), so the path is three launches: prologue, walk, finish.
//
// B200 arithmetic (measured): the FP64 pipe takes one warp instruction per 2 cycles per SM
// sub-partition; an ALU instruction issued between DADDs costs ~0.7 cycle and a broadcast LDS.128 ~2, so the walk's
// ceiling is ~4.9 cycles per warp-candidate-pair-slot, i.e. ~75-80 % FP64-pipe utilisation, not 100 %.
//
// Index convention as in qa_kernels_walk.cu: candidate index = sum_i b_i 2^(n-1-i); low bit j <-> dot n-1-j; high bit j'
// of t <-> dot n-1-NL-j'.
#include "qa_internal.cuh"

namespace {

constexpr int FW_THREADS = 256;
constexpr int FW_PX = 2;  // pixels walked per thread at once

__host__ __device__ constexpr int fw_ctz(int k)
{
    int j = 0;
    while (((k >> j) & 1) == 0) ++j;
    return j;
}

__device__ __forceinline__ double fw_shfl(double x, int src) { return __shfl_sync(0xffffffffu, x, src); }

// Two consecutive walk steps: s (+/-)= ha; e1 = s + q1; s (+/-)= hb; e2 = s + q2; mh = min(mh, hi32(e1), hi32(e2)).
// One asm volatile block per pair keeps the order (and with it the register pressure) the source states.
#define FW_STEP2(OPA, OPB)                                                                                             \
    asm volatile("{ .reg .f64 e1, e2; .reg .b32 l1, h1, l2, h2;\n" OPA " %0, %0, %2; add.f64 e1, %0, %4;\n" OPB        \
                 " %0, %0, %3; add.f64 e2, %0, %5;\n mov.b64 {l1,h1}, e1; mov.b64 {l2,h2}, e2;\n"                      \
                 " min.u32 %1, %1, h1; min.u32 %1, %1, h2; }"                                                          \
                 : "+d"(s), "+r"(mh)                                                                                   \
                 : "d"(ha), "d"(hb), "d"(q1), "d"(q2))

template <bool PA, bool PB>
__device__ __forceinline__ void fw_step2(double &s, unsigned &mh, double ha, double hb, double q1, double q2)
{
    if (PA && PB)
        FW_STEP2("add.f64", "add.f64");
    else if (PA && !PB)
        FW_STEP2("add.f64", "sub.f64");
    else if (!PA && PB)
        FW_STEP2("sub.f64", "add.f64");
    else
        FW_STEP2("sub.f64", "sub.f64");
}

// v_j(t) = sum over the high bits jh of t of M[low dot j][high dot jh], jh ascending (pixel-independent)
template <int NL, int NH>
__device__ __forceinline__ double fw_cross(const double *M, unsigned t, int j)
{
    constexpr int N = NL + NH;
    double s = 0.0;
#pragma unroll
    for (int jh = 0; jh < NH; ++jh)
        if ((t >> jh) & 1u) s += M[(N - 1 - j) * QA_MAXN + (N - 1 - NL - jh)];
    return s;
}

// E_C + pair energy of high pattern t (the positive offset rides along with the high-pattern constant)
template <int NL, int NH>
__device__ __forceinline__ double fw_high_pairs(const double *M, double EC, unsigned t)
{
    constexpr int N = NL + NH;
    double q = EC;
#pragma unroll
    for (int jh = 0; jh < NH; ++jh)
#pragma unroll
        for (int jh2 = jh + 1; jh2 < NH; ++jh2)
            if (((t >> jh) & 1u) && ((t >> jh2) & 1u)) q += M[(N - 1 - NL - jh) * QA_MAXN + (N - 1 - NL - jh2)];
    return q;
}

// ---------------------------------------------------------------------------------------------------------------------
// pass 1
template <int NL, int NH, int MINB>
__global__ void __launch_bounds__(FW_THREADS, MINB) qa_filter_walk_kernel(const QaDevModel *__restrict__ mdl,
                                                                          const __grid_constant__ QaWalkTable tab,
                                                                          QaWorkspace ws)
{
    constexpr int N = NL + NH;
    constexpr int TPP = 1 << NH;             // threads per pixel
    constexpr int WPP = TPP / 32;            // warps per pixel
    constexpr int SLOTS = FW_THREADS / TPP;  // pixel pairs per CTA iteration
    constexpr int NV = N + 1;                // per-pixel inputs: h[0..N-1], E(base)
    constexpr int PX = FW_PX;
    static_assert(NL == 8 && NH >= 5 && NH <= 8 && N <= 31, "one or more whole warps per pixel");

    __shared__ __align__(16) double sT[1 << NL];  // pair table in walk order
    for (int k = threadIdx.x; k < (1 << NL); k += FW_THREADS) sT[k] = tab.QL[k ^ (k >> 1)];
    __syncthreads();

    const unsigned lane = threadIdx.x & 31u;
    const unsigned t = threadIdx.x & (TPP - 1);
    const int slot = threadIdx.x >> NH;
    const unsigned wq = (threadIdx.x >> 5) % WPP;  // this warp's index among the pixel's warps
    const int64_t P = ws.P;

    double v[NL];
#pragma unroll
    for (int j = 0; j < NL; ++j) v[j] = fw_cross<NL, NH>(mdl->M, t, j);
    const double QH = fw_high_pairs<NL, NH>(mdl->M, mdl->EC, t);

    const int64_t groups = (P + (int64_t)SLOTS * PX - 1) / ((int64_t)SLOTS * PX);
    // lane i < NV of every warp carries input i of the warp's pixels; the next group's is fetched one iteration ahead
    auto fetch = [&](int64_t grp, int px) -> double {
        double r = 0.0;
        if (grp < groups && lane < NV) {
            int64_t p = (grp * SLOTS + slot) * PX + px;
            if (p >= P) p = P - 1;
            r = lane < N ? __ldg(ws.h + (int64_t)lane * P + p) : __ldg(ws.e0 + p);
        }
        return r;
    };
    double nextv[PX];
#pragma unroll
    for (int px = 0; px < PX; ++px) nextv[px] = fetch(blockIdx.x, px);

    for (int64_t grp = blockIdx.x; grp < groups; grp += gridDim.x) {
        asm volatile("" ::: "memory");
        double hp[PX][NL], s[PX], be0[PX];
        unsigned mh[PX];
#pragma unroll
        for (int px = 0; px < PX; ++px) {
            const double myv = nextv[px];
            nextv[px] = fetch(grp + gridDim.x, px);
#pragma unroll
            for (int j = 0; j < NL; ++j) hp[px][j] = fw_shfl(myv, N - 1 - j) + v[j];
            double be = fw_shfl(myv, N) + QH;
#pragma unroll
            for (int jh = 0; jh < NH; ++jh) {
                const double hv = fw_shfl(myv, N - 1 - NL - jh);
                if ((t >> jh) & 1u) be += hv;
            }
            s[px] = be;
            be0[px] = be;
            mh[px] = (unsigned)__double2hiint(be);  // k = 0: the all-zero low pattern, T[0] = 0
        }

        // steps k = 1 .. 2^NL - 1; T[k], T[k+1] arrive as one LDS.128 and serve both pixels
#pragma unroll
        for (int k = 0; k < (1 << NL); k += 2) {
            if ((k % 16) == 0) asm volatile("" ::: "memory");  // bounds how far the table loads are hoisted
            const double2 q = *reinterpret_cast<const double2 *>(&sT[k]);
            if (k == 0) {
#pragma unroll
                for (int px = 0; px < PX; ++px) {  // single step k = 1: bit 0 turns on
                    s[px] += hp[px][0];
                    mh[px] = min(mh[px], (unsigned)__double2hiint(s[px] + q.y));
                }
            } else {
                const int ja = fw_ctz(k);  // step k flips bit ctz(k); step k + 1 flips bit 0
                const int ga = k ^ (k >> 1), gb = (k + 1) ^ ((k + 1) >> 1);
                const bool pa = (ga >> ja) & 1, pb = gb & 1;
#pragma unroll
                for (int px = 0; px < PX; ++px) {
                    if (pa && pb)
                        fw_step2<true, true>(s[px], mh[px], hp[px][ja], hp[px][0], q.x, q.y);
                    else if (pa && !pb)
                        fw_step2<true, false>(s[px], mh[px], hp[px][ja], hp[px][0], q.x, q.y);
                    else if (!pa && pb)
                        fw_step2<false, true>(s[px], mh[px], hp[px][ja], hp[px][0], q.x, q.y);
                    else
                        fw_step2<false, false>(s[px], mh[px], hp[px][ja], hp[px][0], q.x, q.y);
                }
            }
        }

        // record of this warp's 32 high patterns: (minimum of hi32(e), lanes attaining it)
#pragma unroll
        for (int px = 0; px < PX; ++px) {
            const unsigned wmin = __reduce_min_sync(0xffffffffu, mh[px]);
            const unsigned ball = __ballot_sync(0xffffffffu, mh[px] == wmin);
            const int64_t p = (grp * SLOTS + slot) * PX + px;
            if (p < P) {
                if (lane == 0) ws.rec[p * WPP + wq] = make_uint2(wmin, ball);
                if (lane == (unsigned)(__ffs(ball) - 1)) {  // the first lane attaining the minimum leaves its walk inputs
                    double *sv = ws.sv + (p * WPP + wq) * (NL + 1);
#pragma unroll
                    for (int j = 0; j < NL; ++j) sv[j] = hp[px][j];
                    sv[NL] = be0[px];
                }
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------------------------------
// pass 2 + S7: one warp per pixel.  The code is executed once per warp, so it is kept short (instruction fetch, not
// arithmetic, is what a 10^4-warp one-shot kernel pays for): each lane scores 2^NL / 32 candidates of a survivor from
// scratch, the warp reduces lexicographically, 16 lanes decode N* and compute E(N*) from the definition.
constexpr int FF_THREADS = 128;

template <int NL, int NH>
__global__ void __launch_bounds__(FF_THREADS) qa_filter_finish_kernel(const QaDevModel *__restrict__ mdl,
                                                                      QaWorkspace ws, int32_t *__restrict__ outN,
                                                                      double *__restrict__ outE)
{
    constexpr int N = NL + NH;
    constexpr int WPP = (1 << NH) / 32;
    constexpr int CPL = (1 << NL) / 32;  // candidates per lane
    __shared__ double sM[N][N + 1];
    __shared__ double sQL[1 << NL];  // QL[b], b = low pattern: per-lane (divergent) indexing
    for (int e = threadIdx.x; e < N * N; e += FF_THREADS) sM[e / N][e % N] = mdl->M[(e / N) * QA_MAXN + (e % N)];
    for (int b = threadIdx.x; b < (1 << NL); b += FF_THREADS) {
        double q = 0.0;  // same order as the host table (qa_api.cu rebuild): j ascending, j2 > j ascending
        for (int j = 0; j < NL; ++j)
            for (int j2 = j + 1; j2 < NL; ++j2)
                if (((b >> j) & 1) && ((b >> j2) & 1)) q += mdl->M[(N - 1 - j) * QA_MAXN + (N - 1 - j2)];
        sQL[b] = q;
    }
    __syncthreads();

    const unsigned lane = threadIdx.x & 31u;
    const int64_t P = ws.P;
    const int64_t p = (int64_t)blockIdx.x * (FF_THREADS / 32) + (threadIdx.x >> 5);
    if (p >= P) return;

    uint2 r = make_uint2(0xffffffffu, 0u);
    if (lane < WPP) r = ws.rec[p * WPP + lane];
    const unsigned H = __reduce_min_sync(0xffffffffu, r.x);
    const unsigned wmask = __ballot_sync(0xffffffffu, r.x == H);                     // warps holding a survivor
    const unsigned multi = __ballot_sync(0xffffffffu, r.x == H && (r.y & (r.y - 1)));  // ... more than one

    double bestE = INFINITY;
    unsigned bestI = 0xffffffffu;
    auto score = [&](unsigned ts, const double *bh, double bs) {
        double e1 = INFINITY;
        unsigned i1 = 0;
#pragma unroll
        for (int c = 0; c < CPL; ++c) {
            const unsigned l = lane * CPL + c;
            double a = bs;
#pragma unroll
            for (int j = NL - 1; j >= 0; --j)
                if ((l >> j) & 1u) a += bh[j];
            a += sQL[l];
            if (a < e1) {  // l ascending within the lane: strict '<' keeps the smallest index
                e1 = a;
                i1 = l;
            }
        }
        i1 |= ts << NL;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const double e2 = fw_shfl(e1, (int)(lane ^ o));
            const unsigned i2 = __shfl_xor_sync(0xffffffffu, i1, o);
            if (e2 < e1 || (e2 == e1 && i2 < i1)) {
                e1 = e2;
                i1 = i2;
            }
        }
        if (e1 < bestE || (e1 == bestE && i1 < bestI)) {
            bestE = e1;
            bestI = i1;
        }
    };

    if ((wmask & (wmask - 1)) == 0 && multi == 0) {
        // the usual case, one survivor: its h' and start value were left behind by pass 1
        const int q = __ffs(wmask) - 1;
        const unsigned ball = __shfl_sync(0xffffffffu, r.y, q);
        const unsigned ts = (unsigned)q * 32u + (unsigned)(__ffs(ball) - 1);
        const double *sv = ws.sv + (p * WPP + q) * (NL + 1);
        double bh[NL];
#pragma unroll
        for (int j = 0; j < NL; ++j) bh[j] = sv[j];
        score(ts, bh, sv[NL]);
    } else {
        // several threads tie in the high word: rebuild each one's inputs as pass 1 did (same operands, same order)
        double hv = 0.0;
        if (lane <= N) hv = lane < N ? ws.h[(int64_t)lane * P + p] : ws.e0[p];
        for (int q = 0; q < WPP; ++q) {
            unsigned surv = __shfl_sync(0xffffffffu, r.y, q);
            if (!((wmask >> q) & 1u)) continue;
            while (surv) {
                const unsigned ts = (unsigned)q * 32u + (unsigned)(__ffs(surv) - 1);
                surv &= surv - 1;
                const double vmine = lane < NL ? fw_cross<NL, NH>(mdl->M, ts, (int)lane) : 0.0;
                double bh[NL];
#pragma unroll
                for (int j = 0; j < NL; ++j) bh[j] = fw_shfl(hv, N - 1 - j) + fw_shfl(vmine, j);
                double bs = fw_shfl(hv, N) + fw_high_pairs<NL, NH>(mdl->M, mdl->EC, ts);
#pragma unroll
                for (int jh = 0; jh < NH; ++jh) {
                    const double hj = fw_shfl(hv, N - 1 - NL - jh);
                    if ((ts >> jh) & 1u) bs += hj;
                }
                score(ts, bh, bs);
            }
        }
    }
    if (!outN) {
        if (lane == 0) ws.best[p] = (uint64_t)bestI;
        return;
    }
    // S7: N* and E(N*) = 1/2 d^T M d from the definition (Eq. (C1)); lane i holds dot i
    int32_t Ni = 0;
    double di = 0.0;
    if (lane < N) {
        Ni = ws.base[(int64_t)lane * P + p] + (int32_t)((bestI >> (N - 1 - lane)) & 1u);
        di = (double)Ni - ws.nc[(int64_t)lane * P + p];
    }
    double row = 0.0;
#pragma unroll
    for (int j = 0; j < N; ++j) {
        const double dj = fw_shfl(di, j);
        if (lane < N) row = fma(sM[lane][j], dj, row);
    }
    double E = di * row;  // lanes >= N contribute 0
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) E += fw_shfl(E, (int)(lane ^ o));
    if (lane < N) outN[p * N + lane] = Ni;
    if (lane == 0) outE[p] = 0.5 * E;
}

// Grid of the walk: every CTA runs ceil(groups / grid) iterations, so among the resident-CTA counts the hardware allows
// pick the one with the least total time, rounds x CTAs per SM / efficiency (measured pass-1 efficiency rises only
// slowly with occupancy: 0.745 / 0.755 / 0.76 at 2 / 3 / 4 CTAs per SM).
int64_t fw_pick_grid(int64_t groups, int sm_count, int per_sm)
{
    static const double eff[5] = {0.0, 0.65, 0.745, 0.755, 0.76};
    int64_t best_grid = sm_count;
    double best_cost = 1e300;
    for (int occ = 1; occ <= per_sm && occ <= 4; ++occ) {
        const int64_t gmax = (int64_t)sm_count * occ;
        const int64_t rounds = (groups + gmax - 1) / gmax;
        const double cost = (double)rounds * occ / eff[occ];
        if (cost < best_cost) {
            best_cost = cost;
            best_grid = (groups + rounds - 1) / rounds;  // same number of rounds, evenly filled
        }
    }
    return best_grid < 1 ? 1 : best_grid;
}

template <int NL, int NH, int MINB>
cudaError_t launch_fw(const QaDevModel *d_model, const QaWalkTable &tab, QaWorkspace ws, const double *d_Vg,
                      int32_t *d_N, double *d_E, double *d_Vs, int sm_count, cudaStream_t stream)
{
    constexpr int SLOTS = FW_THREADS >> NH;
    const int64_t groups = (ws.P + (int64_t)SLOTS * FW_PX - 1) / ((int64_t)SLOTS * FW_PX);
    int per_sm = 0;
    cudaError_t err =
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, qa_filter_walk_kernel<NL, NH, MINB>, FW_THREADS, 0);
    if (err != cudaSuccess) return err;
    if (per_sm < 1) per_sm = 1;
    const int64_t grid = fw_pick_grid(groups, sm_count, per_sm);
    qa_filter_walk_kernel<NL, NH, MINB><<<(unsigned)grid, FW_THREADS, 0, stream>>>(d_model, tab, ws);
    err = cudaGetLastError();
    if (err != cudaSuccess) return err;
    qa_plan_add("qa_filter_finish_kernel");
    qa_timing_mark(stream);
    const int64_t fblocks = (ws.P + FF_THREADS / 32 - 1) / (FF_THREADS / 32);
    qa_filter_finish_kernel<NL, NH><<<(unsigned)fblocks, FF_THREADS, 0, stream>>>(d_model, ws, d_N, d_E);
    return cudaGetLastError();
}

}  // namespace

// d_N == nullptr: the finish kernel only stores the winning index (ws.best) and the caller runs qa_finalize_kernel.
cudaError_t qa_launch_filter_walk(const QaDevModel *d_model, int n, const QaWalkTable &tab, QaWorkspace ws,
                                  const double *d_Vg, int32_t *d_N, double *d_E, double *d_Vs, int sm_count, int variant,
                                  cudaStream_t stream)
{
    qa_plan_add("qa_filter_walk_kernel");
#define FW_CALL(NH, MINB) launch_fw<8, NH, MINB>(d_model, tab, ws, d_Vg, d_N, d_E, d_Vs, sm_count, stream)
    if (variant == 3) {
        switch (n) {
            case 13: return FW_CALL(5, 4);
            case 14: return FW_CALL(6, 4);
            case 15: return FW_CALL(7, 4);
            case 16: return FW_CALL(8, 4);
            default: return cudaErrorInvalidValue;
        }
    }
    switch (n) {
        case 13: return FW_CALL(5, 3);
        case 14: return FW_CALL(6, 3);
        case 15: return FW_CALL(7, 3);
        case 16: return FW_CALL(8, 3);
        default: return cudaErrorInvalidValue;
    }
#undef FW_CALL
}
