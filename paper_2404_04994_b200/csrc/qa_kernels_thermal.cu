// qa_kernels_thermal.cu -- thermal broadening (section IV.B): the arg min of Eq. (5) is replaced by the
// soft arg min of Eq. (10) L157 over the SAME candidate set,
//     <N> = sum_N N exp(-E(N)/kT) / sum_N exp(-E(N)/kT),
// kT = k_B T in the energy units of E (reading R13).  Runs after qa_prologue_kernel (S1-S4: candidate ranges in the
// workspace) in place of the enumeration + finalize kernels.
//
// Same decomposition as qa_enumerate_kernel: the candidate box prod_i [base_i, base_i + cnt_i) is a mixed-radix odometer
// (dot 0 most significant), G threads share a pixel and each walks a contiguous chunk with rank-1 energy updates
//     E(d + delta e_i) = E(d) + delta grad_i + 1/2 delta^2 M_ii,   grad += delta M[:, i]                  (from (C1) L607)
// Two passes over the chunk: (1) E_min of the set (reduced over the G threads), (2) Z = sum w, S_i = sum w N_i with
// w = exp(-(E - E_min)/kT) -- the largest weight is 1 (Eq. (4) and E differ by a per-pixel constant that cancels in the
// ratio).  The G partial sums are combined in a fixed tree order, so the result does not depend on scheduling.  Closed
// arrays keep only candidates with sum N = N_hat (L159).
#include "qa_internal.cuh"

namespace {

constexpr int TH_THREADS = 256;

template <int N, int G>
__global__ void __launch_bounds__(TH_THREADS, 1) qa_thermal_kernel(const QaDevModel *__restrict__ mdl, QaWorkspace ws,
                                                                QaCallArgs args, double kT, double *__restrict__ outNmean,
                                                                double *__restrict__ outEmin, qa_stats *stats)
{
    __shared__ double sM[N * N];
    __shared__ double sRed[TH_THREADS / 32][N + 1];
    __shared__ double sMin;
    for (int e = threadIdx.x; e < N * N; e += TH_THREADS) sM[e] = mdl->M[(e / N) * QA_MAXN + (e % N)];
    __syncthreads();

    const int64_t P = ws.P;
    const int64_t p = (blockIdx.x * (int64_t)TH_THREADS + threadIdx.x) / G;
    const unsigned r = threadIdx.x % G;
    const bool live = p < P;
    const int64_t pp = live ? p : P - 1;
    const bool closed = args.closed != 0;

    // per dot: lowest and highest candidate value and the current one (the odometer digit is cur - lo)
    int32_t lo[N], hi[N], cur[N];
    double grad[N];
#pragma unroll
    for (int i = 0; i < N; ++i) {
        lo[i] = ws.base[i * P + pp];
        hi[i] = lo[i] + ws.cnt[i * P + pp] - 1;
    }
    const uint64_t T = ws.total[pp];
    const uint64_t q = T / G, rem = T % G;
    const uint64_t start = r * q + (r < rem ? r : rem);
    const uint64_t len = live ? q + (r < rem ? 1 : 0) : 0;

    double Emin = INFINITY, Z = 0.0, S[N];
#pragma unroll
    for (int i = 0; i < N; ++i) S[i] = 0.0;
    int64_t scored = 0;

    for (int pass = 0; pass < 2; ++pass) {
        // first candidate of the chunk: digits of `start`, energy and gradient from the definition
        int64_t sumN = 0;
        double E = 0.0;
        {
            uint64_t idx = start;
            double d[N];
#pragma unroll
            for (int i = N - 1; i >= 0; --i) {
                const uint64_t c = (uint64_t)(hi[i] - lo[i] + 1);
                cur[i] = lo[i] + (int32_t)(idx % c);
                idx /= c;
                d[i] = (double)cur[i] - ws.nc[i * P + pp];
                sumN += cur[i];
            }
#pragma unroll
            for (int i = 0; i < N; ++i) {
                double gi = 0.0;
#pragma unroll
                for (int j = 0; j < N; ++j) gi = fma(sM[i * N + j], d[j], gi);
                grad[i] = gi;
                E = fma(d[i], gi, E);
            }
            E *= 0.5;
        }
        for (uint64_t it = 0; it < len; ++it) {
            if (!closed || sumN == args.N_hat) {
                if (pass == 0) {
                    ++scored;
                    Emin = fmin(Emin, E);
                } else {
                    const double w = exp(-(E - Emin) / kT);
                    Z += w;
#pragma unroll
                    for (int i = 0; i < N; ++i) S[i] = fma(w, (double)cur[i], S[i]);
                }
            }
            if (it + 1 == len) break;
            bool carry = true;  // odometer step, least significant digit = dot N-1
#pragma unroll
            for (int i = N - 1; i >= 0; --i) {
                if (carry) {
                    int delta;
                    if (cur[i] == hi[i]) {
                        delta = lo[i] - cur[i];
                        cur[i] = lo[i];
                    } else {
                        delta = 1;
                        ++cur[i];
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
        if (pass == 0 && G > 1) {  // E_min over the G threads of the pixel
            constexpr int W = G < 32 ? G : 32;
#pragma unroll
            for (int o = W / 2; o > 0; o >>= 1) Emin = fmin(Emin, __shfl_xor_sync(0xffffffffu, Emin, o));
            if (G > 32) {  // G == TH_THREADS: the whole block is one pixel
                if ((threadIdx.x & 31) == 0) sRed[threadIdx.x >> 5][0] = Emin;
                __syncthreads();
                if (threadIdx.x == 0) {
                    double mn = sRed[0][0];
                    for (int w = 1; w < TH_THREADS / 32; ++w) mn = fmin(mn, sRed[w][0]);
                    sMin = mn;
                }
                __syncthreads();
                Emin = sMin;
                __syncthreads();
            }
        }
    }

    // Z and S over the G threads, fixed tree order
    if (G > 1) {
        constexpr int W = G < 32 ? G : 32;
#pragma unroll
        for (int o = W / 2; o > 0; o >>= 1) {
            Z += __shfl_xor_sync(0xffffffffu, Z, o);
#pragma unroll
            for (int i = 0; i < N; ++i) S[i] += __shfl_xor_sync(0xffffffffu, S[i], o);
        }
        if (G > 32) {
            if ((threadIdx.x & 31) == 0) {
                sRed[threadIdx.x >> 5][N] = Z;
#pragma unroll
                for (int i = 0; i < N; ++i) sRed[threadIdx.x >> 5][i] = S[i];
            }
            __syncthreads();
            if (threadIdx.x == 0) {
                for (int w = 1; w < TH_THREADS / 32; ++w) {
                    Z += sRed[w][N];
#pragma unroll
                    for (int i = 0; i < N; ++i) S[i] += sRed[w][i];
                }
            }
        }
    }
    if (live && r == 0) {
        const bool empty = !(Z > 0.0);
#pragma unroll
        for (int i = 0; i < N; ++i) outNmean[p * N + i] = empty ? -1.0 : S[i] / Z;
        if (outEmin) outEmin[p] = Emin;
    }
    if (stats && closed) qa_warp_count(&stats->n_candidates_scored, scored);  // open: counted by the prologue
}

// ---------------------------------------------------------------------------------------------------------------------
// Binary candidate sets (default and thresholded algorithm: every dot has one or two values, i.e. lo + a subset of the k
// free dots): the same two passes as a binary-reflected Gray walk over the free dots -- one rank-1 update per candidate
// instead of the odometer's carries, one code path instead of N unrolled odometer levels (which spill at N = 16).
// Occupation sums by prefix bookkeeping: with W_s = sum of the weights of steps <= s, a dot whose bit is on during the
// steps [a, b) collects W_{b-1} - W_{a-1}; so A_i -= W_{s-1} when bit i turns on at step s, A_i += W_{s-1} when it turns
// off, A_i += W_last for the bits still on at the end, and <N_i> = lo_i + A_i / Z: one update per flip instead of N per
// candidate.  A lives in shared memory (indexed by the flipped dot).  G threads share a pixel, each owns a contiguous
// range of Gray indices.  A pixel whose set is not binary (the widened closed set of reading R5, expected never) is
// evaluated from the definition by one thread (qa_thermal_pixel_plain).
__device__ __noinline__ void qa_thermal_pixel_plain(const QaDevModel *__restrict__ mdl, const QaWorkspace &ws, int64_t p,
                                                    bool closed, int N_hat, double kT, double *__restrict__ outNmean,
                                                    double *__restrict__ outEmin, int64_t &scored)
{
    const int n = mdl->n;
    const int64_t P = ws.P;
    int32_t lo[QA_MAXN], hi[QA_MAXN], cur[QA_MAXN];
    double nc[QA_MAXN], S[QA_MAXN];
    for (int i = 0; i < n; ++i) {
        lo[i] = ws.base[i * P + p];
        hi[i] = lo[i] + ws.cnt[i * P + p] - 1;
        nc[i] = ws.nc[i * P + p];
    }
    double Emin = INFINITY, Z = 0.0;
    for (int pass = 0; pass < 2; ++pass) {
        for (int i = 0; i < n; ++i) {
            cur[i] = lo[i];
            S[i] = 0.0;
        }
        for (;;) {
            int64_t sumN = 0;
            for (int i = 0; i < n; ++i) sumN += cur[i];
            if (!closed || sumN == N_hat) {
                double E = 0.0;
                for (int i = 0; i < n; ++i) {
                    double row = 0.0;
                    for (int j = 0; j < n; ++j) row = fma(mdl->M[i * QA_MAXN + j], (double)cur[j] - nc[j], row);
                    E = fma((double)cur[i] - nc[i], row, E);
                }
                E *= 0.5;
                if (pass == 0) {
                    ++scored;
                    Emin = fmin(Emin, E);
                } else {
                    const double w = exp(-(E - Emin) / kT);
                    Z += w;
                    for (int i = 0; i < n; ++i) S[i] = fma(w, (double)cur[i], S[i]);
                }
            }
            int i = n - 1;
            while (i >= 0) {
                if (cur[i] < hi[i]) {
                    ++cur[i];
                    break;
                }
                cur[i] = lo[i];
                --i;
            }
            if (i < 0) break;
        }
    }
    for (int i = 0; i < n; ++i) outNmean[p * n + i] = Z > 0.0 ? S[i] / Z : -1.0;
    if (outEmin) outEmin[p] = Emin;
}

template <int N, int G>
__global__ void __launch_bounds__(TH_THREADS, 3) qa_thermal_gray_kernel(const QaDevModel *__restrict__ mdl, QaWorkspace ws,
                                                                        QaCallArgs args, double kT,
                                                                        double *__restrict__ outNmean,
                                                                        double *__restrict__ outEmin, qa_stats *stats)
{
    __shared__ double sM[N * N];
    __shared__ double sA[N][TH_THREADS];  // per-thread occupation sums, indexed by dot (conflict-free: one column each)
    __shared__ double sRed[TH_THREADS / 32][N + 1];
    __shared__ double sMin;
    for (int e = threadIdx.x; e < N * N; e += TH_THREADS) sM[e] = mdl->M[(e / N) * QA_MAXN + (e % N)];
    __syncthreads();

    const int64_t P = ws.P;
    const int64_t p = (blockIdx.x * (int64_t)TH_THREADS + threadIdx.x) / G;
    const unsigned r = threadIdx.x % G;
    const bool live = p < P;
    const int64_t pp = live ? p : P - 1;
    const bool closed = args.closed != 0;
    const int tid = threadIdx.x;

    int32_t lo[N];
    uint64_t flist = 0;  // 4-bit dot indices of the free dots, Gray bit 0 = the highest free dot
    int k = 0;
    bool binary = true;
#pragma unroll
    for (int i = N - 1; i >= 0; --i) {
        lo[i] = ws.base[i * P + pp];
        const int32_t c = ws.cnt[i * P + pp];
        if (c == 2) flist |= (uint64_t)i << (4 * k++);
        binary &= c <= 2;
    }
    const uint64_t T = binary ? (1ull << k) : 0;  // a non-binary pixel is left to qa_thermal_pixel_plain below
    const uint64_t q = T / G, rem = T % G;
    const uint64_t start = r * q + (r < rem ? r : rem);
    const uint64_t len = live ? q + (r < rem ? 1 : 0) : 0;

    double Emin = INFINITY, Z = 0.0, grad[N];
    int64_t scored = 0;
    unsigned state = 0;  // bit (N-1-i) = dot i is at lo_i + 1

    for (int pass = 0; pass < 2; ++pass) {
        // first candidate of the range: Gray code of `start`; energy and gradient from the definition
        int64_t sumN = 0;
        double E = 0.0;
        state = 0;
        {
            const uint64_t gb = start ^ (start >> 1);
            double d[N];
#pragma unroll
            for (int j = 0; j < N; ++j)
                if (j < k && ((gb >> j) & 1ull)) state |= 1u << (N - 1 - (int)((flist >> (4 * j)) & 15ull));
#pragma unroll
            for (int i = 0; i < N; ++i) {
                const int32_t ci = lo[i] + (int32_t)((state >> (N - 1 - i)) & 1u);
                d[i] = (double)ci - ws.nc[i * P + pp];
                sumN += ci;
                sA[i][tid] = 0.0;
            }
#pragma unroll
            for (int i = 0; i < N; ++i) {
                double gi = 0.0;
#pragma unroll
                for (int j = 0; j < N; ++j) gi = fma(sM[i * N + j], d[j], gi);
                grad[i] = gi;
                E = fma(d[i], gi, E);
            }
            E *= 0.5;
        }
        double Wrun = 0.0;
        for (uint64_t it = 0; it < len; ++it) {
            if (it > 0) {  // step to Gray index start + it: flip the free dot of bit ctz(start + it)
                const uint64_t sidx = start + it;
                const int i = (int)((flist >> (4 * (__ffsll((long long)sidx) - 1))) & 15ull);
                const unsigned bit = 1u << (N - 1 - i);
                const bool on = (state & bit) != 0;
                const double dl = on ? -1.0 : 1.0;
                double gi = 0.0;
#pragma unroll
                for (int j = 0; j < N; ++j)
                    if (j == i) gi = grad[j];
                E += dl * (gi + 0.5 * dl * sM[i * N + i]);
#pragma unroll
                for (int j = 0; j < N; ++j) grad[j] = fma(dl, sM[j * N + i], grad[j]);
                sumN += on ? -1 : 1;
                state ^= bit;
                if (pass == 1) sA[i][tid] += on ? Wrun : -Wrun;  // W_{s-1}: the weights up to the previous step
            }
            if (!closed || sumN == args.N_hat) {
                if (pass == 0) {
                    ++scored;
                    Emin = fmin(Emin, E);
                } else {
                    Wrun += exp(-(E - Emin) / kT);
                }
            }
        }
        if (pass == 1) {
            Z = Wrun;
#pragma unroll
            for (int i = 0; i < N; ++i)
                if ((state >> (N - 1 - i)) & 1u) sA[i][tid] += Wrun;  // bits still on at the end of the range
        }
        if (pass == 0 && G > 1) {  // E_min over the G threads of the pixel
            constexpr int W = G < 32 ? G : 32;
#pragma unroll
            for (int o = W / 2; o > 0; o >>= 1) Emin = fmin(Emin, __shfl_xor_sync(0xffffffffu, Emin, o));
            if (G > 32) {
                if ((threadIdx.x & 31) == 0) sRed[threadIdx.x >> 5][0] = Emin;
                __syncthreads();
                if (threadIdx.x == 0) {
                    double mn = sRed[0][0];
                    for (int w = 1; w < TH_THREADS / 32; ++w) mn = fmin(mn, sRed[w][0]);
                    sMin = mn;
                }
                __syncthreads();
                Emin = sMin;
                __syncthreads();
            }
        }
    }

    // Z and A over the G threads, fixed tree order
    double A[N];
#pragma unroll
    for (int i = 0; i < N; ++i) A[i] = sA[i][tid];
    if (G > 1) {
        constexpr int W = G < 32 ? G : 32;
#pragma unroll
        for (int o = W / 2; o > 0; o >>= 1) {
            Z += __shfl_xor_sync(0xffffffffu, Z, o);
#pragma unroll
            for (int i = 0; i < N; ++i) A[i] += __shfl_xor_sync(0xffffffffu, A[i], o);
        }
        if (G > 32) {
            if ((threadIdx.x & 31) == 0) {
                sRed[threadIdx.x >> 5][N] = Z;
#pragma unroll
                for (int i = 0; i < N; ++i) sRed[threadIdx.x >> 5][i] = A[i];
            }
            __syncthreads();
            if (threadIdx.x == 0) {
                for (int w = 1; w < TH_THREADS / 32; ++w) {
                    Z += sRed[w][N];
#pragma unroll
                    for (int i = 0; i < N; ++i) A[i] += sRed[w][i];
                }
            }
        }
    }
    if (live && r == 0) {
        if (binary) {
            const bool empty = !(Z > 0.0);
#pragma unroll
            for (int i = 0; i < N; ++i) outNmean[p * N + i] = empty ? -1.0 : (double)lo[i] + A[i] / Z;
            if (outEmin) outEmin[p] = Emin;
        } else {
            qa_thermal_pixel_plain(mdl, ws, p, closed, args.N_hat, kT, outNmean, outEmin, scored);
        }
    }
    if (stats && closed) qa_warp_count(&stats->n_candidates_scored, scored);  // open: counted by the prologue
}

template <int N>
cudaError_t launch_thermal_n(const QaDevModel *d_model, QaWorkspace ws, QaCallArgs args, double kT, double expect_cand,
                             double *d_Nmean, double *d_Emin, qa_stats *d_stats, cudaStream_t stream)
{
    const bool gray = args.alg != QA_ALG_BRUTE_FORCE;  // default / thresholded: binary sets (widened pixels handled inside)
    if (expect_cand <= 64.0) {
        const unsigned blocks = (unsigned)((ws.P + TH_THREADS - 1) / TH_THREADS);
        if (gray)
            qa_thermal_gray_kernel<N, 1><<<blocks, TH_THREADS, 0, stream>>>(d_model, ws, args, kT, d_Nmean, d_Emin, d_stats);
        else
            qa_thermal_kernel<N, 1><<<blocks, TH_THREADS, 0, stream>>>(d_model, ws, args, kT, d_Nmean, d_Emin, d_stats);
        qa_plan_add(gray ? "qa_thermal_gray_kernel<G=1>" : "qa_thermal_kernel<G=1>");
    } else if (expect_cand <= 4096.0) {
        const unsigned blocks = (unsigned)((ws.P * 32 + TH_THREADS - 1) / TH_THREADS);
        if (gray)
            qa_thermal_gray_kernel<N, 32><<<blocks, TH_THREADS, 0, stream>>>(d_model, ws, args, kT, d_Nmean, d_Emin, d_stats);
        else
            qa_thermal_kernel<N, 32><<<blocks, TH_THREADS, 0, stream>>>(d_model, ws, args, kT, d_Nmean, d_Emin, d_stats);
        qa_plan_add(gray ? "qa_thermal_gray_kernel<G=32>" : "qa_thermal_kernel<G=32>");
    } else {
        if (gray)
            qa_thermal_gray_kernel<N, TH_THREADS><<<(unsigned)ws.P, TH_THREADS, 0, stream>>>(d_model, ws, args, kT, d_Nmean,
                                                                                            d_Emin, d_stats);
        else
            qa_thermal_kernel<N, TH_THREADS><<<(unsigned)ws.P, TH_THREADS, 0, stream>>>(d_model, ws, args, kT, d_Nmean, d_Emin,
                                                                                       d_stats);
        qa_plan_add(gray ? "qa_thermal_gray_kernel<G=256>" : "qa_thermal_kernel<G=256>");
    }
    return cudaGetLastError();
}

}  // namespace

cudaError_t qa_launch_thermal(const QaDevModel *d_model, int n, QaWorkspace ws, QaCallArgs args, double kT,
                              double expect_cand, double *d_Nmean, double *d_Emin, qa_stats *d_stats, cudaStream_t stream)
{
#define CALL(NN) launch_thermal_n<NN>(d_model, ws, args, kT, expect_cand, d_Nmean, d_Emin, d_stats, stream)
    switch (n) {
        case 1: return CALL(1);
        case 2: return CALL(2);
        case 3: return CALL(3);
        case 4: return CALL(4);
        case 5: return CALL(5);
        case 6: return CALL(6);
        case 7: return CALL(7);
        case 8: return CALL(8);
        case 9: return CALL(9);
        case 10: return CALL(10);
        case 11: return CALL(11);
        case 12: return CALL(12);
        case 13: return CALL(13);
        case 14: return CALL(14);
        case 15: return CALL(15);
        case 16: return CALL(16);
        default: return cudaErrorInvalidValue;
    }
#undef CALL
}
