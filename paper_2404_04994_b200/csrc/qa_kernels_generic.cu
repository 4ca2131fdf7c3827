// qa_kernels_generic.cu -- prologue (steps S1-S4), generic mixed-radix enumeration (S5-S6 for every algorithm / regime)
// and finalize (S7-S8) kernels.  Hand-written CUDA for sm_100a; compiled with --fmad=false so that every fused
// multiply-add in the parity-critical arithmetic (reading R1) is an explicit fma().
//
// "Lnnn" = PAPER.md line; R1..R12 = DESIGN.md readings; S0..S8 = SURVEY.md section 8(a) steps.
#include "qa_internal.cuh"

namespace {

constexpr int PRO_THREADS = 128;
constexpr int ENUM_THREADS = 256;
constexpr int FIN_THREADS = 128;

// ------------------------------------------------------------------------------------------------------------------
// S3: exact QP  min 1/2 (x-c)^T M (x-c)  s.t. x >= 0 [, 1^T x = N_hat]  (Eq. (8) L110-L119 with the 1/2 restored).
// c_dd is a Maxwell matrix (offdiag <= 0, Eq. (B1)), i.e. a Stieltjes matrix, so the KKT system is a linear
// complementarity problem with a K-matrix and the monotone clamp-only active set is exact (reading R3): clamp every
// negative component, re-solve the equality-constrained problem on the free set F, repeat; a clamped dot is never
// released; at most n rounds.  Working in c_dd (size |A|) instead of M (size |F|):
//   y = M (x - c),  y_F = lambda 1_F,  x - c = c_dd y  =>  (x-c)_A = -c_A = C_AA y_A + lambda C_AF 1_F
//   open:   lambda = 0,  y_A = -C_AA^-1 c_A,  x_F = c_F + C_FA y_A
//   closed: y_A = a - lambda b,  a = -C_AA^-1 c_A,  b = C_AA^-1 C_AF 1_F,
//           lambda = (N_hat - sum c_F - 1^T C_FA a) / (1^T C_FF 1 - 1^T C_FA b),  x_F = c_F + C_FA y_A + lambda C_FF 1_F
// Multipliers of the bounds: r_A = y_A - lambda >= 0 is verified (KKT); a violation is counted in n_qp_failed.
// Minimiser of the objective with the dots of A held at 0 (and, closed, 1^T x = N_hat): xe, and the multipliers of the
// held bounds r_i = y_i - lambda, i in A (r of a free dot is 0).  0 < |A| < N.
template <int N>
__device__ void qa_qp_eqp(const double *__restrict__ sC, const double *c, bool closed, double Nhat, unsigned A, double *xe,
                          double *r)
{
    int ia[N], k = 0;
    for (int i = 0; i < N; ++i)
        if ((A >> i) & 1u) ia[k++] = i;
    // Cholesky C_AA = L L^T
    double L[N * N], a[N], b[N], rb[N];
    for (int p = 0; p < k; ++p) {
        for (int q = 0; q <= p; ++q) {
            double s = sC[ia[p] * N + ia[q]];
            for (int t = 0; t < q; ++t) s -= L[p * N + t] * L[q * N + t];
            if (p == q)
                L[p * N + p] = sqrt(s);
            else
                L[p * N + q] = s / L[q * N + q];
        }
    }
    auto solve = [&](const double *rhs, double *out) {
        for (int p = 0; p < k; ++p) {
            double s = rhs[p];
            for (int t = 0; t < p; ++t) s -= L[p * N + t] * out[t];
            out[p] = s / L[p * N + p];
        }
        for (int p = k - 1; p >= 0; --p) {
            double s = out[p];
            for (int t = p + 1; t < k; ++t) s -= L[t * N + p] * out[t];
            out[p] = s / L[p * N + p];
        }
    };
    for (int q = 0; q < k; ++q) rb[q] = -c[ia[q]];
    solve(rb, a);
    double lam = 0.0;
    if (closed) {
        double sumcF = 0.0, t1 = 0.0, t2 = 0.0, t3 = 0.0;
        for (int q = 0; q < k; ++q) {
            double s = 0.0;
            for (int f = 0; f < N; ++f)
                if (!((A >> f) & 1u)) s += sC[ia[q] * N + f];
            rb[q] = s;
        }
        solve(rb, b);
        for (int f = 0; f < N; ++f) {
            if ((A >> f) & 1u) continue;
            sumcF += c[f];
            for (int q = 0; q < k; ++q) {
                t1 += sC[f * N + ia[q]] * a[q];
                t3 += sC[f * N + ia[q]] * b[q];
            }
            for (int f2 = 0; f2 < N; ++f2)
                if (!((A >> f2) & 1u)) t2 += sC[f * N + f2];
        }
        lam = (Nhat - sumcF - t1) / (t2 - t3);
        for (int q = 0; q < k; ++q) a[q] -= lam * b[q];
    }
    for (int f = 0; f < N; ++f) r[f] = 0.0;
    for (int q = 0; q < k; ++q) r[ia[q]] = a[q] - lam;
    for (int f = 0; f < N; ++f) {
        if ((A >> f) & 1u) {
            xe[f] = 0.0;  // clamped components are exactly 0 (R3)
            continue;
        }
        double s = c[f];
        for (int q = 0; q < k; ++q) s += sC[f * N + ia[q]] * a[q];
        if (closed) {
            double rowF = 0.0;
            for (int f2 = 0; f2 < N; ++f2)
                if (!((A >> f2) & 1u)) rowF += sC[f * N + f2];
            s += lam * rowF;
            if (k == N - 1) s = Nhat;  // R3: a single free dot carries the whole charge, exactly
        }
        xe[f] = s;
    }
}

// Phase 1 (every c_dd): the monotone clamp-only active set described above.  For a Maxwell c_dd it ends at the KKT point.
// Phase 2 (only when c_dd has a positive off-diagonal, `general`): phase 1 still ends at a feasible x that minimises the
// objective on its face x_A = 0, but a bound multiplier may be negative; from there the textbook primal active-set method
// continues (release the most negative multiplier, move towards the new face minimiser, stop at the first bound that
// blocks), which terminates at the unique KKT point of the strictly convex problem.
template <int N>
__device__ int qa_qp_clamp(const double *__restrict__ sC, const double *c, bool closed, double Nhat, bool general,
                           double *x, bool &failed)
{
    unsigned A = 0;
    int rounds = 0;
    double scale = 1.0;
    for (int i = 0; i < N; ++i) scale = fmax(scale, fabs(c[i]));
    if (closed && Nhat <= 0.0) {
        for (int i = 0; i < N; ++i) x[i] = 0.0;
        return 1;
    }
    double r[N];
    for (int i = 0; i < N; ++i) r[i] = 0.0;
    for (;;) {
        unsigned neg = 0;
        for (int i = 0; i < N; ++i)
            if (x[i] < 0.0) neg |= 1u << i;
        neg &= ~A;
        if (!neg) break;
        A |= neg;
        if (++rounds > N) {
            failed = true;
            break;
        }
        if (__popc(A) == N) {  // nothing left free: only consistent for an open array
            for (int i = 0; i < N; ++i) x[i] = 0.0;
            if (closed) failed = true;
            break;
        }
        qa_qp_eqp<N>(sC, c, closed, Nhat, A, x, r);
        if (!general)
            for (int i = 0; i < N; ++i)
                if (r[i] < -1e-9 * scale) failed = true;  // KKT: bound multipliers must be >= 0
    }
    if (!general || failed || A == 0) return rounds;
    // phase 2
    const double tol = 1e-13 * scale;
    double xe[N];
    for (int it = 0; it < 50 * N + 50; ++it) {
        if (A != 0) {
            qa_qp_eqp<N>(sC, c, closed, Nhat, A, xe, r);  // |A| = N only for an open array (x = 0, r = -M c)
        } else {  // every bound released: the face minimiser is the analytic minimum of S2
            double lam = 0.0;
            if (closed) {
                double sc = 0.0, sCC = 0.0;
                for (int i = 0; i < N; ++i) {
                    sc += c[i];
                    for (int j = 0; j < N; ++j) sCC += sC[i * N + j];
                }
                lam = (Nhat - sc) / sCC;
            }
            for (int i = 0; i < N; ++i) {
                double row = 0.0;
                for (int j = 0; j < N; ++j) row += sC[i * N + j];
                xe[i] = c[i] + lam * row;
                r[i] = 0.0;
            }
        }
        double pmax = 0.0;
        for (int i = 0; i < N; ++i) pmax = fmax(pmax, fabs(xe[i] - x[i]));
        ++rounds;
        if (pmax <= tol) {
            for (int i = 0; i < N; ++i) x[i] = xe[i];
            int worst = -1;
            double rmin = -1e-12 * scale;
            for (int i = 0; i < N; ++i)
                if (((A >> i) & 1u) && r[i] < rmin) {
                    rmin = r[i];
                    worst = i;
                }
            if (worst < 0) return rounds;  // KKT point
            A &= ~(1u << worst);
            continue;
        }
        double alpha = 1.0;
        int block = -1;
        for (int i = 0; i < N; ++i) {
            if ((A >> i) & 1u) continue;
            const double p = xe[i] - x[i];
            if (p < 0.0) {
                const double al = x[i] / (-p);
                if (al < alpha) {
                    alpha = al;
                    block = i;
                }
            }
        }
        if (block < 0) {
            for (int i = 0; i < N; ++i) x[i] = xe[i];
        } else {
            for (int i = 0; i < N; ++i)
                if (!((A >> i) & 1u)) x[i] += alpha * (xe[i] - x[i]);
            x[block] = 0.0;
            A |= 1u << block;
        }
    }
    failed = true;
    return rounds;
}

// Eq. (9) L137 with the readings R4 / R10: candidate values of dot i are base .. base + cnt - 1.
__device__ __forceinline__ void qa_floor_ceil(double x, double t, bool thresholded, int32_t &base, int32_t &cnt)
{
    const double fl = floor(x);
    const double frac = x - fl;
    const int32_t lo = fl > 0.0 ? (int32_t)fl : 0;
    if (!thresholded || fabs(frac - 0.5) <= t * 0.5) {
        base = lo;
        cnt = 2;
    } else {
        base = frac < 0.5 ? lo : lo + 1;
        cnt = 1;
    }
}

// ------------------------------------------------------------------------------------------------------------------
// Prologue: one thread per pixel.  S1 N_c (fixed fma order, R1), S2 analytic minimum (Eq. (6) L90 / Eq. (7)),
// S3 QP when a component is negative (L82-L84, L106), S4 candidate ranges, and the base-point gradient
// h_i = [M (base - N_c)]_i + 1/2 M_ii = E(base + e_i) - E(base)  (from Eq. (C1)).
template <int N>
__global__ void __launch_bounds__(PRO_THREADS) qa_prologue_kernel(const QaDevModel *__restrict__ mdl,
                                                                  const double *__restrict__ Vg, QaWorkspace ws,
                                                                  QaCallArgs args, double *__restrict__ xcont,
                                                                  qa_stats *stats)
{
    __shared__ double sM[N * N], sC[N * N], sCgd[N * QA_MAXG], sC1[N];
    const int g = mdl->g;
    for (int e = threadIdx.x; e < N * N; e += PRO_THREADS) {
        sM[e] = mdl->M[(e / N) * QA_MAXN + (e % N)];
        sC[e] = mdl->C[(e / N) * QA_MAXN + (e % N)];
    }
    for (int e = threadIdx.x; e < N * g; e += PRO_THREADS) sCgd[e] = mdl->Cgd[(e / g) * QA_MAXG + (e % g)];
    if (threadIdx.x < N) sC1[threadIdx.x] = mdl->C1[threadIdx.x];
    const double oneC1 = mdl->oneC1;
    __syncthreads();
    qa_pdl_launch_dependents();  // the candidate kernel may become resident and load its constants meanwhile

    const int64_t P = ws.P;
    const int64_t p = blockIdx.x * (int64_t)PRO_THREADS + threadIdx.x;
    const bool live = p < P;
    const int64_t pp = live ? p : P - 1;
    const bool closed = args.closed != 0;

    // S1: N_c,i = fma(C_gd[i,k], V[k], acc), k ascending (R1)
    double nc[N];
#pragma unroll
    for (int i = 0; i < N; ++i) nc[i] = 0.0;
    const double *v = Vg + pp * g;
    for (int k = 0; k < g; ++k) {
        const double vk = __ldg(v + k);
#pragma unroll
        for (int i = 0; i < N; ++i) nc[i] = fma(sCgd[i * g + k], vk, nc[i]);
    }
    // S2
    double x[N];
    bool neg = false;
    if (!closed) {
#pragma unroll
        for (int i = 0; i < N; ++i) x[i] = nc[i];
    } else {
        double s = 0.0;
#pragma unroll
        for (int i = 0; i < N; ++i) s = s + nc[i];
        const double lam = ((double)args.N_hat - s) / oneC1;
#pragma unroll
        for (int i = 0; i < N; ++i) x[i] = fma(lam, sC1[i], nc[i]);
    }
#pragma unroll
    for (int i = 0; i < N; ++i) neg |= x[i] < 0.0;
    // S3
    int rounds = 0;
    bool failed = false;
    if (neg) rounds = qa_qp_clamp<N>(sC, nc, closed, (double)args.N_hat, args.general_qp != 0, x, failed);
    // S4
    int32_t base[N], cnt[N];
    int doublings = 0;
    bool widened = false;
    if (args.alg == QA_ALG_BRUTE_FORCE) {
#pragma unroll
        for (int i = 0; i < N; ++i) {
            base[i] = 0;
            cnt[i] = args.n_max + 1;
        }
    } else {
        const bool thr = args.alg == QA_ALG_THRESHOLDED;
        double tt = thr ? args.t : 1.0;
        for (;;) {
            int64_t smin = 0, smax = 0;
#pragma unroll
            for (int i = 0; i < N; ++i) {
                qa_floor_ceil(x[i], tt, thr, base[i], cnt[i]);
                smin += base[i];
                smax += base[i] + cnt[i] - 1;
            }
            if (!closed) break;
            const bool nonempty = smin <= args.N_hat && args.N_hat <= smax;
            if (nonempty) break;
            if (thr && tt < 1.0) {  // L141 + R5: per pixel, t <- min(1, 2t), t = 0 -> 1
                tt = tt > 0.0 ? fmin(1.0, 2.0 * tt) : 1.0;
                ++doublings;
                continue;
            }
            widened = true;  // R5 fallback: {lo-1 .. lo+2} n [0, inf)
#pragma unroll
            for (int i = 0; i < N; ++i) {
                const double fl = floor(x[i]);
                const int32_t lo = fl > 0.0 ? (int32_t)fl : 0;
                base[i] = lo > 0 ? lo - 1 : 0;
                cnt[i] = lo + 2 - base[i] + 1;
            }
            break;
        }
    }
    // base-point gradient
    double d0[N];
    uint64_t total = 1;
#pragma unroll
    for (int i = 0; i < N; ++i) {
        d0[i] = (double)base[i] - nc[i];
        total *= (uint64_t)cnt[i];
    }
    if (live) {
        double e0 = 0.0;
#pragma unroll
        for (int i = 0; i < N; ++i) {
            double gi = 0.0;
#pragma unroll
            for (int j = 0; j < N; ++j) gi = fma(sM[i * N + j], d0[j], gi);
            e0 = fma(d0[i], gi, e0);
            ws.h[i * P + p] = gi + 0.5 * sM[i * N + i];
            ws.nc[i * P + p] = nc[i];
            ws.base[i * P + p] = base[i];
            ws.cnt[i * P + p] = cnt[i];
        }
        ws.total[p] = total;
        ws.e0[p] = 0.5 * e0;
        if (xcont) {
#pragma unroll
            for (int i = 0; i < N; ++i) xcont[p * N + i] = x[i];
        }
    }
    if (stats) {
        qa_warp_count(&stats->n_pixels, live ? 1 : 0);
        qa_warp_count(&stats->n_qp_pixels, (live && neg) ? 1 : 0);
        qa_warp_count(&stats->n_qp_rounds, live ? rounds : 0);
        qa_warp_count(&stats->n_qp_failed, (live && failed) ? 1 : 0);
        qa_warp_count(&stats->n_threshold_doublings, live ? doublings : 0);
        qa_warp_count(&stats->n_widened_pixels, (live && widened) ? 1 : 0);
        qa_warp_count(&stats->n_candidates_enumerated, live ? (int64_t)total : 0);
        qa_warp_count(&stats->n_candidates_scored, (live && !closed) ? (int64_t)total : 0);  // open: all are scored
    }
}

// ------------------------------------------------------------------------------------------------------------------
// Generic enumeration (every algorithm and regime): the candidate set of a pixel is the box prod_i [base_i, base_i +
// cnt_i), enumerated in lexicographic order (dot 0 most significant) as a mixed-radix odometer.  G threads share a pixel;
// each takes a contiguous chunk of the index range, builds its first candidate from the definition (d = N - N_c,
// grad = M d, E = 1/2 d.grad) and then steps the odometer with rank-1 updates
//     E(d + delta e_i) = E(d) + delta grad_i + 1/2 delta^2 M_ii,   grad += delta M[:, i]
// Closed arrays score only candidates with sum N = N_hat (L127, L159).  Ties: strict '<' inside a chunk keeps the
// lexicographically first, and the cross-thread reduction is lexicographic on (E, index) (R6, on the GPU's own energies).
template <int N, int G>
__global__ void __launch_bounds__(ENUM_THREADS) qa_enumerate_kernel(const QaDevModel *__restrict__ mdl, QaWorkspace ws,
                                                                    QaCallArgs args, qa_stats *stats)
{
    __shared__ double sM[N * N];
    __shared__ double sE[ENUM_THREADS / 32];
    __shared__ uint64_t sI[ENUM_THREADS / 32];
    for (int e = threadIdx.x; e < N * N; e += ENUM_THREADS) sM[e] = mdl->M[(e / N) * QA_MAXN + (e % N)];
    __syncthreads();

    const int64_t P = ws.P;
    const int64_t p = (blockIdx.x * (int64_t)ENUM_THREADS + threadIdx.x) / G;
    const unsigned r = threadIdx.x % G;
    const bool live = p < P;
    const int64_t pp = live ? p : P - 1;
    const bool closed = args.closed != 0;

    int32_t base[N], cnt[N], dg[N];
    double d[N], grad[N];
#pragma unroll
    for (int i = 0; i < N; ++i) {
        base[i] = ws.base[i * P + pp];
        cnt[i] = ws.cnt[i * P + pp];
    }
    const uint64_t T = ws.total[pp];
    const uint64_t q = T / G, rem = T % G;
    const uint64_t start = r * q + (r < rem ? r : rem);
    const uint64_t len = live ? q + (r < rem ? 1 : 0) : 0;
    // decode the first index of the chunk
    {
        uint64_t idx = start;
#pragma unroll
        for (int i = N - 1; i >= 0; --i) {
            const uint64_t c = (uint64_t)cnt[i];
            dg[i] = (int32_t)(idx % c);
            idx /= c;
        }
    }
    int64_t sumN = 0;
#pragma unroll
    for (int i = 0; i < N; ++i) {
        d[i] = (double)(base[i] + dg[i]) - ws.nc[i * P + pp];
        sumN += base[i] + dg[i];
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
    for (uint64_t it = 0; it < len; ++it) {
        if (!closed || sumN == args.N_hat) {
            ++scored;
            if (E < best) {
                best = E;
                bidx = start + it;
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
    // reduce (best, bidx) over the G threads of the pixel
    if (G > 1) {
        constexpr int W = G < 32 ? G : 32;
#pragma unroll
        for (int o = W / 2; o > 0; o >>= 1) {
            const double e2 = __shfl_xor_sync(0xffffffffu, best, o);
            const uint64_t i2 = __shfl_xor_sync(0xffffffffu, bidx, o);
            qa_lexmin(best, bidx, e2, i2);
        }
        if (G > 32) {  // G == ENUM_THREADS: the whole block is one pixel
            if ((threadIdx.x & 31) == 0) {
                sE[threadIdx.x >> 5] = best;
                sI[threadIdx.x >> 5] = bidx;
            }
            __syncthreads();
            if (threadIdx.x == 0) {
                for (int w = 1; w < ENUM_THREADS / 32; ++w) qa_lexmin(best, bidx, sE[w], sI[w]);
            }
        }
    }
    if (live && r == 0) ws.best[p] = bidx;
    if (stats && closed) qa_warp_count(&stats->n_candidates_scored, scored);  // open: counted by the prologue
}

// ------------------------------------------------------------------------------------------------------------------
// Finalize: one thread per pixel (qa_finalize_pixel in qa_internal.cuh).
__global__ void __launch_bounds__(FIN_THREADS) qa_finalize_kernel(const QaDevModel *__restrict__ mdl,
                                                                  const double *__restrict__ Vg, QaWorkspace ws,
                                                                  int32_t *__restrict__ outN, double *__restrict__ outE,
                                                                  double *__restrict__ outVs)
{
    const int64_t p = blockIdx.x * (int64_t)FIN_THREADS + threadIdx.x;
    if (p >= ws.P) return;
    qa_finalize_pixel(mdl, Vg, ws, p, ws.best[p], outN, outE, outVs);
}

// FP64 issue-rate probe: 8 independent DFMA chains per thread.
__global__ void __launch_bounds__(256) qa_fp64_probe_kernel(double *sink, int iters)
{
    double a0 = threadIdx.x * 1e-9, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6,
           a7 = a0 + 7;
    const double m = 1.0 + 1e-12 * (blockIdx.x + 1), c = 1e-13;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            a0 = fma(a0, m, c);
            a1 = fma(a1, m, c);
            a2 = fma(a2, m, c);
            a3 = fma(a3, m, c);
            a4 = fma(a4, m, c);
            a5 = fma(a5, m, c);
            a6 = fma(a6, m, c);
            a7 = fma(a7, m, c);
        }
    }
    const double s = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;
    if (s == -1.2345) sink[0] = s;  // never true; keeps the chains alive
}

template <int N>
cudaError_t launch_prologue_n(const QaDevModel *d_model, const double *d_Vg, QaWorkspace ws, QaCallArgs args,
                              double *d_xcont, qa_stats *d_stats, cudaStream_t stream)
{
    const unsigned blocks = (unsigned)((ws.P + PRO_THREADS - 1) / PRO_THREADS);
    qa_prologue_kernel<N><<<blocks, PRO_THREADS, 0, stream>>>(d_model, d_Vg, ws, args, d_xcont, d_stats);
    return cudaGetLastError();
}

template <int N>
cudaError_t launch_enumerate_n(const QaDevModel *d_model, QaWorkspace ws, QaCallArgs args, double expect_cand,
                               qa_stats *d_stats, cudaStream_t stream)
{
    if (expect_cand <= 64.0) {
        const unsigned blocks = (unsigned)((ws.P + ENUM_THREADS - 1) / ENUM_THREADS);
        qa_enumerate_kernel<N, 1><<<blocks, ENUM_THREADS, 0, stream>>>(d_model, ws, args, d_stats);
        qa_plan_add("qa_enumerate_kernel<G=1>");
    } else if (expect_cand <= 4096.0) {
        const unsigned blocks = (unsigned)((ws.P * 32 + ENUM_THREADS - 1) / ENUM_THREADS);
        qa_enumerate_kernel<N, 32><<<blocks, ENUM_THREADS, 0, stream>>>(d_model, ws, args, d_stats);
        qa_plan_add("qa_enumerate_kernel<G=32>");
    } else {
        qa_enumerate_kernel<N, ENUM_THREADS><<<(unsigned)ws.P, ENUM_THREADS, 0, stream>>>(d_model, ws, args, d_stats);
        qa_plan_add("qa_enumerate_kernel<G=256>");
    }
    return cudaGetLastError();
}

}  // namespace

#define QA_DISPATCH_N(n, CALL)                                                                                         \
    switch (n) {                                                                                                       \
        case 1: return CALL(1);                                                                                        \
        case 2: return CALL(2);                                                                                        \
        case 3: return CALL(3);                                                                                        \
        case 4: return CALL(4);                                                                                        \
        case 5: return CALL(5);                                                                                        \
        case 6: return CALL(6);                                                                                        \
        case 7: return CALL(7);                                                                                        \
        case 8: return CALL(8);                                                                                        \
        case 9: return CALL(9);                                                                                        \
        case 10: return CALL(10);                                                                                      \
        case 11: return CALL(11);                                                                                      \
        case 12: return CALL(12);                                                                                      \
        case 13: return CALL(13);                                                                                      \
        case 14: return CALL(14);                                                                                      \
        case 15: return CALL(15);                                                                                      \
        case 16: return CALL(16);                                                                                      \
        default: return cudaErrorInvalidValue;                                                                         \
    }

cudaError_t qa_launch_prologue(const QaDevModel *d_model, int n, int g, const double *d_Vg, QaWorkspace ws,
                               QaCallArgs args, double *d_xcont, qa_stats *d_stats, cudaStream_t stream)
{
    (void)g;
    qa_plan_add("qa_prologue_kernel");
#define CALL(NN) launch_prologue_n<NN>(d_model, d_Vg, ws, args, d_xcont, d_stats, stream)
    QA_DISPATCH_N(n, CALL)
#undef CALL
}

cudaError_t qa_launch_enumerate(const QaDevModel *d_model, int n, QaWorkspace ws, QaCallArgs args, double expect_cand,
                                qa_stats *d_stats, cudaStream_t stream)
{
#define CALL(NN) launch_enumerate_n<NN>(d_model, ws, args, expect_cand, d_stats, stream)
    QA_DISPATCH_N(n, CALL)
#undef CALL
}

cudaError_t qa_launch_finalize(const QaDevModel *d_model, const double *d_Vg, QaWorkspace ws, int32_t *d_N, double *d_E,
                               double *d_Vsensor, qa_stats *d_stats, cudaStream_t stream)
{
    (void)d_stats;
    qa_plan_add("qa_finalize_kernel");
    const unsigned blocks = (unsigned)((ws.P + FIN_THREADS - 1) / FIN_THREADS);
    qa_finalize_kernel<<<blocks, FIN_THREADS, 0, stream>>>(d_model, d_Vg, ws, d_N, d_E, d_Vsensor);
    return cudaGetLastError();
}

cudaError_t qa_launch_fp64_probe(double *d_sink, int blocks, int threads, int iters, cudaStream_t stream)
{
    (void)threads;
    qa_fp64_probe_kernel<<<blocks, 256, 0, stream>>>(d_sink, iters);
    return cudaGetLastError();
}
