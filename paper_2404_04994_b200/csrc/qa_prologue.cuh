// qa_prologue.cuh -- device functions of steps S1-S4 (N_c, analytic minimum, exact QP, candidate ranges), shared by the
// prologue kernel (qa_kernels_generic.cu) and the fused small-array kernel (qa_kernels_fused.cu).  One thread = one pixel.
#pragma once
#include "qa_internal.cuh"

struct QaPixelFlags {
    bool neg, failed;
    int rounds, doublings;
};

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

// Open array, one to three clamped dots A (nearly every QP pixel of a sweep): y_A = -C_AA^-1 c_A from the explicit inverse of
// the 1x1 / 2x2 / 3x3 block (registers only), x_F = c_F + C_FA y_A, x_A = 0 exactly (R3).  Returns false if a bound
// multiplier y_A is negative beyond rounding (KKT violated).  c and x are fully unrolled: static register indices.
template <int N>
__device__ __forceinline__ bool qa_qp_small_open(const double *__restrict__ sC, const double *c, unsigned A, double scale,
                                                 double *x)
{
    const int ia = __ffs(A) - 1;
    const unsigned A2 = A & (A - 1);
    const int ib = A2 ? __ffs(A2) - 1 : ia;
    const unsigned A3 = A2 & (A2 - 1);
    const int ic = A3 ? __ffs(A3) - 1 : ib;
    double ca = 0.0, cb = 0.0, cc = 0.0;
#pragma unroll
    for (int f = 0; f < N; ++f) {
        if (f == ia) ca = c[f];
        if (f == ib) cb = c[f];
        if (f == ic) cc = c[f];
    }
    double ya, yb = 0.0, yc = 0.0;
    if (A3) {
        const double a = sC[ia * N + ia], b = sC[ia * N + ib], cq = sC[ia * N + ic];
        const double d = sC[ib * N + ib], e = sC[ib * N + ic], f = sC[ic * N + ic];
        const double k00 = d * f - e * e, k01 = cq * e - b * f, k02 = b * e - cq * d;
        const double k11 = a * f - cq * cq, k12 = b * cq - a * e, k22 = a * d - b * b;
        const double det = a * k00 + b * k01 + cq * k02;
        ya = -(k00 * ca + k01 * cb + k02 * cc) / det;
        yb = -(k01 * ca + k11 * cb + k12 * cc) / det;
        yc = -(k02 * ca + k12 * cb + k22 * cc) / det;
    } else if (A2) {
        const double Caa = sC[ia * N + ia], Cab = sC[ia * N + ib], Cbb = sC[ib * N + ib];
        const double det = Caa * Cbb - Cab * Cab;
        ya = (cb * Cab - ca * Cbb) / det;
        yb = (ca * Cab - cb * Caa) / det;
    } else {
        ya = -ca / sC[ia * N + ia];
    }
#pragma unroll
    for (int f = 0; f < N; ++f) {
        double s = c[f] + sC[f * N + ia] * ya;
        if (A2) s += sC[f * N + ib] * yb;
        if (A3) s += sC[f * N + ic] * yc;
        x[f] = ((A >> f) & 1u) ? 0.0 : s;  // clamped components are exactly 0 (R3)
    }
    return !(ya < -1e-9 * scale || yb < -1e-9 * scale || yc < -1e-9 * scale);  // KKT: bound multipliers must be >= 0
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
        if (!general && !closed && __popc(A) <= 3) {
            if (!qa_qp_small_open<N>(sC, c, A, scale, x)) failed = true;
            continue;
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
// S1-S4 of one pixel: N_c (fixed fma order, R1), analytic minimum (Eq. (6) L90 / Eq. (7)), QP when a component is
// negative (L82-L84, L106), candidate ranges base_i .. base_i + cnt_i - 1.  sCgd is [N][g] (stride g), sC is [N][N].
template <int N>
__device__ __forceinline__ void qa_prologue_pixel(const double *__restrict__ sCgd, const double *__restrict__ sC,
                                                  const double *__restrict__ sC1, double oneC1, int g,
                                                  const double *__restrict__ v, const QaCallArgs &args, double (&nc)[N],
                                                  double (&x)[N], int32_t (&base)[N], int32_t (&cnt)[N], QaPixelFlags &fl)
{
    const bool closed = args.closed != 0;
    // S1: N_c,i = fma(C_gd[i,k], V[k], acc), k ascending (R1)
#pragma unroll
    for (int i = 0; i < N; ++i) nc[i] = 0.0;
    for (int k = 0; k < g; ++k) {
        const double vk = __ldg(v + k);
#pragma unroll
        for (int i = 0; i < N; ++i) nc[i] = fma(sCgd[i * g + k], vk, nc[i]);
    }
    // S2
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
    int doublings = 0;
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
            // t = 1 is the closed default set, never empty for a feasible x (sum lo <= sum x = N_hat < sum lo + n up to
            // rounding << 1; reading R5).  Were it empty, the search reports an empty set (N = -1, E = inf).
            break;
        }
    }
    fl.neg = neg;
    fl.failed = failed;
    fl.rounds = rounds;
    fl.doublings = doublings;
}
