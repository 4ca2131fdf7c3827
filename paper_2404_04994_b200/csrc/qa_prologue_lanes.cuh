// qa_prologue_lanes.cuh -- steps S1-S4 and the base-point gradient of one pixel with SIXTEEN LANES PER PIXEL (lane i <->
// dot i; a warp carries two pixels), shared by qa_prologue_lanes_kernel (qa_kernels_generic.cu) and the one-kernel path of
// 9..12-dot arrays (qa_kernels_fused_mid.cu).  Open and closed arrays.  N_c,i keeps the fixed fma chain over k (reading R1);
// the other dots' values travel by shuffles inside the 16-lane group; the QP is described at qa_lanes_pixel.
#pragma once
#include "qa_internal.cuh"
#include "qa_prologue.cuh"

// The serial QP of one pixel on its own frame: cx[0..N-1] = N_c, cx[N..2N-1] = the analytic minimum (the solver starts from
// it); the constrained minimum replaces cx[0..N-1].
template <int N>
__device__ __noinline__ void pl_slow_qp(const double *__restrict__ sC, double *cx, bool closed, double Nhat, bool general,
                                        int *st)
{
    double c[N], xs[N];
    for (int j = 0; j < N; ++j) {
        c[j] = cx[j];
        xs[j] = cx[N + j];
    }
    bool failed = false;
    st[0] = qa_qp_clamp<N>(sC, c, closed, Nhat, general, xs, failed);
    st[1] = failed ? 1 : 0;
    for (int j = 0; j < N; ++j) cx[j] = xs[j];
}

// What lane i of a pixel ends up with.
struct QaLaneOut {
    double nc, x, gi, e0;     // N_c,i; continuous minimum x_i; row i of M (base - N_c); E(base) (all lanes of the pixel)
    int32_t base, cnt;        // candidate range of dot i
    uint64_t total;           // product of cnt over the pixel's dots (all lanes)
    int rounds, doublings;
    unsigned neg0;            // dots with a negative analytic minimum (0: no QP)
    bool failed, slow;
};

// sum over the 16 lanes of the pixel's group (fixed butterfly order)
__device__ __forceinline__ double qa_gsum(double v)
{
#pragma unroll
    for (int o = 8; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// sCgT[k*N + i] = C_gd[i][k], sC row-major c_dd, sMT[j*N + i] = M[i][j], sC1 = c_dd 1; sVrow = the pixel's g gate voltages,
// sXrow = 2 N doubles of scratch of the pixel (shared memory).  i = lane & 15, gb = lane & 16, dot = i < N.  All 32 lanes
// of a warp must call (its two pixels run the QP rounds in lockstep).
//
// QP (L106, reading R3), Maxwell c_dd: clamp-only active set A (never released).  Per round the equality-constrained
// problem on the free set F is solved in c_dd:  y_A = a - lambda b,  C_AA a = -c_A,  C_AA b = C_AF 1_F (closed only),
//   lambda = (N_hat - sum c_F - 1^T C_FA a) / (1^T C_FF 1 - 1^T C_FA b)   (open: 0),
//   x_F = c_F + C_FA y_A + lambda C_FF 1_F,   x_A = 0 exactly;   KKT: y_A - lambda >= 0.
// Open arrays with |A| <= 3: explicit inverse in registers (qa_qp_small_open's arithmetic).  Otherwise the two small SPD
// systems are solved by conjugate gradients with lane a <-> unknown a: c_dd is diagonally dominant (condition number 2-3),
// so |A| + 2 iterations reach the rounding floor; every iteration is one 16-wide matrix-vector product out of shared
// memory and two butterfly sums.  A c_dd with a positive off-diagonal, N_hat <= 0 and a fully clamped closed pixel go to
// the serial solver on the pixel's first lane.
template <int N>
__device__ __forceinline__ void qa_lanes_pixel(const double *__restrict__ sCgT, const double *__restrict__ sC,
                                               const double *__restrict__ sMT, const double *__restrict__ sC1, double oneC1,
                                               const double *__restrict__ sVrow, double *__restrict__ sXrow, int g, int i, int gb,
                                               bool dot, const QaCallArgs &args, QaLaneOut &o)
{
    const int ii = dot ? i : 0;
    const bool closed = args.closed != 0;
    const double Nhat = (double)args.N_hat;
    // S1 (R1): N_c,i = fma(C_gd[i,k], V[k], acc), k ascending
    double nc = 0.0;
    for (int k = 0; k < g; ++k) nc = fma(sCgT[k * N + ii], sVrow[k], nc);
    if (!dot) nc = 0.0;
    // S2: open x = N_c; closed Eq. (7) L102 in the fixed order of R1 (s = sum N_c left to right: every lane the same chain)
    double x = nc;
    if (closed) {
        double ssum = 0.0;
#pragma unroll
        for (int j = 0; j < N; ++j) ssum = ssum + __shfl_sync(0xffffffffu, nc, gb + j);
        const double lam = (Nhat - ssum) / oneC1;
        x = fma(lam, sC1[ii], nc);
    }
    const double x0 = x;
    // S3
    int rounds = 0;
    bool failed = false, slow = false;
    const unsigned neg0 = (__ballot_sync(0xffffffffu, dot && x < 0.0) >> gb) & 0xffffu;
    if (__any_sync(0xffffffffu, neg0 != 0u)) {
        double scale = fabs(nc);
#pragma unroll
        for (int o = 8; o > 0; o >>= 1) scale = fmax(scale, __shfl_xor_sync(0xffffffffu, scale, o));
        scale = fmax(scale, 1.0);
        unsigned A = 0;
        bool done = neg0 == 0u;
        slow = !done && (args.general_qp != 0 || (closed && args.N_hat <= 0));
        for (;;) {
            const unsigned negm = (__ballot_sync(0xffffffffu, dot && x < 0.0) >> gb) & 0xffffu & ~A;
            if (!done && !slow) {
                if (!negm) {
                    done = true;
                } else {
                    A |= negm;
                    ++rounds;
                    if (__popc(A) == N) {
                        if (closed) {
                            slow = true;
                        } else {
                            x = 0.0;
                            done = true;
                        }
                    }
                }
            }
            const bool work = !done && !slow;
            if (!__any_sync(0xffffffffu, work)) break;
            const unsigned Aw = work ? A : 1u;
            const bool inA = dot && ((Aw >> i) & 1u);
            // (which of the two solvers a pixel gets depends on that pixel alone, not on the other pixel of its warp)
            const bool small = !closed && __popc(Aw) <= 3;
            const bool workS = work && small, workC = work && !small;
            if (__any_sync(0xffffffffu, workS)) {
                // open, |A| <= 3: explicit inverse (qa_qp_small_open's arithmetic)
                const int ia = __ffs(Aw) - 1;
                const unsigned A2 = Aw & (Aw - 1);
                const int ib = A2 ? __ffs(A2) - 1 : ia;
                const unsigned A3 = A2 & (A2 - 1);
                const int ic = A3 ? __ffs(A3) - 1 : ib;
                const double ca = __shfl_sync(0xffffffffu, nc, gb + ia), cb = __shfl_sync(0xffffffffu, nc, gb + ib),
                             cc = __shfl_sync(0xffffffffu, nc, gb + ic);
                if (workS) {
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
                    double sx = nc + sC[ii * N + ia] * ya;
                    if (A2) sx += sC[ii * N + ib] * yb;
                    if (A3) sx += sC[ii * N + ic] * yc;
                    x = ((A >> i) & 1u) ? 0.0 : sx;  // clamped components are exactly 0 (R3)
                    if (ya < -1e-9 * scale || yb < -1e-9 * scale || yc < -1e-9 * scale) failed = true;  // KKT
                }
            }
            if (!__any_sync(0xffffffffu, workC)) continue;
            // ---- conjugate gradients on C_AA a = -c_A and (closed) C_AA b = C_AF 1_F; lane a <-> unknown a
            double rF = 0.0;  // sum_{f in F} C[i][f]
            if (closed) {
#pragma unroll
                for (int j = 0; j < N; ++j)
                    if (!((Aw >> j) & 1u)) rF += sC[ii * N + j];
            }
            double za = 0.0, zb = 0.0;
            double ra = (workC && inA) ? -nc : 0.0, rb = (workC && inA && closed) ? rF : 0.0;
            double pa = ra, pb = rb;
            double rsa = qa_gsum(ra * ra), rsb = closed ? qa_gsum(rb * rb) : 0.0;
            const double tola = 1e-32 * rsa, tolb = 1e-32 * rsb;
            const int myit = workC ? __popc(Aw) + 2 : 0;  // a pixel's own iteration count (not its warp neighbour's)
            const int itmax = __reduce_max_sync(0xffffffffu, myit);
            for (int it = 0; it < itmax; ++it) {
                __syncwarp();
                if (dot) {
                    sXrow[i] = pa;
                    sXrow[N + i] = pb;
                }
                __syncwarp();
                double Apa = 0.0, Apb = 0.0;
#pragma unroll
                for (int j = 0; j < N; ++j) {
                    const double cij = sC[ii * N + j];
                    Apa = fma(cij, sXrow[j], Apa);
                    Apb = fma(cij, sXrow[N + j], Apb);
                }
                if (!inA) Apa = Apb = 0.0;
                const double da = qa_gsum(pa * Apa);
                const double ala = (it < myit && rsa > tola && da > 0.0) ? rsa / da : 0.0;
                za = fma(ala, pa, za);
                ra = fma(-ala, Apa, ra);
                const double rsa2 = qa_gsum(ra * ra);
                const double bea = (it < myit && rsa > tola && rsa > 0.0) ? rsa2 / rsa : 0.0;
                pa = fma(bea, pa, ra);
                rsa = rsa2;
                if (closed) {
                    const double db = qa_gsum(pb * Apb);
                    const double alb = (it < myit && rsb > tolb && db > 0.0) ? rsb / db : 0.0;
                    zb = fma(alb, pb, zb);
                    rb = fma(-alb, Apb, rb);
                    const double rsb2 = qa_gsum(rb * rb);
                    const double beb = (it < myit && rsb > tolb && rsb > 0.0) ? rsb2 / rsb : 0.0;
                    pb = fma(beb, pb, rb);
                    rsb = rsb2;
                }
            }
            // C_FA a, C_FA b for the free lanes, lambda, x
            __syncwarp();
            if (dot) {
                sXrow[i] = za;
                sXrow[N + i] = zb;
            }
            __syncwarp();
            double Ca = 0.0, Cb = 0.0;
#pragma unroll
            for (int j = 0; j < N; ++j) {
                const double cij = sC[ii * N + j];
                Ca = fma(cij, sXrow[j], Ca);
                Cb = fma(cij, sXrow[N + j], Cb);
            }
            double lam = 0.0;
            const bool fr = dot && !inA;
            if (closed) {
                const double s0 = qa_gsum(fr ? nc : 0.0), s1 = qa_gsum(fr ? Ca : 0.0);
                const double s2 = qa_gsum(fr ? rF : 0.0), s3 = qa_gsum(fr ? Cb : 0.0);
                lam = ((Nhat - s0) - s1) / (s2 - s3);
            }
            if (workC) {
                const double yi = za - lam * zb;  // multiplier direction of a clamped lane
                double sx = nc + Ca;
                if (closed) sx += lam * (rF - Cb);
                if (closed && __popc(Aw) == N - 1) sx = Nhat;  // R3: a single free dot carries the whole charge, exactly
                x = inA ? 0.0 : sx;                            // clamped components are exactly 0 (R3)
                if (inA && yi - lam < -1e-9 * scale) failed = true;  // KKT: multipliers of the clamped bounds >= 0
            }
            failed = ((__ballot_sync(0xffffffffu, failed) >> gb) & 0xffffu) != 0u;  // the pixel fails if any of its lanes does
        }
        // a c_dd with a positive off-diagonal, N_hat <= 0, a fully clamped closed pixel: the serial solver on the first lane
        if (__any_sync(0xffffffffu, slow)) {
            __syncwarp();
            if (slow && dot) {
                sXrow[i] = nc;
                sXrow[N + i] = x0;
            }
            __syncwarp();
            if (slow && i == 0) {
                int st2[2];
                pl_slow_qp<N>(sC, sXrow, closed, Nhat, args.general_qp != 0, st2);
                rounds = st2[0];
                failed = st2[1] != 0;
            }
            __syncwarp();
            if (slow && dot) x = sXrow[i];
            failed = ((__ballot_sync(0xffffffffu, failed) >> gb) & 0xffffu) != 0u;
        }
    }
    // S4: candidate range of dot i; closed + thresholded: per-pixel threshold doubling until the kept set is non-empty
    // (L141, reading R5)
    int32_t base = 0, cnt = 1;
    int doublings = 0;
    if (args.alg == QA_ALG_BRUTE_FORCE) {
        cnt = dot ? args.n_max + 1 : 1;
    } else {
        const bool thr = args.alg == QA_ALG_THRESHOLDED;
        double tt = thr ? args.t : 1.0;
        for (;;) {
            base = 0;
            cnt = 1;
            if (dot) qa_floor_ceil(x, tt, thr, base, cnt);
            if (!closed) break;
            int smin = dot ? base : 0, smax = dot ? base + cnt - 1 : 0;
#pragma unroll
            for (int oo = 8; oo > 0; oo >>= 1) {
                smin += __shfl_xor_sync(0xffffffffu, smin, oo);
                smax += __shfl_xor_sync(0xffffffffu, smax, oo);
            }
            const bool again = !(smin <= args.N_hat && args.N_hat <= smax) && thr && tt < 1.0;
            if (again) {
                tt = tt > 0.0 ? fmin(1.0, 2.0 * tt) : 1.0;
                ++doublings;
            }
            if (!__any_sync(0xffffffffu, again)) break;  // (a finished pixel recomputes the same range)
        }
    }
    const double d0 = dot ? (double)base - nc : 0.0;
    // base-point gradient: row i of M d0 (j ascending), h_i = grad_i + 1/2 M_ii, E(base) = 1/2 sum_i d0_i grad_i
    double gi = 0.0;
#pragma unroll
    for (int j = 0; j < N; ++j) gi = fma(sMT[j * N + ii], __shfl_sync(0xffffffffu, d0, gb + j), gi);
    double e0 = dot ? d0 * gi : 0.0;
    uint64_t total = (uint64_t)cnt;
#pragma unroll
    for (int oo = 8; oo > 0; oo >>= 1) {
        e0 += __shfl_xor_sync(0xffffffffu, e0, oo);
        total *= __shfl_xor_sync(0xffffffffu, total, oo);
    }
    o.nc = nc;
    o.x = x;
    o.gi = gi;
    o.e0 = e0;
    o.base = base;
    o.cnt = cnt;
    o.total = total;
    o.rounds = rounds;
    o.doublings = doublings;
    o.neg0 = neg0;
    o.failed = failed;
    o.slow = slow;
}
