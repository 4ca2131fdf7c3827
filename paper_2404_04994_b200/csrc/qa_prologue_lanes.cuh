// qa_prologue_lanes.cuh -- steps S1-S4 and the base-point gradient of one pixel with SIXTEEN LANES PER PIXEL (lane i <->
// dot i; a warp carries two pixels), shared by qa_prologue_lanes_kernel (qa_kernels_generic.cu) and the one-kernel path of
// 9..12-dot arrays (qa_kernels_fused_mid.cu).  Open arrays.  N_c,i keeps the fixed fma chain over k (reading R1); the other
// dots' values travel by shuffles inside the 16-lane group; the QP (L106, reading R3) is the clamp-only active set with
// every lane of the pixel solving the same 1x1 / 2x2 / 3x3 system in registers (qa_qp_small_open's arithmetic); more than
// three clamped dots or a non-Maxwell c_dd go to the serial solver on the pixel's first lane.
#pragma once
#include "qa_internal.cuh"
#include "qa_prologue.cuh"

// The serial QP of one pixel on its own frame: cx holds N_c on entry and the constrained minimum on return.
template <int N>
__device__ __noinline__ void pl_slow_qp(const double *__restrict__ sC, double *cx, bool general, int *st)
{
    double c[N], xs[N];
    for (int j = 0; j < N; ++j) c[j] = xs[j] = cx[j];
    bool failed = false;
    st[0] = qa_qp_clamp<N>(sC, c, false, 0.0, general, xs, failed);
    st[1] = failed ? 1 : 0;
    for (int j = 0; j < N; ++j) cx[j] = xs[j];
}

// What lane i of a pixel ends up with.
struct QaLaneOut {
    double nc, x, gi, e0;     // N_c,i; continuous minimum x_i; row i of M (base - N_c); E(base) (all lanes of the pixel)
    int32_t base, cnt;        // candidate range of dot i
    uint64_t total;           // product of cnt over the pixel's dots (all lanes)
    int rounds;
    unsigned neg0;            // dots with a negative analytic minimum (0: no QP)
    bool failed, slow;
};

// sCgT[k*N + i] = C_gd[i][k], sC row-major c_dd, sMT[j*N + i] = M[i][j]; sVrow = the pixel's g gate voltages, sXrow = N
// doubles of scratch of the pixel (shared memory).  i = lane & 15, gb = lane & 16, dot = i < N.  All 32 lanes must call.
template <int N>
__device__ __forceinline__ void qa_lanes_pixel(const double *__restrict__ sCgT, const double *__restrict__ sC,
                                               const double *__restrict__ sMT, const double *__restrict__ sVrow,
                                               double *__restrict__ sXrow, int g, int i, int gb, bool dot, const QaCallArgs &args,
                                               QaLaneOut &o)
{
    const int ii = dot ? i : 0;
    // S1 (R1): N_c,i = fma(C_gd[i,k], V[k], acc), k ascending
    double nc = 0.0;
    for (int k = 0; k < g; ++k) nc = fma(sCgT[k * N + ii], sVrow[k], nc);
    // S2 (open): x = N_c.  S3: clamp-only active set
    double x = nc;
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
        slow = !done && args.general_qp != 0;
        for (;;) {
            const unsigned negm = (__ballot_sync(0xffffffffu, dot && x < 0.0) >> gb) & 0xffffu & ~A;
            if (!done && !slow) {
                if (!negm) {
                    done = true;
                } else {
                    A |= negm;
                    ++rounds;
                    if (__popc(A) == N) {
                        x = 0.0;
                        done = true;
                    } else if (__popc(A) > 3) {
                        slow = true;
                    }
                }
            }
            const bool work = !done && !slow;
            if (!__any_sync(0xffffffffu, work)) break;
            // closed form for |A| <= 3 (every lane of the pixel computes the same y): qa_qp_small_open's arithmetic
            const unsigned Aw = work ? A : 1u;
            const int ia = __ffs(Aw) - 1;
            const unsigned A2 = Aw & (Aw - 1);
            const int ib = A2 ? __ffs(A2) - 1 : ia;
            const unsigned A3 = A2 & (A2 - 1);
            const int ic = A3 ? __ffs(A3) - 1 : ib;
            const double ca = __shfl_sync(0xffffffffu, nc, gb + ia), cb = __shfl_sync(0xffffffffu, nc, gb + ib),
                         cc = __shfl_sync(0xffffffffu, nc, gb + ic);
            if (work) {
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
        // more than three clamped dots, or a c_dd with a positive off-diagonal: the serial solver on the pixel's first lane
        if (__any_sync(0xffffffffu, slow)) {
            if (slow && dot) sXrow[i] = nc;
            __syncwarp();
            if (slow && i == 0) {
                int st2[2];
                pl_slow_qp<N>(sC, sXrow, args.general_qp != 0, st2);
                rounds = st2[0];
                failed = st2[1] != 0;
            }
            __syncwarp();
            if (slow && dot) x = sXrow[i];
        }
    }
    // S4: candidate range of dot i
    int32_t base = 0, cnt = 1;
    if (dot) {
        if (args.alg == QA_ALG_BRUTE_FORCE) {
            base = 0;
            cnt = args.n_max + 1;
        } else {
            qa_floor_ceil(x, args.t, args.alg == QA_ALG_THRESHOLDED, base, cnt);
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
    for (int o = 8; o > 0; o >>= 1) {
        e0 += __shfl_xor_sync(0xffffffffu, e0, o);
        total *= __shfl_xor_sync(0xffffffffu, total, o);
    }
    o.nc = nc;
    o.x = x;
    o.gi = gi;
    o.e0 = e0;
    o.base = base;
    o.cnt = cnt;
    o.total = total;
    o.rounds = rounds;
    o.neg0 = neg0;
    o.failed = failed;
    o.slow = slow;
}
