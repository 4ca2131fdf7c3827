// qa_kernels_minplus.cu -- the hot path for n >= 13: default algorithm, open array (S5 + S6 [+ S7] of SURVEY.md section
// 8(a)) as a "min-plus" split of the candidate lattice: ONE FP64-pipe instruction per candidate, every one of them
// independent of the others (no running sum, no dependent chain).
//
// The n bits of a candidate b (N = base + b, L123-L127) are split into three groups (low bit j <-> dot n-1-j):
//     w = bits [0, NW)        u = bits [NW, NL), NL = NU + NW        t = bits [NL, n)  (NH = n - NL of them)
// One thread owns one high pattern t of one pixel and scores its 2^NL candidates (u, w).  With d0 = base - N_c,
// h_i = [M d0]_i + 1/2 M_ii (prologue) and h'_j = h_j + sum_{jh in t} M[j][jh], the energy (C1) L607 separates as
//     e(t,u,w) = A[u] + ( B[w] + QL[u,w] )
//     B[w]     = offW + sum_{j in w} h'_j                 2^NW values, registers, built once per (thread, pixel)
//     A[u]     = be + offU + sum_{j in u} h'_j            (bits of u >> 2 added from the highest down, then {0, h'_NW, h'_NW+1, sum})
//     QL[u,w]  = pair energy sum_{j<j' in (u,w)} M_jj'    pixel- and thread-independent: kernel parameter (constant bank)
//     be       = E(base) + QHT[t] + sum_{jh in t} h_jh    offW = E_C + sum_{j<NW} |h_j|,  offU = sum_{j>=NW} |h_j|
// (VT[t][j] = the cross term of t with low bit j and QHT[t] = E_C + pairs(t) are model tables, qa_api.cu rebuild), so that
// min_w e = A[u] + min_w (B[w] + QL[u,w]):  per candidate ONE DADD  y = B[w] + QL[u,w]  and half an integer min3 on the high
// words.  The offsets make every y and every A positive, so the high 32 bits of the fp64 pattern order like the values; they
// are thread-independent (the bounds L_t are compared across the threads of a pixel).  Table entries reach the DADD through
// uniform registers: a real loop over chunks of 4 u (64 entries) keeps the address "uniform register + immediate"
// (LDCU.64; measured: one indexed LDCU per ~4 cycles per scheduler), and every entry serves the PX = 2 pixels a thread
// walks at once.  DESIGN.md section 6 lists what else was measured (register-bank conflicts of the min3, LDS vs LDCU).
//
//   Keys.  The pruned and the one-kernel variants compare the HIGH words as described below.  qa_minplus_walk_kernel itself
//   (ENC = 1) uses fixed-point keys: a per-pixel constant C' = 1.5 * 2^(52-k) is folded into B[0] and into a0, so every
//   B[w], y and A[u] lies in [2^(52-k), 2^(53-k)) and shares one exponent; the LOW 32 bits of the pattern are then the
//   energy in units of 2^-k rounded to nearest (one rounding of <= 1/2 unit per addition), m_u = min_w lo32(y) and
//   L_t = min_u (lo32(C' + A[u]) + m_u) are integer operations (VIMNMX3, VIADDMNMX), and k is chosen per pixel from a
//   thread-independent bound of A + y (E(base), E_C, |h_j| of all dots, the sum of all pair energies) so that A + y < 2^31
//   units: no wrap.  An estimate passes at most 10 roundings (B: C' + 4 subset adds, y: 1, A: C' + 3 adds, the sum: exact),
//   so |L_t - min e_t| <= 5 units and the thread of the arg min (and of every tie) has L_t <= min L + 10; the kernel keeps
//   the lanes within MP_ENC_SLACK = 16.  One unit is ~2^-30 of the bound (~4e-8 E_C on config 4; the high-word keys resolve
//   2^-20 of the value), so pass 2 sees fewer survivors, and the row bound costs an integer add instead of a DADD.
//   Measured: walk 87.4 -> 85.0 us, identical N and E on every test.  offW, offU and C' are the same for the 256 threads of
//   a pixel: the lanes prologue computes them once per pixel (ws.ext) and the walk reads them with the other inputs
//   (85.0 -> 80.0 us).
//   qa_minplus_walk_kernel (pass 1; a lower bound per thread; the high-word form):
//       m_u  = min_w hi32(y)                               (ALU pipe, VIMNMX3)
//       LB_u = A[u] + double(m_u, 0)   <= min_w e(t,u,w)   (truncation and rounding are monotone)
//       L_t  = min_u hi32(LB_u)
//     and, because A[u] > 0, the candidate that attains m_u has e <= A[u] + double(m_u, 0xffffffff), whose high word
//     is at most hi32(LB_u) + 2.  Hence the thread holding the argmin has L_t <= min_t' L_t' + 2.  Each warp stores
//     (min of L over its lanes, ballot of lanes with L <= that + 2): 8 bytes.  No barrier, no atomics, no shared memory.
//   qa_minplus_finish_kernel (pass 2 + S7; one warp per pixel):
//     survivors = ballot lanes of the warps whose minimum is <= the pixel minimum + 2 (a superset of the threads that can
//     hold the argmin; normally ONE thread).  Their 2^NL candidates are scored again with pass 1's arithmetic
//     (same operands, same order, so bitwise the same e) and an exact lexicographic (e, index) compare (reading R6).
//     The result is therefore exactly the argmin of the pass-1 energies, whose rounding (a few ulp of ~20 E_C) is ten
//     orders of magnitude below the 1e-9 E_C near-tie rule.  The same warp then decodes N* and recomputes E(N*) from the
//     definition (S7), so the path is three launches: prologue, walk, finish.
//
// FP64-pipe instructions per (thread, pixel) at NU = NW = 4, NH = 8: 256 (y) + 20 (A) + 16 (LB) + 15 (B) + 8 (h') + 8
// (offsets) + 11 (be, a0, lo3) = 334 per 256 candidates, i.e. 1.30 per candidate (exact-compare Gray walk: 3).  With the
// fixed-point keys (no LB additions) and offW, offU, C' read from ws.ext (written once per pixel by the lanes prologue,
// qa_kernels_generic.cu) qa_minplus_walk_kernel needs 312 = 1.22 per candidate.
//
// Index convention as in qa_kernels_walk.cu: candidate index = sum_i b_i 2^(n-1-i) = (t << NL) | (u << NW) | w.
#include "qa_internal.cuh"
#include "qa_prologue_lanes.cuh"

namespace {

constexpr int MP_THREADS = 256;
constexpr int MF_THREADS = 256;
constexpr unsigned MP_ENC_SLACK = 16u;  // fixed-point keys: how far above the minimum a bound may lie (see the kernel)

template <int NL>
struct alignas(16) MpTable {
    double q[1 << NL];
};

__host__ __device__ constexpr int mp_ctz(int k)
{
    int j = 0;
    while (((k >> j) & 1) == 0) ++j;
    return j;
}

__device__ __forceinline__ double mp_shfl(double x, int src) { return __shfl_sync(0xffffffffu, x, src); }

// ---- the walk's inner steps, each one asm volatile statement so that the order below (a software pipeline) survives:
// ptxas places a DADD's consumer right behind it and lets every warp sit out the FP64 latency otherwise.
// y[k] = b[k] + q[k], k = 0..7: eight independent DADDs
__device__ __forceinline__ void mp_add8(double (&y)[8], const double (&b)[8], const double (&q)[8])
{
    asm volatile(
        "add.f64 %0, %8, %16; add.f64 %1, %9, %17; add.f64 %2, %10, %18; add.f64 %3, %11, %19;\n"
        " add.f64 %4, %12, %20; add.f64 %5, %13, %21; add.f64 %6, %14, %22; add.f64 %7, %15, %23;"
        : "=d"(y[0]), "=d"(y[1]), "=d"(y[2]), "=d"(y[3]), "=d"(y[4]), "=d"(y[5]), "=d"(y[6]), "=d"(y[7])
        : "d"(b[0]), "d"(b[1]), "d"(b[2]), "d"(b[3]), "d"(b[4]), "d"(b[5]), "d"(b[6]), "d"(b[7]), "d"(q[0]), "d"(q[1]),
          "d"(q[2]), "d"(q[3]), "d"(q[4]), "d"(q[5]), "d"(q[6]), "d"(q[7]));
}
// m0 = min(m0, hi32(y[0..3])), m1 = min(m1, hi32(y[4..7])): four VIMNMX3
__device__ __forceinline__ void mp_min8(unsigned &m0, unsigned &m1, const double (&y)[8])
{
    asm volatile(
        "{ .reg .b32 lo, h0, h1, h2, h3, h4, h5, h6, h7;\n"
        " mov.b64 {lo,h0}, %2; mov.b64 {lo,h1}, %3; mov.b64 {lo,h2}, %4; mov.b64 {lo,h3}, %5;\n"
        " mov.b64 {lo,h4}, %6; mov.b64 {lo,h5}, %7; mov.b64 {lo,h6}, %8; mov.b64 {lo,h7}, %9;\n"
        " min.u32 h0, h0, h1; min.u32 %0, %0, h0; min.u32 h2, h2, h3; min.u32 %0, %0, h2;\n"
        " min.u32 h4, h4, h5; min.u32 %1, %1, h4; min.u32 h6, h6, h7; min.u32 %1, %1, h6; }"
        : "+r"(m0), "+r"(m1)
        : "d"(y[0]), "d"(y[1]), "d"(y[2]), "d"(y[3]), "d"(y[4]), "d"(y[5]), "d"(y[6]), "d"(y[7]));
}
// lb = a + double(m, 0)
__device__ __forceinline__ void mp_lb(double &lb, double a, unsigned m)
{
    asm volatile("{ .reg .f64 z; .reg .b32 zero; mov.b32 zero, 0; mov.b64 z, {zero,%2}; add.f64 %0, %1, z; }"
                 : "=d"(lb)
                 : "d"(a), "r"(m));
}
// L = min(L, hi32(lb))
__device__ __forceinline__ void mp_lmin(unsigned &L, double lb)
{
    asm volatile("{ .reg .b32 lo, hi; mov.b64 {lo,hi}, %1; min.u32 %0, %0, hi; }" : "+r"(L) : "d"(lb));
}

// ---- fixed-point keys (ENC = 1): every y carries the pixel's constant C' = 1.5 * 2^(52 - k) (folded into B[w]), so all of
// them share one exponent and the LOW 32 bits of the pattern are the energy in units of 2^-k, rounded to nearest.
// m0 = min(m0, lo32(y[0..3])), m1 = min(m1, lo32(y[4..7]))
__device__ __forceinline__ void mp_min8_lo(unsigned &m0, unsigned &m1, const double (&y)[8])
{
    asm volatile(
        "{ .reg .b32 hi, l0, l1, l2, l3, l4, l5, l6, l7;\n"
        " mov.b64 {l0,hi}, %2; mov.b64 {l1,hi}, %3; mov.b64 {l2,hi}, %4; mov.b64 {l3,hi}, %5;\n"
        " mov.b64 {l4,hi}, %6; mov.b64 {l5,hi}, %7; mov.b64 {l6,hi}, %8; mov.b64 {l7,hi}, %9;\n"
        " min.u32 l0, l0, l1; min.u32 %0, %0, l0; min.u32 l2, l2, l3; min.u32 %0, %0, l2;\n"
        " min.u32 l4, l4, l5; min.u32 %1, %1, l4; min.u32 l6, l6, l7; min.u32 %1, %1, l6; }"
        : "+r"(m0), "+r"(m1)
        : "d"(y[0]), "d"(y[1]), "d"(y[2]), "d"(y[3]), "d"(y[4]), "d"(y[5]), "d"(y[6]), "d"(y[7]));
}
// L = min(L, alo + m): integer lower bound of a row (alo = lo32(C' + A[u]))
__device__ __forceinline__ void mp_lmin_int(unsigned &L, unsigned alo, unsigned m)
{
    asm volatile("{ .reg .b32 s; add.u32 s, %1, %2; min.u32 %0, %0, s; }" : "+r"(L) : "r"(alo), "r"(m));
}
__device__ __forceinline__ unsigned mp_lo32(double x)
{
    return (unsigned)__double2loint(x);
}

// One chunk of the walk: the four u = 4 i + {0..3} against every w, for PX pixels, as a software pipeline over batches of
// eight DADDs: batch g is issued, then the minima of batch g-1 are taken, then the lower bound of a u whose last batch
// was g-2 is formed, then that of g-3 enters L.  q = the chunk's 4 * 2^NW table entries; a[ul][px] = A[4 i + ul].
template <int NW, int PX, int ENC = 0>
__device__ __forceinline__ void mp_chunk(const double2 *__restrict__ q, const double (&B)[PX][1 << NW],
                                         const double (&a)[4][PX], unsigned (&L)[PX])
{
    constexpr int EPB = 8 / PX;             // table entries per batch
    constexpr int BPU = (1 << NW) / EPB;    // batches per u
    constexpr int G = 4 * BPU;
    static_assert(PX == 1 || PX == 2, "batches of eight DADDs");
    double y[2][8], lb[4][PX];
    unsigned m[4][2];
#pragma unroll
    for (int ul = 0; ul < 4; ++ul) m[ul][0] = m[ul][1] = 0xffffffffu;
#pragma unroll
    for (int g = 0; g < G + 3; ++g) {
        if (g < G) {
            const int ul = g / BPU, w0 = (g % BPU) * EPB;
            double bb[8], qq[8];
#pragma unroll
            for (int k = 0; k < EPB; k += 2) {
                const double2 t2 = q[((ul << NW) | (w0 + k)) >> 1];
#pragma unroll
                for (int px = 0; px < PX; ++px) {
                    qq[px * EPB + k] = t2.x;
                    qq[px * EPB + k + 1] = t2.y;
                    bb[px * EPB + k] = B[px][w0 + k];
                    bb[px * EPB + k + 1] = B[px][w0 + k + 1];
                }
            }
            mp_add8(y[g & 1], bb, qq);
        }
        if (g >= 1 && g <= G) {
            if (ENC)
                mp_min8_lo(m[(g - 1) / BPU][0], m[(g - 1) / BPU][1], y[(g - 1) & 1]);
            else
                mp_min8(m[(g - 1) / BPU][0], m[(g - 1) / BPU][1], y[(g - 1) & 1]);
        }
        if (ENC) {  // a[ul][px] holds C' + A[u]: its low word plus the row minimum is the row's bound, in units of 2^-k
            if (g >= 2 && g - 2 < G && (g - 2) % BPU == BPU - 1) {
                const int ul = (g - 2) / BPU;
                if (PX == 2) {
                    mp_lmin_int(L[0], mp_lo32(a[ul][0]), m[ul][0]);
                    mp_lmin_int(L[PX - 1], mp_lo32(a[ul][PX - 1]), m[ul][1]);
                } else {
                    mp_lmin_int(L[0], mp_lo32(a[ul][0]), min(m[ul][0], m[ul][1]));
                }
            }
            continue;
        }
        if (g >= 2 && g - 2 < G && (g - 2) % BPU == BPU - 1) {
            const int ul = (g - 2) / BPU;
            if (PX == 2) {
                mp_lb(lb[ul][0], a[ul][0], m[ul][0]);
                mp_lb(lb[ul][PX - 1], a[ul][PX - 1], m[ul][1]);
            } else {
                mp_lb(lb[ul][0], a[ul][0], min(m[ul][0], m[ul][1]));
            }
        }
        if (g >= 3 && (g - 3) % BPU == BPU - 1) {
            const int ul = (g - 3) / BPU;
#pragma unroll
            for (int px = 0; px < PX; ++px) mp_lmin(L[px], lb[ul][px]);
        }
    }
}

// ---------------------------------------------------------------------------------------------------------------------
// pass 1.  PX pixels per thread at once: every table entry fetched into a uniform register serves PX DADDs.
template <int NH, int NU, int NW, int PX, int MINB, int ENC_ = 0>
__global__ void __launch_bounds__(MP_THREADS, MINB) qa_minplus_walk_kernel(const QaDevModel *__restrict__ mdl,
                                                                           const __grid_constant__ MpTable<NU + NW> tab,
                                                                           QaWorkspace ws)
{
    constexpr int ENC = ENC_;
    constexpr int NL = NU + NW;
    constexpr int N = NL + NH;
    constexpr int TPP = 1 << NH;             // threads per pixel
    constexpr int WPP = TPP / 32;            // warps per pixel
    constexpr int SLOTS = MP_THREADS / TPP;  // pixel groups in flight per CTA
    constexpr int NV = N + 1 + (ENC_ ? 3 : 0);  // per-pixel inputs: h[0..N-1], E(base) (+ offW, offU, C' from ws.ext)
    constexpr int NCH = 1 << (NU - 2);       // chunks of 4 u each
    static_assert(NH >= 5 && NH <= 8 && N <= 31 && NW >= 2 && NU >= 2, "one or more whole warps per pixel");

    const unsigned lane = threadIdx.x & 31u;
    const unsigned t = threadIdx.x & (TPP - 1);
    const int slot = threadIdx.x >> NH;
    const unsigned wq = (threadIdx.x >> 5) % WPP;  // this warp's index among the pixel's warps
    const int64_t P = ws.P;

    static_assert(NL == QA_WALK_NL, "the model's VT / QHT tables are built for NL = QA_WALK_NL");
    double v[NL];  // pixel-independent per-thread constants (model tables, qa_api.cu rebuild)
#pragma unroll
    for (int j = 0; j < NL; ++j) v[j] = mdl->VT[t * NL + j];
    const double EC = mdl->EC;
    const double QH = mdl->QHT[t];
    // Every slot (the TPP threads of one pixel group) is an independent worker; consecutive workers sit in different
    // CTAs so that a ragged last round is spread over all SMs.
    const int64_t groups = (P + PX - 1) / PX;
    const int64_t workers = (int64_t)gridDim.x * SLOTS;
    const int64_t worker = (int64_t)slot * gridDim.x + blockIdx.x;
    // lane i < NV of every warp carries input i of the warp's pixel; the next group's is fetched one iteration ahead
    auto fetch = [&](int64_t grp, int px) -> double {
        double r = 0.0;
        if (grp < groups && lane < NV) {
            int64_t p = grp * PX + px;
            if (p >= P) p = P - 1;  // ragged last group: the last pixel is walked twice, stored once
            r = lane < N ? __ldg(ws.h + (int64_t)lane * P + p)
                         : (lane == N ? __ldg(ws.e0 + p) : __ldg(ws.ext + (int64_t)(lane - N - 1) * P + p));
        }
        return r;
    };
    qa_pdl_launch_dependents();
    qa_pdl_wait();  // everything above reads model constants only; h / e0 come from the prologue kernel
    double nextv[PX];
#pragma unroll
    for (int px = 0; px < PX; ++px) nextv[px] = fetch(worker, px);

    for (int64_t grp = worker; grp < groups; grp += workers) {
        double B[PX][1 << NW];  // B[w]: bits of w added from the highest to the lowest
        double hu[PX][NU];      // h' of the u bits
        double a0[PX], lo3[PX];
        double Cenc[PX];  // ENC: the pixel's fixed-point constant C' = 1.5 * 2^(52 - k)
#pragma unroll
        for (int px = 0; px < PX; ++px) {
            const double myv = nextv[px];
            nextv[px] = fetch(grp + workers, px);
            // The offsets must be the same for every thread of the pixel (the L_t are compared across threads), so they
            // are built from |h_j|, not |h'_j|: h'_j = h_j + v_j(t) >= h_j because M = c_dd^-1 of a Maxwell matrix is >= 0.
            double hw[NW], offw = EC, offu = 0.0;
#pragma unroll
            for (int j = 0; j < NL; ++j) {
                const double hj = mp_shfl(myv, N - 1 - j);
                if (j < NW) {
                    hw[j] = hj + v[j];
                    if (!ENC) offw += fabs(hj);
                } else {
                    hu[px][j - NW] = hj + v[j];
                    if (!ENC) offu += fabs(hj);
                }
            }
            double be = mp_shfl(myv, N) + QH;
#pragma unroll
            for (int jh = 0; jh < NH; ++jh) {
                const double hv = mp_shfl(myv, N - 1 - NL - jh);
                if ((t >> jh) & 1u) be += hv;
            }
            if (ENC) {  // thread-independent constants of the pixel, computed once by the prologue (ws.ext)
                offw = mp_shfl(myv, N + 1);
                offu = mp_shfl(myv, N + 2);
                Cenc[px] = mp_shfl(myv, N + 3);
            } else {
                Cenc[px] = 0.0;
            }
            a0[px] = be + offu;
            lo3[px] = hu[px][1] + hu[px][0];
            B[px][0] = offw;
            if (ENC) {
                a0[px] += Cenc[px];     // (every A[u] of the chunk loop then carries C': one rounding to the grid per add)
                B[px][0] += Cenc[px];
            }
#pragma unroll
            for (int w = 1; w < (1 << NW); ++w) B[px][w] = B[px][w & (w - 1)] + hw[mp_ctz(w)];
        }

        // A[u] = ah[u >> 2] + lo[u & 3]: ah adds the bits of u >> 2 from the highest down, lo = {0, h'_NW, h'_NW+1, their sum}.
        // A real loop, one iteration per 4 * 2^NW candidates: the table address is a uniform register plus an immediate
        // (LDCU UR, c[0x0][UR + imm]) and ptxas schedules one short basic block.  (Fully unrolled it interleaves the chunks,
        // hoists every table load and spills.)  iv mirrors the loop counter in a vector register the compiler cannot
        // identify with it: a vector use of the counter itself would turn every table load into a per-thread LDC.
        unsigned L[PX];
#pragma unroll
        for (int px = 0; px < PX; ++px) L[px] = 0xffffffffu;
        int iv;
        asm volatile("mov.u32 %0, 0;" : "=r"(iv));
#pragma unroll 1
        for (int i = 0; i < NCH; ++i, ++iv) {
            const double2 *q = reinterpret_cast<const double2 *>(tab.q) + (i << (NW + 1));
            double a[4][PX];
#pragma unroll
            for (int px = 0; px < PX; ++px) {
                double ah = a0[px];
#pragma unroll
                for (int j = NU - 1; j >= 2; --j)
                    if ((iv >> (j - 2)) & 1) ah += hu[px][j];
                a[0][px] = ah;
                a[1][px] = ah + hu[px][0];
                a[2][px] = ah + hu[px][1];
                a[3][px] = ah + lo3[px];
            }
            mp_chunk<NW, PX, ENC>(q, B, a, L);
        }

#pragma unroll
        for (int px = 0; px < PX; ++px) {
            const unsigned wmin = __reduce_min_sync(0xffffffffu, L[px]);
            const unsigned ball = __ballot_sync(0xffffffffu, L[px] <= wmin + (ENC ? MP_ENC_SLACK : 2u));
            const int64_t p = grp * PX + px;
            if (lane == 0 && p < P) ws.rec[p * WPP + wq] = make_uint2(wmin, ball);
        }
    }
}

// ---------------------------------------------------------------------------------------------------------------------
// pass 1 with exact pruning (opt-in: qa_set_walk_variant(2)).  One WARP owns a pair of pixels.
//   bound:   every high pattern t gets LB_t = be_t + sum_{j low} min(0, h'_j) <= every e(t, ., .) (the pair energies are
//            >= 0 because M >= 0 for a Maxwell c_dd), and UB = min_t (LB_t + QL[b_t]), b_t = {j : h'_j < 0}: the energy of a
//            real candidate.  A pattern with LB_t > UB cannot hold the argmin (nor a tie of it).
//   compact: the surviving patterns of the pixel (7 % of the 256 on config 4) are listed in shared memory;
//   walk:    32 of them at a time, one per lane, through the same chunk loop as qa_minplus_walk_kernel (the pair table
//            is lane-independent; VT[t], QHT[t] are gathered per lane);
//   record:  the per-pattern bounds L_t are turned into the same per-32-patterns records (minimum, ballot) the full
//            walk writes, so qa_minplus_finish_kernel runs unchanged.
// Same argmin as the full enumeration; the candidates of the pruned patterns are covered by the bound, not scored.
template <int NH, int NU, int NW, int MINB>
__global__ void __launch_bounds__(MP_THREADS, MINB) qa_minplus_pruned_kernel(const QaDevModel *__restrict__ mdl,
                                                                             const __grid_constant__ MpTable<NU + NW> tab,
                                                                             QaWorkspace ws)
{
    constexpr int PX = 2;
    constexpr int NL = NU + NW;
    constexpr int N = NL + NH;
    constexpr int TP = 1 << NH;          // high patterns per pixel
    constexpr int KP = TP / 32;          // patterns per lane in the bound phase = records per pixel
    constexpr int NCH = 1 << (NU - 2);
    constexpr int WARPS = MP_THREADS / 32;
    static_assert(NH >= 5 && NH <= 8 && NW >= 2 && NU >= 2, "whole groups of 32 patterns");
    __shared__ unsigned sL[WARPS][PX][TP];        // L_t of every pattern (0xffffffff: pruned)
    __shared__ unsigned char sList[WARPS][PX][TP];  // surviving patterns

    const unsigned lane = threadIdx.x & 31u;
    const int wid = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);  // warp-uniform, and ptxas can see it
    const int64_t P = ws.P;
    const double EC = mdl->EC;
    const int64_t groups = (P + PX - 1) / PX;
    const int64_t nwarps = (int64_t)gridDim.x * WARPS;
    // cross terms of the pattern t = 32 k + lane with low bit j: VT[t][j] = VT[lane][j] + VT[32 k][j]
    __shared__ double sVTk[KP][NL];
    for (int e = threadIdx.x; e < KP * NL; e += MP_THREADS) sVTk[e / NL][e % NL] = mdl->VT[((e / NL) << 5) * NL + (e % NL)];
    double vl[NL];
#pragma unroll
    for (int j = 0; j < NL; ++j) vl[j] = mdl->VT[lane * NL + j];
    __syncthreads();
    qa_pdl_launch_dependents();
    qa_pdl_wait();

    // pixel pairs are handed out through a counter (zeroed by the prologue kernel): the survivors per pixel vary
    (void)nwarps;
    for (;;) {
        long long take = 0;
        if (lane == 0) take = (long long)atomicAdd(reinterpret_cast<unsigned long long *>(ws.counter), 1ull);
        const int64_t grp = __shfl_sync(0xffffffffu, take, 0);
        if (grp >= groups) break;
        double myv[PX];
        int S[PX];
#pragma unroll
        for (int px = 0; px < PX; ++px) {
            int64_t p = grp * PX + px;
            if (p >= P) p = P - 1;
            myv[px] = 0.0;
            if (lane <= N) myv[px] = lane < N ? __ldg(ws.h + (int64_t)lane * P + p) : __ldg(ws.e0 + p);
            // ---- bound phase: lane handles the patterns t = 32 k + lane.  Both the cross terms and the high-bit sums split
            // into a lane part (bits 0..4 of t; vl, per kernel / hlane, per pixel) and a k part (bits 5.., uniform: sVTk, hk)
            double hb[NL];
#pragma unroll
            for (int j = 0; j < NL; ++j) hb[j] = mp_shfl(myv[px], N - 1 - j) + vl[j];
            double hk[KP], blane = mp_shfl(myv[px], N);
#pragma unroll
            for (int k = 0; k < KP; ++k) hk[k] = 0.0;
#pragma unroll
            for (int jh = 0; jh < NH; ++jh) {
                const double hv = mp_shfl(myv[px], N - 1 - NL - jh);
                if (jh < 5) {
                    if ((lane >> jh) & 1u) blane += hv;
                } else {
#pragma unroll
                    for (int k = 0; k < KP; ++k)
                        if ((k >> (jh - 5)) & 1) hk[k] += hv;
                }
            }
            double LBk[KP], ub = INFINITY;
#pragma unroll
            for (int k = 0; k < KP; ++k) {
                const unsigned t = (unsigned)k * 32u + lane;
                double lb = (blane + hk[k]) + mdl->QHT[t];
                unsigned bl = 0;
#pragma unroll
                for (int j = 0; j < NL; ++j) {
                    const double hpj = hb[j] + sVTk[k][j];
                    if (hpj < 0.0) {
                        lb += hpj;
                        bl |= 1u << j;
                    }
                }
                LBk[k] = lb;
                ub = fmin(ub, lb + mdl->QL[bl]);
                sL[wid][px][t] = 0xffffffffu;
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) ub = fmin(ub, mp_shfl(ub, (int)(lane ^ o)));
            ub += 1e-9 * EC;  // rounding of the bounds is ~1e-15 relative; the margin keeps every tie of the minimum
            // ---- compaction
            int cnt = 0;
#pragma unroll
            for (int k = 0; k < KP; ++k) {
                const bool keep = LBk[k] <= ub;
                const unsigned bal = __ballot_sync(0xffffffffu, keep);
                if (keep) sList[wid][px][cnt + __popc(bal & ((1u << lane) - 1u))] = (unsigned char)(k * 32 + lane);
                cnt += __popc(bal);
            }
            S[px] = cnt;  // >= 1: the pattern attaining ub is kept
        }
        __syncwarp();
        // ---- walk the survivors, 32 at a time
        const int rounds = __shfl_sync(0xffffffffu, (max(S[0], S[1]) + 31) >> 5, 0);
#pragma unroll 1
        for (int rd = 0; rd < rounds; ++rd) {
            double B[PX][1 << NW], hu[PX][NU], a0[PX], lo3[PX];
            unsigned tt[PX];
            bool valid[PX];
#pragma unroll
            for (int px = 0; px < PX; ++px) {
                const int idx = rd * 32 + (int)lane;
                valid[px] = idx < S[px];
                const unsigned t = sList[wid][px][valid[px] ? idx : 0];
                tt[px] = t;
                double hw[NW], offw = EC, offu = 0.0;
#pragma unroll
                for (int j = 0; j < NL; ++j) {
                    const double hj = mp_shfl(myv[px], N - 1 - j);
                    const double hpj = hj + mdl->VT[t * NL + j];
                    if (j < NW) {
                        hw[j] = hpj;
                        offw += fabs(hj);
                    } else {
                        hu[px][j - NW] = hpj;
                        offu += fabs(hj);
                    }
                }
                double be = mp_shfl(myv[px], N) + mdl->QHT[t];
#pragma unroll
                for (int jh = 0; jh < NH; ++jh) {
                    const double hv = mp_shfl(myv[px], N - 1 - NL - jh);
                    if ((t >> jh) & 1u) be += hv;
                }
                a0[px] = be + offu;
                lo3[px] = hu[px][1] + hu[px][0];
                B[px][0] = offw;
#pragma unroll
                for (int w = 1; w < (1 << NW); ++w) B[px][w] = B[px][w & (w - 1)] + hw[mp_ctz(w)];
            }
            unsigned L[PX];
#pragma unroll
            for (int px = 0; px < PX; ++px) L[px] = 0xffffffffu;
            int iv;
            asm volatile("mov.u32 %0, 0;" : "=r"(iv));
#pragma unroll 1
            for (int i = 0; i < NCH; ++i, ++iv) {
                const double2 *q = reinterpret_cast<const double2 *>(tab.q) + (i << (NW + 1));
                double a[4][PX];
#pragma unroll
                for (int px = 0; px < PX; ++px) {
                    double ah = a0[px];
#pragma unroll
                    for (int j = NU - 1; j >= 2; --j)
                        if ((iv >> (j - 2)) & 1) ah += hu[px][j];
                    a[0][px] = ah;
                    a[1][px] = ah + hu[px][0];
                    a[2][px] = ah + hu[px][1];
                    a[3][px] = ah + lo3[px];
                }
                mp_chunk<NW, PX>(q, B, a, L);
            }
#pragma unroll
            for (int px = 0; px < PX; ++px)
                if (valid[px]) sL[wid][px][tt[px]] = L[px];
        }
        __syncwarp();
        // ---- records in the format of the full walk: one per 32 consecutive patterns
#pragma unroll
        for (int px = 0; px < PX; ++px) {
            const int64_t p = grp * PX + px;
#pragma unroll
            for (int qd = 0; qd < KP; ++qd) {
                const unsigned v = sL[wid][px][qd * 32 + (int)lane];
                const unsigned wmin = __reduce_min_sync(0xffffffffu, v);
                const unsigned ball = __ballot_sync(0xffffffffu, v != 0xffffffffu && v - wmin <= 2u);
                if (lane == 0 && p < P) ws.rec[p * KP + qd] = make_uint2(wmin, ball);
            }
        }
        __syncwarp();
    }
}

// ---------------------------------------------------------------------------------------------------------------------
// pass 2 + S7: one warp per pixel, PERSISTENT warps.  A pixel costs a warp a chain of dependent steps (records -> minimum ->
// survivor -> its constants -> 2^NL candidates -> lexicographic minimum -> N*, E(N*)), so what the kernel pays for is
// latency, not arithmetic.  Hence: every warp walks pixels gw, gw + #warps, ... and requests the inputs of its NEXT pixel
// (one value per lane: h_lane or E(base); the warp records; base and N_c of the lane's dot) before it works on the current
// one, whose inputs sit in shared memory; the survivor's constants (VT[t], QHT[t]) are read from the model tables the walk
// kernel has just left in L2, lane i keeps row i of M in registers for S7, and each lane scores a block of CPL consecutive
// candidates with a static add tree.
// Pass 2 + S7 of ONE pixel by one warp (all 32 lanes call).  h: the pixel's h[0..N-1], E(base) (shared memory); r: the
// record of walk warp `lane` (lanes < WPP); base_i, nc_i: base point and N_c of dot `lane` (lanes < N); ql: the lane's table
// entries QL[lane * CPL ..]; mrow(j) = M[lane][j]; sd: N doubles of scratch of this warp.  outN == nullptr: only best[p].
template <int NH, int NU, int NW, class MRow>
__device__ __forceinline__ void mp_finish_pixel(const QaDevModel *__restrict__ mdl, const double *__restrict__ h, uint2 r,
                                                int32_t base_i, double nc_i, const double2 (&ql)[(1 << (NU + NW - 5)) / 2],
                                                double EC, unsigned slack, double *__restrict__ sd, MRow mrow, int64_t p,
                                                uint64_t *__restrict__ best, int32_t *__restrict__ outN,
                                                double *__restrict__ outE)
{
    constexpr int NL = NU + NW;
    constexpr int N = NL + NH;
    constexpr int WPP = (1 << NH) / 32;
    constexpr int LB = NL - 5;          // log2 of the candidates per lane
    constexpr int CPL = 1 << LB;        // candidates per lane: w = (wb << LB) + c, one u per lane
    static_assert(LB >= 1 && LB <= NW, "a lane's block of candidates lies inside one u");
    const unsigned lane = threadIdx.x & 31u;
    const unsigned u = lane >> (NW - LB);                         // this lane's u
    const unsigned wb = lane & ((1u << (NW - LB)) - 1u);          // ... and the bits of w above its block
    const double e0 = h[N];
    const unsigned H = __reduce_min_sync(0xffffffffu, r.x);
    const unsigned wmask = __ballot_sync(0xffffffffu, lane < (unsigned)WPP && r.x <= H + slack);  // warps that may hold the argmin

    // thread-independent offsets, as pass 1 formed them (j ascending)
    double offw = EC, offu = 0.0;
#pragma unroll
    for (int j = 0; j < NL; ++j) {
        if (j < NW)
            offw += fabs(h[N - 1 - j]);
        else
            offu += fabs(h[N - 1 - j]);
    }

    double bestE = INFINITY;
    unsigned bestI = 0xffffffffu;
    for (int q = 0; q < WPP; ++q) {
        unsigned surv = __shfl_sync(0xffffffffu, r.y, q);
        if (!((wmask >> q) & 1u)) continue;
        while (surv) {
            const unsigned ts = (unsigned)q * 32u + (unsigned)(__ffs(surv) - 1);
            surv &= surv - 1;
            // the survivor's inputs as pass 1 built them (same operands, same order)
            double hp[NL];
#pragma unroll
            for (int j = 0; j < NL; ++j) hp[j] = h[N - 1 - j] + __ldg(mdl->VT + ts * NL + j);
            double be = e0 + __ldg(mdl->QHT + ts);
#pragma unroll
            for (int jh = 0; jh < NH; ++jh)
                if ((ts >> jh) & 1u) be += h[N - 1 - NL - jh];
            // A[u] = ah[u >> 2] + lo[u & 3]
            double a = be + offu;
#pragma unroll
            for (int j = NU - 1; j >= 2; --j)
                if ((u >> j) & 1u) a += hp[NW + j];
            if ((u & 3u) == 1u) a += hp[NW];
            if ((u & 3u) == 2u) a += hp[NW + 1];
            if ((u & 3u) == 3u) a += hp[NW + 1] + hp[NW];
            // B[w] of the lane's block: bits of w from the highest down
            double b[CPL];
            b[0] = offw;
#pragma unroll
            for (int j = NW - 1; j >= LB; --j)
                if ((wb >> (j - LB)) & 1u) b[0] += hp[j];
#pragma unroll
            for (int c = 1; c < CPL; ++c) b[c] = b[c & (c - 1)] + hp[mp_ctz(c)];
            double e1 = INFINITY;
            unsigned i1 = 0;
#pragma unroll
            for (int c = 0; c < CPL; c += 2) {
                const double ea = a + (b[c] + ql[c >> 1].x), eb = a + (b[c + 1] + ql[c >> 1].y);
                if (ea < e1) {  // c ascending within the lane: strict '<' keeps the smallest index
                    e1 = ea;
                    i1 = c;
                }
                if (eb < e1) {
                    e1 = eb;
                    i1 = c + 1;
                }
            }
            i1 |= (ts << NL) | (lane << LB);
            // lexicographic (e, index) minimum over the lanes.  Every e is positive (the offsets), so its bit pattern
            // orders like its value: minimum of the high words, then of the low words among the lanes that hold it,
            // then of the indices among those -- three warp reductions instead of five shuffle rounds.
            const unsigned ehi = (unsigned)__double2hiint(e1), elo = (unsigned)__double2loint(e1);
            const unsigned mhi = __reduce_min_sync(0xffffffffu, ehi);
            const unsigned mlo = __reduce_min_sync(0xffffffffu, ehi == mhi ? elo : 0xffffffffu);
            const bool tie = ehi == mhi && elo == mlo;
            const unsigned mi = __reduce_min_sync(0xffffffffu, tie ? i1 : 0xffffffffu);
            const double em = __hiloint2double((int)mhi, (int)mlo);
            if (em < bestE || (em == bestE && mi < bestI)) {
                bestE = em;
                bestI = mi;
            }
        }
    }
    if (!outN) {
        if (lane == 0) best[p] = (uint64_t)bestI;
        return;
    }
    // S7: N* and E(N*) = 1/2 d^T M d from the definition (Eq. (C1)); lane i holds dot i and row i of M
    int32_t Ni = 0;
    double di = 0.0;
    if (lane < (unsigned)N) {
        Ni = base_i + (int32_t)((bestI >> (N - 1 - lane)) & 1u);
        di = (double)Ni - nc_i;
        sd[lane] = di;
    }
    __syncwarp();
    double row = 0.0;
#pragma unroll
    for (int j = 0; j < N; ++j) row = fma(mrow(j), sd[j], row);
    double E = di * row;  // lanes >= N hold di = 0
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) E += mp_shfl(E, (int)(lane ^ o));
    if (lane < (unsigned)N) outN[p * N + lane] = Ni;
    if (lane == 0) outE[p] = 0.5 * E;
}

template <int NH, int NU, int NW>
__global__ void __launch_bounds__(MF_THREADS) qa_minplus_finish_kernel(const QaDevModel *__restrict__ mdl,
                                                                       QaWorkspace ws, int32_t *__restrict__ outN,
                                                                       double *__restrict__ outE, unsigned slack)
{
    constexpr int NL = NU + NW;
    constexpr int N = NL + NH;
    constexpr int WPP = (1 << NH) / 32;
    constexpr int LB = NL - 5;          // log2 of the candidates per lane
    constexpr int CPL = 1 << LB;        // candidates per lane: w = (wb << LB) + c, one u per lane
    constexpr int WARPS = MF_THREADS / 32;
    static_assert(LB >= 1 && LB <= NW, "a lane's block of candidates lies inside one u");
    __shared__ double sIn[WARPS][N + 1];   // h[0..N-1], E(base) of the warp's current pixel
    __shared__ double sd[WARPS][QA_MAXN];
    const unsigned lane = threadIdx.x & 31u;
    const int wid = threadIdx.x >> 5;
    const int64_t P = ws.P;
    const int64_t gw = (int64_t)wid * gridDim.x + blockIdx.x;   // consecutive warps sit in different CTAs (ragged tail)
    const int64_t tw = (int64_t)gridDim.x * WARPS;

    // model constants: the lane's table entries, row `lane` of M, and the survivor tables in shared memory
    const double EC = mdl->EC;
    double2 ql[CPL / 2];
#pragma unroll
    for (int c = 0; c < CPL / 2; ++c) ql[c] = reinterpret_cast<const double2 *>(mdl->QL + lane * CPL)[c];
    double Mrow[N];
    {
        const int li = lane < (unsigned)N ? (int)lane : 0;
#pragma unroll
        for (int j = 0; j < N; ++j) Mrow[j] = mdl->M[li * QA_MAXN + j];
    }
    qa_pdl_wait();  // model constants above; everything below was written by the prologue / walk kernels

    // inputs of a pixel, one value per lane
    double in_v = 0.0, in_nc = 0.0;
    int32_t in_base = 0;
    uint2 in_r = make_uint2(0xffffffffu, 0u);
    auto request = [&](int64_t p) {
        if (p >= P) return;
        if (lane <= (unsigned)N) in_v = lane < (unsigned)N ? __ldg(ws.h + (int64_t)lane * P + p) : __ldg(ws.e0 + p);
        if (lane < (unsigned)N) {
            in_base = ws.base[(int64_t)lane * P + p];
            in_nc = ws.nc[(int64_t)lane * P + p];
        }
        in_r = lane < (unsigned)WPP ? ws.rec[p * WPP + lane] : make_uint2(0xffffffffu, 0u);
    };
    request(gw);
    for (int64_t p = gw; p < P; p += tw) {
        const uint2 r = in_r;
        const int32_t base_i = in_base;
        const double nc_i = in_nc;
        if (lane <= (unsigned)N) sIn[wid][lane] = in_v;
        __syncwarp();
        request(p + tw);
        const double *__restrict__ h = sIn[wid];
        mp_finish_pixel<NH, NU, NW>(mdl, h, r, base_i, nc_i, ql, EC, slack, sd[wid], [&](int j) { return Mrow[j]; }, p, ws.best,
                                    outN, outE);
        __syncwarp();  // sIn / sd are rewritten by the next iteration
    }
}

// ---------------------------------------------------------------------------------------------------------------------
// The whole path S1-S7 of a 16-dot open array in ONE persistent kernel (NH = 8: a CTA of 256 threads = the 2^8 high
// patterns of one pixel pair).  With three launches the step pays two launch gaps and two cold starts (prologue and finish
// are ~15 us kernels that keep 2-20 % of the machine busy).  Here the walk of pixel pair `it` by all eight warps is pass 1
// exactly as in qa_minplus_walk_kernel, and two small duties ride along in the issue slots the walk leaves idle:
//   * the warp it % 8 first runs S1-S4 of pair it + LA (sixteen lanes per pixel: qa_prologue_lanes.cuh) into a
//     shared-memory ring (h, E(base), base, N_c),
//   * the warps (it + 3) % 8 and (it + 5) % 8 first run pass 2 + S7 (mp_finish_pixel) of the two pixels of pair it - FD from
//     the ring (the eight warps left the records of that pair there).
// There is no CTA barrier in the loop: a barrier per pair makes seven warps wait for the one that has a duty.  The warps
// drift instead, and three counters per ring slot order the data (producer: data, fence, counter; consumer: counter,
// fence, data): fIn = "inputs of pair j are in the slot", fRec = "warps that have left their record of pair j", fFin =
// "pixels of pair j finished" (the slot may be refilled).  Every wait refers to work that other warps do in an EARLIER
// iteration of theirs, so the waits are well-founded (no cycle); all warps of a CTA are resident, so they make progress.
// Nothing but V_g is read from and nothing but N*, E(N*) (and x) is written to global memory; no workspace.
__device__ __forceinline__ void mp_wait_eq(const unsigned *f, unsigned target)
{
    while (*reinterpret_cast<const volatile unsigned *>(f) != target) __nanosleep(40);
    __threadfence_block();
    __syncwarp();
}
__device__ __forceinline__ void mp_signal(unsigned *f, unsigned lane, unsigned value, bool add)
{
    __threadfence_block();
    __syncwarp();
    if (lane == 0) {
        if (add)
            atomicAdd(f, value);
        else
            *reinterpret_cast<volatile unsigned *>(f) = value;
    }
}

template <int NU, int NW, int MINB>
__global__ void __launch_bounds__(MP_THREADS, MINB) qa_minplus_fused_kernel(const QaDevModel *__restrict__ mdl,
                                                                            const __grid_constant__ MpTable<NU + NW> tab,
                                                                            const double *__restrict__ Vg, int64_t P,
                                                                            QaCallArgs args, int32_t *__restrict__ outN,
                                                                            double *__restrict__ outE, double *__restrict__ xcont,
                                                                            qa_stats *stats)
{
    constexpr int NH = 8, PX = 2, RING = 8, LA = 3, FD = 2;
    constexpr int NL = NU + NW;
    constexpr int N = NL + NH;
    constexpr int WPP = 8;
    constexpr int NCH = 1 << (NU - 2);
    constexpr int CPL = 1 << (NL - 5);
    static_assert(NL == QA_WALK_NL && N == 16 && MP_THREADS == 256, "one CTA = the 2^8 high patterns of a pixel pair");
    static_assert(LA + FD < RING, "a slot is refilled only after its pair is finished");
    __shared__ double sCgT[QA_MAXG * N], sC[N * N], sMT[N * N], sC1[N];
    __shared__ double sV[WPP][PX][QA_MAXG], sX[WPP][PX][2 * N];  // scratch of the warp that runs S1-S4
    __shared__ double sIn[RING][PX][N + 1], sNc[RING][PX][N];
    __shared__ int32_t sBase[RING][PX][N];
    __shared__ uint2 sRec[RING][PX][WPP];
    __shared__ double sd[WPP][N];
    __shared__ unsigned fIn[RING], fRec[RING], fFin[RING];

    const int tid = threadIdx.x;
    const unsigned lane = tid & 31u;
    const unsigned t = tid;
    const int wid = tid >> 5;
    const int g = mdl->g;
    for (int e = tid; e < N * N; e += MP_THREADS) {
        sMT[e] = mdl->M[(e % N) * QA_MAXN + (e / N)];
        sC[e] = mdl->C[(e / N) * QA_MAXN + (e % N)];
    }
    for (int e = tid; e < N * g; e += MP_THREADS) sCgT[e] = mdl->Cgd[(e % N) * QA_MAXG + (e / N)];
    if (tid < N) sC1[tid] = mdl->C1[tid];
    if (tid < RING) fIn[tid] = fRec[tid] = fFin[tid] = 0u;
    double v[NL];
#pragma unroll
    for (int j = 0; j < NL; ++j) v[j] = mdl->VT[t * NL + j];
    const double EC = mdl->EC;
    const double QH = mdl->QHT[t];
    __syncthreads();

    const int64_t groups = (P + PX - 1) / PX;
    // (the launcher keeps the pairs per CTA below 2^30: 32-bit loop control)
    const int nit = blockIdx.x < groups ? (int)((groups - blockIdx.x + gridDim.x - 1) / gridDim.x) : 0;
    int64_t st_np = 0, st_nq = 0, st_nr = 0, st_nf = 0;

    // S1-S4 of pixel pair j by the calling warp (sixteen lanes per pixel) into ring slot j % RING
    auto prologue = [&](int j) {
        const int64_t grp = blockIdx.x + j * (int64_t)gridDim.x;
        const int s = (int)(lane >> 4), i = (int)(lane & 15u), gb = (int)(lane & 16u);
        const int64_t p = grp * PX + s;
        const bool live = p < P;
        const int64_t pp = live ? p : P - 1;
        const int slot = j & (RING - 1);
        mp_wait_eq(&fFin[slot], (unsigned)(PX * (j / RING)));  // the pair that used the slot before is finished
        for (int k = i; k < g; k += 16) sV[wid][s][k] = __ldg(Vg + pp * g + k);
        __syncwarp();
        QaLaneOut lo;
        qa_lanes_pixel<N>(sCgT, sC, sMT, sC1, 1.0, sV[wid][s], sX[wid][s], g, i, gb, true, args, lo);
        sIn[slot][s][i] = lo.gi + 0.5 * sMT[i * N + i];
        if (i == 0) sIn[slot][s][N] = 0.5 * lo.e0;
        sNc[slot][s][i] = lo.nc;
        sBase[slot][s][i] = lo.base;
        if (live && xcont) xcont[p * N + i] = lo.x;
        if (live && i == 0) {
            ++st_np;
            st_nq += lo.neg0 != 0u ? 1 : 0;
            st_nr += lo.rounds;
            st_nf += lo.failed ? 1 : 0;
        }
        mp_signal(&fIn[slot], lane, (unsigned)(j + 1), false);
    };
    if (wid < LA && wid < nit) prologue(wid);

    for (int it = 0; it < nit + FD; ++it) {
        // ---- duty: S1-S4 of a pair ahead
        if (it + LA < nit && wid == (it & 7)) prologue(it + LA);
        // ---- duty: pass 2 + S7 of a pair behind
        if (it >= FD) {
            const int px = wid == ((it + 3) & 7) ? 0 : (wid == ((it + 5) & 7) ? 1 : -1);
            if (px >= 0) {
                const int j = it - FD;
                const int slot = j & (RING - 1);
                const int64_t p = (blockIdx.x + j * (int64_t)gridDim.x) * PX + px;
                mp_wait_eq(&fRec[slot], (unsigned)(WPP * (j / RING + 1)));  // all eight warps have left their record
                if (p < P) {
                    const uint2 r = lane < (unsigned)WPP ? sRec[slot][px][lane] : make_uint2(0xffffffffu, 0u);
                    const int li = lane < (unsigned)N ? (int)lane : 0;
                    double2 ql[CPL / 2];
#pragma unroll
                    for (int c = 0; c < CPL / 2; ++c) ql[c] = __ldg(reinterpret_cast<const double2 *>(mdl->QL + lane * CPL) + c);
                    mp_finish_pixel<NH, NU, NW>(mdl, sIn[slot][px], r, sBase[slot][px][li], sNc[slot][px][li], ql, EC, 2u, sd[wid],
                                                [&](int jj) { return sMT[jj * N + li]; }, p, nullptr, outN, outE);
                }
                mp_signal(&fFin[slot], lane, 1u, true);
            }
        }
        // ---- pass 1 of pair `it`: qa_minplus_walk_kernel's arithmetic, inputs from the ring
        if (it < nit) {
            const int slot = it & (RING - 1);
            mp_wait_eq(&fIn[slot], (unsigned)(it + 1));
            double B[PX][1 << NW], hu[PX][NU], a0[PX], lo3[PX];
#pragma unroll
            for (int px = 0; px < PX; ++px) {
                const double *__restrict__ hin = sIn[slot][px];
                double hw[NW], offw = EC, offu = 0.0;
#pragma unroll
                for (int j = 0; j < NL; ++j) {
                    const double hj = hin[N - 1 - j];
                    if (j < NW) {
                        hw[j] = hj + v[j];
                        offw += fabs(hj);
                    } else {
                        hu[px][j - NW] = hj + v[j];
                        offu += fabs(hj);
                    }
                }
                double be = hin[N] + QH;
#pragma unroll
                for (int jh = 0; jh < NH; ++jh) {
                    const double hv = hin[N - 1 - NL - jh];
                    if ((t >> jh) & 1u) be += hv;
                }
                a0[px] = be + offu;
                lo3[px] = hu[px][1] + hu[px][0];
                B[px][0] = offw;
#pragma unroll
                for (int w = 1; w < (1 << NW); ++w) B[px][w] = B[px][w & (w - 1)] + hw[mp_ctz(w)];
            }
            unsigned L[PX];
#pragma unroll
            for (int px = 0; px < PX; ++px) L[px] = 0xffffffffu;
            int iv;
            asm volatile("mov.u32 %0, 0;" : "=r"(iv));
#pragma unroll 1
            for (int i = 0; i < NCH; ++i, ++iv) {
                const double2 *q = reinterpret_cast<const double2 *>(tab.q) + (i << (NW + 1));
                double a[4][PX];
#pragma unroll
                for (int px = 0; px < PX; ++px) {
                    double ah = a0[px];
#pragma unroll
                    for (int j = NU - 1; j >= 2; --j)
                        if ((iv >> (j - 2)) & 1) ah += hu[px][j];
                    a[0][px] = ah;
                    a[1][px] = ah + hu[px][0];
                    a[2][px] = ah + hu[px][1];
                    a[3][px] = ah + lo3[px];
                }
                mp_chunk<NW, PX>(q, B, a, L);
            }
#pragma unroll
            for (int px = 0; px < PX; ++px) {
                const unsigned wmin = __reduce_min_sync(0xffffffffu, L[px]);
                const unsigned ball = __ballot_sync(0xffffffffu, L[px] <= wmin + 2u);
                if (lane == 0) sRec[slot][px][wid] = make_uint2(wmin, ball);
            }
            mp_signal(&fRec[slot], lane, 1u, true);
        }
    }
    if (stats) {
        qa_warp_count(&stats->n_pixels, st_np);
        qa_warp_count(&stats->n_qp_pixels, st_nq);
        qa_warp_count(&stats->n_qp_rounds, st_nr);
        qa_warp_count(&stats->n_qp_failed, st_nf);
        qa_warp_count(&stats->n_candidates_enumerated, st_np << N);
        qa_warp_count(&stats->n_candidates_scored, st_np << N);
    }
}

template <int NH, int NU, int NW>
cudaError_t launch_finish(const QaDevModel *d_model, QaWorkspace ws, int32_t *d_N, double *d_E, int sm_count, cudaStream_t stream,
                          unsigned slack = 2u)
{
    int per_sm = 0;
    cudaError_t err = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, qa_minplus_finish_kernel<NH, NU, NW>, MF_THREADS, 0);
    if (err != cudaSuccess) return err;
    if (per_sm < 1) per_sm = 1;
    int64_t grid = (int64_t)sm_count * per_sm;
    const int64_t need = (ws.P + MF_THREADS / 32 - 1) / (MF_THREADS / 32);
    if (grid > need) grid = need;
    return qa_launch_pdl(qa_minplus_finish_kernel<NH, NU, NW>, dim3((unsigned)grid), dim3(MF_THREADS), stream, d_model, ws, d_N,
                         d_E, slack);
}

template <int NH, int NU, int NW, int PX, int MINB, int ENC = 0>
cudaError_t launch_mp(const QaDevModel *d_model, const double *QLhost, QaWorkspace ws, int32_t *d_N, double *d_E,
                      int sm_count, cudaStream_t stream)
{
    constexpr int NL = NU + NW;
    constexpr int SLOTS = MP_THREADS >> NH;
    MpTable<NL> local;  // the first 2^NL entries of the model's table (the table of fewer low bits is a prefix)
    for (int b = 0; b < (1 << NL); ++b) local.q[b] = QLhost[b];
    int per_sm = 0;
    cudaError_t err = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, qa_minplus_walk_kernel<NH, NU, NW, PX, MINB, ENC>,
                                                                    MP_THREADS, 0);
    if (err != cudaSuccess) return err;
    if (per_sm < 1) per_sm = 1;
    int64_t grid = (int64_t)sm_count * per_sm;
    const int64_t need = ((ws.P + PX - 1) / PX + SLOTS - 1) / SLOTS;
    if (grid > need) grid = need;
    err = qa_launch_pdl(qa_minplus_walk_kernel<NH, NU, NW, PX, MINB, ENC>, dim3((unsigned)grid), dim3(MP_THREADS), stream, d_model,
                        local, ws);
    if (err != cudaSuccess) return err;
    qa_plan_add("qa_minplus_finish_kernel");
    qa_timing_mark(stream);
    return launch_finish<NH, NU, NW>(d_model, ws, d_N, d_E, sm_count, stream, ENC ? MP_ENC_SLACK : 2u);
}

}  // namespace

template <int NH>
cudaError_t launch_mp_pruned(const QaDevModel *d_model, const double *QLhost, QaWorkspace ws, int32_t *d_N, double *d_E,
                             int sm_count, cudaStream_t stream)
{
    MpTable<8> local;
    for (int b = 0; b < 256; ++b) local.q[b] = QLhost[b];
    int per_sm = 0;
    cudaError_t err = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, qa_minplus_pruned_kernel<NH, 4, 4, 2>, MP_THREADS, 0);
    if (err != cudaSuccess) return err;
    if (per_sm < 1) per_sm = 1;
    int64_t grid = (int64_t)sm_count * per_sm;
    const int64_t need = ((ws.P + 1) / 2 + MP_THREADS / 32 - 1) / (MP_THREADS / 32);
    if (grid > need) grid = need;
    err = qa_launch_pdl(qa_minplus_pruned_kernel<NH, 4, 4, 2>, dim3((unsigned)grid), dim3(MP_THREADS), stream, d_model, local, ws);
    if (err != cudaSuccess) return err;
    qa_plan_add("qa_minplus_finish_kernel");
    qa_timing_mark(stream);
    return launch_finish<NH, 4, 4>(d_model, ws, d_N, d_E, sm_count, stream);
}

// d_N == nullptr: the finish kernel only stores the winning index (ws.best) and the caller runs qa_finalize_kernel.
cudaError_t qa_launch_minplus_walk(const QaDevModel *d_model, int n, const double *QLhost, QaWorkspace ws, int32_t *d_N,
                                   double *d_E, int sm_count, int pruned, cudaStream_t stream)
{
    if (pruned) {
        qa_plan_add("qa_minplus_pruned_kernel");
        switch (n) {
            case 13: return launch_mp_pruned<5>(d_model, QLhost, ws, d_N, d_E, sm_count, stream);
            case 14: return launch_mp_pruned<6>(d_model, QLhost, ws, d_N, d_E, sm_count, stream);
            case 15: return launch_mp_pruned<7>(d_model, QLhost, ws, d_N, d_E, sm_count, stream);
            case 16: return launch_mp_pruned<8>(d_model, QLhost, ws, d_N, d_E, sm_count, stream);
            default: return cudaErrorInvalidValue;
        }
    }
    qa_plan_add("qa_minplus_walk_kernel");
    // ENC = 1: fixed-point keys on the low words (see the kernel); the high-word keys (ENC = 0) remain in the pruned and the
    // one-kernel variants
#define MP_CALL(NH) launch_mp<NH, 4, 4, 2, 2, 1>(d_model, QLhost, ws, d_N, d_E, sm_count, stream)
    switch (n) {
        case 13: return MP_CALL(5);
        case 14: return MP_CALL(6);
        case 15: return MP_CALL(7);
        case 16: return MP_CALL(8);
        default: return cudaErrorInvalidValue;
    }
#undef MP_CALL
}

// Pass 2 + S7 on records another pass 1 wrote (qa_kernels_minplus32.cu): `slack` = how far, in units of the record key, a
// thread's bound may lie above the pixel minimum and still hold the argmin.
cudaError_t qa_launch_minplus_finish(const QaDevModel *d_model, int n, QaWorkspace ws, int32_t *d_N, double *d_E, unsigned slack,
                                     int sm_count, cudaStream_t stream)
{
    qa_plan_add("qa_minplus_finish_kernel");
    qa_timing_mark(stream);
    switch (n) {
        case 13: return launch_finish<5, 4, 4>(d_model, ws, d_N, d_E, sm_count, stream, slack);
        case 14: return launch_finish<6, 4, 4>(d_model, ws, d_N, d_E, sm_count, stream, slack);
        case 15: return launch_finish<7, 4, 4>(d_model, ws, d_N, d_E, sm_count, stream, slack);
        case 16: return launch_finish<8, 4, 4>(d_model, ws, d_N, d_E, sm_count, stream, slack);
        default: return cudaErrorInvalidValue;
    }
}

// Open default search of a 16-dot Maxwell array without sensor dots: the whole path in one persistent kernel.
cudaError_t qa_launch_minplus_fused(const QaDevModel *d_model, const double *QLhost, const double *d_Vg, int64_t P, QaCallArgs args,
                                    int32_t *d_N, double *d_E, double *d_xcont, qa_stats *d_stats, int sm_count,
                                    cudaStream_t stream)
{
    qa_plan_add("qa_minplus_fused_kernel");
    MpTable<8> local;
    for (int b = 0; b < 256; ++b) local.q[b] = QLhost[b];
    int per_sm = 0;
    cudaError_t err = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, qa_minplus_fused_kernel<4, 4, 2>, MP_THREADS, 0);
    if (err != cudaSuccess) return err;
    if (per_sm < 1) per_sm = 1;
    int64_t grid = (int64_t)sm_count * per_sm;
    const int64_t need = (P + 1) / 2;
    if (grid > need) grid = need;
    if (need / grid >= ((int64_t)1 << 30)) return cudaErrorInvalidValue;  // (P <= 2^40: only with a grid below 512 CTAs)
    qa_minplus_fused_kernel<4, 4, 2><<<(unsigned)grid, MP_THREADS, 0, stream>>>(d_model, local, d_Vg, P, args, d_N, d_E, d_xcont,
                                                                               d_stats);
    return cudaGetLastError();
}
