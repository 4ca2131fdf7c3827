// qa_kernels_fused_open.cu -- the whole path S1-S7 (S8 for a model with sensor dots) of SURVEY.md section 8(a) in ONE kernel
// for OPEN arrays with n <= 8 dots and a BINARY candidate set: the default algorithm (lo + {0,1}^n, L123-L127) and the
// thresholded one (lo/round + a subset of the free dots, Eq. (9)).  This is the kernel of the dataset batch
// (BASELINE.json configs[4]: 256 arrays x 128x128 pixels x {default, t = 0.2, t = 0.5}); blockIdx.y selects the model.
//
// What bounds it: V_g is the only HBM read (8 g bytes per pixel), N*, E(N*) the only writes, so the
// floor is HBM (104 B per pixel at n = g = 8); the arithmetic next to it is ~140 FP64 instructions of per-pixel prologue
// and epilogue (N_c: n g FMA, M d0: n^2 FMA, E(base): n FMA) plus the candidate walk.  Every FMA
// of the prologue takes one operand from a per-MODEL matrix, i.e. a warp-uniform value that has to come out of shared
// memory (the model differs per CTA, so the constant bank is not available).  The kernel is a template over PX = pixels
// per thread.  PX = 2 halves that operand traffic (every uniform operand serves two FMAs / DADDs) but needs 128 registers
// and 48 KB of shared memory per CTA (N_c and the base point parked there), i.e. 16 warps per SM; measured, the kernels
// then run at 20-45 % of the FP64 pipe with 37-60 % of the issue slots: bound by latency, not by operand bandwidth.
// PX = 1 (64 registers, 20-28 KB, 32 warps per SM) is what the launcher instantiates: config 5 1.49 -> 1.21 ms per step.
//
// Register discipline: nothing in the common path is dynamically indexed, so nothing lives in local memory.  The QP
// (L106, reading R3) is solved in closed form in registers for one to three clamped dots (all but 3 in 10^5 pixels of the
// batch); larger active sets and non-Maxwell models are redone after the kernel's own stores by a __noinline__ function
// with the general solver (fo_slow_pixel), whose work arrays never touch the frame of the common path.
//
// Candidate walk.
//   default:      the static counting-order walk of qa_kernels_walk.cu over all 2^n patterns, the thread's PX pixels at once
//                 (3 FP64 instructions per candidate and pixel, one table entry per candidate for all of them).
//   thresholded:  the number of free dots k differs from pixel to pixel (2^k candidates: 4.3 on average at t = 0.2, 25.6
//                 at t = 0.5, but up to 256), so a warp of neighbouring pixels runs at the pace of its largest set.  For
//                 t <= FO_NOSORT_T = 0.6 that is accepted (every thread walks its own pixels: no sort, no CTA barrier;
//                 measured faster on config 5 up to t ~ 0.6); above, the
//                 pixels of a CTA are bucket-sorted by k in shared memory and every thread walks PX
//                 pixels of (nearly) equal k.  The walk is the counting-order walk restricted to the free dots: with the
//                 free dots f_0 < f_1 < .. (bit positions) the step st-1 -> st sets free bit j = ctz(st) and clears the
//                 free bits below it, so the linear part moves by c_j = h_{f_j} - sum_{i<j} h_{f_i} (stored per pixel in
//                 shared memory, read with a warp-uniform j) and the bit pattern by an XOR mask; ascending st is ascending
//                 pattern, so the strict '<' keeps the lexicographically smallest N among equal energies (reading R6).
//   The winner's energy is E(N*) = E(base) + dE: E(base) = 1/2 d0^T M d0 from the definition (Eq. (C1); the gradient
//   M d0 is already there) and dE = sum_{i in b} h_i + pairs(b), the increment the walk has minimised (the same expansion of
//   (C1) around the base point).  Round 2 recomputed the whole quadratic form for N* instead (n^2 + n more FMAs and N_c parked
//   in shared memory): 10 % of the kernel for the same result to a few ulp of E_C.
#include "qa_internal.cuh"
#include "qa_prologue.cuh"

namespace {

constexpr int FO_THREADS = 128;
// CTAs per SM the min-plus default walk is compiled for: 80 registers instead of 64, so that the table reads of several
// batches are in flight before their DADDs (measured, config 5 default pass: 0.412 -> 0.399 ms)
constexpr int FO_MP_CTAS = 6;
constexpr int FO_MULTI_CTAS = 8;
constexpr double FO_NOSORT_T = QA_FO_NOSORT_T;  // thresholded: at or below this t the pixels are not bucket-sorted (measured on config 5: crossover between 0.5 and 0.7)
constexpr int FO_PX_RUN = 1;  // pixels per thread the launcher instantiates (measured, config 5: 1.21 ms per step vs 1.49 with 2)
// PX = pixels per thread (2: every uniform operand serves two FMAs; 1: half the registers and shared memory per CTA, twice
// the CTAs per SM -- the thresholded kernels are bound by latency, not by the FP64 pipe), PIX = FO_THREADS * PX per CTA

__host__ __device__ constexpr int fo_ctz(int k)
{
    int j = 0;
    while (((k >> j) & 1) == 0) ++j;
    return j;
}

// Sensor step S8 on its own frame (single-model calls with sensor dots only).
__device__ __noinline__ void fo_sensor(const QaDevModel *__restrict__ mdl, const double *__restrict__ Vg, int64_t p,
                                       const int32_t *Ns, int32_t *__restrict__ outN, double *__restrict__ outVs)
{
    qa_sensor_pixel(mdl, Vg, p, Ns, outN, outVs);
}

// Open-array QP of one pixel in registers: clamp-only monotone active set (reading R3), closed form for |A| <= 3.
// x holds the analytic minimum (= c) on entry.  Returns the number of rounds.  slow = true: more than three clamped dots or a
// c_dd with a positive off-diagonal -- the pixel is redone by fo_slow_pixel at the end of the kernel (x is then unusable).
template <int N>
__device__ __forceinline__ int fo_qp_open(const double *__restrict__ sC, const double (&c)[N], int general, double (&x)[N],
                                          bool &failed, bool &slow)
{
    unsigned A = 0;
    int rounds = 0;
    slow = general != 0;
    double scale = 1.0;
#pragma unroll
    for (int i = 0; i < N; ++i) scale = fmax(scale, fabs(c[i]));
    while (!slow) {
        unsigned neg = 0;
#pragma unroll
        for (int i = 0; i < N; ++i)
            if (x[i] < 0.0) neg |= 1u << i;
        neg &= ~A;
        if (!neg) break;
        A |= neg;
        ++rounds;
        const int na = __popc(A);
        if (na == N) {
#pragma unroll
            for (int i = 0; i < N; ++i) x[i] = 0.0;
            break;
        }
        if (na > 3) {
            slow = true;
            break;
        }
        if (!qa_qp_small_open<N>(sC, c, A, scale, x)) failed = true;
    }
    return rounds;
}

// The model's tables into shared memory: QaDevModel::fo_pack holds MT | C | T (contiguous in FoSmem as well) and CgT in the
// kernel's layout, so the CTA copies 16 bytes per thread and step, without index arithmetic.
template <int N>
__device__ __forceinline__ void fo_stage(const QaDevModel *__restrict__ mdl, int g, int tid, double *sMT_C_T, double *sCgT)
{
    constexpr int N1 = (2 * N * N + (1 << N)) / 2;  // double2 entries of MT | C | T (an even number of doubles)
    static_assert((2 * N * N + (1 << N)) % 2 == 0, "16-byte copies");
    const double2 *__restrict__ src = reinterpret_cast<const double2 *>(mdl->fo_pack);
    double2 *dst = reinterpret_cast<double2 *>(sMT_C_T);
    for (int e = tid; e < N1; e += FO_THREADS) dst[e] = __ldg(src + e);
    const int n2 = (g * N + 1) >> 1;  // C_gd^T, zero padded to an even count (both sides have the room)
    double2 *dst2 = reinterpret_cast<double2 *>(sCgT);
    for (int e = tid; e < n2; e += FO_THREADS) dst2[e] = __ldg(src + N1 + e);
}

template <int N, bool THR, int PIX>
struct FoSort {  // thresholded: bookkeeping of the bucket sort and the walk
    unsigned long long xm[THR ? PIX : 1];  // XOR masks of the steps, 8 bits per free dot
    unsigned short order[THR ? PIX : 1];   // pixel slots sorted by the number of free dots, descending
    unsigned char kfree[THR ? PIX : 1];    // number of free dots
    unsigned char wkey[THR ? PIX : 1];     // winning pattern
};

template <int N, bool THR, int PIX, bool KEEP_NC = false>
struct FoSmem {
    double MT[N * N];          // MT[j*N + i] = M[i][j]: the N values a column step needs are contiguous
    double C[N * N];           // c_dd, row-major (QP)
    double T[1 << N];          // pair table of the bit patterns: T[b] = QL[b] (bit j <-> dot N-1-j)
    double nc[KEEP_NC ? N : 1][KEEP_NC ? PIX : 1];  // N_c of every pixel slot (multi-algorithm kernel: read by every pass)
    int32_t base[N][PIX];   // ... and the base point
    double cs[THR ? N : 1][PIX];     // thresholded: c_j of the compacted free dots, per pixel slot
    int bucket[16];                  // thresholded: pixels of the CTA per number of free dots (outside the union below:
                                     // zeroed before the first barrier)
    union alignas(16) {        // C_gd is dead after S1 (a barrier separates it from the sort's first write)
        double CgT[QA_MAXG * N];   // CgT[k*N + i] = C_gd[i][k]
        FoSort<N, THR, PIX> sort;
    };
};

// A pixel the register path defers (more than three clamped dots, or a c_dd with a positive off-diagonal: 3 in 10^5
// pixels of the dataset batch): the whole path S1-S7 once more, by one thread, with the general QP solver of
// qa_prologue.cuh, the same h / c_j / pair-table walk in ascending pattern order, and E(N*) from the definition.
// __noinline__, called after the kernel's own stores: its work arrays never touch the frame of the common path.
template <int N, bool THR>
__device__ __noinline__ void fo_slow_pixel(const double *__restrict__ MT, const double *__restrict__ C,
                                           const double *__restrict__ T,
                                           const QaDevModel *__restrict__ mdl, const double *__restrict__ Vg, int64_t gp,
                                           QaCallArgs args, int32_t *__restrict__ outN, double *__restrict__ outE,
                                           double *__restrict__ xcont, double *__restrict__ outVs, int *stat)
{
    const int g = mdl->g;
    double nc[N], x[N], d0[N], hp[N], cs[N];
    int32_t base[N];
    for (int i = 0; i < N; ++i) {
        double acc = 0.0;
        for (int k = 0; k < g; ++k) acc = fma(mdl->Cgd[i * QA_MAXG + k], __ldg(Vg + gp * g + k), acc);
        nc[i] = acc;
        x[i] = acc;
    }
    bool failed = false;
    const int rounds = qa_qp_clamp<N>(C, nc, false, 0.0, args.general_qp != 0, x, failed);
    unsigned fm = 0;
    for (int i = 0; i < N; ++i) {
        int32_t cn;
        qa_floor_ceil(x[i], args.t, THR, base[i], cn);
        if (cn == 2) fm |= 1u << (N - 1 - i);
        d0[i] = (double)base[i] - nc[i];
    }
    for (int i = 0; i < N; ++i) {
        double gi = 0.0;
        for (int j = 0; j < N; ++j) gi = fma(MT[j * N + i], d0[j], gi);
        hp[N - 1 - i] = gi + 0.5 * MT[i * N + i];
    }
    unsigned long long xm = 0;
    int kf = 0;
    {
        double pre = 0.0;
        unsigned low = 0;
        for (int b = 0; b < N; ++b)
            if ((fm >> b) & 1u) {
                cs[kf] = hp[b] - pre;
                pre += hp[b];
                xm |= (unsigned long long)((1u << b) | low) << (8 * kf);
                low |= 1u << b;
                ++kf;
            }
    }
    double s = 0.0, best = 0.0;
    unsigned key = 0, bkey = 0;
    for (unsigned st = 1; st < (1u << kf); ++st) {
        const int j = __ffs(st) - 1;
        s += cs[j];
        key ^= (unsigned)(xm >> (8 * j)) & 0xffu;
        const double e = s + T[key];
        if (e < best) {
            best = e;
            bkey = key;
        }
    }
    int32_t Ns[N];
    double d[N];
    for (int i = 0; i < N; ++i) {
        Ns[i] = base[i] + (int32_t)((bkey >> (N - 1 - i)) & 1u);
        d[i] = (double)Ns[i] - nc[i];
    }
    double Ed = 0.0;
    for (int i = 0; i < N; ++i) {
        double row = 0.0;
        for (int j = 0; j < N; ++j) row = fma(MT[j * N + i], d[j], row);
        Ed = fma(d[i], row, Ed);
    }
    outE[gp] = 0.5 * Ed;
    if (mdl->ns == 0) {
        for (int i = 0; i < N; ++i) outN[gp * N + i] = Ns[i];
    } else {
        qa_sensor_pixel(mdl, Vg, gp, Ns, outN, outVs);
    }
    if (xcont)
        for (int i = 0; i < N; ++i) xcont[gp * N + i] = x[i];
    stat[0] = rounds;
    stat[1] = failed ? 1 : 0;
    stat[2] = kf;
}

// Rank of the calling thread among the threads of the CTA that pass the same `key` (0..15), any order: one shared-memory
// atomic per distinct key and warp instead of one per thread (all pixels of a CTA often share a key).
__device__ __forceinline__ int fo_bucket_rank(int *bucket, int key)
{
    const unsigned peers = __match_any_sync(0xffffffffu, key);
    const unsigned lane = threadIdx.x & 31u;
    const int leader = __ffs(peers) - 1;
    int start = 0;
    if ((int)lane == leader) start = atomicAdd(&bucket[key], __popc(peers));
    start = __shfl_sync(0xffffffffu, start, leader);
    return start + __popc(peers & ((1u << lane) - 1u));
}

template <int N, bool THR, int PX, bool MP>
__global__ void __launch_bounds__(FO_THREADS, MP ? FO_MP_CTAS : 4 * (3 - PX)) qa_fused_open_kernel(const QaDevModel *const *__restrict__ models,
                                                                   const double *__restrict__ Vg, int64_t P, int g,
                                                                   QaCallArgs args, int32_t *__restrict__ outN,
                                                                   double *__restrict__ outE, double *__restrict__ xcont,
                                                                   double *__restrict__ outVs, qa_stats *stats)
{
    constexpr int FO_PX = PX, FO_PIX = FO_THREADS * PX;
    __shared__ __align__(16) FoSmem<N, THR, FO_PIX> sm;
    const int tid = threadIdx.x;
    // The thread's two pixels: slot = tid + px * FO_THREADS (coalescing: consecutive threads, consecutive rows).  The first
    // eight gate voltages of both rows are requested before anything else: their HBM round trip overlaps the staging of the
    // model tables below (g is a kernel argument so that nothing has to be read to form the addresses).
    int64_t gp[FO_PX];
    bool live[FO_PX];
#pragma unroll
    for (int px = 0; px < FO_PX; ++px) {
        const int64_t p = (int64_t)blockIdx.x * FO_PIX + px * FO_THREADS + tid;
        live[px] = p < P;
        gp[px] = (int64_t)blockIdx.y * P + (live[px] ? p : P - 1);
    }
    const double *vp[FO_PX];
#pragma unroll
    for (int px = 0; px < FO_PX; ++px) vp[px] = Vg + gp[px] * g;
    const bool vec = (g & 1) == 0 && (reinterpret_cast<uintptr_t>(Vg) & 15u) == 0;
    auto load_chunk = [&](int k0, double (&a)[FO_PX][8]) {
#pragma unroll
        for (int px = 0; px < FO_PX; ++px) {
            if (vec) {
#pragma unroll
                for (int k = 0; k < 8; k += 2) {
                    double2 ta = make_double2(0.0, 0.0);
                    if (k0 + k < g) ta = __ldg(reinterpret_cast<const double2 *>(vp[px] + k0 + k));
                    a[px][k] = ta.x, a[px][k + 1] = ta.y;
                }
            } else {
#pragma unroll
                for (int k = 0; k < 8; ++k) a[px][k] = k0 + k < g ? __ldg(vp[px] + k0 + k) : 0.0;
            }
        }
    };
    double va[FO_PX][8];
    load_chunk(0, va);
    const QaDevModel *__restrict__ mdl = models[blockIdx.y];
    fo_stage<N>(mdl, g, tid, sm.MT, sm.CgT);
    if (THR && tid < 16) sm.bucket[tid] = 0;
    const int ns = mdl->ns;
    const double EC = MP ? mdl->EC : 0.0;
    __syncthreads();

    // ---- S1-S4
    double nc[FO_PX][N], hp[FO_PX][N];   // hp[b]: energy increment of raising dot N-1-b at the base point
    unsigned freem[FO_PX];               // bit b set: dot N-1-b has two candidate values
    int rounds[FO_PX], rk[FO_PX];
    bool negf[FO_PX], failed[FO_PX], slowf[FO_PX];
#pragma unroll
    for (int px = 0; px < FO_PX; ++px)
#pragma unroll
        for (int i = 0; i < N; ++i) nc[px][i] = 0.0;
    // S1: N_c,i = fma(C_gd[i,k], V[k], acc), k ascending (R1), in chunks of 8 gates (all loads of a chunk before its FMAs)
    for (int k0 = 0; k0 < g; k0 += 8) {
        if (k0 > 0) load_chunk(k0, va);
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            if (k0 + k < g) {
#pragma unroll
                for (int i = 0; i < N; ++i) {
                    const double cg = sm.CgT[(k0 + k) * N + i];
#pragma unroll
                    for (int px = 0; px < FO_PX; ++px) nc[px][i] = fma(cg, va[px][k], nc[px][i]);
                }
            }
        }
    }
    double d0[FO_PX][N];
    double Ebase[FO_PX], dE[FO_PX];  // E(base) and the winner's energy relative to it: E(N*) = E(base) + dE (see S7 below)
#pragma unroll
    for (int px = 0; px < FO_PX; ++px) {
        // S2 + S3
        double x[N];
        bool neg = false;
#pragma unroll
        for (int i = 0; i < N; ++i) {
            x[i] = nc[px][i];
            neg |= x[i] < 0.0;
        }
        rounds[px] = 0;
        rk[px] = 0;
        failed[px] = false;
        slowf[px] = false;
        if (neg) rounds[px] = fo_qp_open<N>(sm.C, nc[px], args.general_qp, x, failed[px], slowf[px]);
        negf[px] = neg;
        // S4 (Eq. (9), readings R4 / R10)
        unsigned fm = 0;
#pragma unroll
        for (int i = 0; i < N; ++i) {
            int32_t cn, bs;
            qa_floor_ceil(x[i], args.t, THR, bs, cn);
            if (cn == 2) fm |= 1u << (N - 1 - i);
            d0[px][i] = (double)bs - nc[px][i];
            // the base point waits in shared memory while the gradient and the walk have the registers
            sm.base[i][px * FO_THREADS + tid] = bs;
        }
        freem[px] = fm;
        if (xcont && live[px] && !slowf[px]) {
#pragma unroll
            for (int i = 0; i < N; ++i) xcont[gp[px] * N + i] = x[i];
        }
    }
    {   // base-point gradient grad = M d0 (row i: j ascending), h_i = grad_i + 1/2 M_ii
        double grad[FO_PX][N];
#pragma unroll
        for (int px = 0; px < FO_PX; ++px)
#pragma unroll
            for (int i = 0; i < N; ++i) grad[px][i] = 0.0;
#pragma unroll
        for (int j = 0; j < N; ++j) {
#pragma unroll
            for (int i = 0; i < N; ++i) {
                const double mij = sm.MT[j * N + i];
#pragma unroll
                for (int px = 0; px < FO_PX; ++px) grad[px][i] = fma(mij, d0[px][j], grad[px][i]);
            }
        }
#pragma unroll
        for (int b = 0; b < N; ++b) {
            const double hm = 0.5 * sm.MT[(N - 1 - b) * N + (N - 1 - b)];
#pragma unroll
            for (int px = 0; px < FO_PX; ++px) hp[px][b] = grad[px][N - 1 - b] + hm;
        }
        // E(base) = 1/2 d0^T M d0 (Eq. (C1)) from the gradient that is already there
#pragma unroll
        for (int px = 0; px < FO_PX; ++px) {
            double eb = 0.0;
#pragma unroll
            for (int i = 0; i < N; ++i) eb = fma(d0[px][i], grad[px][i], eb);
            Ebase[px] = 0.5 * eb;
        }
    }

    asm volatile("" ::: "memory");
    // ---- S5-S6
    unsigned win[FO_PX];
    if constexpr (!THR && MP) {
        // Maxwell c_dd (pair energies >= 0), N >= 5: the min-plus split of qa_kernels_minplus.cu inside one thread.  With
        // w = bits [0,4), u = bits [4,N):  e(u,w) = A[u] + (B[w] + T[u,w]),  B[w] = offW + sum_{j in w} h'_j,
        // A[u] = offU + sum_{j in u} h'_j,  offW = E_C + sum_{j<4} |h'_j|, offU = E_C + sum_{j>=4} |h'_j| (every y = B + T and
        // every A is positive: the high 32 bits of the patterns order like the values).
        //   pass 1:  m_u = min_w hi32(y)  (one DADD + half an integer min3 per candidate),  L_u = hi32(A[u] + double(m_u, 0))
        //            is a lower bound of the row's energies, and the row of the arg min (and of every tie) has
        //            L_u <= min L + 2 (qa_kernels_minplus.cu header).  Rows are taken four at a time in a real loop; per
        //            group the minimum and the rows within 2 of it are kept (a superset of the rows within 2 of min L).
        //   pass 2:  the rows that can hold the arg min (1.2 on average) are scored with the same arithmetic and the exact
        //            compare, ascending index: the lexicographically smallest N among equal energies (reading R6).
        // 1.3 FP64 instructions per candidate instead of 3, and no dependent chain through the running sum.
        constexpr int NW = 4, NU = N - NW, R = 1 << NU, GS = R < 4 ? R : 4, NG = R / GS;
        static_assert(N > NW, "at least one high bit");
#pragma unroll
        for (int px = 0; px < FO_PX; ++px) {
            double B[1 << NW], hu[NU];
            double offw = EC, offu = EC;
#pragma unroll
            for (int j = 0; j < NW; ++j) offw += fabs(hp[px][j]);
#pragma unroll
            for (int j = 0; j < NU; ++j) {
                hu[j] = hp[px][NW + j];
                offu += fabs(hu[j]);
            }
            B[0] = offw;
#pragma unroll
            for (int w = 1; w < (1 << NW); ++w) B[w] = B[w & (w - 1)] + hp[px][fo_ctz(w)];
            const double lo3 = NU >= 2 ? hu[NU >= 2 ? 1 : 0] + hu[0] : 0.0;
            // A[u] of row u = 4 i + ul (the same expression in both passes: bitwise the same value)
            auto row_a = [&](int i, int ul) -> double {
                double ah = offu;
#pragma unroll
                for (int j = NU - 1; j >= 2; --j)
                    if ((i >> (j - 2)) & 1) ah += hu[j];
                if (NU >= 2) return ul == 0 ? ah : (ul == 1 ? ah + hu[0] : (ul == 2 ? ah + hu[NU >= 2 ? 1 : 0] : ah + lo3));
                return ul == 0 ? ah : ah + hu[0];
            };
            unsigned Lg[NG], rowmask = 0;
#pragma unroll
            for (int k = 0; k < NG; ++k) Lg[k] = 0xffffffffu;
#pragma unroll 1
            for (int i = 0; i < NG; ++i) {
                const double2 *__restrict__ T2 = reinterpret_cast<const double2 *>(sm.T + ((i * GS) << NW));
                unsigned l[GS];
#pragma unroll
                for (int ul = 0; ul < GS; ++ul) {
                    unsigned m0 = 0xffffffffu, m1 = 0xffffffffu;
#pragma unroll
                    for (int w = 0; w < (1 << NW); w += 4) {
                        const double2 ta = T2[((ul << NW) | w) >> 1], tb = T2[((ul << NW) | (w + 2)) >> 1];
                        const double y0 = B[w] + ta.x, y1 = B[w + 1] + ta.y, y2 = B[w + 2] + tb.x, y3 = B[w + 3] + tb.y;
                        m0 = min(m0, min((unsigned)__double2hiint(y0), (unsigned)__double2hiint(y1)));
                        m1 = min(m1, min((unsigned)__double2hiint(y2), (unsigned)__double2hiint(y3)));
                    }
                    const double lb = row_a(i, ul) + __hiloint2double((int)min(m0, m1), 0);
                    l[ul] = (unsigned)__double2hiint(lb);
                }
                unsigned gmin = l[0];
#pragma unroll
                for (int ul = 1; ul < GS; ++ul) gmin = min(gmin, l[ul]);
                unsigned nib = 0;
#pragma unroll
                for (int ul = 0; ul < GS; ++ul) nib |= (l[ul] <= gmin + 2u ? 1u : 0u) << ul;
                rowmask |= nib << (i * GS);
#pragma unroll
                for (int k = 0; k < NG; ++k)
                    if (k == i) Lg[k] = gmin;
            }
            unsigned Lmin = Lg[0];
#pragma unroll
            for (int k = 1; k < NG; ++k) Lmin = min(Lmin, Lg[k]);
            unsigned cand = 0;
#pragma unroll
            for (int k = 0; k < NG; ++k)
                if (Lg[k] <= Lmin + 2u) cand |= rowmask & (((1u << GS) - 1u) << (k * GS));
            double best = __longlong_as_double(0x7ff0000000000000ll);
            unsigned bkey = 0;
            while (cand) {
                const int u = __ffs(cand) - 1;
                cand &= cand - 1u;
                const double a = row_a(u / GS, u % GS);
                const double *__restrict__ T = sm.T + (u << NW);
#pragma unroll
                for (int w = 0; w < (1 << NW); ++w) {
                    const double e = a + (B[w] + T[w]);
                    if (e < best) {
                        best = e;
                        bkey = ((unsigned)u << NW) | (unsigned)w;
                    }
                }
            }
            win[px] = bkey;
            dE[px] = best - (offw + offu);  // (the offsets are exact sums of |h| and E_C: their rounding is that of best itself)
        }
    } else if constexpr (!THR) {
        // counting-order walk over all 2^N patterns, both pixels at once (qa_kernels_walk.cu).  A real loop over chunks of
        // 2^LB patterns (the fully unrolled walk is 60 KB of code and stalls on instruction fetch): inside a chunk every
        // index is static; the step into chunk i sets bit LB + ctz(i), picked from registers by a short select chain.
        constexpr int LB = N < 4 ? N : 4;
        constexpr int NHI = N - LB;
        double cl[FO_PX][LB], ch[FO_PX][NHI > 0 ? NHI : 1], s[FO_PX], m[FO_PX];
#pragma unroll
        for (int px = 0; px < FO_PX; ++px) {
            double pre = 0.0;
#pragma unroll
            for (int j = 0; j < N; ++j) {
                if (j < LB)
                    cl[px][j] = hp[px][j] - pre;
                else
                    ch[px][j - LB] = hp[px][j] - pre;
                pre += hp[px][j];
            }
            s[px] = 0.0;
            m[px] = 0.0;
            win[px] = 0;
        }
#pragma unroll 1
        for (int i = 0; i < (1 << NHI); ++i) {
            const double *__restrict__ T = sm.T + (i << LB);
            const unsigned kb = (unsigned)i << LB;
            if (i > 0) {
                const double q = T[0];
#pragma unroll
                for (int px = 0; px < FO_PX; ++px) {
                    double c = ch[px][NHI > 0 ? NHI - 1 : 0];
#pragma unroll
                    for (int j = NHI - 2; j >= 0; --j)
                        if ((i >> j) & 1) c = ch[px][j];
                    s[px] += c;
                    const double e = s[px] + q;
                    if (e < m[px]) {
                        m[px] = e;
                        win[px] = kb;
                    }
                }
            }
#pragma unroll
            for (int w = 1; w < (1 << LB); ++w) {
                const double q = T[w];
#pragma unroll
                for (int px = 0; px < FO_PX; ++px) {
                    s[px] += cl[px][fo_ctz(w)];
                    const double e = s[px] + q;
                    if (e < m[px]) {
                        m[px] = e;
                        win[px] = kb + w;
                    }
                }
            }
        }
#pragma unroll
        for (int px = 0; px < FO_PX; ++px) dE[px] = m[px];
    } else if (args.t <= FO_NOSORT_T) {
        // small thresholds (few free dots per pixel: 2^k = 4.3 candidates on average at t = 0.2, rarely more than 16): every
        // thread walks its own pixels; the warp runs at the pace of its largest set, but there is no sort and no CTA barrier
#pragma unroll
        for (int px = 0; px < FO_PX; ++px) {
            const int slot = px * FO_THREADS + tid;
            double pre = 0.0;
            int jj = 0;
            unsigned low = 0;
            unsigned long long xm = 0;
#pragma unroll
            for (int b = 0; b < N; ++b) {
                if ((freem[px] >> b) & 1u) {
                    sm.cs[jj][slot] = hp[px][b] - pre;
                    pre += hp[px][b];
                    xm |= (unsigned long long)((1u << b) | low) << (8 * jj);
                    low |= 1u << b;
                    ++jj;
                }
            }
            const unsigned nst = live[px] ? 1u << jj : 1u;
            double s = 0.0, best = 0.0;
            unsigned key = 0, bkey = 0;
            for (unsigned st = 1; st < nst; ++st) {
                const int j = __ffs(st) - 1;
                s += sm.cs[j][slot];
                key ^= (unsigned)(xm >> (8 * j)) & 0xffu;
                const double e = s + sm.T[key];
                if (e < best) {
                    best = e;
                    bkey = key;
                }
            }
            win[px] = bkey;
            dE[px] = best;
        }
    } else {
        // compaction of the free dots (ascending bit position), bucket sort of the CTA's pixels by k, walk, hand back
        __syncthreads();  // every warp is done with C_gd: its storage becomes the sort's
#pragma unroll
        for (int px = 0; px < FO_PX; ++px) {
            const int slot = px * FO_THREADS + tid;
            double pre = 0.0;
            int jj = 0;
            unsigned low = 0;
            unsigned long long xm = 0;
#pragma unroll
            for (int b = 0; b < N; ++b) {
                if ((freem[px] >> b) & 1u) {
                    sm.cs[jj][slot] = hp[px][b] - pre;
                    pre += hp[px][b];
                    xm |= (unsigned long long)((1u << b) | low) << (8 * jj);
                    low |= 1u << b;
                    ++jj;
                }
            }
            const int kf = live[px] ? jj : 0;
            sm.sort.xm[slot] = xm;
            sm.sort.kfree[slot] = (unsigned char)kf;
            sm.sort.wkey[slot] = 0;
            rk[px] = fo_bucket_rank(sm.bucket, N - kf);
        }
        __syncthreads();
#pragma unroll
        for (int px = 0; px < FO_PX; ++px) {
            const int slot = px * FO_THREADS + tid;
            const int kf = sm.sort.kfree[slot];
            int start = 0;
#pragma unroll
            for (int bkt = 0; bkt <= N; ++bkt)
                if (bkt < N - kf) start += sm.bucket[bkt];
            sm.sort.order[start + rk[px]] = (unsigned short)slot;
        }
        __syncthreads();
        // thread tid walks the pixels of rank tid (large sets first) and FO_PIX-1-tid (small sets): balanced pairs
#pragma unroll 1
        for (int half = 0; half < FO_PX; ++half) {
            const int slot = sm.sort.order[half == 0 ? tid : FO_PIX - 1 - tid];
            const unsigned nst = 1u << sm.sort.kfree[slot];
            const unsigned long long xm = sm.sort.xm[slot];
            double s = 0.0, best = 0.0;
            unsigned key = 0, bkey = 0;
            for (unsigned st = 1; st < nst; ++st) {
                const int j = __ffs(st) - 1;
                s += sm.cs[j][slot];
                key ^= (unsigned)(xm >> (8 * j)) & 0xffu;
                const double e = s + sm.T[key];
                if (e < best) {
                    best = e;
                    bkey = key;
                }
            }
            sm.sort.wkey[slot] = (unsigned char)bkey;
            sm.cs[0][slot] = best;  // (the slot's c_j are dead: this thread was their only reader)
        }
        __syncthreads();
#pragma unroll
        for (int px = 0; px < FO_PX; ++px) {
            win[px] = sm.sort.wkey[px * FO_THREADS + tid];
            dE[px] = sm.cs[0][px * FO_THREADS + tid];
        }
    }

    // (compiler barrier: without it the M values the gradient phase loaded are kept for the epilogue -- in local memory)
    asm volatile("" ::: "memory");
    // ---- S7 (+ S8): N* = base + bits of the winner.  E(N*) = E(base) + dE: E(base) from the definition (Eq. (C1)) and dE
    // the increment the walk has minimised (Eq. (C1) expanded around the base point: dE = sum_{i in b} h_i + pairs(b)); the
    // rounding of both is a few ulp of E_C-sized terms, far inside the 1e-9 max(|E|, E_C) of the parity tests
    int32_t Ns[FO_PX][N];
#pragma unroll
    for (int px = 0; px < FO_PX; ++px)
#pragma unroll
        for (int i = 0; i < N; ++i) Ns[px][i] = sm.base[i][px * FO_THREADS + tid] + (int32_t)((win[px] >> (N - 1 - i)) & 1u);
#pragma unroll
    for (int px = 0; px < FO_PX; ++px) {
        if (live[px]) {
            outE[gp[px]] = Ebase[px] + dE[px];
            if (ns == 0) {
                if constexpr (N % 4 == 0) {
                    if ((reinterpret_cast<uintptr_t>(outN) & 15u) == 0) {
#pragma unroll
                        for (int i = 0; i < N; i += 4)
                            *reinterpret_cast<int4 *>(outN + gp[px] * N + i) =
                                make_int4(Ns[px][i], Ns[px][i + 1], Ns[px][i + 2], Ns[px][i + 3]);
                    } else {
#pragma unroll
                        for (int i = 0; i < N; ++i) outN[gp[px] * N + i] = Ns[px][i];
                    }
                } else {
#pragma unroll
                    for (int i = 0; i < N; ++i) outN[gp[px] * N + i] = Ns[px][i];
                }
            } else {  // S8: sensor dots in the full model (single-model calls only: gp = p)
                int32_t Nl[N];
#pragma unroll
                for (int i = 0; i < N; ++i) Nl[i] = Ns[px][i];
                fo_sensor(mdl, Vg, gp[px], Nl, outN, outVs);
            }
        }
    }
    // deferred pixels (see fo_slow_pixel): redone from scratch, overwriting what the register path stored
#pragma unroll
    for (int px = 0; px < FO_PX; ++px) {  // (unrolled: a dynamic px would put every per-pixel array in local memory)
        if (live[px] && slowf[px]) {
            int st3[3];
            fo_slow_pixel<N, THR>(sm.MT, sm.C, sm.T, mdl, Vg, gp[px], args, outN, outE, xcont, outVs, st3);
            rounds[px] = st3[0];
            failed[px] = st3[1] != 0;
            freem[px] = (1u << st3[2]) - 1u;  // only its population count is used below
        }
    }
    if (stats) {
        int64_t np = 0, nq = 0, nr = 0, nf = 0, ne = 0;
#pragma unroll
        for (int px = 0; px < FO_PX; ++px) {
            if (!live[px]) continue;
            ++np;
            nq += negf[px] ? 1 : 0;
            nr += rounds[px];
            nf += failed[px] ? 1 : 0;
            ne += (int64_t)1 << __popc(freem[px]);
        }
        qa_warp_count(&stats->n_pixels, np);
        qa_warp_count(&stats->n_qp_pixels, nq);
        qa_warp_count(&stats->n_qp_rounds, nr);
        qa_warp_count(&stats->n_qp_failed, nf);
        qa_warp_count(&stats->n_candidates_enumerated, ne);
        qa_warp_count(&stats->n_candidates_scored, ne);
    }
}

// ---------------------------------------------------------------------------------------------------------------------
// Several algorithms on the SAME sweep in one launch (qa_ground_state_batch_multi: a dataset run searches every diagram with
// the default algorithm and with one or more thresholds, PAPER.md L500 / BASELINE.json configs[4]).  V_g is read once, the
// model tables are staged once, N_c (S1) and the continuous minimum x (S2-S3, the QP) are computed once per pixel; S4-S7 then
// run once per algorithm on the same x, with exactly the arithmetic of qa_fused_open_kernel (same order: the results are
// bit-identical to separate calls, tests).  One pixel per thread; THR is a run-time, CTA-uniform switch per pass.
template <int N, bool MP>
__global__ void __launch_bounds__(FO_THREADS, FO_MULTI_CTAS) qa_fused_open_multi_kernel(const QaDevModel *const *__restrict__ models,
                                                                            const double *__restrict__ Vg, int64_t P, int g,
                                                                            int general_qp, QaMultiArgs ma,
                                                                            double *__restrict__ xcont, qa_stats *stats)
{
    constexpr int PIX = FO_THREADS;
    // 27 KB at N = 8: eight CTAs per SM.  N_c and x of every pixel slot wait here for every pass; the base point is not
    // parked (the epilogue recomputes floor(x) and keeps one bit per dot for "rounded up")
    struct Smem {
        double MT[N * N], C[N * N], T[1 << N];  // contiguous: fo_stage
        double nc[N][PIX];
        double x[N][PIX];
        union alignas(16) {
            double CgT[QA_MAXG * N];  // dead after S1
            double cs[N][PIX];        // thresholded passes: c_j of the compacted free dots of the thread's own pixel
        };
    };
    __shared__ __align__(16) Smem sm;
    double(*sx)[PIX] = sm.x;
    const int tid = threadIdx.x;
    const int64_t p = (int64_t)blockIdx.x * PIX + tid;
    const bool live = p < P;
    const int64_t gp = (int64_t)blockIdx.y * P + (live ? p : P - 1);
    const double *vp = Vg + gp * g;
    const bool vec = (g & 1) == 0 && (reinterpret_cast<uintptr_t>(Vg) & 15u) == 0;
    auto load_chunk = [&](int k0, double (&a)[8]) {
        if (vec) {
#pragma unroll
            for (int k = 0; k < 8; k += 2) {
                double2 ta = make_double2(0.0, 0.0);
                if (k0 + k < g) ta = __ldg(reinterpret_cast<const double2 *>(vp + k0 + k));
                a[k] = ta.x, a[k + 1] = ta.y;
            }
        } else {
#pragma unroll
            for (int k = 0; k < 8; ++k) a[k] = k0 + k < g ? __ldg(vp + k0 + k) : 0.0;
        }
    };
    double va[8];
    load_chunk(0, va);
    const QaDevModel *__restrict__ mdl = models[blockIdx.y];
    fo_stage<N>(mdl, g, tid, sm.MT, sm.CgT);
    const double EC = MP ? mdl->EC : 0.0;
    __syncthreads();

    // ---- S1-S3, once per pixel
    double x[N];
    {
        double nc[N];
#pragma unroll
        for (int i = 0; i < N; ++i) nc[i] = 0.0;
        for (int k0 = 0; k0 < g; k0 += 8) {
            if (k0 > 0) load_chunk(k0, va);
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                if (k0 + k < g) {
#pragma unroll
                    for (int i = 0; i < N; ++i) nc[i] = fma(sm.CgT[(k0 + k) * N + i], va[k], nc[i]);
                }
            }
        }
#pragma unroll
        for (int i = 0; i < N; ++i) {
            x[i] = nc[i];
            sm.nc[i][tid] = nc[i];
        }
    }
    bool neg = false;
#pragma unroll
    for (int i = 0; i < N; ++i) neg |= x[i] < 0.0;
    int rounds0 = 0;
    bool failed0 = false, slowf = false;
    if (neg) {
        double nc[N];
#pragma unroll
        for (int i = 0; i < N; ++i) nc[i] = x[i];
        rounds0 = fo_qp_open<N>(sm.C, nc, general_qp, x, failed0, slowf);
    }
    if (xcont && live && !slowf) {
#pragma unroll
        for (int i = 0; i < N; ++i) xcont[gp * N + i] = x[i];
    }
#pragma unroll
    for (int i = 0; i < N; ++i) sx[i][tid] = x[i];
    __syncthreads();  // every warp is done with C_gd: its storage becomes the c_j columns of the thresholded passes

#pragma unroll 1
    for (int a = 0; a < ma.n_alg; ++a) {
        const bool thr = ma.thr[a] != 0;
        const double tt = ma.t[a];
        int32_t *__restrict__ outN = ma.N[a];
        double *__restrict__ outE = ma.E[a];
        // ---- S4 (Eq. (9), readings R4 / R10) and the base-point gradient
        double hp[N], Ebase, dE;  // E(N*) = E(base) + dE, as in qa_fused_open_kernel
        unsigned fm = 0, up = 0;
        {
            double d0[N], grad[N];
#pragma unroll
            for (int i = 0; i < N; ++i) {
                int32_t cn, bs;
                const double xi = sx[i][tid];
                qa_floor_ceil(xi, tt, thr, bs, cn);
                if (cn == 2) fm |= 1u << (N - 1 - i);
                const double fl = floor(xi);
                const int32_t lo = fl > 0.0 ? (int32_t)fl : 0;
                up |= (unsigned)(bs - lo) << (N - 1 - i);  // 1: the base point is lo + 1 (thresholded, fraction >= 1/2)
                d0[i] = (double)bs - sm.nc[i][tid];
                grad[i] = 0.0;
            }
#pragma unroll
            for (int j = 0; j < N; ++j) {
#pragma unroll
                for (int i = 0; i < N; ++i) grad[i] = fma(sm.MT[j * N + i], d0[j], grad[i]);
            }
#pragma unroll
            for (int b = 0; b < N; ++b) hp[b] = grad[N - 1 - b] + 0.5 * sm.MT[(N - 1 - b) * N + (N - 1 - b)];
            double eb = 0.0;
#pragma unroll
            for (int i = 0; i < N; ++i) eb = fma(d0[i], grad[i], eb);
            Ebase = 0.5 * eb;
        }
        unsigned win = 0;
        asm volatile("" ::: "memory");
        if (!thr) {
            if constexpr (MP) {
                // min-plus split inside the thread (see qa_fused_open_kernel): pass 1 lower bounds per row of 16, pass 2 exact
                constexpr int NW = 4, NU = N - NW, R = 1 << NU, GS = R < 4 ? R : 4, NG = R / GS;
                double B[1 << NW], hu[NU];
                double offw = EC, offu = EC;
#pragma unroll
                for (int j = 0; j < NW; ++j) offw += fabs(hp[j]);
#pragma unroll
                for (int j = 0; j < NU; ++j) {
                    hu[j] = hp[NW + j];
                    offu += fabs(hu[j]);
                }
                B[0] = offw;
#pragma unroll
                for (int w = 1; w < (1 << NW); ++w) B[w] = B[w & (w - 1)] + hp[fo_ctz(w)];
                const double lo3 = NU >= 2 ? hu[NU >= 2 ? 1 : 0] + hu[0] : 0.0;
                auto row_a = [&](int i, int ul) -> double {
                    double ah = offu;
#pragma unroll
                    for (int j = NU - 1; j >= 2; --j)
                        if ((i >> (j - 2)) & 1) ah += hu[j];
                    if (NU >= 2) return ul == 0 ? ah : (ul == 1 ? ah + hu[0] : (ul == 2 ? ah + hu[NU >= 2 ? 1 : 0] : ah + lo3));
                    return ul == 0 ? ah : ah + hu[0];
                };
                unsigned Lg[NG], rowmask = 0;
#pragma unroll
                for (int k = 0; k < NG; ++k) Lg[k] = 0xffffffffu;
#pragma unroll 1
                for (int i = 0; i < NG; ++i) {
                    const double2 *__restrict__ T2 = reinterpret_cast<const double2 *>(sm.T + ((i * GS) << NW));
                    unsigned l[GS];
#pragma unroll
                    for (int ul = 0; ul < GS; ++ul) {
                        unsigned m0 = 0xffffffffu, m1 = 0xffffffffu;
#pragma unroll
                        for (int w = 0; w < (1 << NW); w += 4) {
                            const double2 ta = T2[((ul << NW) | w) >> 1], tb = T2[((ul << NW) | (w + 2)) >> 1];
                            const double y0 = B[w] + ta.x, y1 = B[w + 1] + ta.y, y2 = B[w + 2] + tb.x, y3 = B[w + 3] + tb.y;
                            m0 = min(m0, min((unsigned)__double2hiint(y0), (unsigned)__double2hiint(y1)));
                            m1 = min(m1, min((unsigned)__double2hiint(y2), (unsigned)__double2hiint(y3)));
                        }
                        const double lb = row_a(i, ul) + __hiloint2double((int)min(m0, m1), 0);
                        l[ul] = (unsigned)__double2hiint(lb);
                    }
                    unsigned gmin = l[0];
#pragma unroll
                    for (int ul = 1; ul < GS; ++ul) gmin = min(gmin, l[ul]);
                    unsigned nib = 0;
#pragma unroll
                    for (int ul = 0; ul < GS; ++ul) nib |= (l[ul] <= gmin + 2u ? 1u : 0u) << ul;
                    rowmask |= nib << (i * GS);
#pragma unroll
                    for (int k = 0; k < NG; ++k)
                        if (k == i) Lg[k] = gmin;
                }
                unsigned Lmin = Lg[0];
#pragma unroll
                for (int k = 1; k < NG; ++k) Lmin = min(Lmin, Lg[k]);
                unsigned cand = 0;
#pragma unroll
                for (int k = 0; k < NG; ++k)
                    if (Lg[k] <= Lmin + 2u) cand |= rowmask & (((1u << GS) - 1u) << (k * GS));
                double best = __longlong_as_double(0x7ff0000000000000ll);
                unsigned bkey = 0;
                while (cand) {
                    const int u = __ffs(cand) - 1;
                    cand &= cand - 1u;
                    const double av = row_a(u / GS, u % GS);
                    const double *__restrict__ T = sm.T + (u << NW);
#pragma unroll
                    for (int w = 0; w < (1 << NW); ++w) {
                        const double e = av + (B[w] + T[w]);
                        if (e < best) {
                            best = e;
                            bkey = ((unsigned)u << NW) | (unsigned)w;
                        }
                    }
                }
                win = bkey;
                dE = best - (offw + offu);
            } else {
                // counting-order walk over all 2^N patterns (qa_fused_open_kernel, plain form)
                constexpr int LB = N < 4 ? N : 4;
                constexpr int NHI = N - LB;
                double cl[LB], ch[NHI > 0 ? NHI : 1];
                {
                    double pre = 0.0;
#pragma unroll
                    for (int j = 0; j < N; ++j) {
                        if (j < LB)
                            cl[j] = hp[j] - pre;
                        else
                            ch[j - LB] = hp[j] - pre;
                        pre += hp[j];
                    }
                }
                double sl = 0.0, m = 0.0;
#pragma unroll 1
                for (int i = 0; i < (1 << NHI); ++i) {
                    const double *__restrict__ T = sm.T + (i << LB);
                    const unsigned kb = (unsigned)i << LB;
                    if (i > 0) {
                        double c = ch[NHI > 0 ? NHI - 1 : 0];
#pragma unroll
                        for (int j = NHI - 2; j >= 0; --j)
                            if ((i >> j) & 1) c = ch[j];
                        sl += c;
                        const double e = sl + T[0];
                        if (e < m) {
                            m = e;
                            win = kb;
                        }
                    }
#pragma unroll
                    for (int w = 1; w < (1 << LB); ++w) {
                        sl += cl[fo_ctz(w)];
                        const double e = sl + T[w];
                        if (e < m) {
                            m = e;
                            win = kb + w;
                        }
                    }
                }
                dE = m;
            }
        } else {
            // thresholded (the launcher admits t <= QA_FO_NOSORT_T only): every thread walks its own pixel, no sort, no barrier
            double pre = 0.0;
            int jj = 0;
            unsigned low = 0;
            unsigned long long xm = 0;
#pragma unroll
            for (int b = 0; b < N; ++b) {
                if ((fm >> b) & 1u) {
                    sm.cs[jj][tid] = hp[b] - pre;
                    pre += hp[b];
                    xm |= (unsigned long long)((1u << b) | low) << (8 * jj);
                    low |= 1u << b;
                    ++jj;
                }
            }
            const unsigned nst = live ? 1u << jj : 1u;
            double sl = 0.0, best = 0.0;
            unsigned key = 0, bkey = 0;
            for (unsigned st = 1; st < nst; ++st) {
                const int j = __ffs(st) - 1;
                sl += sm.cs[j][tid];
                key ^= (unsigned)(xm >> (8 * j)) & 0xffu;
                const double e = sl + sm.T[key];
                if (e < best) {
                    best = e;
                    bkey = key;
                }
            }
            win = bkey;
            dE = best;
        }
        // (compiler barriers: without them the M values the gradient phase loaded are kept for the epilogue, in local memory)
        asm volatile("" ::: "memory");
        // ---- S7: N* = base + bits of the winner; E(N*) = E(base) + dE
        {
            int32_t Ns[N];
#pragma unroll
            for (int i = 0; i < N; ++i) {
                const double fl = floor(sx[i][tid]);
                const int32_t lo = fl > 0.0 ? (int32_t)fl : 0;
                Ns[i] = lo + (int32_t)((up >> (N - 1 - i)) & 1u) + (int32_t)((win >> (N - 1 - i)) & 1u);
            }
            if (live) {
                outE[gp] = Ebase + dE;
                if (N % 4 == 0 && (reinterpret_cast<uintptr_t>(outN) & 15u) == 0) {
#pragma unroll
                    for (int i = 0; i + 3 < N; i += 4)
                        *reinterpret_cast<int4 *>(outN + gp * N + i) = make_int4(Ns[i], Ns[i + 1], Ns[i + 2], Ns[i + 3]);
                } else {
#pragma unroll
                    for (int i = 0; i < N; ++i) outN[gp * N + i] = Ns[i];
                }
            }
        }
        asm volatile("" ::: "memory");
        int rounds = rounds0, kfree = __popc(fm);
        bool failed = failed0;
        if (live && slowf) {  // deferred pixel (see fo_slow_pixel): redone from scratch with this pass's algorithm
            int st3[3];
            QaCallArgs sa{0, 0, thr ? (int)QA_ALG_THRESHOLDED : (int)QA_ALG_DEFAULT, tt, 0, general_qp, 0};
            if (thr)
                fo_slow_pixel<N, true>(sm.MT, sm.C, sm.T, mdl, Vg, gp, sa, outN, outE, xcont, nullptr, st3);
            else
                fo_slow_pixel<N, false>(sm.MT, sm.C, sm.T, mdl, Vg, gp, sa, outN, outE, xcont, nullptr, st3);
            rounds = st3[0];
            failed = st3[1] != 0;
            kfree = st3[2];
        }
        if (stats) {
            qa_warp_count(&stats->n_pixels, live ? 1 : 0);
            qa_warp_count(&stats->n_qp_pixels, (live && neg) ? 1 : 0);
            qa_warp_count(&stats->n_qp_rounds, live ? rounds : 0);
            qa_warp_count(&stats->n_qp_failed, (live && failed) ? 1 : 0);
            const int64_t ne = live ? (int64_t)1 << kfree : 0;
            qa_warp_count(&stats->n_candidates_enumerated, ne);
            qa_warp_count(&stats->n_candidates_scored, ne);
        }
    }
}

template <int N>
cudaError_t launch_fused_open_n(const QaDevModel *const *d_models, int n_models, const double *d_Vg, int64_t P, int g,
                                QaCallArgs args, int32_t *d_N, double *d_E, double *d_xcont, double *d_Vs,
                                qa_stats *d_stats, cudaStream_t stream)
{
    const dim3 grid((unsigned)((P + FO_THREADS * FO_PX_RUN - 1) / (FO_THREADS * FO_PX_RUN)), (unsigned)n_models);
    if (args.alg == QA_ALG_DEFAULT) {
        // Maxwell models (every model of the call) with at least five dots: the min-plus form of the walk
        if (N >= 5 && args.general_qp == 0)
            qa_fused_open_kernel<N, false, FO_PX_RUN, (N >= 5)><<<grid, FO_THREADS, 0, stream>>>(d_models, d_Vg, P, g, args, d_N, d_E,
                                                                                              d_xcont, d_Vs, d_stats);
        else
            qa_fused_open_kernel<N, false, FO_PX_RUN, false><<<grid, FO_THREADS, 0, stream>>>(d_models, d_Vg, P, g, args, d_N, d_E,
                                                                                           d_xcont, d_Vs, d_stats);
    } else
        qa_fused_open_kernel<N, true, FO_PX_RUN, false><<<grid, FO_THREADS, 0, stream>>>(d_models, d_Vg, P, g, args, d_N, d_E,
                                                                                      d_xcont, d_Vs, d_stats);
    return cudaGetLastError();
}

}  // namespace

// Open arrays, default or thresholded algorithm, n <= QA_FUSED_MAXN.  Arguments as qa_launch_fused_small.
cudaError_t qa_launch_fused_open(const QaDevModel *const *d_models, int n_models, int n, int g, const double *d_Vg,
                                 int64_t P, QaCallArgs args, int32_t *d_N, double *d_E, double *d_xcont, double *d_Vs,
                                 qa_stats *d_stats, cudaStream_t stream)
{
    qa_plan_add("qa_fused_open_kernel");
    if (n_models > 65535 || args.closed || args.alg == QA_ALG_BRUTE_FORCE) return cudaErrorInvalidValue;
#define CALL(NN) launch_fused_open_n<NN>(d_models, n_models, d_Vg, P, g, args, d_N, d_E, d_xcont, d_Vs, d_stats, stream)
    switch (n) {
        case 1: return CALL(1);
        case 2: return CALL(2);
        case 3: return CALL(3);
        case 4: return CALL(4);
        case 5: return CALL(5);
        case 6: return CALL(6);
        case 7: return CALL(7);
        case 8: return CALL(8);
        default: return cudaErrorInvalidValue;
    }
#undef CALL
}

// Open arrays, n <= QA_FUSED_MAXN, no sensor dots: ma.n_alg passes (default / thresholded) over one sweep in one launch.
cudaError_t qa_launch_fused_open_multi(const QaDevModel *const *d_models, int n_models, int n, int g, const double *d_Vg,
                                       int64_t P, int general_qp, const QaMultiArgs &ma, double *d_xcont, qa_stats *d_stats,
                                       cudaStream_t stream)
{
    qa_plan_add("qa_fused_open_multi_kernel");
    if (n_models > 65535 || ma.n_alg < 1 || ma.n_alg > QA_MULTI_MAX) return cudaErrorInvalidValue;
    const dim3 grid((unsigned)((P + FO_THREADS - 1) / FO_THREADS), (unsigned)n_models);
#define CALL(NN)                                                                                                         \
    do {                                                                                                                 \
        if (NN >= 5 && general_qp == 0)                                                                                  \
            qa_fused_open_multi_kernel<NN, (NN >= 5)><<<grid, FO_THREADS, 0, stream>>>(d_models, d_Vg, P, g, general_qp, ma, \
                                                                                    d_xcont, d_stats);                  \
        else                                                                                                             \
            qa_fused_open_multi_kernel<NN, false><<<grid, FO_THREADS, 0, stream>>>(d_models, d_Vg, P, g, general_qp, ma,  \
                                                                                d_xcont, d_stats);                      \
    } while (0)
    switch (n) {
        case 1: CALL(1); break;
        case 2: CALL(2); break;
        case 3: CALL(3); break;
        case 4: CALL(4); break;
        case 5: CALL(5); break;
        case 6: CALL(6); break;
        case 7: CALL(7); break;
        case 8: CALL(8); break;
        default: return cudaErrorInvalidValue;
    }
#undef CALL
    return cudaGetLastError();
}
