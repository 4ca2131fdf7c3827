// qa_kernels_minplus32.cu -- MIXED-PRECISION pass 1 of the min-plus walk ("fp32 walk, fp64
// re-score"): open array, default algorithm, 13 <= n <= 16, Maxwell c_dd; selected with qa_model_set_walk_variant(m, 3).
//
// Pass 1 of qa_kernels_minplus.cu only has to produce, per thread (= high pattern t of a pixel), a LOWER BOUND L_t of the
// thread's smallest energy that is tight enough for pass 2 to re-score very few threads exactly.  Here that estimate is
// formed in fp32 with an explicit error bound:
//     h'_j, offW, offU + be -> fp32;  B32[w], A32[u] by fp32 subset sums;  y = B32[w] + q32[u,w] (two per packed add,
//     add.rn.f32x2);  m_u = min_w y  (positive floats order like their bit patterns: integer min3);
//     LB_u = A32[u] + m_u;  L_t = min_u bits(LB_u).
// Every partial sum is positive and at most the energy it belongs to, and a candidate goes through at most 21 roundings
// of at most one ulp32 each (conversions round down, additions to nearest), so  |e_t - L_t| <= 21 ulp32(e_t)  for the
// thread's smallest energy e_t.  With t* the thread of the argmin e* and t' the thread of the smallest L:
//     L_t* <= e* + 21 ulp <= e_t' + 21 ulp <= L_t' + 42 ulp,
// so the argmin (and every tie of it) lies in a thread with bits(L_t) <= min bits(L) + 42.  The kernel keeps the lanes
// within MP32_SLACK = 48 of the warp minimum in the same 8-byte record as the fp64 pass 1, and qa_minplus_finish_kernel
// re-scores those threads with the fp64 arithmetic of pass 1 and the exact lexicographic compare.  The charge map and the
// energies are therefore BIT-IDENTICAL to the fp64 walk's (tests: variants 1 and 3 agree exactly); what changes is the
// pipe that does the 2^n additions: FP32 (two table entries per packed add, four pixels per thread) instead of FP64.
#include "qa_internal.cuh"

constexpr unsigned MP32_SLACK = 48u;

namespace {

constexpr int M32_THREADS = 256;

struct alignas(16) Mp32Table {
    float q[256];  // pair energies of the low 8 bits, rounded down
};

__device__ __forceinline__ float f32_down(double x)
{
    float r;
    asm("cvt.rm.f32.f64 %0, %1;" : "=f"(r) : "d"(x));
    return r;
}
__device__ __forceinline__ float addf(float a, float b) { return __fadd_rn(a, b); }

// two fp32 additions in one instruction (sm_100 packed add): {a.x + b.x, a.y + b.y}, round to nearest
__device__ __forceinline__ unsigned long long add2(unsigned long long a, unsigned long long b)
{
    unsigned long long r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ unsigned long long pack2(float lo, float hi)
{
    return (unsigned long long)__float_as_uint(lo) | ((unsigned long long)__float_as_uint(hi) << 32);
}

__host__ __device__ constexpr int m32_ctz(int k)
{
    int j = 0;
    while (((k >> j) & 1) == 0) ++j;
    return j;
}

__device__ __forceinline__ double m32_shfl(double x, int src) { return __shfl_sync(0xffffffffu, x, src); }

template <int NH, int PX, int MINB>
__global__ void __launch_bounds__(M32_THREADS, MINB) qa_minplus_walk32_kernel(const QaDevModel *__restrict__ mdl,
                                                                             const __grid_constant__ Mp32Table tab,
                                                                             QaWorkspace ws)
{
    constexpr int NU = 4, NW = 4, NL = 8;
    constexpr int N = NL + NH;
    constexpr int TPP = 1 << NH;
    constexpr int WPP = TPP / 32;
    constexpr int SLOTS = M32_THREADS / TPP;
    constexpr int NV = N + 1;
    static_assert(NH >= 5 && NH <= 8 && QA_WALK_NL == NL, "one or more whole warps per pixel");

    const unsigned lane = threadIdx.x & 31u;
    const unsigned t = threadIdx.x & (TPP - 1);
    const int slot = threadIdx.x >> NH;
    const unsigned wq = (threadIdx.x >> 5) % WPP;
    const int64_t P = ws.P;

    double v[NL];
#pragma unroll
    for (int j = 0; j < NL; ++j) v[j] = mdl->VT[t * NL + j];
    const double EC = mdl->EC;
    const double QH = mdl->QHT[t];

    const int64_t groups = (P + PX - 1) / PX;
    const int64_t workers = (int64_t)gridDim.x * SLOTS;
    const int64_t worker = (int64_t)slot * gridDim.x + blockIdx.x;
    auto fetch = [&](int64_t grp, int px) -> double {
        double r = 0.0;
        if (grp < groups && lane < NV) {
            int64_t p = grp * PX + px;
            if (p >= P) p = P - 1;
            r = lane < N ? __ldg(ws.h + (int64_t)lane * P + p) : __ldg(ws.e0 + p);
        }
        return r;
    };
    qa_pdl_launch_dependents();
    qa_pdl_wait();
    double nextv[PX];
#pragma unroll
    for (int px = 0; px < PX; ++px) nextv[px] = fetch(worker, px);

    for (int64_t grp = worker; grp < groups; grp += workers) {
        float B[PX][16], hu[PX][NU], a0[PX];
        unsigned long long B2[PX][8];  // (B[2k], B[2k+1]) packed
#pragma unroll
        for (int px = 0; px < PX; ++px) {
            const double myv = nextv[px];
            nextv[px] = fetch(grp + workers, px);
            // fp64 exactly as pass 1 forms them (the offsets are thread-independent), then converted to fp32
            float hw[NW];
            double offw = EC, offu = 0.0;
#pragma unroll
            for (int j = 0; j < NL; ++j) {
                const double hj = m32_shfl(myv, N - 1 - j);
                if (j < NW) {
                    hw[j] = f32_down(hj + v[j]);
                    offw += fabs(hj);
                } else {
                    hu[px][j - NW] = f32_down(hj + v[j]);
                    offu += fabs(hj);
                }
            }
            double be = m32_shfl(myv, N) + QH;
#pragma unroll
            for (int jh = 0; jh < NH; ++jh) {
                const double hv = m32_shfl(myv, N - 1 - NL - jh);
                if ((t >> jh) & 1u) be += hv;
            }
            a0[px] = f32_down(be + offu);
            B[px][0] = f32_down(offw);
#pragma unroll
            for (int w = 1; w < 16; ++w) B[px][w] = addf(B[px][w & (w - 1)], hw[m32_ctz(w)]);
#pragma unroll
            for (int k = 0; k < 8; ++k) B2[px][k] = pack2(B[px][2 * k], B[px][2 * k + 1]);
        }

        unsigned L[PX];
#pragma unroll
        for (int px = 0; px < PX; ++px) L[px] = 0xffffffffu;
        // a real loop over the 16 rows u: the table address stays "uniform register + immediate"; iv mirrors the counter in
        // a vector register (see qa_kernels_minplus.cu)
        int iv;
        asm volatile("mov.u32 %0, 0;" : "=r"(iv));
#pragma unroll 1
        for (int u = 0; u < 16; ++u, ++iv) {
            const unsigned long long *q = reinterpret_cast<const unsigned long long *>(tab.q) + (u << 3);
            unsigned m[PX];
#pragma unroll
            for (int px = 0; px < PX; ++px) m[px] = 0xffffffffu;
#pragma unroll
            for (int w = 0; w < 16; w += 2) {
                const unsigned long long t2 = q[w >> 1];
#pragma unroll
                for (int px = 0; px < PX; ++px) {
                    const unsigned long long y = add2(B2[px][w >> 1], t2);
                    m[px] = min(m[px], min((unsigned)y, (unsigned)(y >> 32)));
                }
            }
#pragma unroll
            for (int px = 0; px < PX; ++px) {
                float a = a0[px];
#pragma unroll
                for (int j = NU - 1; j >= 0; --j)
                    if ((iv >> j) & 1) a = addf(a, hu[px][j]);
                const float lb = addf(a, __uint_as_float(m[px]));
                L[px] = min(L[px], __float_as_uint(lb));
            }
        }

#pragma unroll
        for (int px = 0; px < PX; ++px) {
            const unsigned wmin = __reduce_min_sync(0xffffffffu, L[px]);
            const unsigned ball = __ballot_sync(0xffffffffu, L[px] <= wmin + MP32_SLACK);
            const int64_t p = grp * PX + px;
            if (lane == 0 && p < P) ws.rec[p * WPP + wq] = make_uint2(wmin, ball);
        }
    }
}

template <int NH, int PX, int MINB>
cudaError_t launch_mp32(const QaDevModel *d_model, const double *QLhost, QaWorkspace ws, int sm_count, cudaStream_t stream)
{
    constexpr int SLOTS = M32_THREADS >> NH;
    Mp32Table local;
    for (int b = 0; b < 256; ++b) {  // round down: the largest float <= QL[b] (QL >= 0)
        float f = (float)QLhost[b];
        if ((double)f > QLhost[b]) f = nextafterf(f, -1.0f);
        local.q[b] = f;
    }
    int per_sm = 0;
    cudaError_t err =
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, qa_minplus_walk32_kernel<NH, PX, MINB>, M32_THREADS, 0);
    if (err != cudaSuccess) return err;
    if (per_sm < 1) per_sm = 1;
    int64_t grid = (int64_t)sm_count * per_sm;
    const int64_t need = ((ws.P + PX - 1) / PX + SLOTS - 1) / SLOTS;
    if (grid > need) grid = need;
    return qa_launch_pdl(qa_minplus_walk32_kernel<NH, PX, MINB>, dim3((unsigned)grid), dim3(M32_THREADS), stream, d_model, local,
                         ws);
}

}  // namespace

// fp32 lower-bound pass 1 + the fp64 finish kernel (pass 2 + S7); d_N == nullptr: the finish kernel only stores ws.best
cudaError_t qa_launch_minplus_walk32(const QaDevModel *d_model, int n, const double *QLhost, QaWorkspace ws, int32_t *d_N,
                                     double *d_E, int sm_count, cudaStream_t stream)
{
    qa_plan_add("qa_minplus_walk32_kernel");
    cudaError_t err;
    switch (n) {
        case 13: err = launch_mp32<5, 4, 2>(d_model, QLhost, ws, sm_count, stream); break;
        case 14: err = launch_mp32<6, 4, 2>(d_model, QLhost, ws, sm_count, stream); break;
        case 15: err = launch_mp32<7, 4, 2>(d_model, QLhost, ws, sm_count, stream); break;
        case 16: err = launch_mp32<8, 4, 2>(d_model, QLhost, ws, sm_count, stream); break;
        default: return cudaErrorInvalidValue;
    }
    if (err != cudaSuccess) return err;
    return qa_launch_minplus_finish(d_model, n, ws, d_N, d_E, MP32_SLACK, sm_count, stream);
}
