// qa_kernels_thermal_sp.cu -- thermal broadening (Eq. (10)) of the open default set of 9..16 dots as a SUM-PRODUCT over
// the same split of the candidate lattice the min-plus walk uses (qa_kernels_minplus.cu): bits w = [0,4), u = [4,8),
// t = [8,n), one thread per high pattern t of a pixel.  From (C1) L607
//     E(t,u,w) = A[u] + B[w] + QL[u,w],   A[u] = be_t + sum_{j in u} h'_j,   B[w] = sum_{j in w} h'_j,
// so the Boltzmann weight factorises,  exp(-beta (E - ref_t)) = a[u] b[w] q[u,w]  with  q = exp(-beta QL)  a pixel- and
// thread-independent table (kernel parameter) and a, b products of per-bit factors normalised to max 1:
//     bit j off: exp(-beta max(0, -h'_j)),  on: exp(-beta max(0, h'_j))      (one exp per low bit and thread),
//     ref_t = be_t + sum_j min(0, h'_j)  <=  every E(t, ., .).
// Then  R[u] = sum_w b[w] q[u,w]  and  C[w] = sum_u a[u] q[u,w]  cost ONE DFMA per candidate each, and
//     Z_t = sum_u a[u] R[u];   (u-bit j) sum_{u has j} a[u] R[u];   (w-bit j) sum_{w has j} b[w] C[w];   (t-bit) Z_t itself.
// Threads are combined relative to a reference every thread can form alone: ref_pix = E(base) + E_C + sum_i min(0, h_i)
// <= ref_t (h' >= h and the pair energies are >= 0 for a Maxwell c_dd), scale_t = exp(-beta (ref_t - ref_pix)) <= 1.  The true
// minimum lies at most G = sum_{i<j} M_ij above ref_pix, so Z >= exp(-beta G): the launcher uses this kernel only while
// beta G <= 600 (far from underflow; a factor that does underflow belongs to weights < e^-100 of the dominant one) and
// for Maxwell models; everything else runs the two-pass Gray kernel of qa_kernels_thermal.cu.
// E_min (optional output): a lower bound per thread exactly as pass 1 of the min-plus walk forms it (1 DADD + 1/2 integer
// min3 per candidate), then the threads within 2 units of the pixel's smallest bound (normally one) are re-scored exactly
// by all threads of the pixel together.
// FP64-pipe instructions per candidate: 2 DFMA (+ 1 DADD for E_min); per thread 8 exp + ~150 for the factors and marginals.
// Deterministic: fixed shuffle / shared-memory reduction order.
#include "qa_internal.cuh"

namespace {

constexpr int SP_THREADS = 256;

struct SpTable {
    double q[256];   // exp(-beta QL[u,w])
    double QL[256];  // pair energies of the low 8 bits (E_min pass)
};

__host__ __device__ constexpr int sp_ctz(int k)
{
    int j = 0;
    while (((k >> j) & 1) == 0) ++j;
    return j;
}

template <int NH, bool EMIN>
__global__ void __launch_bounds__(SP_THREADS, 2) qa_thermal_sp_kernel(const QaDevModel *__restrict__ mdl,
                                                                     const __grid_constant__ SpTable tab, QaWorkspace ws,
                                                                     double beta, double *__restrict__ outNmean,
                                                                     double *__restrict__ outEmin)
{
    constexpr int NL = QA_WALK_NL;
    constexpr int N = NL + NH;
    constexpr int TPP = 1 << NH;              // threads per pixel
    constexpr int PPB = SP_THREADS / TPP;     // pixels per CTA iteration
    constexpr int W = TPP < 32 ? TPP : 32;    // lanes of a shuffle group
    constexpr int GPP = TPP / W;              // groups per pixel
    constexpr int NG = SP_THREADS / W;        // groups per CTA
    constexpr int NHW = NH < 5 ? NH : 5;      // t-bits that live inside a group
    constexpr int NR = 9 + NHW;               // values reduced inside a group: Z, 8 low-bit marginals, NHW t-bit marginals
    static_assert(NL == 8 && NH >= 1 && NH <= 8, "low bits = two groups of four");
    __shared__ double sIn[PPB][N + 1];
    __shared__ double sRed[NG][NR];
    __shared__ double sMin[NG];
    __shared__ unsigned sLmin[NG];
    __shared__ int sCnt[PPB];
    __shared__ double sSurv[EMIN ? SP_THREADS : 1][NL + 1];  // survivors of the E_min bound: h'_0..7, be

    const unsigned t = threadIdx.x & (TPP - 1);
    const int slot = threadIdx.x >> NH;
    const int grp_id = threadIdx.x / W;
    const int64_t P = ws.P;
    double v[NL];
#pragma unroll
    for (int j = 0; j < NL; ++j) v[j] = mdl->VT[t * NL + j];
    const double QH = mdl->QHT[t];
    const double EC = mdl->EC;
    qa_pdl_launch_dependents();
    qa_pdl_wait();

    const int64_t groups = (P + PPB - 1) / PPB;
    for (int64_t grp = blockIdx.x; grp < groups; grp += gridDim.x) {
        const int64_t p0 = grp * PPB;
        __syncthreads();  // the previous iteration's sIn / sRed have been read
        for (int e = threadIdx.x; e < PPB * (N + 1); e += SP_THREADS) {
            const int s = e / (N + 1), i = e % (N + 1);
            int64_t p = p0 + s;
            if (p >= P) p = P - 1;
            sIn[s][i] = i < N ? __ldg(ws.h + (int64_t)i * P + p) : __ldg(ws.e0 + p);
        }
        __syncthreads();

        // per-thread inputs, as the min-plus walk forms them
        double hp[NL];
        double refpix = sIn[slot][N] + EC;
#pragma unroll
        for (int i = 0; i < N; ++i) refpix += fmin(0.0, sIn[slot][i]);
#pragma unroll
        for (int j = 0; j < NL; ++j) hp[j] = sIn[slot][N - 1 - j] + v[j];
        double be = sIn[slot][N] + QH;
#pragma unroll
        for (int jh = 0; jh < NH; ++jh)
            if ((t >> jh) & 1u) be += sIn[slot][N - 1 - NL - jh];
        double ref = be;
#pragma unroll
        for (int j = 0; j < NL; ++j) ref += fmin(0.0, hp[j]);

        // ---- weights: per-bit factors normalised to max 1
        double on[NL], off[NL];
#pragma unroll
        for (int j = 0; j < NL; ++j) {
            const double x = exp(-beta * fabs(hp[j]));
            on[j] = hp[j] >= 0.0 ? x : 1.0;
            off[j] = hp[j] >= 0.0 ? 1.0 : x;
        }
        double b[16], a[16];
#pragma unroll
        for (int w = 0; w < 16; ++w) {
            b[w] = ((w & 1) ? on[0] : off[0]) * ((w & 2) ? on[1] : off[1]);
            b[w] *= ((w & 4) ? on[2] : off[2]) * ((w & 8) ? on[3] : off[3]);
            a[w] = ((w & 1) ? on[4] : off[4]) * ((w & 2) ? on[5] : off[5]);
            a[w] *= ((w & 4) ? on[6] : off[6]) * ((w & 8) ? on[7] : off[7]);
        }
        // phase 1, rows: R[u] = sum_w b[w] q[u,w] -> Z_t and the marginals of the u bits
        double zt = 0.0, su[4] = {0.0, 0.0, 0.0, 0.0}, sw[4] = {0.0, 0.0, 0.0, 0.0};
#pragma unroll
        for (int u = 0; u < 16; ++u) {
            double r0 = 0.0, r1 = 0.0;
#pragma unroll
            for (int w = 0; w < 16; w += 2) {
                r0 = fma(b[w], tab.q[(u << 4) | w], r0);
                r1 = fma(b[w + 1], tab.q[(u << 4) | (w + 1)], r1);
            }
            const double ar = a[u] * (r0 + r1);
            zt += ar;
#pragma unroll
            for (int j = 0; j < 4; ++j)
                if ((u >> j) & 1) su[j] += ar;
        }
        // phase 2, columns: C[w] = sum_u a[u] q[u,w] -> the marginals of the w bits
#pragma unroll
        for (int w = 0; w < 16; ++w) {
            double c0 = 0.0, c1 = 0.0;
#pragma unroll
            for (int u = 0; u < 16; u += 2) {
                c0 = fma(a[u], tab.q[(u << 4) | w], c0);
                c1 = fma(a[u + 1], tab.q[((u + 1) << 4) | w], c1);
            }
            const double bc = b[w] * (c0 + c1);
#pragma unroll
            for (int j = 0; j < 4; ++j)
                if ((w >> j) & 1) sw[j] += bc;
        }
        // values this thread contributes, relative to ref_pix: Z, marginals of low bits 0..7, marginals of t-bits < NHW
        const double scale = exp(-beta * (ref - refpix));
        double val[NR];
        val[0] = zt * scale;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            val[1 + j] = sw[j] * scale;
            val[5 + j] = su[j] * scale;
        }
#pragma unroll
        for (int jh = 0; jh < NHW; ++jh) val[9 + jh] = ((t >> jh) & 1u) ? val[0] : 0.0;

        // ---- reduce inside the group (fixed butterfly order), then across the groups of the pixel through shared memory
#pragma unroll
        for (int o = W / 2; o > 0; o >>= 1) {
#pragma unroll
            for (int k = 0; k < NR; ++k) val[k] += __shfl_xor_sync(0xffffffffu, val[k], o);
        }
        if ((threadIdx.x & (W - 1)) == 0) {
#pragma unroll
            for (int k = 0; k < NR; ++k) sRed[grp_id][k] = val[k];
        }
        // ---- E_min, step 1: a lower bound of the thread's smallest energy as in pass 1 of the min-plus walk (positivity
        // offsets from |h_j|, one DADD per candidate, integer minima on the high words: qa_kernels_minplus.cu); the threads
        // within 2 of the pixel's smallest bound are re-scored exactly below
        unsigned Lb = 0xffffffffu;
        if (EMIN) {
            double offw = EC, offu = 0.0;
#pragma unroll
            for (int j = 0; j < NL; ++j) {
                if (j < 4)
                    offw += fabs(sIn[slot][N - 1 - j]);
                else
                    offu += fabs(sIn[slot][N - 1 - j]);
            }
            double B[16];
            B[0] = offw;
#pragma unroll
            for (int w = 1; w < 16; ++w) B[w] = B[w & (w - 1)] + hp[sp_ctz(w)];
#pragma unroll
            for (int u = 0; u < 16; ++u) {
                unsigned m = 0xffffffffu;
#pragma unroll
                for (int w = 0; w < 16; w += 2)
                    m = min(m, min((unsigned)__double2hiint(B[w] + tab.QL[(u << 4) | w]),
                                   (unsigned)__double2hiint(B[w + 1] + tab.QL[(u << 4) | (w + 1)])));
                double a = be + offu;
#pragma unroll
                for (int j = 3; j >= 0; --j)
                    if ((u >> j) & 1) a += hp[4 + j];
                Lb = min(Lb, (unsigned)__double2hiint(a + __hiloint2double((int)m, 0)));
            }
        }

        unsigned Lg = Lb;
        if (EMIN) {
#pragma unroll
            for (int o = W / 2; o > 0; o >>= 1) Lg = min(Lg, __shfl_xor_sync(0xffffffffu, Lg, o));
        }
        if ((threadIdx.x & (W - 1)) == 0) sLmin[grp_id] = Lg;
        if (EMIN && threadIdx.x < PPB) sCnt[threadIdx.x] = 0;
        __syncthreads();
        const int64_t p = p0 + slot;
        const int g0 = slot * GPP;
        if (EMIN) {
            // ---- E_min, step 2: the survivors publish (h'_0..7, be); every thread of the pixel then scores its share of a
            // survivor's 2^8 candidates from the definition of the split, e = be + sum_{j in c} h'_j + QL[c]
            unsigned Lp = 0xffffffffu;
#pragma unroll
            for (int gq = 0; gq < GPP; ++gq) Lp = min(Lp, sLmin[g0 + gq]);
            if (Lb <= Lp + 2u) {
                const int pos = atomicAdd(&sCnt[slot], 1);
                double *dst = sSurv[slot * TPP + pos];
#pragma unroll
                for (int j = 0; j < NL; ++j) dst[j] = sIn[slot][N - 1 - j] + v[j];
                double be2 = sIn[slot][N] + QH;
#pragma unroll
                for (int jh = 0; jh < NH; ++jh)
                    if ((t >> jh) & 1u) be2 += sIn[slot][N - 1 - NL - jh];
                dst[NL] = be2;
            }
            __syncthreads();
            double em = INFINITY;
            const int ns = sCnt[slot];
            for (int sv = 0; sv < ns; ++sv) {
                const double *src = sSurv[slot * TPP + sv];
                for (int c = (int)t; c < 256; c += TPP) {
                    double e = src[NL];
#pragma unroll
                    for (int j = NL - 1; j >= 0; --j)
                        if ((c >> j) & 1) e += src[j];
                    em = fmin(em, e + tab.QL[c]);
                }
            }
#pragma unroll
            for (int o = W / 2; o > 0; o >>= 1) em = fmin(em, __shfl_xor_sync(0xffffffffu, em, o));
            if ((threadIdx.x & (W - 1)) == 0) sMin[grp_id] = em;
            __syncthreads();
        }
        for (int q = (int)t; q <= N && p < P; q += TPP) {  // output q < N: dot q; q = N: E_min
            if (q < N) {
                double Z = 0.0;
#pragma unroll
                for (int gq = 0; gq < GPP; ++gq) Z += sRed[g0 + gq][0];
                // dot q: low bit j = N-1-q (j < 8) or t-bit jh = N-1-8-q
                const int bit = N - 1 - q;
                double S = 0.0;
                if (bit < NL) {
#pragma unroll
                    for (int gq = 0; gq < GPP; ++gq) S += sRed[g0 + gq][1 + bit];
                } else if (bit - NL < NHW) {
#pragma unroll
                    for (int gq = 0; gq < GPP; ++gq) S += sRed[g0 + gq][9 + bit - NL];
                } else {  // a t-bit that selects whole groups
#pragma unroll
                    for (int gq = 0; gq < GPP; ++gq)
                        if ((gq >> (bit - NL - 5)) & 1) S += sRed[g0 + gq][0];
                }
                const double lo = (double)ws.base[(int64_t)q * P + p];
                outNmean[p * N + q] = Z > 0.0 ? lo + S / Z : -1.0;
            } else if (EMIN) {
                double m = INFINITY;
#pragma unroll
                for (int gq = 0; gq < GPP; ++gq) m = fmin(m, sMin[g0 + gq]);
                outEmin[p] = m - EC;  // QHT carries + E_C (a positivity offset of the min-plus walk)
            }
        }
    }
}

template <int NH>
cudaError_t launch_sp(const QaDevModel *d_model, const SpTable &tab, QaWorkspace ws, double beta, double *d_Nmean,
                      double *d_Emin, int sm_count, cudaStream_t stream)
{
    constexpr int PPB = SP_THREADS >> NH;
    const int64_t groups = (ws.P + PPB - 1) / PPB;
    int per_sm = 0;
    cudaError_t err;
    if (d_Emin)
        err = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, qa_thermal_sp_kernel<NH, true>, SP_THREADS, 0);
    else
        err = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, qa_thermal_sp_kernel<NH, false>, SP_THREADS, 0);
    if (err != cudaSuccess) return err;
    if (per_sm < 1) per_sm = 1;
    int64_t grid = (int64_t)sm_count * per_sm;
    if (grid > groups) grid = groups;
    if (d_Emin)
        return qa_launch_pdl(qa_thermal_sp_kernel<NH, true>, dim3((unsigned)grid), dim3(SP_THREADS), stream, d_model, tab, ws,
                             beta, d_Nmean, d_Emin);
    return qa_launch_pdl(qa_thermal_sp_kernel<NH, false>, dim3((unsigned)grid), dim3(SP_THREADS), stream, d_model, tab, ws, beta,
                         d_Nmean, d_Emin);
}

}  // namespace

// QLhost: the model's pair table of the low 8 bits (host copy).  The caller has checked beta * sum_{i<j} M_ij <= 600.
cudaError_t qa_launch_thermal_sp(const QaDevModel *d_model, int n, const double *QLhost, QaWorkspace ws, double kT,
                                 double *d_Nmean, double *d_Emin, int sm_count, cudaStream_t stream)
{
    qa_plan_add("qa_thermal_sp_kernel");
    SpTable tab;
    const double beta = 1.0 / kT;
    for (int b = 0; b < 256; ++b) {
        tab.QL[b] = QLhost[b];
        tab.q[b] = exp(-beta * QLhost[b]);
    }
    switch (n) {
        case 9: return launch_sp<1>(d_model, tab, ws, beta, d_Nmean, d_Emin, sm_count, stream);
        case 10: return launch_sp<2>(d_model, tab, ws, beta, d_Nmean, d_Emin, sm_count, stream);
        case 11: return launch_sp<3>(d_model, tab, ws, beta, d_Nmean, d_Emin, sm_count, stream);
        case 12: return launch_sp<4>(d_model, tab, ws, beta, d_Nmean, d_Emin, sm_count, stream);
        case 13: return launch_sp<5>(d_model, tab, ws, beta, d_Nmean, d_Emin, sm_count, stream);
        case 14: return launch_sp<6>(d_model, tab, ws, beta, d_Nmean, d_Emin, sm_count, stream);
        case 15: return launch_sp<7>(d_model, tab, ws, beta, d_Nmean, d_Emin, sm_count, stream);
        case 16: return launch_sp<8>(d_model, tab, ws, beta, d_Nmean, d_Emin, sm_count, stream);
        default: return cudaErrorInvalidValue;
    }
}
