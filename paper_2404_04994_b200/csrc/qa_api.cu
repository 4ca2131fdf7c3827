// qa_api.cu -- host side of the C ABI (include/qarray_b200.h): model validation and setup (S0), argument checks,
// workspace carving and kernel dispatch.  No compute on the host beyond S0; no CPU fallback.
#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <string>

#include "qa_internal.cuh"
#include "../../include/qarray_b200_aids.h"

struct qa_batch {
    int n_models, n, g, general;
    int device;
    const QaDevModel **dev_list;  // device array of the models' device pointers
    qa_model **members;           // host: the models (their in_batches count is held until qa_batch_destroy)
};

struct qa_model {
    int nf, g, ns;          // full model
    int device;
    int sm_count;
    bool is_z;              // every off-diagonal of c_dd <= 0 (Maxwell, Eq. (B1))
    double Cf[QA_MAXN * QA_MAXN];    // full c_dd, stride nf
    double Cgdf[QA_MAXN * QA_MAXG];  // full c_gd, stride g
    double Mf[QA_MAXN * QA_MAXN];    // full inverse, stride nf
    double ECf;
    int sens[QA_MAXN];
    QaDevModel host;        // mirror of the device constants
    QaDevModel *dev;        // device copy
    const QaDevModel **dev_self;  // device array of one pointer (= dev): the model list of a single-model fused launch
    QaWalkTable walk;       // pair table of the low bits of the search model
    std::atomic<int> walk_variant;  // kernel selection (qa_model_set_walk_variant; cross-check aid)
    std::atomic<int> in_batches;    // qa_batch objects holding this model's device pointer
    // qa_ground_state_host: a private stream and a grow-only device staging buffer, reused from call to call (creating
    // a stream and going through the allocator cost more than the search itself on a 100x100 diagram)
    std::mutex host_mu;
    cudaStream_t host_stream;
    char *host_buf;
    size_t host_buf_bytes;
};

namespace {

thread_local std::string g_plan;
thread_local int g_plan_count = 0;
thread_local char g_cuda_err[256] = "";
thread_local bool g_timing = false;           // measurement aid: CUDA events around every kernel of a call
thread_local cudaEvent_t g_events[8];
thread_local int g_n_events_created = 0, g_n_marks = 0;

void timing_mark(cudaStream_t stream)
{
    if (!g_timing || g_n_marks >= 8) return;
    if (g_n_marks >= g_n_events_created) {
        if (cudaEventCreate(&g_events[g_n_events_created]) != cudaSuccess) return;
        ++g_n_events_created;
    }
    cudaEventRecord(g_events[g_n_marks++], stream);
}

qa_status cuda_fail(cudaError_t e, const char *where)
{
    std::snprintf(g_cuda_err, sizeof(g_cuda_err), "%s: %s", where, cudaGetErrorString(e));
    return QA_ERR_CUDA;
}
#define QA_CUDA(call)                                                                                                  \
    do {                                                                                                               \
        cudaError_t e__ = (call);                                                                                      \
        if (e__ != cudaSuccess) return cuda_fail(e__, #call);                                                          \
    } while (0)

// Cholesky-based inverse of an SPD matrix (k x k, row-major, stride k).  Returns false if not positive definite.
bool spd_inverse(const double *A, int k, double *inv)
{
    double L[QA_MAXN * QA_MAXN];
    for (int i = 0; i < k; ++i) {
        for (int j = 0; j <= i; ++j) {
            double s = A[i * k + j];
            for (int q = 0; q < j; ++q) s -= L[i * k + q] * L[j * k + q];
            if (i == j) {
                if (!(s > 0.0) || !std::isfinite(s)) return false;
                L[i * k + i] = std::sqrt(s);
            } else {
                L[i * k + j] = s / L[j * k + j];
            }
        }
    }
    for (int c = 0; c < k; ++c) {
        double y[QA_MAXN], x[QA_MAXN];
        for (int i = 0; i < k; ++i) {
            double s = (i == c) ? 1.0 : 0.0;
            for (int q = 0; q < i; ++q) s -= L[i * k + q] * y[q];
            y[i] = s / L[i * k + i];
        }
        for (int i = k - 1; i >= 0; --i) {
            double s = y[i];
            for (int q = i + 1; q < k; ++q) s -= L[q * k + i] * x[q];
            x[i] = s / L[i * k + i];
        }
        for (int i = 0; i < k; ++i) inv[i * k + c] = x[i];
    }
    return true;
}

// (Re)build the search model (full model minus sensor dots), its tables, and upload.
qa_status rebuild(qa_model *m)
{
    QaDevModel &h = m->host;
    std::memset(&h, 0, sizeof(h));
    const int nf = m->nf, g = m->g, ns = m->ns;
    bool is_s[QA_MAXN] = {false};
    for (int a = 0; a < ns; ++a) is_s[m->sens[a]] = true;
    int n = 0;
    for (int i = 0; i < nf; ++i)
        if (!is_s[i]) h.arr_idx[n++] = i;
    for (int a = 0; a < ns; ++a) h.sens_idx[a] = m->sens[a];
    h.n = n;
    h.g = g;
    h.nf = nf;
    h.ns = ns;
    double Csub[QA_MAXN * QA_MAXN], Msub[QA_MAXN * QA_MAXN];
    for (int a = 0; a < n; ++a)
        for (int b = 0; b < n; ++b) Csub[a * n + b] = m->Cf[h.arr_idx[a] * nf + h.arr_idx[b]];
    if (!spd_inverse(Csub, n, Msub)) return QA_ERR_NOT_POSDEF;
    double tot = 0.0, mn = 0.0;
    for (int a = 0; a < n; ++a) {
        double s = 0.0;  // c_dd 1: plain left-to-right sum (reading R1)
        for (int b = 0; b < n; ++b) {
            h.C[a * QA_MAXN + b] = Csub[a * n + b];
            h.M[a * QA_MAXN + b] = Msub[a * n + b];
            s = s + Csub[a * n + b];
        }
        h.C1[a] = s;
        tot = tot + s;
        for (int k = 0; k < g; ++k) h.Cgd[a * QA_MAXG + k] = m->Cgdf[h.arr_idx[a] * g + k];
        if (a == 0 || Msub[a * n + a] < mn) mn = Msub[a * n + a];
    }
    h.oneC1 = tot;
    h.EC = 0.5 * mn;
    for (int i = 0; i < nf; ++i) {
        for (int j = 0; j < nf; ++j) h.Mf[i * QA_MAXN + j] = m->Mf[i * nf + j];
        for (int k = 0; k < g; ++k) h.Cgdf[i * QA_MAXG + k] = m->Cgdf[i * g + k];
    }
    // pair table of the low bits: low bit j <-> search dot n-1-j
    const int nl = n < QA_PAIR_NL ? n : QA_PAIR_NL;
    for (int b = 0; b < (1 << QA_PAIR_NL); ++b) {
        double s = 0.0;
        if (b < (1 << nl))
            for (int j = 0; j < nl; ++j)
                for (int j2 = j + 1; j2 < nl; ++j2)
                    if (((b >> j) & 1) && ((b >> j2) & 1)) s += Msub[(n - 1 - j) * n + (n - 1 - j2)];
        h.QL[b] = s;
        if (b < (1 << QA_WALK_NL)) m->walk.QL[b] = s;
    }
    // tables of the min-plus walk: high pattern t of the NH = n - QA_WALK_NL high bits (high bit jh <-> dot n-1-NL-jh)
    if (n > QA_WALK_NL) {
        const int NL = QA_WALK_NL, NH = n - NL;
        for (int t = 0; t < (1 << NH); ++t) {
            for (int j = 0; j < NL; ++j) {
                double s = 0.0;
                for (int jh = 0; jh < NH; ++jh)
                    if ((t >> jh) & 1) s += Msub[(n - 1 - j) * n + (n - 1 - NL - jh)];
                h.VT[t * NL + j] = s;
                h.VTt[j * (1 << QA_WALK_NL) + t] = s;
            }
            double q = h.EC;
            for (int jh = 0; jh < NH; ++jh)
                for (int jh2 = jh + 1; jh2 < NH; ++jh2)
                    if (((t >> jh) & 1) && ((t >> jh2) & 1)) q += Msub[(n - 1 - NL - jh) * n + (n - 1 - NL - jh2)];
            h.QHT[t] = q;
        }
    }
    h.qsum = 0.0;
    for (int i = 0; i < n; ++i)
        for (int j = i + 1; j < n; ++j) h.qsum += std::fabs(h.M[i * QA_MAXN + j]);
    if (n <= 8) {  // staging block of the one-kernel path (layout: QaDevModel::fo_pack)
        double *pk = h.fo_pack;
        for (int j = 0; j < n; ++j)
            for (int i = 0; i < n; ++i) pk[j * n + i] = h.M[i * QA_MAXN + j];
        pk += n * n;
        for (int i = 0; i < n; ++i)
            for (int j = 0; j < n; ++j) pk[i * n + j] = h.C[i * QA_MAXN + j];
        pk += n * n;
        for (int b = 0; b < (1 << n); ++b) pk[b] = h.QL[b];
        pk += 1 << n;
        for (int k = 0; k < m->g; ++k)
            for (int i = 0; i < n; ++i) pk[k * n + i] = h.Cgd[i * QA_MAXG + k];
    }
    // The source is pageable and the kernels run on non-blocking streams, which are not ordered against the legacy
    // stream: wait until the copy has landed and nothing else on the device can still read the old constants.
    QA_CUDA(cudaMemcpy(m->dev, &h, sizeof(h), cudaMemcpyHostToDevice));
    QA_CUDA(cudaDeviceSynchronize());
    return QA_OK;
}

// Initial kernel selection of a model (qa_model_set_walk_variant): environment variable QA_WALK_VARIANT, default 1.
int initial_walk_variant()
{
    const char *e = std::getenv("QA_WALK_VARIANT");
    const int v = e ? std::atoi(e) : 1;
    return (v < 0 || v > 4) ? 1 : v;
}

// A model (batch) belongs to the device that was current when it was created.
bool on_device(int device)
{
    int cur = -1;
    return cudaGetDevice(&cur) == cudaSuccess && cur == device;
}

size_t align256(size_t b) { return (b + 255) & ~(size_t)255; }

size_t carve(const qa_model *m, int64_t P, void *base, QaWorkspace *ws)
{
    const size_t n = (size_t)m->host.n, Pz = (size_t)P;
    char *p = static_cast<char *>(base);
    size_t off = 0;
    auto take = [&](size_t bytes) {
        void *r = p ? p + off : nullptr;
        off += align256(bytes);
        return r;
    };
    double *h = static_cast<double *>(take(n * Pz * 8));
    double *nc = static_cast<double *>(take(n * Pz * 8));
    int32_t *bs = static_cast<int32_t *>(take(n * Pz * 4));
    int32_t *ct = static_cast<int32_t *>(take(n * Pz * 4));
    uint64_t *tt = static_cast<uint64_t *>(take(Pz * 8));
    uint64_t *be = static_cast<uint64_t *>(take(Pz * 8));
    double *e0 = static_cast<double *>(take(Pz * 8));
    // records of the min-plus walk (n >= 13: 8 bytes per warp of a pixel) or of the closed walk (n >= 9: 16 bytes per block)
    size_t rec_bytes = n >= 13 ? Pz * 8 * ((size_t)1 << (n - 13)) : 0;
    if (n > QA_WALK_NL && rec_bytes < Pz * 16 * (size_t)QA_CLOSED_MAXB) rec_bytes = Pz * 16 * (size_t)QA_CLOSED_MAXB;
    uint2 *rec = static_cast<uint2 *>(take(rec_bytes));
    unsigned long long *counter = static_cast<unsigned long long *>(take(256));
    if (ws) {
        ws->h = h;
        ws->nc = nc;
        ws->base = bs;
        ws->cnt = ct;
        ws->total = tt;
        ws->best = be;
        ws->e0 = e0;
        ws->rec = rec;
        ws->rec2 = reinterpret_cast<double2 *>(rec);
        // n >= 13: the walk's records take 8 * 2^(n-13) <= 64 bytes per pixel of the 256 the region has
        ws->ext = n >= 13 ? reinterpret_cast<double *>(reinterpret_cast<char *>(rec) + Pz * 64) : nullptr;
        ws->counter = counter;
        ws->P = P;
    }
    return off;
}

qa_status ground_state(const qa_model *m, const double *d_Vg, int64_t P, int closed, int N_hat, qa_algorithm alg,
                       double t, int n_max, int32_t *d_N, double *d_E, double *d_xcont, double *d_Vsensor,
                       qa_stats *d_stats, void *d_ws, size_t ws_bytes, void *stream_v)
{
    qa_plan_reset();
    if (!m || P < 0 || (P > 0 && (!d_Vg || !d_N || !d_E))) return QA_ERR_INVALID_ARG;
    if (P > 0 && !on_device(m->device)) return QA_ERR_INVALID_ARG;
    const int variant = m->walk_variant.load(std::memory_order_relaxed);
    if (alg != QA_ALG_DEFAULT && alg != QA_ALG_THRESHOLDED && alg != QA_ALG_BRUTE_FORCE) return QA_ERR_INVALID_ARG;
    if (alg == QA_ALG_THRESHOLDED && !(t >= 0.0 && t <= 1.0)) return QA_ERR_INVALID_ARG;
    if (alg == QA_ALG_BRUTE_FORCE && n_max < 0) return QA_ERR_INVALID_ARG;
    const int n = m->host.n;
    if (closed && N_hat < 0) return QA_ERR_INFEASIBLE;
    if (alg == QA_ALG_BRUTE_FORCE) {
        if (std::pow((double)n_max + 1.0, (double)n) >= 4.611686018427388e18) return QA_ERR_OVERFLOW;
        if (closed && (int64_t)n * n_max < N_hat) return QA_ERR_INFEASIBLE;
    }
    if (P == 0) return QA_OK;
    if (P > (int64_t)1 << 40) return QA_ERR_INVALID_ARG;
    if (!d_ws || ws_bytes < carve(m, P, nullptr, nullptr) || (reinterpret_cast<uintptr_t>(d_ws) & 255u))
        return QA_ERR_INVALID_ARG;
    QaWorkspace ws;
    carve(m, P, d_ws, &ws);
    cudaStream_t stream = static_cast<cudaStream_t>(stream_v);
    QaCallArgs a{closed, N_hat, (int)alg, t, n_max, m->is_z ? 0 : 1, 0};
    // the min-plus walk follows the prologue: have it write the walk's per-pixel constants as well (ws.ext)
    if (alg == QA_ALG_DEFAULT && !closed && n >= 13 && variant == 1 && m->is_z) a.walk_ext = 1;
    g_n_marks = 0;
    timing_mark(stream);
    // small arrays with small candidate sets: the whole path in one kernel, one thread per pixel (no workspace traffic)
    {
        const double expect = alg == QA_ALG_BRUTE_FORCE ? std::pow((double)n_max + 1.0, (double)n) : std::pow(2.0, (double)n);
        if (n <= QA_FUSED_MAXN && !closed && alg != QA_ALG_BRUTE_FORCE && variant != 0) {  // binary set of an open array
            QA_CUDA(qa_launch_fused_open(m->dev_self, 1, n, m->g, d_Vg, P, a, d_N, d_E, d_xcont, m->ns > 0 ? d_Vsensor : nullptr,
                                         d_stats, stream));
            timing_mark(stream);
            return QA_OK;
        }
        if (n <= QA_FUSED_MAXN && expect <= 256.0 && variant != 0) {
            QA_CUDA(qa_launch_fused_small(m->dev_self, 1, n, d_Vg, P, a, d_N, d_E, d_xcont, m->ns > 0 ? d_Vsensor : nullptr,
                                          d_stats, stream));
            timing_mark(stream);
            return QA_OK;
        }
    }
    // open default search of 9..12 dots without sensor dots: the whole path in one kernel, a warp per two pixels
    if (!closed && alg == QA_ALG_DEFAULT && n > QA_FUSED_MAXN && n <= 12 && m->ns == 0 && variant != 0) {
        QA_CUDA(qa_launch_fused_mid(m->dev, n, m->walk, d_Vg, P, a, d_N, d_E, d_xcont, d_stats, stream));
        timing_mark(stream);
        return QA_OK;
    }
    // open default search of a 16-dot Maxwell array without sensor dots (variant 4): S1-S7 in one persistent kernel
    if (!closed && alg == QA_ALG_DEFAULT && n == 16 && m->ns == 0 && m->is_z && variant == 4) {
        QA_CUDA(qa_launch_minplus_fused(m->dev, m->host.QL, d_Vg, P, a, d_N, d_E, d_xcont, d_stats, m->sm_count, stream));
        timing_mark(stream);
        return QA_OK;
    }
    QA_CUDA(qa_launch_prologue(m->dev, n, m->g, d_Vg, ws, a, d_xcont, d_stats, stream, variant != 0));
    timing_mark(stream);
    // the min-plus walk needs M >= 0 entrywise (its positivity offsets), which holds for a Maxwell c_dd
    if (alg == QA_ALG_DEFAULT && !closed && n >= 13 && variant != 0 && m->is_z) {
        const bool fuse = m->ns == 0;  // S7 runs inside the finish kernel: no finalize launch
        if (variant == 3)  // mixed precision: fp32 lower-bound pass 1, fp64 exact pass 2 (same charge map, bit for bit)
            QA_CUDA(qa_launch_minplus_walk32(m->dev, n, m->host.QL, ws, fuse ? d_N : nullptr, d_E, m->sm_count, stream));
        else
            QA_CUDA(qa_launch_minplus_walk(m->dev, n, m->host.QL, ws, fuse ? d_N : nullptr, d_E, m->sm_count,
                                           variant == 2, stream));
        timing_mark(stream);
        if (fuse) return QA_OK;
    } else if (alg == QA_ALG_DEFAULT && closed && n > QA_WALK_NL && variant != 0) {
        // closed default set of a larger array: only the C(n, k) states with the right total are visited (NEXT-3)
        int nb = 0;
        QA_CUDA(qa_launch_closed_walk(m->dev, n, m->walk, ws, a, m->sm_count, stream, &nb));
        timing_mark(stream);
        QA_CUDA(qa_launch_finalize(m->dev, d_Vg, ws, d_N, d_E, m->ns > 0 ? d_Vsensor : nullptr, d_stats, stream, nb, N_hat,
                                   (m->ns == 0 && variant != 0) ? n : 0));
        timing_mark(stream);
        return QA_OK;
    } else if (alg == QA_ALG_DEFAULT && !closed) {
        QA_CUDA(qa_launch_walk(m->dev, n, m->walk, ws, d_stats, m->sm_count, stream));
        timing_mark(stream);
    } else {
        double expect = alg == QA_ALG_BRUTE_FORCE ? std::pow((double)n_max + 1.0, (double)n)
                        : alg == QA_ALG_DEFAULT   ? std::pow(2.0, (double)n)
                                                  : std::pow(1.0 + t, (double)n);
        QA_CUDA(qa_launch_enumerate(m->dev, n, ws, a, expect, d_stats, stream));
        timing_mark(stream);
    }
    QA_CUDA(qa_launch_finalize(m->dev, d_Vg, ws, d_N, d_E, m->ns > 0 ? d_Vsensor : nullptr, d_stats, stream, 0, 0,
                               (m->ns == 0 && variant != 0) ? n : 0));
    timing_mark(stream);
    return QA_OK;
}

// Thermal broadening (Eq. (10)): prologue (S1-S4) + qa_thermal_kernel.
qa_status thermal(const qa_model *m, const double *d_Vg, int64_t P, int closed, int N_hat, qa_algorithm alg, double t,
                  int n_max, double kT, double *d_Nmean, double *d_Emin, qa_stats *d_stats, void *d_ws, size_t ws_bytes,
                  void *stream_v)
{
    qa_plan_reset();
    if (!m || P < 0 || (P > 0 && (!d_Vg || !d_Nmean))) return QA_ERR_INVALID_ARG;
    if (P > 0 && !on_device(m->device)) return QA_ERR_INVALID_ARG;
    if (!(kT > 0.0) || !std::isfinite(kT)) return QA_ERR_INVALID_ARG;
    if (alg != QA_ALG_DEFAULT && alg != QA_ALG_THRESHOLDED && alg != QA_ALG_BRUTE_FORCE) return QA_ERR_INVALID_ARG;
    if (alg == QA_ALG_THRESHOLDED && !(t >= 0.0 && t <= 1.0)) return QA_ERR_INVALID_ARG;
    if (alg == QA_ALG_BRUTE_FORCE && n_max < 0) return QA_ERR_INVALID_ARG;
    const int n = m->host.n;
    if (closed && N_hat < 0) return QA_ERR_INFEASIBLE;
    if (alg == QA_ALG_BRUTE_FORCE) {
        if (std::pow((double)n_max + 1.0, (double)n) >= 4.611686018427388e18) return QA_ERR_OVERFLOW;
        if (closed && (int64_t)n * n_max < N_hat) return QA_ERR_INFEASIBLE;
    }
    if (P == 0) return QA_OK;
    if (P > (int64_t)1 << 40) return QA_ERR_INVALID_ARG;
    if (!d_ws || ws_bytes < carve(m, P, nullptr, nullptr) || (reinterpret_cast<uintptr_t>(d_ws) & 255u))
        return QA_ERR_INVALID_ARG;
    QaWorkspace ws;
    carve(m, P, d_ws, &ws);
    cudaStream_t stream = static_cast<cudaStream_t>(stream_v);
    QaCallArgs a{closed, N_hat, (int)alg, t, n_max, m->is_z ? 0 : 1, 0};
    g_n_marks = 0;
    timing_mark(stream);
    QA_CUDA(qa_launch_prologue(m->dev, n, m->g, d_Vg, ws, a, nullptr, d_stats, stream,
                               m->walk_variant.load(std::memory_order_relaxed) != 0));
    timing_mark(stream);
    const double expect = alg == QA_ALG_BRUTE_FORCE ? std::pow((double)n_max + 1.0, (double)n)
                          : alg == QA_ALG_DEFAULT   ? std::pow(2.0, (double)n)
                                                    : std::pow(1.0 + t, (double)n);
    // open default set of a larger Maxwell array: sum-product over the min-plus split, while the factorised weights stay
    // far from underflow (beta * sum_{i<j} M_ij <= 600, qa_kernels_thermal_sp.cu); otherwise the two-pass kernels
    double gsum = 0.0;
    for (int i = 0; i < n; ++i)
        for (int j = i + 1; j < n; ++j) gsum += std::fabs(m->host.M[i * QA_MAXN + j]);
    if (!closed && alg == QA_ALG_DEFAULT && n > QA_WALK_NL && m->is_z && gsum / kT <= 600.0 &&
        m->walk_variant.load(std::memory_order_relaxed) != 0) {
        QA_CUDA(qa_launch_thermal_sp(m->dev, n, m->host.QL, ws, kT, d_Nmean, d_Emin, m->sm_count, stream));
        timing_mark(stream);
        return QA_OK;
    }
    QA_CUDA(qa_launch_thermal(m->dev, n, ws, a, kT, expect, d_Nmean, d_Emin, d_stats, stream));
    timing_mark(stream);
    return QA_OK;
}

}  // namespace

void qa_timing_mark(cudaStream_t stream) { timing_mark(stream); }
void qa_plan_reset()
{
    g_plan.clear();
    g_plan_count = 0;
}
void qa_plan_add(const char *name)
{
    if (!g_plan.empty()) g_plan += ",";
    g_plan += name;
    ++g_plan_count;
}

extern "C" {

qa_status qa_model_create(const double *C_dd, const double *C_gd, int n_dot, int n_gate, qa_model **out)
{
    if (out) *out = nullptr;
    if (!C_dd || !C_gd || !out || n_dot < 1 || n_gate < 1) return QA_ERR_INVALID_ARG;
    if (n_dot > QA_MAXN || n_gate > QA_MAXG) return QA_ERR_UNSUPPORTED_SIZE;
    double amax = 0.0;
    for (int i = 0; i < n_dot * n_dot; ++i) {
        if (!std::isfinite(C_dd[i])) return QA_ERR_INVALID_ARG;
        amax = std::fmax(amax, std::fabs(C_dd[i]));
    }
    for (int i = 0; i < n_dot * n_gate; ++i)
        if (!std::isfinite(C_gd[i])) return QA_ERR_INVALID_ARG;
    bool is_z = true;
    for (int i = 0; i < n_dot; ++i)
        for (int j = 0; j < i; ++j) {
            if (std::fabs(C_dd[i * n_dot + j] - C_dd[j * n_dot + i]) > 1e-12 * amax) return QA_ERR_NOT_SYMMETRIC;
            if (C_dd[i * n_dot + j] > 0.0) is_z = false;
        }
    qa_model *m = new (std::nothrow) qa_model();  // value-initialised: every plain member zero
    if (!m) return QA_ERR_INVALID_ARG;
    m->nf = n_dot;
    m->g = n_gate;
    m->ns = 0;
    m->is_z = is_z;
    m->walk_variant.store(initial_walk_variant());
    m->in_batches.store(0);
    std::memcpy(m->Cf, C_dd, sizeof(double) * n_dot * n_dot);
    std::memcpy(m->Cgdf, C_gd, sizeof(double) * n_dot * n_gate);
    if (!spd_inverse(m->Cf, n_dot, m->Mf)) {
        delete m;
        return QA_ERR_NOT_POSDEF;
    }
    double mn = m->Mf[0];
    for (int i = 1; i < n_dot; ++i) mn = std::fmin(mn, m->Mf[i * n_dot + i]);
    m->ECf = 0.5 * mn;
    cudaError_t e = cudaGetDevice(&m->device);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&m->sm_count, cudaDevAttrMultiProcessorCount, m->device);
    if (e == cudaSuccess) e = cudaMalloc(reinterpret_cast<void **>(&m->dev), sizeof(QaDevModel));
    if (e == cudaSuccess) e = cudaMalloc(reinterpret_cast<void **>(&m->dev_self), sizeof(QaDevModel *));
    if (e == cudaSuccess) e = cudaMemcpy(m->dev_self, &m->dev, sizeof(QaDevModel *), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) {
        if (m->dev) cudaFree(m->dev);
        if (m->dev_self) cudaFree(m->dev_self);
        delete m;
        return cuda_fail(e, "qa_model_create");
    }
    qa_status s = rebuild(m);
    if (s != QA_OK) {
        cudaFree(m->dev);
        cudaFree(m->dev_self);
        delete m;
        return s;
    }
    *out = m;
    return QA_OK;
}

qa_status qa_model_set_sensor_dots(qa_model *m, const int *dot_idx, int n_sensor)
{
    if (!m || n_sensor < 0 || n_sensor >= m->nf || (n_sensor > 0 && !dot_idx)) return QA_ERR_INVALID_ARG;
    if (m->in_batches.load() != 0 || !on_device(m->device)) return QA_ERR_INVALID_ARG;  // a batch holds the old constants
    bool seen[QA_MAXN] = {false};
    for (int a = 0; a < n_sensor; ++a) {
        if (dot_idx[a] < 0 || dot_idx[a] >= m->nf || seen[dot_idx[a]]) return QA_ERR_INVALID_ARG;
        seen[dot_idx[a]] = true;
    }
    int old_ns = m->ns, old[QA_MAXN];
    std::memcpy(old, m->sens, sizeof(old));
    m->ns = n_sensor;
    for (int a = 0; a < n_sensor; ++a) m->sens[a] = dot_idx[a];
    qa_status s = rebuild(m);
    if (s != QA_OK) {
        m->ns = old_ns;
        std::memcpy(m->sens, old, sizeof(old));
        rebuild(m);
    }
    return s;
}

qa_status qa_model_destroy(qa_model *m)
{
    if (!m) return QA_OK;
    cudaError_t e = cudaFree(m->dev);
    if (m->dev_self) cudaFree(m->dev_self);
    if (m->host_buf) cudaFree(m->host_buf);
    if (m->host_stream) cudaStreamDestroy(m->host_stream);
    delete m;
    return e == cudaSuccess ? QA_OK : cuda_fail(e, "qa_model_destroy");
}

int qa_model_n_dot(const qa_model *m) { return m ? m->nf : 0; }
int qa_model_n_gate(const qa_model *m) { return m ? m->g : 0; }
int qa_model_n_sensor(const qa_model *m) { return m ? m->ns : 0; }
int qa_model_n_search(const qa_model *m) { return m ? m->host.n : 0; }

qa_status qa_model_get_inverse(const qa_model *m, double *M_host, double *E_C)
{
    if (!m) return QA_ERR_INVALID_ARG;
    if (M_host) std::memcpy(M_host, m->Mf, sizeof(double) * m->nf * m->nf);
    if (E_C) *E_C = m->ECf;
    return QA_OK;
}

size_t qa_workspace_bytes(const qa_model *m, int64_t P)
{
    if (!m || P < 0) return 0;
    return carve(m, P < 1 ? 1 : P, nullptr, nullptr);
}

qa_status qa_ground_state_open(const qa_model *m, const double *d_Vg, int64_t P, qa_algorithm alg, double t, int n_max,
                               int32_t *d_N, double *d_E, double *d_xcont, double *d_Vsensor, qa_stats *d_stats,
                               void *d_workspace, size_t workspace_bytes, void *cuda_stream)
{
    return ground_state(m, d_Vg, P, 0, 0, alg, t, n_max, d_N, d_E, d_xcont, d_Vsensor, d_stats, d_workspace,
                        workspace_bytes, cuda_stream);
}

qa_status qa_ground_state_closed(const qa_model *m, const double *d_Vg, int64_t P, int N_hat, qa_algorithm alg, double t,
                                 int n_max, int32_t *d_N, double *d_E, double *d_xcont, double *d_Vsensor,
                                 qa_stats *d_stats, void *d_workspace, size_t workspace_bytes, void *cuda_stream)
{
    return ground_state(m, d_Vg, P, 1, N_hat, alg, t, n_max, d_N, d_E, d_xcont, d_Vsensor, d_stats, d_workspace,
                        workspace_bytes, cuda_stream);
}

qa_status qa_ground_state_host(const qa_model *mc, const double *h_Vg, int64_t P, int closed, int N_hat, qa_algorithm alg,
                               double t, int n_max, int32_t *h_N, double *h_E, double *h_xcont, double *h_Vsensor,
                               qa_stats *h_stats)
{
    if (!mc || P < 0 || (P > 0 && (!h_Vg || !h_N || !h_E))) return QA_ERR_INVALID_ARG;
    if (P == 0) return QA_OK;
    if (!on_device(mc->device)) return QA_ERR_INVALID_ARG;
    qa_model *m = const_cast<qa_model *>(mc);  // only the host-call staging state below is touched, under its mutex
    std::lock_guard<std::mutex> lock(m->host_mu);
    const size_t Pz = (size_t)P, nf = (size_t)m->nf, n = (size_t)m->host.n, g = (size_t)m->g, ns = (size_t)m->ns;
    const size_t bVg = align256(Pz * g * 8), bN = align256(Pz * nf * 4), bE = align256(Pz * 8);
    const size_t bX = h_xcont ? align256(Pz * n * 8) : 0, bVs = (h_Vsensor && ns) ? align256(Pz * ns * 8) : 0;
    const size_t bS = h_stats ? align256(sizeof(qa_stats)) : 0, bW = qa_workspace_bytes(m, P);
    const size_t need = bVg + bN + bE + bX + bVs + bS + bW;
    if (!m->host_stream) QA_CUDA(cudaStreamCreateWithFlags(&m->host_stream, cudaStreamNonBlocking));
    cudaStream_t stream = m->host_stream;
    if (m->host_buf_bytes < need) {
        if (m->host_buf) QA_CUDA(cudaFree(m->host_buf));
        m->host_buf = nullptr;
        m->host_buf_bytes = 0;
        QA_CUDA(cudaMalloc(reinterpret_cast<void **>(&m->host_buf), need));
        m->host_buf_bytes = need;
    }
    char *buf = m->host_buf;
    qa_status st = QA_OK;
    double *dVg = reinterpret_cast<double *>(buf);
    int32_t *dN = reinterpret_cast<int32_t *>(buf + bVg);
    double *dE = reinterpret_cast<double *>(buf + bVg + bN);
    double *dX = bX ? reinterpret_cast<double *>(buf + bVg + bN + bE) : nullptr;
    double *dVs = bVs ? reinterpret_cast<double *>(buf + bVg + bN + bE + bX) : nullptr;
    qa_stats *dS = bS ? reinterpret_cast<qa_stats *>(buf + bVg + bN + bE + bX + bVs) : nullptr;
    void *dW = buf + bVg + bN + bE + bX + bVs + bS;
    cudaError_t e = cudaMemcpyAsync(dVg, h_Vg, Pz * g * 8, cudaMemcpyHostToDevice, stream);
    if (e == cudaSuccess && dS) e = cudaMemsetAsync(dS, 0, sizeof(qa_stats), stream);
    if (e == cudaSuccess) {
        st = ground_state(m, dVg, P, closed, N_hat, alg, t, n_max, dN, dE, dX, dVs, dS, dW, bW, stream);
        if (st == QA_OK) {
            e = cudaMemcpyAsync(h_N, dN, Pz * nf * 4, cudaMemcpyDeviceToHost, stream);
            if (e == cudaSuccess) e = cudaMemcpyAsync(h_E, dE, Pz * 8, cudaMemcpyDeviceToHost, stream);
            if (e == cudaSuccess && dX) e = cudaMemcpyAsync(h_xcont, dX, Pz * n * 8, cudaMemcpyDeviceToHost, stream);
            if (e == cudaSuccess && dVs)
                e = cudaMemcpyAsync(h_Vsensor, dVs, Pz * ns * 8, cudaMemcpyDeviceToHost, stream);
            if (e == cudaSuccess && dS)
                e = cudaMemcpyAsync(h_stats, dS, sizeof(qa_stats), cudaMemcpyDeviceToHost, stream);
        }
    }
    cudaError_t e2 = cudaStreamSynchronize(stream);
    if (st != QA_OK) return st;
    if (e != cudaSuccess) return cuda_fail(e, "qa_ground_state_host");
    if (e2 != cudaSuccess) return cuda_fail(e2, "qa_ground_state_host sync");
    return QA_OK;
}

qa_status qa_thermal_open(const qa_model *m, const double *d_Vg, int64_t P, qa_algorithm alg, double t, int n_max, double kT,
                          double *d_Nmean, double *d_Emin, qa_stats *d_stats, void *d_workspace, size_t workspace_bytes,
                          void *cuda_stream)
{
    return thermal(m, d_Vg, P, 0, 0, alg, t, n_max, kT, d_Nmean, d_Emin, d_stats, d_workspace, workspace_bytes, cuda_stream);
}

qa_status qa_thermal_closed(const qa_model *m, const double *d_Vg, int64_t P, int N_hat, qa_algorithm alg, double t, int n_max,
                            double kT, double *d_Nmean, double *d_Emin, qa_stats *d_stats, void *d_workspace,
                            size_t workspace_bytes, void *cuda_stream)
{
    return thermal(m, d_Vg, P, 1, N_hat, alg, t, n_max, kT, d_Nmean, d_Emin, d_stats, d_workspace, workspace_bytes,
                   cuda_stream);
}

size_t qa_sensor_response_workspace_bytes(int64_t P, int n_sensor)
{
    if (P < 0 || n_sensor < 1 || n_sensor > QA_MAXN) return 0;
    return qa_sensor_workspace_bytes_impl(P, n_sensor);
}

qa_status qa_sensor_response(const double *d_Vsensor, int64_t P, int n_sensor, int64_t W, const qa_sensor_params *params,
                             double *d_signal, double *d_gradient, void *d_workspace, size_t workspace_bytes, void *cuda_stream)
{
    qa_plan_reset();
    if (P < 0 || n_sensor < 1 || n_sensor > QA_MAXN || !params || W < 1 || (P % W) != 0) return QA_ERR_INVALID_ARG;
    if (P > 0 && (!d_Vsensor || !d_signal)) return QA_ERR_INVALID_ARG;
    for (int a = 0; a < n_sensor; ++a) {
        const qa_sensor_params &q = params[a];
        if (q.profile < 0 || q.profile > 2 || !(q.width > 0.0) || !std::isfinite(q.width) || q.pink_octaves < 0 ||
            q.pink_octaves > 30 || !(q.white_sigma >= 0.0) || !(q.pink_sigma >= 0.0) || !(q.jump_sigma >= 0.0) ||
            !(q.jump_rate >= 0.0 && q.jump_rate <= 1.0) || !std::isfinite(q.v0) || !std::isfinite(q.amplitude))
            return QA_ERR_INVALID_ARG;
    }
    if (P == 0) return QA_OK;
    if (P > (int64_t)1 << 40) return QA_ERR_INVALID_ARG;
    if (!d_workspace || workspace_bytes < qa_sensor_workspace_bytes_impl(P, n_sensor) ||
        (reinterpret_cast<uintptr_t>(d_workspace) & 255u))
        return QA_ERR_INVALID_ARG;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    g_n_marks = 0;
    timing_mark(stream);
    QA_CUDA(qa_launch_sensor_response(params, n_sensor, d_Vsensor, P, W, d_signal, d_gradient,
                                      static_cast<double *>(d_workspace), stream));
    timing_mark(stream);
    return QA_OK;
}

qa_status qa_batch_create(const qa_model *const *models, int n_models, qa_batch **out)
{
    if (out) *out = nullptr;
    if (!models || !out || n_models < 1 || n_models > 65535) return QA_ERR_INVALID_ARG;
    for (int b = 0; b < n_models; ++b) {
        if (!models[b]) return QA_ERR_INVALID_ARG;
        if (models[b]->ns != 0 || models[b]->host.n > QA_FUSED_MAXN) return QA_ERR_UNSUPPORTED_SIZE;
        if (models[b]->host.n != models[0]->host.n || models[b]->g != models[0]->g ||
            models[b]->device != models[0]->device)
            return QA_ERR_INVALID_ARG;
    }
    qa_batch *bt = new (std::nothrow) qa_batch();
    if (!bt) return QA_ERR_INVALID_ARG;
    bt->n_models = n_models;
    bt->n = models[0]->host.n;
    bt->g = models[0]->g;
    bt->device = models[0]->device;
    const QaDevModel **list = new (std::nothrow) const QaDevModel *[n_models];
    if (!list) {
        delete bt;
        return QA_ERR_INVALID_ARG;
    }
    bt->members = new (std::nothrow) qa_model *[n_models];
    if (!bt->members) {
        delete[] list;
        delete bt;
        return QA_ERR_INVALID_ARG;
    }
    for (int b = 0; b < n_models; ++b) {
        list[b] = models[b]->dev;
        bt->members[b] = const_cast<qa_model *>(models[b]);
        if (!models[b]->is_z) bt->general = 1;
    }
    cudaError_t e = cudaMalloc(reinterpret_cast<void **>(&bt->dev_list), sizeof(QaDevModel *) * n_models);
    if (e == cudaSuccess) e = cudaMemcpy(bt->dev_list, list, sizeof(QaDevModel *) * n_models, cudaMemcpyHostToDevice);
    delete[] list;
    if (e == cudaSuccess) e = cudaDeviceSynchronize();  // pageable source, non-blocking consumer streams (as in rebuild)
    if (e != cudaSuccess) {
        if (bt->dev_list) cudaFree(bt->dev_list);
        delete[] bt->members;
        delete bt;
        return cuda_fail(e, "qa_batch_create");
    }
    for (int b = 0; b < n_models; ++b) bt->members[b]->in_batches.fetch_add(1);
    *out = bt;
    return QA_OK;
}

qa_status qa_batch_destroy(qa_batch *bt)
{
    if (!bt) return QA_OK;
    cudaError_t e = cudaFree(bt->dev_list);
    for (int b = 0; b < bt->n_models; ++b) bt->members[b]->in_batches.fetch_sub(1);
    delete[] bt->members;
    delete bt;
    return e == cudaSuccess ? QA_OK : cuda_fail(e, "qa_batch_destroy");
}

qa_status qa_ground_state_batch(const qa_batch *bt, const double *d_Vg, int64_t P, int closed, int N_hat, qa_algorithm alg,
                                double t, int n_max, int32_t *d_N, double *d_E, double *d_xcont, qa_stats *d_stats,
                                void *cuda_stream)
{
    qa_plan_reset();
    if (!bt || P < 0 || (P > 0 && (!d_Vg || !d_N || !d_E))) return QA_ERR_INVALID_ARG;
    if (P > 0 && !on_device(bt->device)) return QA_ERR_INVALID_ARG;
    if (alg != QA_ALG_DEFAULT && alg != QA_ALG_THRESHOLDED && alg != QA_ALG_BRUTE_FORCE) return QA_ERR_INVALID_ARG;
    if (alg == QA_ALG_THRESHOLDED && !(t >= 0.0 && t <= 1.0)) return QA_ERR_INVALID_ARG;
    if (alg == QA_ALG_BRUTE_FORCE && n_max < 0) return QA_ERR_INVALID_ARG;
    if (closed && N_hat < 0) return QA_ERR_INFEASIBLE;
    if (alg == QA_ALG_BRUTE_FORCE) {
        if (std::pow((double)n_max + 1.0, (double)bt->n) >= 4.611686018427388e18) return QA_ERR_OVERFLOW;
        if (closed && (int64_t)bt->n * n_max < N_hat) return QA_ERR_INFEASIBLE;
    }
    if (P == 0) return QA_OK;
    if (P > (int64_t)1 << 40) return QA_ERR_INVALID_ARG;
    QaCallArgs a{closed, N_hat, (int)alg, t, n_max, bt->general, 0};
    if (!closed && alg != QA_ALG_BRUTE_FORCE)
        QA_CUDA(qa_launch_fused_open(bt->dev_list, bt->n_models, bt->n, bt->g, d_Vg, P, a, d_N, d_E, d_xcont, nullptr, d_stats,
                                     static_cast<cudaStream_t>(cuda_stream)));
    else
        QA_CUDA(qa_launch_fused_small(bt->dev_list, bt->n_models, bt->n, d_Vg, P, a, d_N, d_E, d_xcont, nullptr, d_stats,
                                      static_cast<cudaStream_t>(cuda_stream)));
    return QA_OK;
}

qa_status qa_ground_state_batch_multi(const qa_batch *bt, const double *d_Vg, int64_t P, int n_alg, const qa_algorithm *algs,
                                      const double *ts, int32_t *const *d_N, double *const *d_E, double *d_xcont,
                                      qa_stats *d_stats, void *cuda_stream)
{
    qa_plan_reset();
    if (!bt || P < 0 || n_alg < 1 || n_alg > QA_MULTI_MAX || !algs || !ts || !d_N || !d_E) return QA_ERR_INVALID_ARG;
    if (P > 0 && !d_Vg) return QA_ERR_INVALID_ARG;
    if (P > 0 && !on_device(bt->device)) return QA_ERR_INVALID_ARG;
    QaMultiArgs ma{};
    ma.n_alg = n_alg;
    for (int a = 0; a < n_alg; ++a) {
        if (algs[a] != QA_ALG_DEFAULT && algs[a] != QA_ALG_THRESHOLDED) return QA_ERR_INVALID_ARG;
        if (algs[a] == QA_ALG_THRESHOLDED && !(ts[a] >= 0.0 && ts[a] <= 1.0)) return QA_ERR_INVALID_ARG;
        if (P > 0 && (!d_N[a] || !d_E[a])) return QA_ERR_INVALID_ARG;
        ma.thr[a] = algs[a] == QA_ALG_THRESHOLDED ? 1 : 0;
        ma.t[a] = algs[a] == QA_ALG_THRESHOLDED ? ts[a] : 1.0;
        ma.N[a] = d_N[a];
        ma.E[a] = d_E[a];
    }
    if (P == 0) return QA_OK;
    if (P > (int64_t)1 << 40) return QA_ERR_INVALID_ARG;
    bool one_launch = true;  // the one-launch kernel has the sort-free thresholded walk only
    for (int a = 0; a < n_alg; ++a)
        if (ma.thr[a] && ma.t[a] > QA_FO_NOSORT_T) one_launch = false;
    if (one_launch) {
        QA_CUDA(qa_launch_fused_open_multi(bt->dev_list, bt->n_models, bt->n, bt->g, d_Vg, P, bt->general, ma, d_xcont,
                                           d_stats, static_cast<cudaStream_t>(cuda_stream)));
        return QA_OK;
    }
    for (int a = 0; a < n_alg; ++a) {  // a large threshold among them: one launch per algorithm, same results
        QaCallArgs ca{0, 0, ma.thr[a] ? (int)QA_ALG_THRESHOLDED : (int)QA_ALG_DEFAULT, ma.t[a], 0, bt->general, 0};
        QA_CUDA(qa_launch_fused_open(bt->dev_list, bt->n_models, bt->n, bt->g, d_Vg, P, ca, ma.N[a], ma.E[a], d_xcont, nullptr,
                                     d_stats, static_cast<cudaStream_t>(cuda_stream)));
    }
    return QA_OK;
}

int qa_batch_size(const qa_batch *bt) { return bt ? bt->n_models : 0; }

qa_status qa_measure_fp64_rate(double seconds, double *thread_inst_per_s, void *cuda_stream)
{
    if (!thread_inst_per_s || !(seconds > 0.0)) return QA_ERR_INVALID_ARG;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    int dev = 0, sms = 0;
    QA_CUDA(cudaGetDevice(&dev));
    QA_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    double *sink = nullptr;
    QA_CUDA(cudaMalloc(reinterpret_cast<void **>(&sink), 8));
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const int blocks = sms * 8, threads = 256;
    int iters = 2000;
    double rate = 0.0;
    qa_status st = QA_OK;
    for (int pass = 0; pass < 3 && st == QA_OK; ++pass) {  // warm-up / calibrate / measure
        cudaEventRecord(e0, stream);
        cudaError_t e = qa_launch_fp64_probe(sink, blocks, threads, iters, stream);
        cudaEventRecord(e1, stream);
        if (e == cudaSuccess) e = cudaEventSynchronize(e1);
        if (e != cudaSuccess) {
            st = cuda_fail(e, "qa_measure_fp64_rate");
            break;
        }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        rate = (double)blocks * threads * (double)iters * 64.0 / (ms * 1e-3);
        if (pass == 1 || pass == 0) {
            double want = (pass == 0 ? 0.05 : seconds) / (ms * 1e-3) * iters;
            iters = want > 2e9 ? 2000000000 : (want < 100 ? 100 : (int)want);
        }
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(sink);
    *thread_inst_per_s = rate;
    return st;
}

qa_status qa_set_kernel_timing(int enable)
{
    g_timing = enable != 0;
    g_n_marks = 0;
    return QA_OK;
}

qa_status qa_model_set_walk_variant(qa_model *m, int variant)
{
    if (!m || variant < 0 || variant > 4) return QA_ERR_INVALID_ARG;
    m->walk_variant.store(variant, std::memory_order_relaxed);
    return QA_OK;
}

qa_status qa_get_kernel_timings(int max_kernels, float *ms, int *n_kernels)
{
    if (!ms || !n_kernels || max_kernels < 0) return QA_ERR_INVALID_ARG;
    *n_kernels = 0;
    if (g_n_marks < 2) return QA_OK;
    QA_CUDA(cudaEventSynchronize(g_events[g_n_marks - 1]));
    for (int k = 0; k + 1 < g_n_marks && k < max_kernels; ++k) {
        QA_CUDA(cudaEventElapsedTime(&ms[k], g_events[k], g_events[k + 1]));
        *n_kernels = k + 1;
    }
    return QA_OK;
}

const char *qa_last_launch_plan(void) { return g_plan.c_str(); }
int qa_last_launch_count(void) { return g_plan_count; }

const char *qa_status_string(qa_status s)
{
    switch (s) {
        case QA_OK: return "ok";
        case QA_ERR_INVALID_ARG: return "invalid argument";
        case QA_ERR_NOT_SYMMETRIC: return "c_dd is not symmetric";
        case QA_ERR_NOT_POSDEF: return "c_dd is not positive definite";
        case QA_ERR_UNSUPPORTED_SIZE: return "n_dot > 16 or n_gate > 64";
        case QA_ERR_INFEASIBLE: return "closed array: no admissible charge state";
        case QA_ERR_OVERFLOW: return "brute force: (n_max+1)^n_dot >= 2^62";
        case QA_ERR_CUDA: return "CUDA error";
        case QA_ERR_UNSUPPORTED: return "unsupported (reserved; not returned by this version)";
        case QA_ERR_STATIC_WORKSPACE: return "sweep too large for the static workspace (qa_static_workspace_last_error)";
    }
    return "unknown status";
}
const char *qa_last_cuda_error(void) { return g_cuda_err; }
const char *qa_version(void) { return "qarray_b200 0.1 (sm_100a)"; }

}  // extern "C"
