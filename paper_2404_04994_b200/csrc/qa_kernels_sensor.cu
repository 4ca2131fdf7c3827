// qa_kernels_sensor.cu -- charge-sensor response, noise and gradient (PAPER.md L149 last two sentences, Fig. 3;
// SURVEY.md section 8(f) NEXT-2; reading R14).  Input: the sensor potentials V_s[P, n_sensor] the ground-state
// search wrote (step S8).  Per sensor a and pixel p (p = iy W + ix, the raster is the time axis):
//     S = profile(V_s)                      Lorentzian A / (1 + x^2), Gaussian A exp(-x^2 / 2), linear A x;  x = (V_s - v0) / w
//       + sigma_w z(0, p)                   white noise
//       + sigma_p / sqrt(K) sum_{j<K} z(1 + j, p >> j)        1/f noise (Voss-McCartney: source j redrawn every 2^j pixels)
//       + J(p) = sum_{q<=p} [u(62, q) < rate] sigma_j z(31, q)   sensor jumps: the baseline keeps every shift
// with counter-based random numbers r(stream, idx) = mix(mix(seed + G (stream + 1)) + G (idx + 1)) (SplitMix64 finaliser),
// u = ((r >> 11) + 1/2) 2^-53, z = Box-Muller of the uniforms of streams 2s and 2s + 1; sensor a uses streams 128 a + ...
// Every pixel draws its own numbers, so the only sequential part is the prefix sum of the jumps: per-chunk sums
// (qa_sensor_jump_partials_kernel), an exclusive scan of the chunk sums (qa_sensor_jump_scan_kernel, one CTA per sensor)
// and a block scan inside the signal kernel.  The gradient along the fast axis (central differences inside a row,
// one-sided at its ends; L464 "derivative of the sensor signal with respect to V_P1") is a second elementwise kernel.
// Bound: latency / HBM (16-32 bytes per pixel and sensor); the noise costs ~2 (K + 2) transcendental evaluations per pixel.
#include "qa_internal.cuh"

namespace {

constexpr int SR_THREADS = 256;
constexpr int SR_PPT = 4;                       // consecutive pixels per thread
constexpr int SR_CHUNK = SR_THREADS * SR_PPT;   // pixels per CTA

struct SrPack {
    qa_sensor_params p[QA_MAXN];
};

constexpr uint64_t SR_GOLDEN = 0x9E3779B97F4A7C15ull;

__device__ __forceinline__ uint64_t sr_mix64(uint64_t z)
{
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}
__device__ __forceinline__ double sr_uniform(uint64_t seed, uint64_t stream, uint64_t idx)
{
    const uint64_t r = sr_mix64(sr_mix64(seed + SR_GOLDEN * (stream + 1)) + SR_GOLDEN * (idx + 1));
    return ((double)(r >> 11) + 0.5) * 0x1.0p-53;
}
__device__ __forceinline__ double sr_normal(uint64_t seed, uint64_t stream, uint64_t idx)
{
    const double u1 = sr_uniform(seed, 2 * stream, idx), u2 = sr_uniform(seed, 2 * stream + 1, idx);
    return sqrt(-2.0 * log(u1)) * cospi(2.0 * u2);
}
__device__ __forceinline__ double sr_jump(const qa_sensor_params &q, uint64_t st, uint64_t p)
{
    if (sr_uniform(q.seed, 2 * (st + 62), p) < q.jump_rate) return q.jump_sigma * sr_normal(q.seed, st + 31, p);
    return 0.0;
}

// deterministic block sum / exclusive block scan over SR_THREADS values
__device__ __forceinline__ double sr_block_exclusive_scan(double v, double *sWarp, double &total)
{
    const unsigned lane = threadIdx.x & 31u, wid = threadIdx.x >> 5;
    double inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const double t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= (unsigned)o) inc += t;
    }
    if (lane == 31) sWarp[wid] = inc;
    __syncthreads();
    double woff = 0.0, tot = 0.0;
#pragma unroll
    for (int w = 0; w < SR_THREADS / 32; ++w) {
        const double s = sWarp[w];
        if ((unsigned)w < wid) woff += s;
        tot += s;
    }
    __syncthreads();
    total = tot;
    return woff + inc - v;
}

// sum of the jumps of every chunk of SR_CHUNK pixels: partial[a][chunk]
__global__ void __launch_bounds__(SR_THREADS) qa_sensor_jump_partials_kernel(const __grid_constant__ SrPack pk, int64_t P,
                                                                             int64_t nchunk, double *__restrict__ partial)
{
    __shared__ double sWarp[SR_THREADS / 32];
    const int a = blockIdx.y;
    const qa_sensor_params &q = pk.p[a];
    if (!(q.jump_rate > 0.0 && q.jump_sigma > 0.0)) return;
    const uint64_t st = 128ull * (uint64_t)a;
    const int64_t p0 = (int64_t)blockIdx.x * SR_CHUNK + (int64_t)threadIdx.x * SR_PPT;
    double v = 0.0;
#pragma unroll
    for (int k = 0; k < SR_PPT; ++k)
        if (p0 + k < P) v += sr_jump(q, st, (uint64_t)(p0 + k));
    double total;
    (void)sr_block_exclusive_scan(v, sWarp, total);
    if (threadIdx.x == 0) partial[(int64_t)a * nchunk + blockIdx.x] = total;
}

// exclusive scan of the chunk sums of one sensor, in place (one CTA per sensor; chunk order = time order)
__global__ void __launch_bounds__(SR_THREADS) qa_sensor_jump_scan_kernel(const __grid_constant__ SrPack pk, int64_t nchunk,
                                                                         double *__restrict__ partial)
{
    __shared__ double sWarp[SR_THREADS / 32];
    const int a = blockIdx.x;
    const qa_sensor_params &q = pk.p[a];
    if (!(q.jump_rate > 0.0 && q.jump_sigma > 0.0)) return;
    double *row = partial + (int64_t)a * nchunk;
    double carry = 0.0;
    for (int64_t c0 = 0; c0 < nchunk; c0 += SR_THREADS) {
        const int64_t c = c0 + threadIdx.x;
        const double v = c < nchunk ? row[c] : 0.0;
        double total;
        const double ex = sr_block_exclusive_scan(v, sWarp, total);
        if (c < nchunk) row[c] = carry + ex;
        carry += total;
    }
}

__global__ void __launch_bounds__(SR_THREADS) qa_sensor_signal_kernel(const __grid_constant__ SrPack pk,
                                                                      const double *__restrict__ Vs, int64_t P, int ns,
                                                                      int64_t nchunk, const double *__restrict__ partial,
                                                                      double *__restrict__ S)
{
    __shared__ double sWarp[SR_THREADS / 32];
    const int a = blockIdx.y;
    const qa_sensor_params &q = pk.p[a];
    const uint64_t st = 128ull * (uint64_t)a;
    const int64_t p0 = (int64_t)blockIdx.x * SR_CHUNK + (int64_t)threadIdx.x * SR_PPT;
    const bool jumps = q.jump_rate > 0.0 && q.jump_sigma > 0.0;
    double jv[SR_PPT], J = 0.0;
    if (jumps) {
        double v = 0.0;
#pragma unroll
        for (int k = 0; k < SR_PPT; ++k) {
            jv[k] = p0 + k < P ? sr_jump(q, st, (uint64_t)(p0 + k)) : 0.0;
            v += jv[k];
        }
        double total;
        J = partial[(int64_t)a * nchunk + blockIdx.x] + sr_block_exclusive_scan(v, sWarp, total);
    }
    const double pink_scale = q.pink_octaves > 0 ? q.pink_sigma / sqrt((double)q.pink_octaves) : 0.0;
#pragma unroll
    for (int k = 0; k < SR_PPT; ++k) {
        const int64_t p = p0 + k;
        if (p >= P) break;
        const double x = (Vs[p * ns + a] - q.v0) / q.width;
        double s;
        if (q.profile == 0)
            s = q.amplitude / (1.0 + x * x);
        else if (q.profile == 1)
            s = q.amplitude * exp(-0.5 * x * x);
        else
            s = q.amplitude * x;
        if (q.white_sigma > 0.0) s += q.white_sigma * sr_normal(q.seed, st, (uint64_t)p);
        if (q.pink_sigma > 0.0 && q.pink_octaves > 0) {
            double acc = 0.0;
            for (int j = 0; j < q.pink_octaves; ++j) acc += sr_normal(q.seed, st + 1 + (uint64_t)j, (uint64_t)p >> j);
            s += pink_scale * acc;
        }
        if (jumps) {
            J += jv[k];
            s += J;
        }
        S[p * ns + a] = s;
    }
}

__global__ void __launch_bounds__(SR_THREADS) qa_sensor_gradient_kernel(const double *__restrict__ S, int64_t P, int ns,
                                                                        int64_t W, double *__restrict__ G)
{
    qa_pdl_wait();
    const int64_t e = (int64_t)blockIdx.x * SR_THREADS + threadIdx.x;  // element (p, a)
    if (e >= P * ns) return;
    const int64_t p = e / ns, ix = p % W;
    double g;
    if (W == 1)
        g = 0.0;
    else if (ix == 0)
        g = S[e + ns] - S[e];
    else if (ix == W - 1)
        g = S[e] - S[e - ns];
    else
        g = 0.5 * (S[e + ns] - S[e - ns]);
    G[e] = g;
}

}  // namespace

size_t qa_sensor_workspace_bytes_impl(int64_t P, int ns)
{
    const int64_t nchunk = (P + SR_CHUNK - 1) / SR_CHUNK;
    return (size_t)((nchunk > 0 ? nchunk : 1) * (int64_t)ns * 8 + 255) & ~(size_t)255;
}

cudaError_t qa_launch_sensor_response(const qa_sensor_params *params, int ns, const double *d_Vs, int64_t P, int64_t W,
                                      double *d_S, double *d_G, double *d_partial, cudaStream_t stream)
{
    SrPack pk;
    bool any_jumps = false;
    for (int a = 0; a < QA_MAXN; ++a) {
        pk.p[a] = params[a < ns ? a : 0];
        if (a < ns && params[a].jump_rate > 0.0 && params[a].jump_sigma > 0.0) any_jumps = true;
    }
    const int64_t nchunk = (P + SR_CHUNK - 1) / SR_CHUNK;
    const dim3 grid((unsigned)nchunk, (unsigned)ns);
    if (any_jumps) {
        qa_plan_add("qa_sensor_jump_partials_kernel");
        qa_sensor_jump_partials_kernel<<<grid, SR_THREADS, 0, stream>>>(pk, P, nchunk, d_partial);
        qa_timing_mark(stream);
        qa_plan_add("qa_sensor_jump_scan_kernel");
        qa_sensor_jump_scan_kernel<<<(unsigned)ns, SR_THREADS, 0, stream>>>(pk, nchunk, d_partial);
        qa_timing_mark(stream);
    }
    qa_plan_add("qa_sensor_signal_kernel");
    qa_sensor_signal_kernel<<<grid, SR_THREADS, 0, stream>>>(pk, d_Vs, P, ns, nchunk, d_partial, d_S);
    cudaError_t err = cudaGetLastError();
    if (err != cudaSuccess || !d_G) return err;
    qa_timing_mark(stream);
    qa_plan_add("qa_sensor_gradient_kernel");
    const int64_t blocks = (P * ns + SR_THREADS - 1) / SR_THREADS;
    return qa_launch_pdl(qa_sensor_gradient_kernel, dim3((unsigned)blocks), dim3(SR_THREADS), stream, d_S, P, ns, W, d_G);
}
