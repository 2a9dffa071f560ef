// gwi_whiten.cu -- whitening front end (PSD estimate of the strain, whitening with
// it, standard deviation normalised to one; parameters by reading A35).
//
// One segment of n raw samples -> whitened samples ready for gwi_stream_push / gwi_infer:
//   1. Welch estimate: frames of nper samples every nper/2, symmetric Hann window, P = mean |rfft(frame)|^2
//   2. P interpolated linearly to the n/2+1 frequencies of the segment
//   3. Y = rfft(x) / sqrt(P_interp), y = irfft(Y)
//   4. out = y / std(y)  (population standard deviation), written as float or __half
// The FFTs are plain library transforms (cuFFT: a batched R2C of the frames, one R2C and one C2R of the segment); the
// windowing, the periodogram mean, the interpolation + division, the statistics and the output scaling are kernels of
// this file.  cuFFT is loaded with dlopen on first use, so that libgwi.so itself has no link-time dependency on it:
// without the library gwi_whiten returns GWI_ERR_UNSUPPORTED and nothing else is affected.
#include <cufft.h>
#include <dlfcn.h>

#include <array>
#include <map>
#include <mutex>
#include <tuple>

#include <algorithm>

#include "gwi_internal.h"

namespace {

struct CufftApi {
    cufftResult (*Plan1d)(cufftHandle*, int, cufftType, int) = nullptr;
    cufftResult (*SetStream)(cufftHandle, cudaStream_t) = nullptr;
    cufftResult (*ExecR2C)(cufftHandle, cufftReal*, cufftComplex*) = nullptr;
    cufftResult (*ExecC2R)(cufftHandle, cufftComplex*, cufftReal*) = nullptr;
    cufftResult (*Destroy)(cufftHandle) = nullptr;
    bool ok = false;
};

CufftApi& cufft_api()
{
    static CufftApi api;
    static bool tried = false;
    if (tried) return api;
    tried = true;
    void* h = nullptr;
    for (const char* name : {"libcufft.so.11", "libcufft.so", "/usr/local/cuda/lib64/libcufft.so.11"}) {
        h = dlopen(name, RTLD_NOW | RTLD_LOCAL);
        if (h) break;
    }
    if (!h) return api;
    api.Plan1d = (decltype(api.Plan1d))dlsym(h, "cufftPlan1d");
    api.SetStream = (decltype(api.SetStream))dlsym(h, "cufftSetStream");
    api.ExecR2C = (decltype(api.ExecR2C))dlsym(h, "cufftExecR2C");
    api.ExecC2R = (decltype(api.ExecC2R))dlsym(h, "cufftExecC2R");
    api.Destroy = (decltype(api.Destroy))dlsym(h, "cufftDestroy");
    api.ok = api.Plan1d && api.SetStream && api.ExecR2C && api.ExecC2R && api.Destroy;
    return api;
}

// 1 / rms of the raw segment: raw strain is ~1e-21, whose squares underflow fp32; the whitened output does not depend
// on the input's scale, so everything is computed on x / rms(x)
__device__ __forceinline__ float raw_scale(const double* stats, int64_t n)
{
    const double ms = stats[1] / (double)n;
    return ms > 0.0 ? (float)(1.0 / sqrt(ms)) : 1.0f;
}

// win[i] = hann(i), once per call (the frames repeat it K times)
__global__ void k_window(int nper, float* __restrict__ win)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < nper) win[i] = 0.5f - 0.5f * cospif(2.0f * (float)i / (float)(nper - 1));
}

// frames[k][i] = scale * x[k * step + i] * hann(i); a block = 1024 samples of one frame, four per thread (the first
// version took a 64-bit division, the window's cosine and the fp64 scale per sample and was instruction-bound at 5 x its
// HBM time)
__global__ void k_frames(const float* __restrict__ x, int nper, int K, float* __restrict__ frames, const double* __restrict__ rs,
                         int64_t n, const float* __restrict__ win)
{
    __shared__ float s_scale;
    if (threadIdx.x == 0) s_scale = raw_scale(rs, n);
    __syncthreads();
    const float sc = s_scale;
    const unsigned bpf = (unsigned)(nper + 1023) / 1024;   // blocks per frame
    const int k = (int)(blockIdx.x / bpf), i0 = (int)((blockIdx.x % bpf) * blockDim.x + threadIdx.x) * 4;
    if (i0 >= nper) return;
    const float* xs = x + (int64_t)k * (nper / 2) + i0;
    float* fr = frames + (int64_t)k * nper + i0;
    if ((nper & 7) == 0 && (reinterpret_cast<uintptr_t>(x) & 15) == 0) {   // every frame starts on a 16-byte boundary
        const float4 v = *reinterpret_cast<const float4*>(xs), w = *reinterpret_cast<const float4*>(win + i0);
        *reinterpret_cast<float4*>(fr) = make_float4(v.x * sc * w.x, v.y * sc * w.y, v.z * sc * w.z, v.w * sc * w.w);
    } else {
        for (int e = 0; e < 4 && i0 + e < nper; e++) fr[e] = xs[e] * sc * win[i0 + e];
    }
}

// P[j] = mean over frames of |F[k][j]|^2, in two steps with a fixed summation order (a thread per bin walking all K frames
// kept 33 CTAs busy for 0.59 ms on a 4096 s segment: half of the whole call): blockIdx.y = y sums the frames y, y + PG_Y, ...
constexpr int PG_Y = 128;
__global__ void k_periodogram_part(const float2* __restrict__ F, int nf, int K, double* __restrict__ part)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= nf) return;
    double acc = 0.0;
#pragma unroll 4
    for (int k = blockIdx.y; k < K; k += PG_Y) {
        float2 v = F[(int64_t)k * nf + j];
        acc += (double)v.x * v.x + (double)v.y * v.y;
    }
    part[(int64_t)blockIdx.y * nf + j] = acc;
}
__global__ void k_periodogram_sum(const double* __restrict__ part, int nf, int K, float* __restrict__ P)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= nf) return;
    double acc = 0.0;
    for (int y = 0; y < PG_Y; y++) acc += part[(int64_t)y * nf + j];
    P[j] = (float)(acc / K);
}

// X[i] /= sqrt(P interpolated at i * nper / n); four consecutive bins per thread, the fp64 ratio nper / n once per thread
// (one fp64 division per bin made the pass instruction-bound)
__global__ void k_divide(float2* __restrict__ X, int64_t nx, int64_t n, int nper, const float* __restrict__ P,
                         const double* __restrict__ rs)
{
    const int64_t i0 = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) * 4;
    if (i0 >= nx) return;
    const double ratio = (double)nper / (double)n;
    const float sc = raw_scale(rs, n);
    auto factor = [&](int64_t i) {
        const double pos = (double)i * ratio;
        int j = (int)pos;
        if (j > nper / 2 - 1) j = nper / 2 - 1;
        const float frac = (float)(pos - j);
        const float p = P[j] * (1.0f - frac) + P[j + 1] * frac;
        return rsqrtf(fmaxf(p, 1e-30f)) * sc;
    };
    if (i0 + 3 < nx) {   // X is 256-byte aligned (workspace layout), i0 a multiple of 4
        float4* X4 = reinterpret_cast<float4*>(X + i0);
        float4 a = X4[0], b = X4[1];
        const float s0 = factor(i0), s1 = factor(i0 + 1), s2 = factor(i0 + 2), s3 = factor(i0 + 3);
        X4[0] = make_float4(a.x * s0, a.y * s0, a.z * s1, a.w * s1);
        X4[1] = make_float4(b.x * s2, b.y * s2, b.z * s3, b.w * s3);
    } else {
        for (int64_t i = i0; i < nx; i++) {
            const float s = factor(i);
            float2 v = X[i];
            X[i] = make_float2(v.x * s, v.y * s);
        }
    }
}

// stats[0] += sum y, stats[1] += sum y^2 (double)
__global__ void k_stats_y(const float* __restrict__ y, int64_t n, double* __restrict__ stats)
{
    __shared__ double s0[256], s1[256];
    double a = 0.0, b = 0.0;
    const int64_t tid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x, nth = (int64_t)gridDim.x * blockDim.x;
    int64_t done = 0;
    if ((reinterpret_cast<uintptr_t>(y) & 15) == 0) {   // 16-byte loads over the whole groups of four, the tail below
        const int64_t n4 = n >> 2;
#pragma unroll 4
        for (int64_t i = tid; i < n4; i += nth) {
            const float4 q = reinterpret_cast<const float4*>(y)[i];
            const double v0 = q.x, v1 = q.y, v2 = q.z, v3 = q.w;
            a += (v0 + v1) + (v2 + v3), b += (v0 * v0 + v1 * v1) + (v2 * v2 + v3 * v3);
        }
        done = n4 << 2;
    }
    for (int64_t i = done + tid; i < n; i += nth) {
        double v = y[i];
        a += v, b += v * v;
    }
    s0[threadIdx.x] = a, s1[threadIdx.x] = b;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) s0[threadIdx.x] += s0[threadIdx.x + o], s1[threadIdx.x] += s1[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        atomicAdd(&stats[0], s0[0]);
        atomicAdd(&stats[1], s1[0]);
    }
}

// eight consecutive outputs (i0 a multiple of 8) with vector stores where the caller's pointer allows it
__device__ __forceinline__ void store8(float* o, float a, float b, float c, float d, float e, float f, float g, float h)
{
    if ((reinterpret_cast<uintptr_t>(o) & 15) == 0) {
        *reinterpret_cast<float4*>(o) = make_float4(a, b, c, d), *reinterpret_cast<float4*>(o + 4) = make_float4(e, f, g, h);
    } else {
        o[0] = a, o[1] = b, o[2] = c, o[3] = d, o[4] = e, o[5] = f, o[6] = g, o[7] = h;
    }
}
__device__ __forceinline__ void store8(__half* o, float a, float b, float c, float d, float e, float f, float g, float h)
{
    if ((reinterpret_cast<uintptr_t>(o) & 15) == 0) {
        union { __half2 h2[4]; uint4 u; } pk;
        pk.h2[0] = __halves2half2((__half)a, (__half)b), pk.h2[1] = __halves2half2((__half)c, (__half)d);
        pk.h2[2] = __halves2half2((__half)e, (__half)f), pk.h2[3] = __halves2half2((__half)g, (__half)h);
        *reinterpret_cast<uint4*>(o) = pk.u;
    } else {
        o[0] = (__half)a, o[1] = (__half)b, o[2] = (__half)c, o[3] = (__half)d;
        o[4] = (__half)e, o[5] = (__half)f, o[6] = (__half)g, o[7] = (__half)h;
    }
}

template <typename OT>
__global__ void k_scale_out(const float* __restrict__ y, int64_t n, const double* __restrict__ stats, OT* __restrict__ out)
{
    // the fp64 scale once per thread, eight samples per thread
    const double mean = stats[0] / (double)n;
    const double var = stats[1] / (double)n - mean * mean;
    const float inv = (float)(1.0 / sqrt(var > 0.0 ? var : 1.0));
    const int64_t i0 = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) * 8;
    if (i0 + 7 < n) {
        const float4 a = *reinterpret_cast<const float4*>(y + i0), b = *reinterpret_cast<const float4*>(y + i0 + 4);
        store8(out + i0, a.x * inv, a.y * inv, a.z * inv, a.w * inv, b.x * inv, b.y * inv, b.z * inv, b.w * inv);
    } else {
        for (int64_t i = i0; i < n; i++) out[i] = (OT)(y[i] * inv);
    }
}

struct WsLayout {
    size_t frames, spec, P, X, y, stats, win, total;
    int K;
};
WsLayout ws_layout(int64_t n, int nper)
{
    WsLayout L;
    L.K = (int)((n - nper) / (nper / 2) + 1);
    size_t o = 0;
    auto take = [&](size_t b) { size_t at = o; o += (b + 255) & ~(size_t)255; return at; };
    L.frames = take(std::max((size_t)L.K * nper * 4, (size_t)PG_Y * (nper / 2 + 1) * 8));   // frames, then the periodogram's partial sums
    L.spec = take((size_t)L.K * (nper / 2 + 1) * 8);
    L.P = take((size_t)(nper / 2 + 2) * 4);
    L.X = take((size_t)(n / 2 + 1) * 8);
    L.y = take((size_t)n * 4);
    L.stats = take(32);
    L.win = take((size_t)nper * 4);
    L.total = o;
    return L;
}

} // namespace

extern "C" size_t gwi_whiten_workspace_bytes(int64_t n, int32_t nper)
{
    if (n < 4 || nper < 4 || (n & 1) || (nper & 1) || nper > n) return 0;
    return ws_layout(n, nper).total;
}

extern "C" gwi_status gwi_whiten(const float* d_raw, int64_t n, int32_t nper, void* d_out, int out_is_half, void* d_workspace,
                                 size_t workspace_bytes, void* cuda_stream)
{
    if (!d_raw || !d_out || !d_workspace || n < 4 || nper < 4 || (n & 1) || (nper & 1) || nper > n || n > (1LL << 30) ||
        ((uintptr_t)d_workspace & 255)) {
        gwi_set_error("gwi_whiten: bad argument (n and nper even, 4 <= nper <= n <= 2^30)");
        return GWI_ERR_ARG;
    }
    WsLayout L = ws_layout(n, nper);
    if (workspace_bytes < L.total) {
        gwi_set_error("gwi_whiten: workspace %zu < %zu bytes", workspace_bytes, L.total);
        return GWI_ERR_NOMEM;
    }
    CufftApi& fft = cufft_api();
    if (!fft.ok) {
        gwi_set_error("gwi_whiten: cuFFT (libcufft.so.11) could not be loaded");
        return GWI_ERR_UNSUPPORTED;
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    char* ws = (char*)d_workspace;
    float* frames = (float*)(ws + L.frames);
    float2* spec = (float2*)(ws + L.spec);
    float* P = (float*)(ws + L.P);
    float2* X = (float2*)(ws + L.X);
    float* y = (float*)(ws + L.y);
    double* stats = (double*)(ws + L.stats);
    float* win = (float*)(ws + L.win);
    const int K = L.K, nf = nper / 2 + 1;
    // The three plans (and the work areas they own) are cached per (device, n, nper, stream) for the life of the process,
    // so the call only enqueues work and returns: segment after segment of the same length re-uses them.
    int device = 0;
    GWI_CUDA_CHECK(cudaGetDevice(&device));
    cufftHandle pf = 0, pr = 0, pi = 0;
    {
        static std::mutex mu;
        static std::map<std::tuple<int, int64_t, int, void*>, std::array<cufftHandle, 3>> cache;
        std::lock_guard<std::mutex> lock(mu);
        auto key = std::make_tuple(device, n, (int)nper, cuda_stream);
        auto it = cache.find(key);
        if (it == cache.end()) {
            auto fail = [&](const char* what) {
                if (pf) fft.Destroy(pf);
                if (pr) fft.Destroy(pr);
                if (pi) fft.Destroy(pi);
                gwi_set_error("gwi_whiten: cuFFT %s failed", what);
                return GWI_ERR_CUDA;
            };
            if (fft.Plan1d(&pf, nper, CUFFT_R2C, K) != CUFFT_SUCCESS) return fail("plan (frames)");
            if (fft.Plan1d(&pr, (int)n, CUFFT_R2C, 1) != CUFFT_SUCCESS) return fail("plan (forward)");
            if (fft.Plan1d(&pi, (int)n, CUFFT_C2R, 1) != CUFFT_SUCCESS) return fail("plan (inverse)");
            fft.SetStream(pf, st), fft.SetStream(pr, st), fft.SetStream(pi, st);
            cache[key] = {pf, pr, pi};
        } else {
            pf = it->second[0], pr = it->second[1], pi = it->second[2];
        }
    }
    auto fail = [&](const char* what) {
        gwi_set_error("gwi_whiten: cuFFT %s failed", what);
        return GWI_ERR_CUDA;
    };
    cudaMemsetAsync(stats, 0, 32, st);
    k_stats_y<<<592, 256, 0, st>>>(d_raw, n, stats + 2);          // stats[2..3]: sum and sum of squares of the raw input
    k_window<<<(nper + 255) / 256, 256, 0, st>>>(nper, win);
    k_frames<<<(unsigned)((int64_t)K * ((nper + 1023) / 1024)), 256, 0, st>>>(d_raw, nper, K, frames, stats + 2, n, win);
    if (fft.ExecR2C(pf, frames, (cufftComplex*)spec) != CUFFT_SUCCESS) return fail("exec (frames)");
    // (the time-domain frames are dead once transformed: their buffer holds the partial sums, PG_Y x nf doubles)
    k_periodogram_part<<<dim3((nf + 127) / 128, PG_Y), 128, 0, st>>>(spec, nf, K, (double*)frames);
    k_periodogram_sum<<<(nf + 127) / 128, 128, 0, st>>>((const double*)frames, nf, K, P);
    // cuFFT R2C is out of place here: the raw input stays untouched
    // (an input off a 16-byte boundary goes through y first: the transform wants its vector alignment)
    const float* fwd_in = d_raw;
    if ((uintptr_t)d_raw & 15) {
        GWI_CUDA_CHECK(cudaMemcpyAsync(y, d_raw, (size_t)n * 4, cudaMemcpyDeviceToDevice, st));
        fwd_in = y;
    }
    if (fft.ExecR2C(pr, const_cast<float*>(fwd_in), (cufftComplex*)X) != CUFFT_SUCCESS) return fail("exec (forward)");
    k_divide<<<(unsigned)((n / 2 + 1 + 1023) / 1024), 256, 0, st>>>(X, n / 2 + 1, n, nper, P, stats + 2);
    if (fft.ExecC2R(pi, (cufftComplex*)X, y) != CUFFT_SUCCESS) return fail("exec (inverse)");
    k_stats_y<<<592, 256, 0, st>>>(y, n, stats);
    if (out_is_half) k_scale_out<__half><<<(unsigned)((n + 2047) / 2048), 256, 0, st>>>(y, n, stats, (__half*)d_out);
    else k_scale_out<float><<<(unsigned)((n + 2047) / 2048), 256, 0, st>>>(y, n, stats, (float*)d_out);
    gwi_count_launch(8);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) {
        gwi_set_error("gwi_whiten: %s", cudaGetErrorString(e));
        return GWI_ERR_CUDA;
    }
    return GWI_OK;
}
