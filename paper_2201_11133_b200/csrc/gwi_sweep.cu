// gwi_sweep.cu -- trigger counts at MANY thresholds in one pass over the probabilities (gwi_threshold_sweep).
//
// The paper's ROC curve sweeps the height threshold of its peak finder between 0 and 0.9998 with the width kept at
// >= 0.5 s; its post-processing of the stored network output was the part that did not scale
// (PAPER.md:110-112).  With the trigger rule of this library (readings A19-A21: maximal runs of pbar > theta of at
// least L_min samples) the count at every threshold follows from ONE sliding-window minimum:
//     m[t] = min(pbar[t - L_min + 1 .. t])            (t >= L_min - 1)
//     a run of >= L_min samples above theta contains t  <=>  m[t] > theta,
// and distinct qualifying runs give distinct maximal runs of {m > theta}, so
//     count(theta) = number of rising edges of (m[t] > theta)  (a window at t = L_min - 1 above theta counts as one).
// For sorted thresholds an edge from m[t-1] to m[t] > m[t-1] raises exactly the thresholds theta_j with
// m[t-1] <= theta_j < m[t]: a range, recorded in a difference array and prefix-summed at the end.
//
// k_sweep / k_sweep_vh: each CTA loads TT + L_min samples of the ensemble mean (fixed fp32 expression, as in
// gwi_post.cu) into shared memory, builds the window minimum (k_sweep: by doubling, min over 2^k then two overlapping
// 2^k windows; k_sweep_vh: prefix / suffix minima per block of L_min), and scans its outputs for rising edges.
// HBM-bound by design: 4 M bytes per sample, read (1 + L_min / TT) times.
#include "gwi_internal.h"

namespace {

constexpr int SW_THREADS = 512;
constexpr int SW_MAXK = 1024;

struct SwPtrs {
    const float* p[GWI_MAX_MODELS];
};

__global__ void __launch_bounds__(SW_THREADS) k_sweep(SwPtrs P, int M, int64_t N, int L, int TT, const float* __restrict__ thr, int K,
                                                      int* __restrict__ diff)
{
    extern __shared__ float sm[];
    float* a = sm;                       // [TT + L]: pbar over [t_lo - L, t_hi), then in-place window minima
    float* b = sm + (TT + L);            // ping-pong buffer
    float* th = b + (TT + L);            // [K]
    const int64_t t_lo = (int64_t)blockIdx.x * TT + (L - 1);   // outputs t in [t_lo, t_hi), plus m[t_lo - 1] for the edge
    if (t_lo >= N) return;
    const int64_t t_hi = min(t_lo + TT, N);
    const int64_t base = t_lo - L;                               // sample index of a[0] (may be -1 for the first CTA)
    const int len = (int)(t_hi - base);
    const float fM = (float)M;
    for (int i = threadIdx.x; i < K; i += SW_THREADS) th[i] = thr[i];
#pragma unroll 4
    for (int i = threadIdx.x; i < len; i += SW_THREADS) {
        int64_t t = base + i;
        float v = INFINITY;                                      // the element before the stream never lowers a minimum
        if (t >= 0) {
            float s = P.p[0][t];
            for (int j = 1; j < M; j++) s = __fadd_rn(s, P.p[j][t]);
            v = __fdiv_rn(s, fM);
        }
        a[i] = v;
    }
    __syncthreads();
    // doubling: after step k, cur[i] = min over [i, i + 2^k)
    float *cur = a, *nxt = b;
    int w = 1;
    while (2 * w <= L) {
        for (int i = threadIdx.x; i + 2 * w <= len; i += SW_THREADS) nxt[i] = fminf(cur[i], cur[i + w]);
        __syncthreads();
        float* tmp = cur;
        cur = nxt, nxt = tmp;
        w *= 2;
    }
    // window of length L ending at sample base + e:  min(cur[e - L + 1], cur[e - w + 1])
    auto wmin = [&](int e) { return fminf(cur[e - L + 1], cur[e - w + 1]); };
    auto idx = [&](float v) {   // number of thresholds strictly below v
        int lo = 0, hi = K;
        while (lo < hi) {
            int mid = (lo + hi) >> 1;
            if (th[mid] < v) lo = mid + 1;
            else hi = mid;
        }
        return lo;
    };
    for (int o = threadIdx.x; o < (int)(t_hi - t_lo); o += SW_THREADS) {
        const int e = L + o;                                     // a-index of output t = t_lo + o
        const float cur_m = wmin(e);
        const bool first = !(t_lo + o > L - 1);                  // the very first window has no predecessor
        const float prev_m = first ? -INFINITY : wmin(e - 1);
        if (!(cur_m > prev_m)) continue;                         // only a rising minimum can raise a threshold
        const int i0 = first ? 0 : idx(prev_m);
        const int i1 = idx(cur_m);
        if (i1 > i0) {
            atomicAdd(&diff[i0], 1);
            atomicAdd(&diff[i1], -1);
        }
    }
}

// van Herk / Gil-Werman form for long windows: the tile is cut into blocks of L samples; G = prefix minimum inside each
// block, H = suffix minimum inside each block; the window [e - L + 1, e] spans at most two blocks, so
// m = min(H[e - L + 1], G[e]).  One warp per (block, direction): every lane scans its own contiguous chunk twice
// (chunk minimum, warp scan of the 32 chunk minima, then the running minimum).  The arrays are padded by one word per
// 32 so that the lanes' strided chunk walks spread over the banks.
__device__ __forceinline__ int padi(int j) { return j + (j >> 5); }

__global__ void __launch_bounds__(SW_THREADS) k_sweep_vh(SwPtrs P, int M, int64_t N, int L, int TT, const float* __restrict__ thr, int K,
                                                         int* __restrict__ diff, int vec)
{
    extern __shared__ float sm[];
    constexpr int OFF = 3;               // a-index 0 is sample blockIdx * TT - 4: 16-byte aligned tiles when TT % 4 == 0
    const int cap = padi(TT + L + OFF) + 1;
    float* G = sm;
    float* H = sm + cap;
    float* th = H + cap;
    const int64_t t_lo = (int64_t)blockIdx.x * TT + (L - 1);
    if (t_lo >= N) return;
    const int64_t t_hi = min(t_lo + TT, N);
    const int64_t base = t_lo - L - OFF;                         // sample index of a-index 0
    const int len = (int)(t_hi - base);
    const float fM = (float)M;
    for (int i = threadIdx.x; i < K; i += SW_THREADS) th[i] = thr[i];
    if (vec) {
        // four samples per thread and load instruction (all pointers 16-byte aligned, TT % 4 == 0)
        int i4 = threadIdx.x;
        if (base >= 0 && base + len + 3 < N && M == 4) {
            // interior tile of a 4-model ensemble: no bounds, three iterations of loads (12 x 16 bytes per thread) in flight
            const float inv = 0.25f;                              // s * 0.25f is the correctly rounded s / 4
#pragma unroll 3
            for (; 4 * i4 + 3 < len; i4 += SW_THREADS) {
                const int64_t t = base + 4 * i4;
                float4 s = __ldg(reinterpret_cast<const float4*>(P.p[0] + t));
                const float4 q1 = __ldg(reinterpret_cast<const float4*>(P.p[1] + t));
                const float4 q2 = __ldg(reinterpret_cast<const float4*>(P.p[2] + t));
                const float4 q3 = __ldg(reinterpret_cast<const float4*>(P.p[3] + t));
                s.x = __fadd_rn(__fadd_rn(__fadd_rn(s.x, q1.x), q2.x), q3.x), s.y = __fadd_rn(__fadd_rn(__fadd_rn(s.y, q1.y), q2.y), q3.y);
                s.z = __fadd_rn(__fadd_rn(__fadd_rn(s.z, q1.z), q2.z), q3.z), s.w = __fadd_rn(__fadd_rn(__fadd_rn(s.w, q1.w), q2.w), q3.w);
                const int p0 = padi(4 * i4);
                G[p0] = H[p0] = __fmul_rn(s.x, inv), G[p0 + 1] = H[p0 + 1] = __fmul_rn(s.y, inv);
                G[p0 + 2] = H[p0 + 2] = __fmul_rn(s.z, inv), G[p0 + 3] = H[p0 + 3] = __fmul_rn(s.w, inv);
            }
        }
        for (; 4 * i4 < len; i4 += SW_THREADS) {
            const int64_t t = base + 4 * i4;
            float v[4] = {INFINITY, INFINITY, INFINITY, INFINITY};
            if (t >= 0 && t + 3 < N) {
                float4 s = *reinterpret_cast<const float4*>(P.p[0] + t);
                for (int j = 1; j < M; j++) {
                    float4 q = *reinterpret_cast<const float4*>(P.p[j] + t);
                    s.x = __fadd_rn(s.x, q.x), s.y = __fadd_rn(s.y, q.y), s.z = __fadd_rn(s.z, q.z), s.w = __fadd_rn(s.w, q.w);
                }
                v[0] = __fdiv_rn(s.x, fM), v[1] = __fdiv_rn(s.y, fM), v[2] = __fdiv_rn(s.z, fM), v[3] = __fdiv_rn(s.w, fM);
            } else {
                for (int e = 0; e < 4; e++)
                    if (t + e >= 0 && t + e < N) {
                        float s = P.p[0][t + e];
                        for (int j = 1; j < M; j++) s = __fadd_rn(s, P.p[j][t + e]);
                        v[e] = __fdiv_rn(s, fM);
                    }
            }
            for (int e = 0; e < 4; e++)
                if (4 * i4 + e < len) G[padi(4 * i4 + e)] = v[e], H[padi(4 * i4 + e)] = v[e];
        }
    } else {
#pragma unroll 4
        for (int i = threadIdx.x; i < len; i += SW_THREADS) {
            int64_t t = base + i;
            float v = INFINITY;
            if (t >= 0) {
                float s = P.p[0][t];
                for (int j = 1; j < M; j++) s = __fadd_rn(s, P.p[j][t]);
                v = __fdiv_rn(s, fM);
            }
            G[padi(i)] = v;
            H[padi(i)] = v;
        }
    }
    __syncthreads();
    {
        const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
        const int nbk = (len - OFF + L - 1) / L, C = ((L + 31) / 32) | 1;   // odd chunk length: the lanes' walks fall on different banks
        for (int task = warp; task < 2 * nbk; task += SW_THREADS / 32) {
            const int q = task >> 1, back = task & 1;
            const int b0 = OFF + q * L, b1 = min(b0 + L, len);         // block [b0, b1)
            const int c0 = min(b0 + lane * C, b1), c1 = min(c0 + C, b1);   // this lane's chunk [c0, c1)
            float* A = back ? H : G;
            float tot = INFINITY;
            for (int j = c0; j < c1; j++) tot = fminf(tot, A[padi(j)]);
            // exclusive scan of the chunk minima over the lanes (forward: lanes below, backward: lanes above)
            float inc = tot;
            for (int o = 1; o < 32; o <<= 1) {
                float v = back ? __shfl_down_sync(0xffffffffu, inc, o) : __shfl_up_sync(0xffffffffu, inc, o);
                if (back ? (lane + o < 32) : (lane >= o)) inc = fminf(inc, v);
            }
            float carry = back ? __shfl_down_sync(0xffffffffu, inc, 1) : __shfl_up_sync(0xffffffffu, inc, 1);
            if (back ? lane == 31 : lane == 0) carry = INFINITY;
            float run = carry;
            if (!back) {
                for (int j = c0; j < c1; j++) {
                    run = fminf(run, A[padi(j)]);
                    A[padi(j)] = run;
                }
            } else {
                for (int j = c1 - 1; j >= c0; j--) {
                    run = fminf(run, A[padi(j)]);
                    A[padi(j)] = run;
                }
            }
        }
    }
    __syncthreads();
    auto wmin = [&](int e) { return fminf(H[padi(e - L + 1)], G[padi(e)]); };
    auto idx = [&](float v) {
        int lo = 0, hi = K;
        while (lo < hi) {
            int mid = (lo + hi) >> 1;
            if (th[mid] < v) lo = mid + 1;
            else hi = mid;
        }
        return lo;
    };
    for (int o = threadIdx.x; o < (int)(t_hi - t_lo); o += SW_THREADS) {
        const int e = OFF + L + o;
        const float cur_m = wmin(e);
        const bool first = !(t_lo + o > L - 1);                  // the very first window has no predecessor
        const float prev_m = first ? -INFINITY : wmin(e - 1);
        if (!(cur_m > prev_m)) continue;                         // only a rising minimum can raise a threshold
        const int i0 = first ? 0 : idx(prev_m);
        const int i1 = idx(cur_m);
        if (i1 > i0) {
            atomicAdd(&diff[i0], 1);
            atomicAdd(&diff[i1], -1);
        }
    }
}

__global__ void k_sweep_scan(const int* __restrict__ diff, int K, int64_t* __restrict__ counts)
{
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    int64_t run = 0;
    for (int j = 0; j < K; j++) {
        run += diff[j];
        counts[j] = run;
    }
}

} // namespace

extern "C" size_t gwi_sweep_workspace_bytes(int32_t n_thresholds) { return n_thresholds < 1 ? 0 : ((size_t)(n_thresholds + 1) * 4 + 255) & ~(size_t)255; }

extern "C" gwi_status gwi_threshold_sweep(const float* const* d_prob, int32_t n_models, int64_t N, const float* d_thresholds,
                                          int32_t n_thresholds, int64_t min_len, int64_t* d_counts, void* d_workspace,
                                          size_t workspace_bytes, void* cuda_stream)
{
    if (!d_prob || n_models < 1 || n_models > GWI_MAX_MODELS || N < 1 || !d_thresholds || n_thresholds < 1 ||
        n_thresholds > SW_MAXK || min_len < 1 || !d_counts || !d_workspace || ((uintptr_t)d_workspace & 255)) {
        gwi_set_error("gwi_threshold_sweep: bad argument (1 <= n_thresholds <= %d)", SW_MAXK);
        return GWI_ERR_ARG;
    }
    if (workspace_bytes < gwi_sweep_workspace_bytes(n_thresholds)) {
        gwi_set_error("gwi_threshold_sweep: workspace too small");
        return GWI_ERR_NOMEM;
    }
    if (min_len > 16384) {
        gwi_set_error("gwi_threshold_sweep: min_len %lld > 16384 is not covered by the shared-memory window", (long long)min_len);
        return GWI_ERR_UNSUPPORTED;
    }
    SwPtrs P;
    for (int j = 0; j < GWI_MAX_MODELS; j++) P.p[j] = j < n_models ? d_prob[j] : nullptr;
    for (int j = 0; j < n_models; j++)
        if (!d_prob[j]) {
            gwi_set_error("gwi_threshold_sweep: d_prob[%d] is null", j);
            return GWI_ERR_ARG;
        }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int* diff = (int*)d_workspace;
    GWI_CUDA_CHECK(cudaMemsetAsync(diff, 0, (size_t)(n_thresholds + 1) * 4, st));
    const int L = (int)min_len;
    if (N >= L) {
        // 2 (TT + L) floats + thresholds: two CTAs per SM (2 x ~108 KB) when the window allows, else one
        const int budget = L <= 6144 ? 13000 : 26000;
        int64_t nout = N - (L - 1);
        if (L >= 256 && L <= 8192) {
            // long windows: prefix / suffix minima per block of L, TT a multiple of L (>= L for these L)
            const int TT = (budget - L) / L * L;
            size_t smem = (size_t)(2 * ((TT + L + 3) + ((TT + L + 3) >> 5) + 1) + n_thresholds) * sizeof(float);
            int vec = (TT & 3) == 0;
            for (int j = 0; j < n_models; j++) vec = vec && (((uintptr_t)d_prob[j] & 15) == 0);
            GWI_CUDA_CHECK(cudaFuncSetAttribute(k_sweep_vh, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            unsigned grid = (unsigned)((nout + TT - 1) / TT);
            k_sweep_vh<<<grid, SW_THREADS, smem, st>>>(P, n_models, N, L, TT, d_thresholds, n_thresholds, diff, vec);
        } else {
            const int TT = (budget - L) / 256 * 256;
            size_t smem = (size_t)(2 * (TT + L) + n_thresholds) * sizeof(float);
            GWI_CUDA_CHECK(cudaFuncSetAttribute(k_sweep, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            unsigned grid = (unsigned)((nout + TT - 1) / TT);
            k_sweep<<<grid, SW_THREADS, smem, st>>>(P, n_models, N, L, TT, d_thresholds, n_thresholds, diff);
        }
        gwi_count_launch(1);
    }
    k_sweep_scan<<<1, 32, 0, st>>>(diff, n_thresholds, d_counts);
    gwi_count_launch(1);
    GWI_CUDA_CHECK(cudaGetLastError());
    return GWI_OK;
}
