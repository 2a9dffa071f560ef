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
// k_sweep: each CTA loads TT + L_min - 1 samples of the ensemble mean (fixed fp32 expression, as in gwi_post.cu) into
// shared memory, builds the window minimum by doubling (min over 2^k, then two overlapping 2^k windows), and scans
// its outputs for rising edges.  HBM-bound: 4 M bytes per sample, read (1 + (L_min - 1) / TT) times.
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
        int i0 = 0;
        if (t_lo + o > L - 1) i0 = idx(wmin(e - 1));             // the very first window has no predecessor
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
        const int TT = ((L <= 6144 ? 13500 : 27000) - L) / 256 * 256;
        size_t smem = (size_t)(2 * (TT + L) + n_thresholds) * sizeof(float);
        GWI_CUDA_CHECK(cudaFuncSetAttribute(k_sweep, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        int64_t nout = N - (L - 1);
        unsigned grid = (unsigned)((nout + TT - 1) / TT);
        k_sweep<<<grid, SW_THREADS, smem, st>>>(P, n_models, N, L, TT, d_thresholds, n_thresholds, diff);
        gwi_count_launch(1);
    }
    k_sweep_scan<<<1, 32, 0, st>>>(diff, n_thresholds, d_counts);
    gwi_count_launch(1);
    GWI_CUDA_CHECK(cudaGetLastError());
    return GWI_OK;
}
