// gwi_peaks.cu -- gwi_find_peaks: the paper's post-processing rule as stated, SciPy's find_peaks(x, height, width) on a
// model's per-timestep probabilities, on the GPU.
//
// Definition (scipy.signal.find_peaks with height and width; the oracle restates it and is pinned against SciPy):
//   1. local maxima with flat tops (a flat top counts once, at the floor of its middle; the array ends are never peaks)
//   2. x[p] >= height
//   3. prominence = x[p] - max(min over the stretch to the left up to the nearest higher sample, same to the right)
//   4. width at half prominence: crossings of level = x[p] - prominence / 2, linearly interpolated; width >= min_width
//
// The nearest-higher searches and the level crossings can reach across the whole array (the paper ran this offline over
// ~500 GB of stored outputs per month), so they run on two pyramids of 32-ary block maxima / minima:
// a search walks at most 32 entries per level.  The array is read ONCE, coalesced: the pass that builds level 1 of the
// pyramids (one warp per 32 samples, warp-wide integer max / min on order-preserving keys) also marks, one bit per
// sample, where a (flat-topped) local maximum that satisfies the height condition starts; the peak pass then walks that
// bit mask (3 % of the array) and evaluates steps 3 and 4 for the marked samples only.  Decisions are taken on the fp32 samples exactly
// as the oracle takes them in fp64 (differences and half-prominences of fp32 numbers are exact in fp64), so the peak
// list is the oracle's; accepted peaks are appended with an atomic counter and sorted by position afterwards.
#include <cfloat>
#include <climits>

#include "gwi_internal.h"

namespace {

constexpr int PK_MAX_LEVELS = 6;   // 32^6 > 10^9 samples

struct Pyr {
    const float* mx[PK_MAX_LEVELS + 1];   // mx[0] = mn[0] = x; level k: maxima / minima of 32^k samples
    const float* mn[PK_MAX_LEVELS + 1];
    int64_t size[PK_MAX_LEVELS + 1];
    int top;                              // highest level (size[top] <= 32 or PK_MAX_LEVELS)
};

__global__ void k_pyr_level(const float* __restrict__ inmx, const float* __restrict__ inmn, int64_t nin, float* __restrict__ outmx,
                            float* __restrict__ outmn, int64_t nout)
{
    // one warp per output: 32 coalesced entries of each input array, warp-wide max / min on order-preserving keys
    const int64_t o = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    if (o >= nout) return;                                       // warp-uniform
    const int lane = threadIdx.x & 31;
    const int64_t i = o * 32 + lane;
    const int b = __float_as_int(i < nin ? inmx[i] : -FLT_MAX), c = __float_as_int(i < nin ? inmn[i] : FLT_MAX);
    const int kmax = __reduce_max_sync(0xffffffffu, b >= 0 ? b : b ^ 0x7fffffff);
    const int kmin = __reduce_min_sync(0xffffffffu, c >= 0 ? c : c ^ 0x7fffffff);
    if (lane == 0) outmx[o] = __int_as_float(kmax >= 0 ? kmax : kmax ^ 0x7fffffff), outmn[o] = __int_as_float(kmin >= 0 ? kmin : kmin ^ 0x7fffffff);
}

// Leftward search from `pos` (inclusive): the largest j <= pos whose sample satisfies pred, -1 if none.  BLK(l, i) must be
// true iff block i of level l MAY contain such a sample (exact at level 0).  The siblings of a 32-block are tested with
// independent loads in flight (all at once above level 0, eight then the rest at level 0): a search that climbs several
// levels is a chain of one or two load latencies per level instead of ~31.
template <class BLK>
__device__ __forceinline__ int64_t search_left(const Pyr& P, int64_t pos, BLK blk)
{
    int l = 0;
    int64_t i = pos;
    while (i >= 0) {
        const int64_t e = i & ~(int64_t)31;                   // first sibling of the 32-block
        int64_t found = -1;
        if (l == 0) {
            // the first eight (on noise-like data the answer is among them), then the other siblings at once: the samples
            // themselves come from DRAM, a microsecond per dependent step
            uint32_t m = 0;
#pragma unroll
            for (int u = 0; u < 8; u++) m |= (uint32_t)((i - u >= e) && blk(l, i - u)) << u;
            if (!m && i - 8 >= e) {
#pragma unroll
                for (int u = 8; u < 32; u++) m |= (uint32_t)((i - u >= e) && blk(l, i - u)) << u;
            }
            if (m) found = i - (__ffs(m) - 1);                // the largest index wins
        } else {                                              // climbing: all siblings at once (one load latency per level)
            uint32_t m = 0;
#pragma unroll
            for (int u = 0; u < 32; u++) m |= (uint32_t)((i - u >= e) && blk(l, i - u)) << u;
            if (m) found = i - (__ffs(m) - 1);
        }
        if (found >= 0) {
            if (l == 0) return found;
            l--;
            i = min(found * 32 + 31, P.size[l] - 1);          // rightmost child
            continue;
        }
        if (l < P.top) i = (e >> 5) - 1, l++;                 // the parent's left part is done: previous parent-level block
        else i = e - 1;
    }
    return -1;
}
// Rightward search from `pos` (inclusive): the smallest j >= pos whose sample satisfies pred, N if none.
template <class BLK>
__device__ __forceinline__ int64_t search_right(const Pyr& P, int64_t pos, BLK blk)
{
    int l = 0;
    int64_t i = pos;
    while (i < P.size[l]) {
        const int64_t e = min(i | 31, P.size[l] - 1);         // last sibling of the 32-block (or of the level)
        int64_t found = -1;
        if (l == 0) {
            uint32_t m = 0;
#pragma unroll
            for (int u = 0; u < 8; u++) m |= (uint32_t)((i + u <= e) && blk(l, i + u)) << u;
            if (!m && i + 8 <= e) {
#pragma unroll
                for (int u = 8; u < 32; u++) m |= (uint32_t)((i + u <= e) && blk(l, i + u)) << u;
            }
            if (m) found = i + (__ffs(m) - 1);                // the smallest index wins
        } else {
            uint32_t m = 0;
#pragma unroll
            for (int u = 0; u < 32; u++) m |= (uint32_t)((i + u <= e) && blk(l, i + u)) << u;
            if (m) found = i + (__ffs(m) - 1);
        }
        if (found >= 0) {
            if (l == 0) return found;
            l--;
            i = found * 32;                                   // leftmost child
            continue;
        }
        if (l < P.top) i = (e >> 5) + 1, l++;
        else i = e + 1;
    }
    return P.size[0];
}
// minimum of x[a..b] (inclusive, a <= b)
__device__ __forceinline__ float range_min(const Pyr& P, int64_t a, int64_t b)
{
    float m = FLT_MAX;
    int l = 0;
    auto span = [&](int64_t lo, int64_t hi) {                 // min over entries lo..hi of level l, 32 loads in flight
        for (int64_t c = lo; c <= hi; c += 32) {
            float t[32];
#pragma unroll
            for (int u = 0; u < 32; u++) t[u] = c + u <= hi ? P.mn[l][c + u] : FLT_MAX;
#pragma unroll
            for (int u = 0; u < 32; u++) m = fminf(m, t[u]);
        }
    };
    while (a <= b) {
        if (l == P.top || (a >> 5) == (b >> 5)) {             // one block, or no level above: the entries themselves
            span(a, b);
            break;
        }
        if (a & 31) {
            span(a, a | 31);
            a = (a | 31) + 1;
        }
        if ((b & 31) != 31) {
            span(b & ~(int64_t)31, b);
            b = (b & ~(int64_t)31) - 1;
        }
        if (a > b) break;
        a >>= 5, b >>= 5, l++;
    }
    return m;
}

// order-preserving map of the non-NaN floats onto the signed integers (and back): warp-wide max / min run on REDUX
__device__ __forceinline__ int f2key(float f)
{
    const int b = __float_as_int(f);
    return b >= 0 ? b : b ^ 0x7fffffff;
}
__device__ __forceinline__ float key2f(int k) { return __int_as_float(k >= 0 ? k : k ^ 0x7fffffff); }

// One pass over x: level 1 of both pyramids (group g = samples [32 g, 32 g + 32)) and the candidate word of the group:
// bit l set iff sample i = 32 g + l starts a rise (x[i-1] < x[i]), reaches the height, and 1 <= i < N - 1.
__global__ void __launch_bounds__(256) k_level1_cand(const float* __restrict__ x, int64_t N, float hmin, float* __restrict__ mx1,
                                                     float* __restrict__ mn1, int64_t n1, uint32_t* __restrict__ cand)
{
    const int lane = threadIdx.x & 31;
    const int64_t warp0 = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarp = ((int64_t)gridDim.x * blockDim.x) >> 5;
    for (int64_t g0 = warp0 * 4; g0 < n1; g0 += nwarp * 4) {
        float v[4], pv[4];
#pragma unroll
        for (int u = 0; u < 4; u++) {                              // four independent 128-byte loads in flight per warp
            const int64_t i = (g0 + u) * 32 + lane;
            v[u] = i < N ? __ldg(x + i) : 0.f;
            pv[u] = (lane == 0 && i >= 1 && i < N) ? __ldg(x + i - 1) : 0.f;
        }
#pragma unroll
        for (int u = 0; u < 4; u++) {
            const int64_t g = g0 + u, i = g * 32 + lane;
            if (g >= n1) break;                                     // warp-uniform
            const bool in = i < N;
            float prev = __shfl_up_sync(0xffffffffu, v[u], 1);
            if (lane == 0) prev = pv[u];
            const bool c = in && i >= 1 && i < N - 1 && prev < v[u] && !(v[u] < hmin);
            const uint32_t w = __ballot_sync(0xffffffffu, c);
            const int kmax = __reduce_max_sync(0xffffffffu, in ? f2key(v[u]) : INT_MIN);
            const int kmin = __reduce_min_sync(0xffffffffu, in ? f2key(v[u]) : INT_MAX);
            if (lane == 0) {
                cand[g] = w;
                if (mx1) mx1[g] = key2f(kmax), mn1[g] = key2f(kmin);
            }
        }
    }
}

// The same for a 16-byte aligned x, without cross-lane reductions (REDUX is what bounds the kernel above: 150 us for
// 2^26 samples): a CTA stages a tile of 256 groups (8192 samples, coalesced 16-byte loads) in shared memory, groups 33
// words apart, and thread g then walks its own group (bank = (g + k) mod 32: conflict-free both ways).
constexpr int L1_GROUPS = 256, L1_PITCH = 33;
__global__ void __launch_bounds__(L1_GROUPS) k_level1_cand_v4(const float* __restrict__ x, int64_t N, float hmin, float* __restrict__ mx1,
                                                              float* __restrict__ mn1, int64_t n1, uint32_t* __restrict__ cand)
{
    __shared__ float sm[L1_GROUPS * L1_PITCH];
    const int64_t base = (int64_t)blockIdx.x * (L1_GROUPS * 32);   // first sample of the tile
    const int tid = threadIdx.x;
    const bool interior = base >= 1 && base + L1_GROUPS * 32 < N - 1;   // no sample of the tile is a boundary case
#pragma unroll
    for (int u = 0; u < 8; u++) {
        const int f = (u * L1_GROUPS + tid) * 4;                   // float index inside the tile
        const int64_t i = base + f;
        float4 v;
        if (interior || i + 3 < N) {
            v = __ldg(reinterpret_cast<const float4*>(x + i));
        } else {
            v.x = i < N ? __ldg(x + i) : 0.f, v.y = i + 1 < N ? __ldg(x + i + 1) : 0.f;
            v.z = i + 2 < N ? __ldg(x + i + 2) : 0.f, v.w = 0.f;
        }
        float* d = sm + (f >> 5) * L1_PITCH + (f & 31);
        d[0] = v.x, d[1] = v.y, d[2] = v.z, d[3] = v.w;
    }
    const float first_prev = (tid == 0 && base >= 1) ? __ldg(x + base - 1) : 0.f;
    __syncthreads();
    const int64_t g = (int64_t)blockIdx.x * L1_GROUPS + tid;
    if (g >= n1) return;
    const float* s = sm + tid * L1_PITCH;
    float prev = tid == 0 ? first_prev : s[-2];                    // last sample of the group before (pitch 33: one pad word)
    float fmx = -FLT_MAX, fmn = FLT_MAX;
    uint32_t w = 0;
    if (interior) {
#pragma unroll
        for (int k = 0; k < 32; k++) {
            const float v = s[k];
            fmx = fmaxf(fmx, v), fmn = fminf(fmn, v);
            w |= (uint32_t)(prev < v && !(v < hmin)) << k;
            prev = v;
        }
    } else {
        for (int k = 0; k < 32; k++) {
            const int64_t t = g * 32 + k;
            if (t >= N) break;
            const float v = s[k];
            fmx = fmaxf(fmx, v), fmn = fminf(fmn, v);
            w |= (uint32_t)(t >= 1 && t < N - 1 && prev < v && !(v < hmin)) << k;
            prev = v;
        }
    }
    cand[g] = w;
    if (mx1) mx1[g] = fmx, mn1[g] = fmn;
}

__device__ __noinline__ void eval_peak(const Pyr& P, int64_t N, int64_t i, double wmin, gwi_peak* __restrict__ out, int capacity, int32_t* __restrict__ count);

// The candidate mask is walked by a small persistent grid, 16 words per thread and step (the evaluation below is heavy in
// registers: one CTA of it per 32 words meant 55 waves of CTAs for 2^26 samples)
__global__ void __launch_bounds__(256) k_find_peaks(Pyr P, int64_t N, double wmin, const uint32_t* __restrict__ cand, int64_t n1,
                                                    gwi_peak* __restrict__ out, int capacity, int32_t* __restrict__ count)
{
    const int64_t nq = (n1 + 3) / 4;                               // 16-byte chunks (the workspace slot is padded to 256 bytes)
    const uint4* c4 = reinterpret_cast<const uint4*>(cand);
    const int64_t nthr = (int64_t)gridDim.x * blockDim.x;
    for (int64_t q0 = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; q0 < nq; q0 += 4 * nthr) {
        uint4 w[4];
#pragma unroll
        for (int u = 0; u < 4; u++) w[u] = q0 + u * nthr < nq ? __ldg(c4 + q0 + u * nthr) : make_uint4(0, 0, 0, 0);
#pragma unroll
        for (int u = 0; u < 4; u++) {
            if (!(w[u].x | w[u].y | w[u].z | w[u].w)) continue;
            const uint32_t ww[4] = {w[u].x, w[u].y, w[u].z, w[u].w};
            for (int j = 0; j < 4; j++) {
                const int64_t g = (q0 + u * nthr) * 4 + j;
                uint32_t m = g < n1 ? ww[j] : 0u;
                while (m) {
                    const int l = __ffs(m) - 1;
                    m &= m - 1;
                    eval_peak(P, N, g * 32 + l, wmin, out, capacity, count);
                }
            }
        }
    }
}

// sample i starts a rise and reaches the height (steps 1 and 2 of the definition): the rest
__device__ __noinline__ void eval_peak(const Pyr& P, int64_t N, int64_t i, double wmin, gwi_peak* __restrict__ out, int capacity, int32_t* __restrict__ count)
{
    const float* x = P.mx[0];
    const float v = x[i];
    // end of the flat top that starts at i: first sample to the right that differs
    const int64_t jn = search_right(P, i + 1, [&](int l, int64_t k) { return P.mx[l][k] != v || P.mn[l][k] != v; });
    if (jn >= N || !(x[jn] < v)) return;                           // reaches the array end, or rises further
    const int64_t p = (i + jn - 1) / 2;
    // step 3: nearest higher sample on either side, minima of the stretches in between
    const int64_t L = search_left(P, p - 1, [&](int l, int64_t k) { return P.mx[l][k] > v; });
    const int64_t R = search_right(P, p + 1, [&](int l, int64_t k) { return P.mx[l][k] > v; });
    const float lmin = range_min(P, L + 1, p), rmin = range_min(P, p, R - 1);
    const double prom = (double)v - (double)fmaxf(lmin, rmin);
    // step 4: crossings of the half-prominence level
    const double level = (double)v - prom * 0.5;
    const int64_t kl = search_left(P, p, [&](int l, int64_t k) { return (double)P.mn[l][k] <= level; });
    const int64_t kr = search_right(P, p, [&](int l, int64_t k) { return (double)P.mn[l][k] <= level; });
    double lip = (double)kl, rip = (double)kr;
    if ((double)x[kl] < level) lip += (level - (double)x[kl]) / ((double)x[kl + 1] - (double)x[kl]);
    if ((double)x[kr] < level) rip -= (level - (double)x[kr]) / ((double)x[kr - 1] - (double)x[kr]);
    const double width = rip - lip;
    if (!(width >= wmin)) return;
    const int slot = atomicAdd(count, 1);
    if (slot < capacity) {
        gwi_peak r;
        r.index = p, r.height = v, r.prominence = (float)prom, r.width = width, r.left_ip = lip, r.right_ip = rip;
        out[slot] = r;
    }
}

// sorts the first min(*count, capacity) records by position: rank by counting (the lists are short)
__global__ void k_sort_peaks(const gwi_peak* __restrict__ in, gwi_peak* __restrict__ out, int capacity, const int32_t* __restrict__ count)
{
    const int n = min(*count, capacity);
    for (int a = blockIdx.x * blockDim.x + threadIdx.x; a < n; a += gridDim.x * blockDim.x) {
        const int64_t key = in[a].index;
        int rank = 0;
        for (int b = 0; b < n; b++) rank += in[b].index < key;
        out[rank] = in[a];
    }
}

struct PkLayout {
    size_t lvl_mx[PK_MAX_LEVELS + 1], lvl_mn[PK_MAX_LEVELS + 1], tmp, cand, total;
    int64_t size[PK_MAX_LEVELS + 1];
    int top;
};
PkLayout pk_layout(int64_t N, int capacity)
{
    PkLayout L;
    size_t o = 0;
    auto take = [&](size_t bytes) { size_t at = o; o += (bytes + 255) & ~(size_t)255; return at; };
    L.size[0] = N, L.top = 0;
    for (int l = 1; l <= PK_MAX_LEVELS; l++) {
        if (L.size[l - 1] <= 32) break;
        L.size[l] = (L.size[l - 1] + 31) / 32;
        L.lvl_mx[l] = take((size_t)L.size[l] * 4), L.lvl_mn[l] = take((size_t)L.size[l] * 4);
        L.top = l;
    }
    L.tmp = take((size_t)(capacity > 0 ? capacity : 1) * sizeof(gwi_peak));
    L.cand = take((size_t)((N + 31) / 32) * 4);
    L.total = o;
    return L;
}

} // namespace

extern "C" size_t gwi_find_peaks_workspace_bytes(int64_t N, int32_t capacity)
{
    return (N < 1 || capacity < 0) ? 0 : pk_layout(N, capacity).total;
}

extern "C" gwi_status gwi_find_peaks(const float* d_x, int64_t N, float height, double min_width, gwi_peak* d_peaks,
                                     int32_t capacity, int32_t* d_count, void* d_workspace, size_t workspace_bytes,
                                     void* cuda_stream)
{
    if (!d_x || N < 1 || capacity < 0 || (capacity > 0 && !d_peaks) || !d_count || !d_workspace || ((uintptr_t)d_workspace & 255) ||
        !(min_width >= 0.0)) {
        gwi_set_error("gwi_find_peaks: bad argument");
        return GWI_ERR_ARG;
    }
    const PkLayout L = pk_layout(N, capacity);
    if (workspace_bytes < L.total) {
        gwi_set_error("gwi_find_peaks: workspace %zu < %zu bytes", workspace_bytes, L.total);
        return GWI_ERR_NOMEM;
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    char* ws = (char*)d_workspace;
    Pyr P;
    P.top = L.top;
    P.mx[0] = P.mn[0] = d_x, P.size[0] = N;
    // level 1 and the candidate mask in one coalesced pass over x (N <= 32: no level 1, the mask alone)
    const int64_t n1 = (N + 31) / 32;
    uint32_t* cand = (uint32_t*)(ws + L.cand);
    {
        float *omx = L.top >= 1 ? (float*)(ws + L.lvl_mx[1]) : nullptr, *omn = L.top >= 1 ? (float*)(ws + L.lvl_mn[1]) : nullptr;
        const int64_t want = (n1 + 31) / 32;                       // CTAs of 8 warps x 4 groups
        if (((uintptr_t)d_x & 15) == 0) {
            k_level1_cand_v4<<<(unsigned)((n1 + L1_GROUPS - 1) / L1_GROUPS), L1_GROUPS, 0, st>>>(d_x, N, height, omx, omn, n1, cand);
        } else {
            k_level1_cand<<<(unsigned)(want < 148 * 8 ? want : 148 * 8), 256, 0, st>>>(d_x, N, height, omx, omn, n1, cand);
        }
        if (L.top >= 1) P.mx[1] = omx, P.mn[1] = omn, P.size[1] = L.size[1];
    }
    for (int l = 2; l <= L.top; l++) {
        float *omx = (float*)(ws + L.lvl_mx[l]), *omn = (float*)(ws + L.lvl_mn[l]);
        k_pyr_level<<<(unsigned)((L.size[l] + 7) / 8), 256, 0, st>>>(P.mx[l - 1], P.mn[l - 1], L.size[l - 1], omx, omn, L.size[l]);
        P.mx[l] = omx, P.mn[l] = omn, P.size[l] = L.size[l];
    }
    for (int l = L.top + 1; l <= PK_MAX_LEVELS; l++) P.mx[l] = P.mn[l] = nullptr, P.size[l] = 0;
    GWI_CUDA_CHECK(cudaMemsetAsync(d_count, 0, 4, st));
    gwi_peak* tmp = (gwi_peak*)(ws + L.tmp);
    if (N >= 3) {
        const int64_t wantp = ((n1 + 3) / 4 + 255) / 256;
        k_find_peaks<<<(unsigned)(wantp < 148 * 4 ? wantp : 148 * 4), 256, 0, st>>>(P, N, min_width, cand, n1, tmp, capacity, d_count);
        if (capacity > 0) k_sort_peaks<<<64, 256, 0, st>>>(tmp, d_peaks, capacity, d_count);
    }
    gwi_count_launch(L.top + 2);
    GWI_CUDA_CHECK(cudaGetLastError());
    return GWI_OK;
}
