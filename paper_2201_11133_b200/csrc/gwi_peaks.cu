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
// a search walks at most 32 entries per level.  One thread per sample decides whether it starts a (flat-topped) local
// maximum and, if the height condition holds, evaluates steps 3 and 4.  Decisions are taken on the fp32 samples exactly
// as the oracle takes them in fp64 (differences and half-prominences of fp32 numbers are exact in fp64), so the peak
// list is the oracle's; accepted peaks are appended with an atomic counter and sorted by position afterwards.
#include <cfloat>

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
    const int64_t o = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (o >= nout) return;
    float a = -FLT_MAX, b = FLT_MAX;
    const int64_t i0 = o * 32, i1 = min(i0 + 32, nin);
    for (int64_t i = i0; i < i1; i++) a = fmaxf(a, inmx[i]), b = fminf(b, inmn[i]);
    outmx[o] = a, outmn[o] = b;
}

// Leftward search from `pos` (inclusive): the largest j <= pos whose sample satisfies pred, -1 if none.  BLK(l, i) must be
// true iff block i of level l MAY contain such a sample (exact at level 0).
template <class BLK>
__device__ __forceinline__ int64_t search_left(const Pyr& P, int64_t pos, BLK blk)
{
    int l = 0;
    int64_t i = pos;
    while (i >= 0) {
        if (blk(l, i)) {
            if (l == 0) return i;
            l--;
            i = min(i * 32 + 31, P.size[l] - 1);   // rightmost child
            continue;
        }
        if ((i & 31) == 0 && l < P.top) {
            i = (i >> 5) - 1, l++;                 // the parent's left part is done: previous parent-level block
        } else {
            i--;
        }
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
        if (blk(l, i)) {
            if (l == 0) return i;
            l--;
            i = i * 32;                            // leftmost child
            continue;
        }
        if ((i & 31) == 31 && l < P.top) {
            i = (i >> 5) + 1, l++;
        } else {
            i++;
        }
    }
    return P.size[0];
}
// minimum of x[a..b] (inclusive, a <= b)
__device__ __forceinline__ float range_min(const Pyr& P, int64_t a, int64_t b)
{
    float m = FLT_MAX;
    int l = 0;
    while (a <= b) {
        while (a <= b && (a & 31)) m = fminf(m, P.mn[l][a++]);
        while (a <= b && (b & 31) != 31) m = fminf(m, P.mn[l][b--]);
        if (a > b) break;
        if (l == P.top) {
            for (int64_t i = a; i <= b; i++) m = fminf(m, P.mn[l][i]);
            break;
        }
        a >>= 5, b >>= 5, l++;
    }
    return m;
}

__global__ void k_find_peaks(Pyr P, int64_t N, float hmin, double wmin, gwi_peak* __restrict__ out, int capacity,
                             int32_t* __restrict__ count)
{
    const float* x = P.mx[0];
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x + 1;
    if (i >= N - 1) return;
    const float v = x[i];
    if (!(x[i - 1] < v) || v < hmin) return;                       // steps 1 (rising edge) and 2
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
    size_t lvl_mx[PK_MAX_LEVELS + 1], lvl_mn[PK_MAX_LEVELS + 1], tmp, total;
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
    for (int l = 1; l <= L.top; l++) {
        float *omx = (float*)(ws + L.lvl_mx[l]), *omn = (float*)(ws + L.lvl_mn[l]);
        k_pyr_level<<<(unsigned)((L.size[l] + 255) / 256), 256, 0, st>>>(P.mx[l - 1], P.mn[l - 1], L.size[l - 1], omx, omn, L.size[l]);
        P.mx[l] = omx, P.mn[l] = omn, P.size[l] = L.size[l];
    }
    for (int l = L.top + 1; l <= PK_MAX_LEVELS; l++) P.mx[l] = P.mn[l] = nullptr, P.size[l] = 0;
    GWI_CUDA_CHECK(cudaMemsetAsync(d_count, 0, 4, st));
    gwi_peak* tmp = (gwi_peak*)(ws + L.tmp);
    if (N >= 3) {
        k_find_peaks<<<(unsigned)((N - 2 + 255) / 256), 256, 0, st>>>(P, N, height, min_width, tmp, capacity, d_count);
        if (capacity > 0) k_sort_peaks<<<64, 256, 0, st>>>(tmp, d_peaks, capacity, d_count);
    }
    gwi_count_launch(L.top + 2);
    GWI_CUDA_CHECK(cudaGetLastError());
    return GWI_OK;
}
