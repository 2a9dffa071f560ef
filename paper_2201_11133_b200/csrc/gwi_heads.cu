// gwi_heads.cu -- time-slide heads of the narrow-architecture ensemble, fused with the ensemble mean and the threshold
// (the per-timestep outputs of every slide are what
// did not scale in the paper's post-processing).
//
//   p_{m,k}[t] = sigmoid(b2 + W2 . ReLU(W1 [u_H[t]; u_L[t - lag_k]] + b1))              (reading A24, C.1 step 5)
//
// W1 [u_H; u_L] + b1 = v_H[t] + v_L[t - lag_k] with v_H = W1[:, :32] u_H + b1 and v_L = W1[:, 32:] u_L, which the branch
// kernel (gwi_tiny_tc.cu, time-slide mode) has already written per sample, in fp16.  What is left per (sample, lag,
// model) is element-wise: 16 fused add-ReLU on half2 pairs, 16 half2 multiply-adds with W2, one sigmoid.  The kernel
// loops over the models in order and forms pbar = (((p0 + p1) + p2) + ...) / M in the fixed fp32 expression of tier T1,
// compares with the threshold and writes, per slide, the bit mask the run clustering works on, pbar (the statistics of
// the few triggers are taken from it) and one byte per sample saying which models exceeded the threshold on their own --
// no per-model, per-slide probability array exists (it was 7.8 GB per hour of data at 33 slides and 4 models).
#include <cstring>
#include <vector>

#include <cuda_fp16.h>

#include "gwi_internal.h"

namespace {

constexpr int HF_MAX_M = 8;

struct HeadsFusedArgs {
    const __half* v[HF_MAX_M];   // per model: row 0 of this chunk inside its [2][lds][32] fp16 buffer (v_H rows, then v_L rows)
    int64_t lds;
    int n, M, n_lags;
    const int64_t* lags;         // device, lags[0] = 0
    float theta;
    uint32_t* bits;              // [n_lags][bits_stride] words, bit i of word w = sample 32 w + i of the chunk
    int64_t bits_stride;
    float* pbar;                 // [n_lags][row_stride]
    uint8_t* mm;                 // [n_lags][row_stride]: bit j = model j alone above the threshold
    int64_t row_stride;
    float* prob;                 // per-model rule: [n_lags][M][row_stride] probabilities instead of the three above (else null)
    uint32_t w2[HF_MAX_M][16];   // W2 as half2 pairs (channels 2c, 2c + 1)
    float b2[HF_MAX_M];
};

__device__ __forceinline__ uint32_t add_relu2(uint32_t a, uint32_t b)
{
    // relu(a * 1 + b) on a half2 pair, one rounding
    uint32_t d;
    asm("fma.rn.relu.f16x2 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(0x3C003C00u), "r"(b));
    return d;
}
__device__ __forceinline__ uint32_t fma2h(uint32_t a, uint32_t b, uint32_t c)
{
    uint32_t d;
    asm("fma.rn.f16x2 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(c));
    return d;
}
__device__ __forceinline__ uint32_t mul2h(uint32_t a, uint32_t b)
{
    uint32_t d;
    asm("mul.rn.f16x2 %0, %1, %2;" : "=r"(d) : "r"(a), "r"(b));
    return d;
}
// sigmoid(y) = 0.5 + 0.5 tanh(y / 2): one MUFU op (tanh.approx.f32, relative error 2^-11: 2.5e-4 absolute at most on p)
__device__ __forceinline__ float sigmoid_fast(float y)
{
    float t;
    asm("tanh.approx.f32 %0, %1;" : "=f"(t) : "f"(0.5f * y));
    return fmaf(0.5f, t, 0.5f);
}
__device__ __forceinline__ float2 h2f2(uint32_t a)
{
    __half2 h = *reinterpret_cast<__half2*>(&a);
    return __half22float2(h);
}

// y = b2 + W2 . relu(vh + vl): four half2 accumulators of four products each, combined in fp32
__device__ __forceinline__ float head_y(const uint4 (&vh)[4], const uint4 (&vl)[4], const uint32_t (&w2)[16], float b2)
{
    float y = b2;
#pragma unroll
    for (int c = 0; c < 4; c++) {
        uint32_t acc = mul2h(add_relu2(vl[c].x, vh[c].x), w2[4 * c]);
        acc = fma2h(add_relu2(vl[c].y, vh[c].y), w2[4 * c + 1], acc);
        acc = fma2h(add_relu2(vl[c].z, vh[c].z), w2[4 * c + 2], acc);
        acc = fma2h(add_relu2(vl[c].w, vh[c].w), w2[4 * c + 3], acc);
        const float2 f = h2f2(acc);
        y += f.x + f.y;
    }
    return y;
}

__global__ void __launch_bounds__(256) k_heads_fused(const __grid_constant__ HeadsFusedArgs a)
{
    const int64_t t = (int64_t)blockIdx.x * 256 + threadIdx.x;
    const bool live = t < a.n;
    const int64_t tc = live ? t : a.n - 1;                            // clamp the loads of the ragged tail
    const int lane = threadIdx.x & 31;
    const float fM = (float)a.M;
    for (int k = 0; k < a.n_lags; k++) {
        const int64_t lag = __ldg(a.lags + k);
        float s = 0.f;
        uint32_t mk = 0;
        for (int m = 0; m < a.M; m++) {
            const uint4* vH = reinterpret_cast<const uint4*>(a.v[m]) + tc * 4;
            const uint4* vL = reinterpret_cast<const uint4*>(a.v[m] + a.lds * 32) + (tc - lag) * 4;
            uint4 h[4], l[4];
#pragma unroll
            for (int c = 0; c < 4; c++) h[c] = __ldg(vH + c), l[c] = __ldg(vL + c);
            const float y = head_y(h, l, a.w2[m], a.b2[m]);
            const float p = sigmoid_fast(y);
            if (a.prob) {
                if (live) a.prob[((size_t)k * a.M + m) * a.row_stride + t] = p;
            } else {
                s = m == 0 ? p : __fadd_rn(s, p);
                mk |= (uint32_t)(p > a.theta) << m;
            }
        }
        if (a.prob) continue;
        const float pb = __fdiv_rn(s, fM);
        const uint32_t w = __ballot_sync(0xffffffffu, live && pb > a.theta);
        if (lane == 0 && (t >> 5) < a.bits_stride) a.bits[(size_t)k * a.bits_stride + (t >> 5)] = w;
        if (live) {
            a.pbar[(size_t)k * a.row_stride + t] = pb;
            a.mm[(size_t)k * a.row_stride + t] = (uint8_t)mk;
        }
    }
}

// ---- regular lag lists (lag_k = k G, BASELINE.json configs[3]: k x 1 s): the "comb" schedule ------------------------------
// A lagged L1 row s is used by every (t, k) with t - k G = s.  A CTA therefore takes a comb of CJ blocks of 16 samples G
// apart, t = (c CJ + j) G + 16 r + [0, 16), j < CJ: for all K lags it needs only the CJ + K - 1 blocks of v_L rows at
// (c CJ + i) G + 16 r, -K < i < CJ, which it stages in shared memory once per model (double-buffered over the models, the
// next model's blocks arrive by cp.async while this one is evaluated): 48 KB feed 8448 evaluations, 8 x fewer bytes from L2
// than one row per evaluation.  512 threads = 16 rows x CJ blocks x 2 interleaved halves of the lag list; a thread keeps
// the running sums of its <= 17 lags in registers across the models (fixed order m = 0, 1, ...: the T1 expression).
constexpr int CJ = 16, CK_MAX = 34, CKH = CK_MAX / 2;
constexpr int COMB_THREADS = 512;

__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}

__global__ void __launch_bounds__(COMB_THREADS, 2) k_heads_comb(const __grid_constant__ HeadsFusedArgs a, const int K, const int64_t G)
{
    extern __shared__ __align__(128) uint8_t smem[];
    const int nblk = CJ + K - 1;                                        // staged v_L blocks per model
    const uint32_t sbase = (uint32_t)__cvta_generic_to_shared(smem);
    const uint32_t stage_bytes = (uint32_t)nblk * 1024;
    const int tid = threadIdx.x, row = tid & 15, j = (tid >> 4) & (CJ - 1), kh = tid >> 8;
    const int64_t G16 = G >> 4;
    const int64_t c = blockIdx.x / G16, r = blockIdx.x % G16;
    const int64_t t = (c * CJ + j) * G + 16 * r + row;                  // this thread's sample
    const bool live = t < a.n;
    const int64_t tc = live ? t : a.n - 1;
    const int64_t lo_row = -(int64_t)(K - 1) * G;                       // oldest ring row
    auto stage_load = [&](int m, int buf) {
        const __half* vL = a.v[m] + a.lds * 32;
        for (int e = tid; e < nblk * 64; e += COMB_THREADS) {           // (block i, row rr, chunk cc)
            const int i = e >> 6, rr = (e >> 2) & 15, cc = e & 3;
            int64_t s = (c * CJ + i - (K - 1)) * G + 16 * r + rr;
            s = s < lo_row ? lo_row : (s > a.n - 1 ? a.n - 1 : s);
            cp_async16(sbase + buf * stage_bytes + i * 1024 + cc * 256 + rr * 16, vL + s * 32 + cc * 8);
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };
    float sum[CKH];
    uint32_t mk[(CKH + 3) / 4];
#pragma unroll
    for (int q = 0; q < CKH; q++) sum[q] = 0.f;
#pragma unroll
    for (int q = 0; q < (CKH + 3) / 4; q++) mk[q] = 0u;
    for (int e = tid; e < a.M * 16; e += COMB_THREADS) reinterpret_cast<uint32_t*>(smem + 2 * stage_bytes)[e] = a.w2[e >> 4][e & 15];
    stage_load(0, 0);
    for (int m = 0; m < a.M; m++) {
        if (m + 1 < a.M) {
            stage_load(m + 1, (m + 1) & 1);
            asm volatile("cp.async.wait_group 1;" ::: "memory");
        } else {
            asm volatile("cp.async.wait_group 0;" ::: "memory");
        }
        __syncthreads();
        uint4 h[4];
        {
            const uint4* vH = reinterpret_cast<const uint4*>(a.v[m]) + tc * 4;
#pragma unroll
            for (int cc = 0; cc < 4; cc++) h[cc] = __ldg(vH + cc);
        }
        // W2 of this model as broadcast shared-memory loads; the address of the thread's row in the block of lag k = 2 q + kh
        // is sa0 - 2048 q (immediate offsets once the q loop is unrolled).  Lags past the list (k >= K, one of 34 at most)
        // are evaluated on block 0 and dropped at the end: no branch in the loop.
        const uint32_t sw = sbase + 2 * stage_bytes + m * 64;
        const uint32_t sa0 = sbase + (m & 1) * stage_bytes + row * 16 + (uint32_t)(j - kh + K - 1) * 1024;
        const float b2 = a.b2[m];
#pragma unroll
        for (int q = 0; q < CKH; q++) {
            const uint32_t sa = (2 * q + kh < K) ? sa0 - 2048u * q : sbase + (m & 1) * stage_bytes + row * 16;
            float y = b2;
#pragma unroll
            for (int cc = 0; cc < 4; cc++) {
                uint4 l, w;
                asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(l.x), "=r"(l.y), "=r"(l.z), "=r"(l.w) : "r"(sa + cc * 256));
                asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(w.x), "=r"(w.y), "=r"(w.z), "=r"(w.w) : "r"(sw + cc * 16));
                uint32_t acc = mul2h(add_relu2(l.x, h[cc].x), w.x);
                acc = fma2h(add_relu2(l.y, h[cc].y), w.y, acc);
                acc = fma2h(add_relu2(l.z, h[cc].z), w.z, acc);
                acc = fma2h(add_relu2(l.w, h[cc].w), w.w, acc);
                const float2 f = h2f2(acc);
                y += f.x + f.y;
            }
            const float p = sigmoid_fast(y);
            sum[q] = __fadd_rn(sum[q], p);                               // 0 + p0 = p0 exactly: the T1 expression
            if (p > a.theta) mk[q >> 2] |= 1u << (8 * (q & 3) + m);
        }
        __syncthreads();                                                // the stage is refilled two models later
    }
    const float fM = (float)a.M;
    const int lane = tid & 31;
    const int64_t blk16 = t >> 4;                                        // 16-sample block of this thread (same for its 16 rows)
#pragma unroll
    for (int q = 0; q < CKH; q++) {
        const int k = 2 * q + kh;
        if (k < K) {                                                     // warp-uniform (kh is)
            const float pb = __fdiv_rn(sum[q], fM);
            const uint32_t w = __ballot_sync(0xffffffffu, live && pb > a.theta);
            if ((lane & 15) == 0 && blk16 < 2 * a.bits_stride)
                reinterpret_cast<uint16_t*>(a.bits + (size_t)k * a.bits_stride)[blk16] = (uint16_t)(w >> (lane & 16));
            if (live) {
                a.pbar[(size_t)k * a.row_stride + t] = pb;
                a.mm[(size_t)k * a.row_stride + t] = (uint8_t)(mk[q >> 2] >> (8 * (q & 3)));
            }
        }
    }
}

} // namespace

// packs W2 / b2 of the models and launches; d_v[m] = row 0 of the chunk inside model m's [2][lds][32] buffer
gwi_status gwi_heads_fused(const gwi_model* const* models, int M, const __half* const* d_v, int64_t lds, int n, const int64_t* d_lags,
                           int n_lags, const int64_t* h_lags, float theta, uint32_t* d_bits, int64_t bits_stride, float* d_pbar,
                           uint8_t* d_mm, int64_t row_stride, float* d_prob, cudaStream_t st)
{
    if (M < 1 || M > HF_MAX_M) {
        gwi_set_error("gwi_heads_fused: 1..%d models", HF_MAX_M);
        return GWI_ERR_UNSUPPORTED;
    }
    HeadsFusedArgs a;
    for (int m = 0; m < M; m++) {
        a.v[m] = d_v[m];
        const float* W = models[m]->host_blob.data();
        for (int c = 0; c < 16; c++) {
            __half lo = __float2half_rn(W[models[m]->off.W2 + 2 * c]), hi = __float2half_rn(W[models[m]->off.W2 + 2 * c + 1]);
            uint16_t ul, uh;
            memcpy(&ul, &lo, 2), memcpy(&uh, &hi, 2);
            a.w2[m][c] = (uint32_t)ul | ((uint32_t)uh << 16);
        }
        a.b2[m] = W[models[m]->off.b2];
    }
    a.lds = lds, a.n = n, a.M = M, a.n_lags = n_lags, a.lags = d_lags, a.theta = theta;
    a.bits = d_bits, a.bits_stride = bits_stride, a.pbar = d_pbar, a.mm = d_mm, a.row_stride = row_stride, a.prob = d_prob;
    // regular lag list k G (G a multiple of 16, at most CK_MAX slides, mean rule): the comb schedule
    std::vector<int64_t> hl((size_t)n_lags);
    bool comb = !d_prob && n_lags >= 2 && n_lags <= CK_MAX && h_lags != nullptr;
    int64_t G = 0;
    if (comb) {
        G = h_lags[1];
        comb = G > 0 && G % 16 == 0;
        for (int k = 0; k < n_lags && comb; k++) comb = h_lags[k] == (int64_t)k * G;
    }
    if (comb) {
        const int64_t nG = (n + G - 1) / G, groups = (nG + CJ - 1) / CJ;
        const size_t smem = (size_t)2 * (CJ + n_lags - 1) * 1024 + HF_MAX_M * 64;
        static bool attr = false;
        if (!attr) {
            GWI_CUDA_CHECK(cudaFuncSetAttribute(k_heads_comb, cudaFuncAttributeMaxDynamicSharedMemorySize, 2 * (CJ + CK_MAX - 1) * 1024 + HF_MAX_M * 64));
            attr = true;
        }
        k_heads_comb<<<(unsigned)(groups * (G / 16)), COMB_THREADS, smem, st>>>(a, n_lags, G);
    } else {
        k_heads_fused<<<(n + 255) / 256, 256, 0, st>>>(a);
    }
    gwi_count_launch(1);
    GWI_CUDA_CHECK(cudaGetLastError());
    return GWI_OK;
}
