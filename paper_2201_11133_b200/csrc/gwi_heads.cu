// gwi_heads.cu -- time-slide heads of the ensemble (narrow architecture: 32 head channels; paper scale: 128), fused with
// the ensemble mean and the threshold
// (the per-timestep outputs of every slide are what
// did not scale in the paper's post-processing).
//
//   p_{m,k}[t] = sigmoid(b2 + W2 . ReLU(W1 [u_H[t]; u_L[t - lag_k]] + b1))              (reading A24, C.1 step 5)
//
// W1 [u_H; u_L] + b1 = v_H[t] + v_L[t - lag_k] with v_H = W1[:, :Hh] u_H + b1 and v_L = W1[:, Hh:] u_L, which the branch
// kernel (gwi_tiny_tc.cu in time-slide mode; gwi_tc.cu k_vhalf_tc for paper-scale models) has already written per
// sample, in fp16.  What is left per (sample, lag, model) is element-wise: Hh / 2 fused add-ReLU on half2 pairs, Hh / 2
// half2 multiply-adds with W2, one sigmoid.  The kernel
// loops over the models in order and forms pbar = (((p0 + p1) + p2) + ...) / M in the fixed fp32 expression of tier T1,
// compares with the threshold and writes, per slide, the bit mask the run clustering works on, pbar (the statistics of
// the few triggers are taken from it) and one byte per sample saying which models exceeded the threshold on their own --
// no per-model, per-slide probability array exists (it was 7.8 GB per hour of data at 33 slides and 4 models).
#include <algorithm>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <vector>

#include <cuda_fp16.h>

#include "gwi_internal.h"
#include "gwi_tc_ptx.h"

#ifndef GWI_COMB_MINB
#define GWI_COMB_MINB 2
#endif

namespace {

constexpr int HF_MAX_M = 8;

struct HeadsFusedArgs {
    const __half* v[HF_MAX_M];   // per model: row 0 of this chunk inside its [2][lds][CH] fp16 buffer (v_H rows, then v_L rows)
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
    uint32_t w2[HF_MAX_M][64];   // W2 as half2 pairs (channels 2c, 2c + 1), CH / 2 of them used
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
__device__ __forceinline__ uint4 lds128(uint32_t addr)
{
    uint4 v;
    asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr));
    return v;
}
// lo + hi of a half2 accumulator added to y in fp32: two mixed-precision multiply-adds by one (FHFMA)
__device__ __forceinline__ float acc_to_y(uint32_t acc, float y)
{
    asm("{ .reg .f16 lo, hi, one;\n\t"
        "mov.b32 {lo, hi}, %1;\n\t"
        "mov.b16 one, 0x3C00;\n\t"
        "fma.rn.f32.f16 %0, lo, one, %0;\n\t"
        "fma.rn.f32.f16 %0, hi, one, %0; }"
        : "+f"(y)
        : "r"(acc));
    return y;
}
// y + the contribution of 8 channels (one 16-byte chunk of v_H, v_L and W2): a half2 accumulator of four products
__device__ __forceinline__ float chunk_acc(float y, uint4 h, uint4 l, uint4 w)
{
    uint32_t acc = mul2h(add_relu2(l.x, h.x), w.x);
    acc = fma2h(add_relu2(l.y, h.y), w.y, acc);
    acc = fma2h(add_relu2(l.z, h.z), w.z, acc);
    acc = fma2h(add_relu2(l.w, h.w), w.w, acc);
    return acc_to_y(acc, y);
}

// ---- any lag list: one thread per sample, the lagged row of every evaluation comes from global memory / L2 ---------------
template <int CH>
__global__ void __launch_bounds__(256) k_heads_fused(const __grid_constant__ HeadsFusedArgs a)
{
    constexpr int CHC = CH / 8;                                          // 16-byte chunks per row
    __shared__ uint4 sw[HF_MAX_M * CHC];
    for (int e = threadIdx.x; e < a.M * CHC * 4; e += 256) reinterpret_cast<uint32_t*>(sw)[e] = a.w2[e / (CHC * 4)][e % (CHC * 4)];
    __syncthreads();
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
            const uint4* vH = reinterpret_cast<const uint4*>(a.v[m]) + tc * CHC;
            const uint4* vL = reinterpret_cast<const uint4*>(a.v[m] + a.lds * CH) + (tc - lag) * CHC;
            float y = a.b2[m];
#pragma unroll 4
            for (int c = 0; c < CHC; c++) y = chunk_acc(y, __ldg(vH + c), __ldg(vL + c), sw[m * CHC + c]);
            const float p = sigmoid_fast(y);
            if (a.prob) {
                if (live) a.prob[((size_t)k * a.M + m) * a.row_stride + t] = p;
            } else {
                s = __fadd_rn(s, p);                                  // 0 + p0 = p0 exactly: the T1 expression
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
// A lagged L1 row s is used by every (t, k) with t - k G = s.  A CTA therefore takes a comb of CJ blocks of T samples G
// apart, t = (c CJ + j) G + T r + [0, T), j < CJ: for all K lags it needs only the CJ + K - 1 blocks of v_L rows at
// (c CJ + i) G + T r, -K < i < CJ, which it stages in shared memory once per model: with T = 16 rows of 32 channels, 48 KB
// feed 8448 evaluations, 8 x fewer bytes from L2 than one row per evaluation (double-buffered over the models: the next
// model's blocks arrive by cp.async while this one is evaluated).  (128-channel rows and longer lists: k_heads_diag below.)
// Threads = T rows x CJ blocks x NG interleaved groups of the lag list; a thread
// keeps the running sums of its <= KQ lags in registers across the models (fixed order m = 0, 1, ...: the T1 expression).

__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}

template <int CH, int T, int CJ, int NG, int KQ, int NBUF, int MINB>
__global__ void __launch_bounds__(T * CJ * NG, MINB) k_heads_comb(const __grid_constant__ HeadsFusedArgs a, const int K, const int64_t G)
{
    constexpr int CHC = CH / 8, BLK = T * CHC * 16, NTHR = T * CJ * NG;
    extern __shared__ __align__(128) uint8_t smem[];
    const int nblk = CJ + K - 1;                                        // staged v_L blocks per model
    const uint32_t sbase = (uint32_t)__cvta_generic_to_shared(smem);
    const uint32_t stage_bytes = (uint32_t)nblk * BLK;
    const int tid = threadIdx.x, row = tid % T, j = (tid / T) % CJ, kg = tid / (T * CJ);
    const int64_t GT = G / T;
    const int64_t c = blockIdx.x / GT, r = blockIdx.x % GT;
    const int64_t t = (c * CJ + j) * G + T * r + row;                   // this thread's sample
    const bool live = t < a.n;
    const int64_t tc = live ? t : a.n - 1;
    const int64_t lo_row = -(int64_t)(K - 1) * G;                       // oldest ring row
    auto stage_load = [&](int m, int buf) {
        const __half* vL = a.v[m] + a.lds * CH;
        for (int e = tid; e < nblk * T * CHC; e += NTHR) {              // (block i, row rr, chunk cc)
            const int i = e / (T * CHC), rr = (e / CHC) % T, cc = e % CHC;
            int64_t s = (c * CJ + i - (K - 1)) * G + T * r + rr;
            s = s < lo_row ? lo_row : (s > a.n - 1 ? a.n - 1 : s);
            cp_async16(sbase + buf * stage_bytes + i * BLK + cc * (T * 16) + rr * 16, vL + s * CH + cc * 8);
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };
    float sum[KQ];
    uint32_t mk[(KQ + 3) / 4];
#pragma unroll
    for (int q = 0; q < KQ; q++) sum[q] = 0.f;
#pragma unroll
    for (int q = 0; q < (KQ + 3) / 4; q++) mk[q] = 0u;
    const uint32_t swb = sbase + NBUF * stage_bytes;                     // W2 of all models, CH / 2 words each
    for (int e = tid; e < a.M * CHC * 4; e += NTHR) reinterpret_cast<uint32_t*>(smem + NBUF * stage_bytes)[e] = a.w2[e / (CHC * 4)][e % (CHC * 4)];
    stage_load(0, 0);
    for (int m = 0; m < a.M; m++) {
        if (NBUF == 2 && m + 1 < a.M) {
            stage_load(m + 1, (m + 1) & 1);
            asm volatile("cp.async.wait_group 1;" ::: "memory");
        } else {
            asm volatile("cp.async.wait_group 0;" ::: "memory");
        }
        __syncthreads();
        uint4 h[CHC];
        {
            const uint4* vH = reinterpret_cast<const uint4*>(a.v[m]) + tc * CHC;
#pragma unroll
            for (int cc = 0; cc < CHC; cc++) h[cc] = __ldg(vH + cc);
        }
        // W2 of this model as broadcast shared-memory loads; the address of the thread's row in the block of lag
        // k = NG q + kg is sa0 - NG BLK q (immediate offsets once the q loop is unrolled).  Lags past the list (k >= K) are
        // evaluated on block 0 and dropped at the end: no branch in the loop.
        const uint32_t sw = swb + m * (CHC * 16);
        const uint32_t st0 = sbase + (NBUF == 2 ? (m & 1) : 0) * stage_bytes + row * 16;
        const uint32_t sa0 = st0 + (uint32_t)(j - kg + K - 1) * BLK;
        const float b2 = a.b2[m];
#pragma unroll
        for (int q = 0; q < KQ; q++) {
            const uint32_t sa = (NG * q + kg < K) ? sa0 - (uint32_t)(NG * BLK) * q : st0;
            float y = b2;
#pragma unroll
            for (int cc = 0; cc < CHC; cc++) y = chunk_acc(y, h[cc], lds128(sa + cc * (T * 16)), lds128(sw + cc * 16));
            const float p = sigmoid_fast(y);
            sum[q] = __fadd_rn(sum[q], p);                               // 0 + p0 = p0 exactly: the T1 expression
            if (p > a.theta) mk[q >> 2] |= 1u << (8 * (q & 3) + m);
        }
        __syncthreads();                                                // the stage is refilled by a later model
        if (NBUF == 1 && m + 1 < a.M) stage_load(m + 1, 0);
    }
    const float fM = (float)a.M;
    const int lane = tid & 31;
#pragma unroll
    for (int q = 0; q < KQ; q++) {
        const int k = NG * q + kg;
        if (k < K) {                                                     // warp-uniform (kg is)
            const float pb = __fdiv_rn(sum[q], fM);
            const uint32_t w = __ballot_sync(0xffffffffu, live && pb > a.theta);
            // the warp holds 32 / T blocks of T samples: each writes its T mask bits
            if ((lane % T) == 0) {
                if (T == 16) {
                    if ((t >> 4) < 2 * a.bits_stride) reinterpret_cast<uint16_t*>(a.bits + (size_t)k * a.bits_stride)[t >> 4] = (uint16_t)(w >> (lane & 16));
                } else {
                    if ((t >> 3) < 4 * a.bits_stride) reinterpret_cast<uint8_t*>(a.bits + (size_t)k * a.bits_stride)[t >> 3] = (uint8_t)(w >> (lane & 24));
                }
            }
            if (live) {
                a.pbar[(size_t)k * a.row_stride + t] = pb;
                a.mm[(size_t)k * a.row_stride + t] = (uint8_t)(mk[q >> 2] >> (8 * (q & 3)));
            }
        }
    }
}

// ---- the comb schedule for 128-channel rows (paper-scale models, up to 64 slides) ---------------------------------------
// The work is cut along the diagonals: a staged v_L block i serves every item (j, k) with j - k = i - (K - 1), so a warp =
// 8 rows x 4 channel quarters keeps the v_H quarter rows of JB = 4 neighbouring comb blocks in registers, walks the staged
// blocks (i = slot, slot + 8, ...) and evaluates up to four items per 64 bytes read from shared memory.  The quarter sums
// of the four items are reduced across the four lanes with a transposing butterfly (3 shuffles) that leaves item jj on
// the lane of quarter jj, which adds its sigmoid to the running sum of the item in shared memory (each item belongs to
// one lane for all models: the T1 expression in model order, no atomics).
//
// Persistent CTAs (one per SM) walk the work items (comb group c fastest, so that the CTAs running at the same time
// share their v_L rows in L2; then the lag pass; then the row group r); one step = one model of one item.  The rows of a
// step (v_L blocks and the CJ v_H blocks) are fetched with 16-byte cp.async copies into one of two stages while the
// step before is evaluated (256-byte bulk copies, one per row, ran at a third of this: the copy engine's cost per
// request); rows sit 272 bytes apart, which makes the quarter-warp's 16-byte reads of eight neighbouring rows
// conflict-free.  Lag lists longer than 33 are evaluated in passes of at most 33 lags, so that
// two stages always fit.
//
// The same kernel serves the 32-channel rows of the narrow architecture: there a lane holds whole rows (no quarters, no
// butterfly), a warp = 16 rows x 2 groups of four comb blocks, blocks are 16 rows, CJ = 16 and rows sit 80 bytes apart.
constexpr int DG_THREADS = 512, DG_KS_MAX = 33;

template <int CH>
struct DiagGeom {
    static constexpr int QN = CH / 32;                  // lanes per row (channel quarters)
    static constexpr int T = CH == 128 ? 8 : 16;        // rows per block
    static constexpr int CJ = CH == 128 ? 8 : 16;       // comb blocks per item
    static constexpr int ROWB = CH * 2 + 16;            // row pitch in shared memory
    static constexpr int BLKB = T * ROWB;
    static constexpr size_t smem_bytes(int KS)
    {
        return (size_t)2 * (CJ + KS - 1 + CJ) * BLKB + (size_t)CJ * KS * T * 5 + HF_MAX_M * CH * 2 + 16;
    }
};

struct DiagItem {
    int c, r, ka, Kp;      // comb group, row group, first lag and number of lags of the pass
};

// warp-level tensor-core pieces of the MMA variant below
__device__ __forceinline__ void ldmatrix_x4(uint32_t (&r)[4], uint32_t addr)
{
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0, %1, %2, %3}, [%4];" : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(addr));
}
__device__ __forceinline__ void mma16816(float (&c)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1)
{
    asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0, %1, %2, %3}, {%4, %5, %6, %7}, {%8, %9}, {%0, %1, %2, %3};"
                 : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
                 : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}

// MMA = true (32-channel rows): the element-wise work is bound by the fp16 pipe (HFMA2 issues every other clock per
// scheduler; measured on B200: HFMA2 / HFMA2.RELU / HADD2 0.5 per clock and scheduler, FFMA / FHFMA / HMNMX2 1.0), and two
// thirds of it is the dot product with W2.  That part moves to the (otherwise idle) warp-level tensor path: a tile = the 16
// samples of a comb block x one lag; z = ReLU(v_H + v_L) is formed on ldmatrix fragments (A operand, 16 x CH) and
// multiplied by a B operand that holds W2 in column n for the n-th tile of a group of eight lags, so that eight tiles
// accumulate into ONE 16 x 8 fp32 accumulator whose lane (g, t) ends up with y of lags 2t, 2t + 1 for samples g, g + 8:
// every lane owns four evaluations of the group for all models (T1's model order in registers, no shared-memory sums).
template <int CH, bool MMA>
__global__ void __launch_bounds__(DG_THREADS, 1) k_heads_diag(const __grid_constant__ HeadsFusedArgs a, const int K, const int KS,
                                                             const int npass, const int G, const int groups, const int nitems)
{
    using namespace tc;
    using GEO = DiagGeom<CH>;
    constexpr int T = GEO::T, CJ = GEO::CJ, JB = 4, NS = 8, QN = GEO::QN, ROWB = GEO::ROWB, BLKB = GEO::BLKB, CHC = CH / 8;
    extern __shared__ __align__(128) uint8_t smem[];
    const int nblk_max = CJ + KS - 1;
    const uint32_t sbase = smem_u32(smem);
    const uint32_t stage_bytes = (uint32_t)(nblk_max + CJ) * BLKB;
    const int nsum = CJ * KS * T;
    float* sums = reinterpret_cast<float*>(smem + 2 * (size_t)stage_bytes);             // [j][k'][row]
    uint8_t* smm = reinterpret_cast<uint8_t*>(sums + nsum);                             // same order
    const uint32_t w2off = 2 * stage_bytes + nsum * 5;                                  // W2 of all models, 256 B each
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    // CH = 128: lane = (quarter, row), the warp serves one group of JB comb blocks; CH = 32: lane = (group, row)
    const int q = QN == 4 ? lane >> 3 : 0, row = lane & (T - 1);
    const int j0 = (QN == 4 ? (warp & 1) : (warp & 1) * 2 + (lane >> 4)) * JB, slot = warp >> 1;
    const int64_t lo_row = -(int64_t)(K - 1) * G;
    for (int e = tid; e < nsum; e += DG_THREADS) sums[e] = 0.f, smm[e] = 0;
    for (int e = tid; e < a.M * (CH / 2); e += DG_THREADS) reinterpret_cast<uint32_t*>(smem + w2off)[e] = a.w2[e / (CH / 2)][e % (CH / 2)];
    __syncthreads();

    auto decode = [&](int wi) {
        DiagItem it;
        it.c = wi % groups;
        const int x = wi / groups, p = x % npass;
        it.r = x / npass;
        it.ka = p * KS, it.Kp = min(KS, K - it.ka);
        return it;
    };
    // all warps: the rows of model m of an item into stage buf, 16 bytes per cp.async.  A block = T consecutive rows,
    // contiguous in global memory (2 KB or 1 KB): a warp-wide copy moves 512 bytes of it.  128-channel rows: blocks
    // start at multiples of 8 and n is one, so a block is inside the rows or outside (then any block will do: its items
    // are dropped); 32-channel rows (any n): every row is clamped.  One commit group per step.
    auto stage_load = [&](const DiagItem& it, int m, int buf) {
        constexpr int RW = 32 / CHC, NX = T / RW;                       // rows per warp-wide copy, copies per block
        const int nblk = CJ + it.Kp - 1;
        const int cr = lane / CHC, ch = lane % CHC;
        const __half* vH = a.v[m] + ch * 8;
        const __half* vL = vH + a.lds * CH;
        const uint32_t dst0 = sbase + buf * stage_bytes + cr * ROWB + ch * 16;
        const int gL = it.c * CJ - (it.Kp - 1) - it.ka, gH = it.c * CJ - nblk;
        for (int blk = warp; blk < nblk + CJ; blk += DG_THREADS / 32) {
            const bool isL = blk < nblk;
            int64_t s0 = (int64_t)((isL ? gL : gH) + blk) * G + T * it.r;
            const int64_t lo = isL ? lo_row : 0;
            const uint32_t dst = dst0 + (isL ? blk : nblk_max + blk - nblk) * BLKB;
            const __half* base = isL ? vL : vH;
            if (CH == 128) {
                s0 = s0 < lo ? lo : (s0 > a.n - T ? a.n - T : s0);
                const __half* src = base + (s0 + cr) * CH;
#pragma unroll
                for (int x = 0; x < NX; x++) cp_async16(dst + x * RW * ROWB, src + x * RW * CH);
            } else if (s0 >= lo && s0 + T <= a.n) {                 // warp-uniform: the whole block is inside the rows
                const __half* src = base + (s0 + cr) * CH;
#pragma unroll
                for (int x = 0; x < NX; x++) cp_async16(dst + x * RW * ROWB, src + x * RW * CH);
            } else {
#pragma unroll
                for (int x = 0; x < NX; x++) {
                    int64_t sr = s0 + cr + x * RW;
                    sr = sr < lo ? lo : (sr > a.n - 1 ? a.n - 1 : sr);
                    cp_async16(dst + x * RW * ROWB, base + sr * CH);
                }
            }
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };

    // one model of an item on the rows of stage buf
    auto compute = [&](const DiagItem& it, int m, int buf) {
        const int Kp = it.Kp, nblk = CJ + Kp - 1;
        const uint32_t bb = sbase + buf * stage_bytes + row * ROWB + q * 64;
        uint4 h[JB][4], w[4];
#pragma unroll
        for (int jj = 0; jj < JB; jj++)
#pragma unroll
            for (int cc = 0; cc < 4; cc++) h[jj][cc] = lds128(bb + (nblk_max + j0 + jj) * BLKB + cc * 16);
#pragma unroll
        for (int cc = 0; cc < 4; cc++) w[cc] = lds128(sbase + w2off + m * (CH * 2) + q * 64 + cc * 16);
        const float b2 = a.b2[m];
        const bool hi = q & 2, od = q & 1;
        for (int i = slot; i < nblk; i += NS) {
            uint4 l[4];
#pragma unroll
            for (int cc = 0; cc < 4; cc++) l[cc] = lds128(bb + i * BLKB + cc * 16);
            const int kb = j0 - i + Kp - 1;                             // lag (within the pass) of item jj = kb + jj
            float y[JB];
            if (kb >= 0 && kb + JB <= Kp) {                             // warp-uniform: the whole diagonal piece is inside
#pragma unroll
                for (int jj = 0; jj < JB; jj++) {
                    y[jj] = 0.f;
#pragma unroll
                    for (int cc = 0; cc < 4; cc++) y[jj] = chunk_acc(y[jj], h[jj][cc], l[cc], w[cc]);
                }
            } else {
#pragma unroll
                for (int jj = 0; jj < JB; jj++) {
                    y[jj] = 0.f;
                    if (kb + jj >= 0 && kb + jj < Kp) {
#pragma unroll
                        for (int cc = 0; cc < 4; cc++) y[jj] = chunk_acc(y[jj], h[jj][cc], l[cc], w[cc]);
                    }
                }
            }
            if (QN == 4) {
                // transposing butterfly over the four quarters: the lane of quarter jj ends with the whole sum of item jj
                float k0 = hi ? y[2] : y[0], k1 = hi ? y[3] : y[1];
                k0 += __shfl_xor_sync(0xffffffffu, hi ? y[0] : y[2], 16);
                k1 += __shfl_xor_sync(0xffffffffu, hi ? y[1] : y[3], 16);
                float yy = od ? k1 : k0;
                yy += __shfl_xor_sync(0xffffffffu, od ? k0 : k1, 8);
                const int k = kb + q;
                if (k >= 0 && k < Kp) {
                    const float p = sigmoid_fast(yy + b2);
                    const int idx = ((j0 + q) * KS + k) * T + row;
                    sums[idx] = __fadd_rn(sums[idx], p);                // 0 + p0 = p0 exactly: the T1 expression
                    if (p > a.theta) smm[idx] |= (uint8_t)(1u << m);
                }
            } else {
#pragma unroll
                for (int jj = 0; jj < JB; jj++) {
                    const int k = kb + jj;
                    if (k >= 0 && k < Kp) {
                        const float p = sigmoid_fast(y[jj] + b2);
                        const int idx = ((j0 + jj) * KS + k) * T + row;
                        sums[idx] = __fadd_rn(sums[idx], p);
                        if (p > a.theta) smm[idx] |= (uint8_t)(1u << m);
                    }
                }
            }
        }
    };
    // ---- MMA variant: warp = comb block j, lane (g, t) owns the evaluations (lag 8 gq + 2 t + (e & 1), row g + 8 (e >> 1))
    constexpr int NGRP = (DG_KS_MAX + 7) / 8;
    float rsum[NGRP][4];
    uint32_t rmk[NGRP];
#pragma unroll
    for (int gq = 0; gq < NGRP; gq++) {
        rmk[gq] = 0;
#pragma unroll
        for (int e = 0; e < 4; e++) rsum[gq][e] = 0.f;
    }
    const int fg = lane >> 2, ft = lane & 3;                        // fragment coordinates of the lane
    const uint32_t frag_off = ((lane & 7) + ((lane >> 3) & 1) * 8) * ROWB + (lane >> 4) * 16;   // ldmatrix row address of the lane
    auto mma_compute = [&](const DiagItem& it, int m, int buf) {
        constexpr int KST = CH / 16;                                 // k-steps of a tile
        const int Kp = it.Kp;
        const uint32_t stage = sbase + buf * stage_bytes;
        uint32_t hf[KST][4], wf[KST][2];
#pragma unroll
        for (int s = 0; s < KST; s++) {
            ldmatrix_x4(hf[s], stage + (nblk_max + warp) * BLKB + frag_off + s * 32);
            const uint32_t* w2s = reinterpret_cast<const uint32_t*>(smem + w2off) + m * (CH / 2) + s * 8 + ft;
            wf[s][0] = w2s[0], wf[s][1] = w2s[4];
        }
        const float hb2 = 0.5f * a.b2[m];
        // B operand of tile n of a group: W2 in column n, i.e. on the lanes with g == n
        auto tile = [&](float (&c)[4], uint32_t lb, int n) {
            const bool mine = fg == n;
#pragma unroll
            for (int s = 0; s < KST; s++) {
                uint32_t z[4];
                ldmatrix_x4(z, lb + s * 32);
#pragma unroll
                for (int x = 0; x < 4; x++) z[x] = add_relu2(z[x], hf[s][x]);
                mma16816(c, z, mine ? wf[s][0] : 0u, mine ? wf[s][1] : 0u);
            }
        };
        auto epilogue = [&](int gq, int e, float y) {              // sigmoid(y + b2) = 0.5 + 0.5 tanh((y + b2) / 2)
            float th;
            asm("tanh.approx.f32 %0, %1;" : "=f"(th) : "f"(fmaf(0.5f, y, hb2)));
            const float p = fmaf(0.5f, th, 0.5f);
            rsum[gq][e] = __fadd_rn(rsum[gq][e], p);               // 0 + p0 = p0 exactly: the T1 expression
            if (p > a.theta) rmk[gq] |= 1u << (8 * e + m);
        };
#pragma unroll
        for (int gq = 0; gq < NGRP; gq++) {
            if (8 * gq >= Kp) break;                                 // warp-uniform
            if ((gq & 1) == 0 && gq + 1 < NGRP && 8 * gq + 16 <= Kp) {
                // two whole groups at once: four independent accumulator chains and twice the ldmatrix loads in flight (the
                // kernel runs four warps per scheduler and waits on those latencies)
                float c0[4] = {0.f, 0.f, 0.f, 0.f}, d0[4] = {0.f, 0.f, 0.f, 0.f}, c1[4] = {0.f, 0.f, 0.f, 0.f}, d1[4] = {0.f, 0.f, 0.f, 0.f};
                const uint32_t la = stage + (warp - 8 * gq + Kp - 1) * BLKB + frag_off, lb = la - 8 * BLKB;
#pragma unroll
                for (int n = 0; n < 8; n += 2) {
                    tile(c0, la - n * BLKB, n), tile(c1, lb - n * BLKB, n);
                    tile(d0, la - (n + 1) * BLKB, n + 1), tile(d1, lb - (n + 1) * BLKB, n + 1);
                }
#pragma unroll
                for (int e = 0; e < 4; e++) epilogue(gq, e, c0[e] + d0[e]), epilogue(gq + 1 < NGRP ? gq + 1 : gq, e, c1[e] + d1[e]);
                continue;
            }
            if ((gq & 1) == 1 && 8 * gq + 8 <= Kp) continue;         // done with the group before
            // two accumulators (even / odd tiles: they fill different columns): half the chain of dependent HMMAs
            float c[4] = {0.f, 0.f, 0.f, 0.f}, d[4] = {0.f, 0.f, 0.f, 0.f};
            const uint32_t lb0 = stage + (warp - 8 * gq + Kp - 1) * BLKB + frag_off;   // staged block of the group's first lag
            if (8 * gq + 8 <= Kp) {                                  // a whole group: no checks inside
#pragma unroll
                for (int n = 0; n < 8; n += 2) tile(c, lb0 - n * BLKB, n), tile(d, lb0 - (n + 1) * BLKB, n + 1);
#pragma unroll
                for (int e = 0; e < 4; e++) epilogue(gq, e, c[e] + d[e]);
            } else {
#pragma unroll
                for (int n = 0; n < 8; n++)
                    if (8 * gq + n < Kp) tile(c, lb0 - n * BLKB, n);
#pragma unroll
                for (int e = 0; e < 4; e++)
                    if (8 * gq + 2 * ft + (e & 1) < Kp) epilogue(gq, e, c[e]);
            }
        }
    };
    auto mma_finalize = [&](const DiagItem& it) {
        const float fM = (float)a.M;
        const int64_t tb = (int64_t)(it.c * CJ + warp) * G + T * it.r;   // first sample of the comb block (a multiple of 16)
#pragma unroll
        for (int gq = 0; gq < NGRP; gq++) {
            if (8 * gq >= it.Kp) break;
            bool pr[4];
#pragma unroll
            for (int e = 0; e < 4; e++) {
                const int kk = 8 * gq + 2 * ft + (e & 1);
                const int64_t t = tb + fg + 8 * (e >> 1);
                const bool live = kk < it.Kp && t < a.n;
                const float pb = __fdiv_rn(rsum[gq][e], fM);
                pr[e] = live && pb > a.theta;
                if (live) {
                    a.pbar[(size_t)(it.ka + kk) * a.row_stride + t] = pb;
                    a.mm[(size_t)(it.ka + kk) * a.row_stride + t] = (uint8_t)(rmk[gq] >> (8 * e));
                }
                rsum[gq][e] = 0.f;
            }
            rmk[gq] = 0;
            // mask bits: the 16 samples of (lag 2 t + par) sit on the lanes with this t, rows g (e = par) and g + 8 (e = par + 2)
#pragma unroll
            for (int par = 0; par < 2; par++) {
                const uint32_t lo = __ballot_sync(0xffffffffu, pr[par]), hi = __ballot_sync(0xffffffffu, pr[par + 2]);
                const int kk = 8 * gq + 2 * ft + par;
                if (fg == 0 && kk < it.Kp && (tb >> 4) < 2 * a.bits_stride) {
                    // bits 4 g + t of the ballots -> bits g: three shift-or steps
                    auto gather = [&](uint32_t x) {
                        x = (x >> ft) & 0x11111111u;
                        x = (x | (x >> 3)) & 0x03030303u;
                        x = (x | (x >> 6)) & 0x000f000fu;
                        return (x | (x >> 12)) & 0xffu;
                    };
                    reinterpret_cast<uint16_t*>(a.bits + (size_t)(it.ka + kk) * a.bits_stride)[tb >> 4] = (uint16_t)(gather(lo) | (gather(hi) << 8));
                }
            }
        }
    };
    // ---- MMA variant for 8-row blocks (128-channel rows): a 16-row tile = the 8 samples of comb block j at TWO consecutive
    // lags (rows 0-7: lag 2 tau from staged block i, rows 8-15: lag 2 tau + 1 from block i - 1; ldmatrix takes any row
    // addresses), v_H of the 8 samples serves both halves.  Two warps per comb block j = warp & 7 take the tiles of even /
    // odd tau; a warp accumulates eight of its tiles (local index n -> column n) per accumulator pair, so lane (g, t) owns
    // the evaluations (tile n = 2 t + (e & 1), lag 2 tau + (e >> 1), sample g) of the group, tau = 16 lg + 2 n + (warp >> 3).
    constexpr int NGRP8 = 2;                                        // <= 9 tiles per warp and pass of <= 33 lags
    const int jw8 = warp & 7, hh8 = warp >> 3;
    const uint32_t frag8 = (lane & 7) * ROWB + (lane >> 4) * 16;    // (the second-lag lanes 8-15, 24-31 go one block back)
    const bool second8 = (lane >> 3) & 1;
    auto mma_compute8 = [&](const DiagItem& it, int m, int buf) {
        constexpr int KST = CH / 16;
        const int Kp = it.Kp, ntile = (Kp + 1) >> 1;
        const uint32_t stage = sbase + buf * stage_bytes;
        uint32_t hf[KST][2], wf[KST][2];
#pragma unroll
        for (int s2 = 0; s2 < KST / 2; s2++) {                       // v_H: one ldmatrix.x4 = the (a0, a2) pairs of two k-steps
            uint32_t r4[4];
            ldmatrix_x4(r4, stage + (nblk_max + jw8) * BLKB + (lane & 7) * ROWB + (lane >> 3) * 16 + s2 * 64);
            hf[2 * s2][0] = r4[0], hf[2 * s2][1] = r4[1], hf[2 * s2 + 1][0] = r4[2], hf[2 * s2 + 1][1] = r4[3];
        }
#pragma unroll
        for (int s = 0; s < KST; s++) {
            const uint32_t* w2s = reinterpret_cast<const uint32_t*>(smem + w2off) + m * (CH / 2) + s * 8 + ft;
            wf[s][0] = w2s[0], wf[s][1] = w2s[4];
        }
        const float hb2 = 0.5f * a.b2[m];
        auto tile = [&](float (&c)[4], uint32_t lb, int n) {
            const bool mine = fg == n;
#pragma unroll
            for (int s = 0; s < KST; s++) {
                uint32_t z[4];
                ldmatrix_x4(z, lb + s * 32);
                z[0] = add_relu2(z[0], hf[s][0]), z[1] = add_relu2(z[1], hf[s][0]);
                z[2] = add_relu2(z[2], hf[s][1]), z[3] = add_relu2(z[3], hf[s][1]);
                mma16816(c, z, mine ? wf[s][0] : 0u, mine ? wf[s][1] : 0u);
            }
        };
        auto epilogue = [&](int lg, int e, float y) {
            float th;
            asm("tanh.approx.f32 %0, %1;" : "=f"(th) : "f"(fmaf(0.5f, y, hb2)));
            const float p = fmaf(0.5f, th, 0.5f);
            rsum[lg][e] = __fadd_rn(rsum[lg][e], p);               // 0 + p0 = p0 exactly: the T1 expression
            if (p > a.theta) rmk[lg] |= 1u << (8 * e + m);
        };
#pragma unroll
        for (int lg = 0; lg < NGRP8; lg++) {
            const int tau0 = 16 * lg + hh8;                          // first tile of the group
            if (tau0 >= ntile) break;                                // warp-uniform
            float c[4] = {0.f, 0.f, 0.f, 0.f}, d[4] = {0.f, 0.f, 0.f, 0.f};
            // staged block of the first lag of tile n: i = j - 2 tau + Kp - 1, tau = tau0 + 2 n
            const uint32_t lb0 = stage + (jw8 - 2 * tau0 + Kp - 1) * BLKB + frag8;
            if (2 * (tau0 + 14) + 1 < Kp) {                          // a whole group, every second lag inside: no checks
                const uint32_t lbs = lb0 - (second8 ? BLKB : 0);
#pragma unroll
                for (int n = 0; n < 8; n += 2) tile(c, lbs - 4 * n * BLKB, n), tile(d, lbs - 4 * (n + 1) * BLKB, n + 1);
#pragma unroll
                for (int e = 0; e < 4; e++) epilogue(lg, e, c[e] + d[e]);
            } else {
#pragma unroll
                for (int n = 0; n < 8; n++) {
                    const int k0 = 2 * (tau0 + 2 * n);
                    if (k0 < Kp) tile(c, lb0 - 4 * n * BLKB - ((second8 && k0 + 1 < Kp) ? BLKB : 0), n);   // (a missing second lag re-reads the first)
                }
#pragma unroll
                for (int e = 0; e < 4; e++)
                    if (2 * (tau0 + 2 * (2 * ft + (e & 1))) + (e >> 1) < Kp) epilogue(lg, e, c[e]);
            }
        }
    };
    auto mma_finalize8 = [&](const DiagItem& it) {
        const float fM = (float)a.M;
        const int64_t tb = (int64_t)(it.c * CJ + jw8) * G + T * it.r;    // first sample of the comb block (a multiple of 8)
        const int64_t t = tb + fg;
        auto gather = [&](uint32_t x) {                              // bits 4 g + t of a ballot -> bits g
            x = (x >> ft) & 0x11111111u;
            x = (x | (x >> 3)) & 0x03030303u;
            x = (x | (x >> 6)) & 0x000f000fu;
            return (x | (x >> 12)) & 0xffu;
        };
#pragma unroll
        for (int lg = 0; lg < NGRP8; lg++) {
            const int tau0 = 16 * lg + hh8;
            if (2 * tau0 >= it.Kp) break;
#pragma unroll
            for (int e = 0; e < 4; e++) {
                const int kk = 2 * (tau0 + 2 * (2 * ft + (e & 1))) + (e >> 1);
                const bool live = kk < it.Kp && t < a.n;
                const float pb = __fdiv_rn(rsum[lg][e], fM);
                if (live) {
                    a.pbar[(size_t)(it.ka + kk) * a.row_stride + t] = pb;
                    a.mm[(size_t)(it.ka + kk) * a.row_stride + t] = (uint8_t)(rmk[lg] >> (8 * e));
                }
                rsum[lg][e] = 0.f;
                const uint32_t bal = __ballot_sync(0xffffffffu, live && pb > a.theta);
                if (fg == 0 && kk < it.Kp && (tb >> 3) < 4 * a.bits_stride)
                    reinterpret_cast<uint8_t*>(a.bits + (size_t)(it.ka + kk) * a.bits_stride)[tb >> 3] = (uint8_t)gather(bal);
            }
            rmk[lg] = 0;
        }
    };
    // mean, threshold, outputs of the item; the sums go back to zero.  Thread = (row, comb block j, lag slot)
    auto finalize = [&](const DiagItem& it) {
        const float fM = (float)a.M;
        const int rr = tid % T, j = (tid / T) % CJ;
        const int64_t t = (int64_t)(it.c * CJ + j) * G + T * it.r + rr;
        const bool live = t < a.n;
        for (int kk = tid / (T * CJ); kk < it.Kp; kk += DG_THREADS / (T * CJ)) {   // warp-uniform
            const int idx = (j * KS + kk) * T + rr, k = it.ka + kk;
            const float pb = __fdiv_rn(sums[idx], fM);
            const uint32_t wd = __ballot_sync(0xffffffffu, live && pb > a.theta);
            // the warp holds 32 / T blocks of T samples: each writes its T mask bits
            if (rr == 0) {
                if (T == 16) {
                    if ((t >> 4) < 2 * a.bits_stride) reinterpret_cast<uint16_t*>(a.bits + (size_t)k * a.bits_stride)[t >> 4] = (uint16_t)(wd >> (lane & 16));
                } else {
                    if ((t >> 3) < 4 * a.bits_stride) reinterpret_cast<uint8_t*>(a.bits + (size_t)k * a.bits_stride)[t >> 3] = (uint8_t)(wd >> (lane & 24));
                }
            }
            if (live) {
                a.pbar[(size_t)k * a.row_stride + t] = pb;
                a.mm[(size_t)k * a.row_stride + t] = smm[idx];
            }
            sums[idx] = 0.f, smm[idx] = 0;
        }
    };

    int wi = blockIdx.x;
    if (wi >= nitems) return;
    DiagItem cur = decode(wi), nxt = cur;
    uint32_t step = 0;
    stage_load(cur, 0, 0);
    for (; wi < nitems; wi += gridDim.x) {
        const bool more = wi + (int)gridDim.x < nitems;
        if (more) nxt = decode(wi + gridDim.x);
        for (int m = 0; m < a.M; m++, step++) {
            const int buf = step & 1;
            // the next step's rows go to the other stage (released by the barrier that ended the step before this one)
            if (m + 1 < a.M || more) {
                if (m + 1 < a.M) stage_load(cur, m + 1, buf ^ 1);
                else stage_load(nxt, 0, buf ^ 1);
                asm volatile("cp.async.wait_group 1;" ::: "memory");
            } else {
                asm volatile("cp.async.wait_group 0;" ::: "memory");
            }
            __syncthreads();
            if (MMA && T == 16) mma_compute(cur, m, buf);
            else if (MMA) mma_compute8(cur, m, buf);
            else compute(cur, m, buf);
            __syncthreads();
        }
        if (MMA && T == 16) mma_finalize(cur);
        else if (MMA) mma_finalize8(cur);
        else finalize(cur);
        __syncthreads();
        cur = nxt;
    }
}

} // namespace

// packs W2 / b2 of the models and launches; d_v[m] = row 0 of the chunk inside model m's [2][lds][CH] buffer, CH = Hh = 32
// (narrow architecture) or 128 (paper scale)
gwi_status gwi_heads_fused(const gwi_model* const* models, int M, const __half* const* d_v, int64_t lds, int n, const int64_t* d_lags,
                           int n_lags, const int64_t* h_lags, float theta, uint32_t* d_bits, int64_t bits_stride, float* d_pbar,
                           uint8_t* d_mm, int64_t row_stride, float* d_prob, cudaStream_t st)
{
    const int CH = models[0]->arch.Hh;
    if (M < 1 || M > HF_MAX_M || (CH != 32 && CH != 128)) {
        gwi_set_error("gwi_heads_fused: 1..%d models with 32 or 128 head channels", HF_MAX_M);
        return GWI_ERR_UNSUPPORTED;
    }
    HeadsFusedArgs a;
    memset(a.w2, 0, sizeof(a.w2));
    for (int m = 0; m < M; m++) {
        a.v[m] = d_v[m];
        const float* W = models[m]->host_blob.data();
        for (int c = 0; c < CH / 2; c++) {
            __half lo = __float2half_rn(W[models[m]->off.W2 + 2 * c]), hi = __float2half_rn(W[models[m]->off.W2 + 2 * c + 1]);
            uint16_t ul, uh;
            memcpy(&ul, &lo, 2), memcpy(&uh, &hi, 2);
            a.w2[m][c] = (uint32_t)ul | ((uint32_t)uh << 16);
        }
        a.b2[m] = W[models[m]->off.b2];
    }
    a.lds = lds, a.n = n, a.M = M, a.n_lags = n_lags, a.lags = d_lags, a.theta = theta;
    a.bits = d_bits, a.bits_stride = bits_stride, a.pbar = d_pbar, a.mm = d_mm, a.row_stride = row_stride, a.prob = d_prob;
    // regular lag list k G (G a multiple of 16, mean rule): the comb schedule, in passes of at most DG_KS_MAX lags
    bool comb = !d_prob && n_lags >= 2 && h_lags != nullptr;
    int64_t G = 0;
    if (comb) {
        G = h_lags[1];
        comb = G > 0 && G % 16 == 0;
        for (int k = 0; k < n_lags && comb; k++) comb = h_lags[k] == (int64_t)k * G;
    }
    // 32-channel rows, up to 34 slides: the thread-per-item comb kernel below (measured 9 % faster per hour than the
    // diagonal kernel there: 18.9 against 20.7 ms with 33 lags, the per-item work is too small to pay for the running sums
    // in shared memory); longer lists and 128-channel rows: the diagonal kernel
    // GWI_HEADS_IMPL (A/B runs, 32-channel rows): 0 = the tensor-core variant of the diagonal kernel (default), 1 = the
    // element-wise diagonal kernel, 2 = the thread-per-item comb kernel (up to 34 slides)
    static const int impl = [] { const char* e = getenv("GWI_HEADS_IMPL"); return e ? atoi(e) : 0; }();
    if (comb && (CH == 32 ? (impl != 2 || n_lags > 34) : n % 8 == 0)) {
        const int T = CH == 32 ? DiagGeom<32>::T : DiagGeom<128>::T, CJ = CH == 32 ? DiagGeom<32>::CJ : DiagGeom<128>::CJ;
        const int64_t nG = (n + G - 1) / G, groups = (nG + CJ - 1) / CJ;
        const int npass = (n_lags + DG_KS_MAX - 1) / DG_KS_MAX, KS = (n_lags + npass - 1) / npass;
        const int64_t nitems = groups * npass * (G / T);
        comb = nitems <= INT32_MAX && G <= INT32_MAX;                    // 32-bit item arithmetic in the kernel
        if (comb) {
            // once per device (the attribute belongs to the device's copy of the kernel)
            static int sms_of[64] = {};
            int dev = 0;
            GWI_CUDA_CHECK(cudaGetDevice(&dev));
            int& sms = sms_of[dev & 63];
            if (!sms) {
                GWI_CUDA_CHECK(cudaFuncSetAttribute(k_heads_diag<32, false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                                    (int)DiagGeom<32>::smem_bytes(DG_KS_MAX)));
                GWI_CUDA_CHECK(cudaFuncSetAttribute(k_heads_diag<32, true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                                    (int)DiagGeom<32>::smem_bytes(DG_KS_MAX)));
                GWI_CUDA_CHECK(cudaFuncSetAttribute(k_heads_diag<128, true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                                    (int)DiagGeom<128>::smem_bytes(DG_KS_MAX)));
                GWI_CUDA_CHECK(cudaFuncSetAttribute(k_heads_diag<128, false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                                    (int)DiagGeom<128>::smem_bytes(DG_KS_MAX)));
                GWI_CUDA_CHECK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
            }
            const unsigned grid = (unsigned)std::min<int64_t>(nitems, sms);
            if (CH == 32 && impl == 1)
                k_heads_diag<32, false><<<grid, DG_THREADS, DiagGeom<32>::smem_bytes(KS), st>>>(a, n_lags, KS, npass, (int)G, (int)groups, (int)nitems);
            else if (CH == 32)
                k_heads_diag<32, true><<<grid, DG_THREADS, DiagGeom<32>::smem_bytes(KS), st>>>(a, n_lags, KS, npass, (int)G, (int)groups, (int)nitems);
            else if (impl == 1)
                k_heads_diag<128, false><<<grid, DG_THREADS, DiagGeom<128>::smem_bytes(KS), st>>>(a, n_lags, KS, npass, (int)G, (int)groups, (int)nitems);
            else
                k_heads_diag<128, true><<<grid, DG_THREADS, DiagGeom<128>::smem_bytes(KS), st>>>(a, n_lags, KS, npass, (int)G, (int)groups, (int)nitems);
            gwi_count_launch(1);
            GWI_CUDA_CHECK(cudaGetLastError());
            return GWI_OK;
        }
    }
    if (comb && CH == 32 && n_lags <= 34) {
        constexpr int CJ = 16;
        auto kern = k_heads_comb<32, 16, CJ, 2, 17, 2, GWI_COMB_MINB>;
        const int64_t nG = (n + G - 1) / G, groups = (nG + CJ - 1) / CJ;
        const size_t smem = (size_t)2 * (CJ + n_lags - 1) * 1024 + HF_MAX_M * 64;
        static bool attr_of[64] = {};
        int dev = 0;
        GWI_CUDA_CHECK(cudaGetDevice(&dev));
        if (!attr_of[dev & 63]) {
            GWI_CUDA_CHECK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 2 * (CJ + 34 - 1) * 1024 + HF_MAX_M * 64));
            attr_of[dev & 63] = true;
        }
        kern<<<(unsigned)(groups * (G / 16)), 512, smem, st>>>(a, n_lags, G);
    } else if (CH == 32) {
        k_heads_fused<32><<<(n + 255) / 256, 256, 0, st>>>(a);
    } else {
        k_heads_fused<128><<<(n + 255) / 256, 256, 0, st>>>(a);
    }
    gwi_count_launch(1);
    GWI_CUDA_CHECK(cudaGetLastError());
    return GWI_OK;
}
