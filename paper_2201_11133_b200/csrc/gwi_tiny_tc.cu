// gwi_tiny_tc.cu -- tcgen05 stream kernel for the narrow ("config-1") architecture: n_branch = 2, c_in = 1, R = 16,
// S = Hh = 32, k = 2 (the ensembles of BASELINE.json configs 3-5), FP16 mode.
//
// The path is bound by MUFU (256 tanh per output sample and model; SURVEY.md section 8(d) cfg 3).  The first kernel for
// this architecture (gwi_tiny.cu, warp-level mma.sync) spends as long in the legacy tensor path as in MUFU (a
// m16n8k16 mma.sync runs at a quarter of the tcgen05 rate) and is latency-bound between the two.  Here every
// contraction is a tcgen05.mma on a 128-row tile with the accumulators in tensor memory:
//
//   per (tile of 128 stream samples, branch):  lift -> L x [ GEMM1 -> gate -> GEMM2 ] -> u = ReLU(skip sum)
//     GEMM1  f|g/2 [128 x 32]   = [h(t-d) | h(t)] [128 x 32] . Wfg^T      A, B in shared memory (a dilation = a row offset
//                                                                         of the A descriptor, as in gwi_tc.cu)
//     gate   z' = tanh(f) (1 + tanh(g/2)) = 2 tanh(f) sigmoid(g)          one row per thread, 32 MUFU
//     GEMM2  [h | skip] [128 x 48] += z' [128 x 16] . [Wr/2 | Ws/2]^T     A = z' in tensor memory (written by the gate
//                                                                         over the g columns), fp32 master of h and the
//                                                                         skip sum ACCUMULATE in tensor memory
//     operand of the next block = fp16(h), one 32-byte row per thread to shared memory
//   Biases ride in the MMAs (one more K step per GEMM: a constant A tile with 1 in its first column times a B row that
//   holds the biases), so the epilogue threads neither load nor add them.
//   per tile: head  [128 x 32] = [u_H | u_L] [128 x 64] . W1^T  (A in tensor memory), ReLU, dot W2, sigmoid  (C.1 step 5)
//
// One persistent CTA per SM holds six tiles ("slots") in flight, four warps each (one per TMEM lane quadrant, a thread
// = one time step).  There is no dedicated MMA warp: after the slot's named barrier an elected lane of its first warp
// issues the slot's MMAs and commits them to the slot's mbarrier, on which the four warps then wait; six slots of
// independent work hide the ~400-clock issue -> complete -> wake latency of each tiny GEMM.  The weights of the model
// (52 KB with the bias steps) stay in shared memory for the whole launch.
//
// Overlap reuse: a slot works through a contiguous span of tiles; the last SR = 16 operand rows of every (branch, block)
// are kept in a shared-memory stash and put in front of the next tile's operand rows (all d <= 16), so a tile is 128
// output samples.  A span starts with one warm-up tile (the 128 samples before it, nothing stored) that fills the
// stash; before a chunk it is fed from the carried last `halo` input samples of the previous chunk, which is all the
// stashed rows depend on (receptive field <= halo + 1).  With a dilation > 16 the kernel falls back to recomputing a
// halo of `halo` rows per tile, as gwi_tiny.cu does.  Rows at global time t < 0 are forced to zero at every layer input
// (reading A4).  Every output sample is a fixed-order computation that does not depend on the tile it falls in, so
// chunked == unchunked bit for bit (reading A17).
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <vector>

#include "gwi_internal.h"
#include "gwi_tc_ptx.h"

using namespace tc;

namespace {

#ifndef GWI_TT_NSLOT
#define GWI_TT_NSLOT 6
#endif
constexpr int NSLOT = GWI_TT_NSLOT;
constexpr int TT_THREADS = NSLOT * 128;
constexpr int TT_MAX_L = 8;
constexpr int PADR = 64;                        // zero rows in front of a tile (past-tap reads of its first rows)
constexpr int X_CH = (PADR + 128) * 16;         // chunk-column stride of a slot's operand buffer (8 channels per chunk)
constexpr int X_SLOT = 2 * X_CH;                // 16 channels
// Biases ride in the MMAs: every B operand has one more K step whose first row holds the bias of its N columns, and
// the matching A operand is a constant tile with 1 in its first K column, so the epilogue threads add nothing
constexpr int WFG_L = 32 * 48 * 2;              // per (branch, layer): N = 32 (f | g/2) x K = 48 (past | current | bias step)
constexpr int WRS_L = 48 * 32 * 2;              // N = 48 (res | skip) x K = 32 (z' | bias step: br, bs)
constexpr int W1_B = 32 * 80 * 2;               // N = 32 x K = 80 ([u_H | u_L] | bias step: b1)
constexpr int ONES_B = 2 * 128 * 16;            // A operand of the bias steps: 128 rows x K = 16, element (r, 0) = 1
constexpr int SR = 16;                          // stashed operand rows per (branch, block)
constexpr int STASH_SLOT = 2 * TT_MAX_L * 2 * SR * 16;   // [branch][block][chunk][SR rows] x 16 B = 8 KB
constexpr int TCOLS = 80;                       // TMEM columns per slot: f 0-15, g 16-31 (z' over 16-23), h 32-47, skip 48-79

struct TtArgs {
    const uint8_t* w;     // [nb][L][WFG_L] | [nb][L][WRS_L] | W1_B, packed for the MMA B operand
    const __half* x;      // planar strain chunk: channel c at x + c * ldx, n samples
    const __half* xh;     // [2][halo] last halo samples of the previous chunk (zeros at the stream start)
    int64_t ldx, t0;      // t0 = global index of sample 0 of this chunk
    int n, L, halo, ntiles;
    int stash;            // 1: 128-sample tiles with stashed operand rows, 0: tiles of 128 - halo samples with recomputed halo
    int dil[TT_MAX_L];
    float* prob;          // fused head: [n] probabilities (null in time-slide mode)
    __half* u16;          // time-slide mode: [2][lds][32] half-head pre-activations v_b = W1_b u_b (+ b1), fp16, time-major; row 0 = sample 0
    int64_t lds;
    // constant-bank operands
    float lift[2][32];            // W_in[16], b_in[16]
    float head[33];               // W2[32], b2
};

__device__ __forceinline__ void named_bar(int id, int nthreads) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory"); }
__device__ __forceinline__ void tmem_st16(uint32_t taddr, const uint32_t (&v)[16])
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16};" ::"r"(taddr),
                 "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]), "r"(v[8]), "r"(v[9]),
                 "r"(v[10]), "r"(v[11]), "r"(v[12]), "r"(v[13]), "r"(v[14]), "r"(v[15])
                 : "memory");
}
__device__ __forceinline__ void tmem_st8(uint32_t taddr, const uint32_t (&v)[8])
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};" ::"r"(taddr), "r"(v[0]), "r"(v[1]),
                 "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7])
                 : "memory");
}

#ifdef GWI_TT_TRACE
__device__ unsigned long long g_tt_trace[8192];
#define TT_TRACE(code)                                                                          \
    do {                                                                                        \
        if (blockIdx.x == 0 && slot == 0 && q == TT_TRACE_Q && lane == 0 && tt_k < 8190) g_tt_trace[tt_k++] = ((unsigned long long)(code) << 48) | (clock64() & 0xffffffffffffull); \
    } while (0)
#ifndef TT_TRACE_Q
#define TT_TRACE_Q 0
#endif
#else
#define TT_TRACE(code)
#endif

#ifndef GWI_TT_ARRIVE
#define GWI_TT_ARRIVE 1
#endif
#ifndef GWI_TT_SPIN
#define GWI_TT_SPIN 0
#endif
#ifndef GWI_TT_SLEEP_NS
#define GWI_TT_SLEEP_NS 4000
#endif

// LT = compile-time number of blocks (the layer loop is unrolled, descriptor offsets become constants), 0 = any (a.L)
template <int LT>
__global__ void __launch_bounds__(TT_THREADS, 1) k_tiny_tc(const __grid_constant__ TtArgs a)
{
    extern __shared__ __align__(1024) uint8_t smem[];
    const int L = LT ? LT : a.L;
    const int OFF_WRS = 2 * L * WFG_L, OFF_W1 = OFF_WRS + 2 * L * WRS_L, OFF_ONES = OFF_W1 + W1_B,
              OFF_X = (OFF_ONES + ONES_B + 1023) & ~1023;
    const int OFF_STASH = OFF_X + NSLOT * X_SLOT;
    const int OFF_BAR = OFF_STASH + NSLOT * STASH_SLOT;
    const uint32_t sbase = smem_u32(smem);
    // warp index through a broadcast shuffle: the compiler then knows that everything derived from it (slot, TMEM and
    // shared-memory addresses, MMA descriptors) is warp-uniform and keeps it in uniform registers, which is what the
    // single-lane tcgen05.mma issue wants (no per-MMA vector -> uniform moves)
    const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0), lane = threadIdx.x & 31;
    const int slot = warp >> 2, q = warp & 3;
    const int r = q * 32 + lane;                                  // row of the tile = TMEM lane
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + OFF_BAR + 8 * NSLOT);

    // ---- one-time setup: weights -> shared memory, operand buffers zeroed (their pad rows stay zero), barriers, TMEM
    {
        const uint4* src = reinterpret_cast<const uint4*>(a.w);
        uint4* dst = reinterpret_cast<uint4*>(smem);
        for (int i = threadIdx.x; i < (OFF_W1 + W1_B) / 16; i += TT_THREADS) dst[i] = __ldg(src + i);
        uint4* on = reinterpret_cast<uint4*>(smem + OFF_ONES);
        for (int i = threadIdx.x; i < ONES_B / 16; i += TT_THREADS) on[i] = make_uint4(i < 128 ? 0x3C00u : 0u, 0, 0, 0);   // half(1.0) at k = 0
        uint4* zx = reinterpret_cast<uint4*>(smem + OFF_X);
        for (int i = threadIdx.x; i < NSLOT * (X_SLOT + STASH_SLOT) / 16; i += TT_THREADS) zx[i] = make_uint4(0, 0, 0, 0);
        if (threadIdx.x == 0) {
            for (int i = 0; i < NSLOT; i++) mbar_init(sbase + OFF_BAR + 8 * i, 1);
            mbar_fence_init();
        }
    }
    if (warp == 0) tmem_alloc(smem_u32(tmem_slot), 512);
    fence_proxy_async_smem();
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = __shfl_sync(0xffffffffu, *tmem_slot, 0);
    const uint32_t tcol = tmem + TCOLS * slot;                    // the slot's columns (lane field 0: MMA operands)
    const uint32_t tlane = tcol + ((uint32_t)(q * 32) << 16);     // this warp's lane quadrant (tcgen05.ld / st)
    const uint32_t mbar = sbase + OFF_BAR + 8 * slot;
    const uint32_t xs = sbase + OFF_X + slot * X_SLOT;            // the slot's operand buffer; row 0 of the tile at + PADR * 16
    const uint32_t xrow = xs + (PADR + r) * 16;
    const bool leader = q == 0;
    uint32_t ph = 0;                                              // phase of the slot's MMA barrier
    const uint32_t idesc32 = make_idesc_f16(128, 32), idesc48 = make_idesc_f16(128, 48);
    const uint64_t dX = make_sdesc(xs + PADR * 16, X_CH, 128);
    const uint64_t dWfg = make_sdesc(sbase, 32 * 16, 128), dWrs = make_sdesc(sbase + OFF_WRS, 48 * 16, 128),
                   dW1 = make_sdesc(sbase + OFF_W1, 32 * 16, 128), dOnes = make_sdesc(sbase + OFF_ONES, 128 * 16, 128);
    const int valid = a.stash ? 128 : 128 - a.halo;
    // stash mode: rows 128 - SR .. 127 exchange their operand row with the stash of (branch, block): the row kept from the
    // previous tile goes in front of the tile (rows -SR .. -1 of the operand buffer), the new one is kept for the next tile
    const bool tail = a.stash && r >= 128 - SR;
    const uint32_t stash0 = sbase + OFF_STASH + slot * STASH_SLOT + (r - (128 - SR)) * 16;
    const uint32_t xpre = xs + (PADR - SR + (r - (128 - SR))) * 16;
    auto put_operand = [&](int bi, const uint32_t (&pk)[8]) {
        st_shared_v4(xrow, pk[0], pk[1], pk[2], pk[3]);
        st_shared_v4(xrow + X_CH, pk[4], pk[5], pk[6], pk[7]);
        if (tail) {
            const uint32_t sa = stash0 + bi * (2 * SR * 16);
            const uint4 o0 = ld_shared_v4(sa), o1 = ld_shared_v4(sa + SR * 16);
            st_shared_v4(xpre, o0.x, o0.y, o0.z, o0.w);
            st_shared_v4(xpre + X_CH, o1.x, o1.y, o1.z, o1.w);
            st_shared_v4(sa, pk[0], pk[1], pk[2], pk[3]);
            st_shared_v4(sa + SR * 16, pk[4], pk[5], pk[6], pk[7]);
        }
    };

    // the leader's elected lane issues `f` (the slot's MMAs) and commits; everybody waits for the completion
#ifdef GWI_TT_TRACE
    int tt_k = 0;
#endif
    auto mma_round = [&](auto&& f) {
        TT_TRACE(1);
#if GWI_TT_ARRIVE
        if (leader) named_bar(1 + slot, 128);
        else asm volatile("bar.arrive %0, %1;" ::"r"(1 + slot), "r"(128) : "memory");
#else
        named_bar(1 + slot, 128);
#endif
        TT_TRACE(2);
        if (leader) {
            if (elect_one()) {
                TT_TRACE(11);
                tc_fence_after();
                TT_TRACE(12);
                f();
                TT_TRACE(13);
                tc_commit(mbar);
                TT_TRACE(14);
            }
            __syncwarp();
        }
        TT_TRACE(3);
#if GWI_TT_SPIN
        {
            uint32_t spins = 0;
            while (!mbar_test(mbar, ph))
                if (++spins > (1u << 26)) __trap();
        }
#else
        mbar_wait_sleep(mbar, ph, GWI_TT_SLEEP_NS);
#endif
        ph ^= 1;
        tc_fence_after();
        TT_TRACE(4);
    };

    // halo mode: tiles blockIdx * NSLOT + slot, + gridDim * NSLOT, ...; stash mode: the slot's span [k0, k1) of the tiles,
    // preceded by the warm-up tile k0 - 1
    const int64_t gs = (int64_t)blockIdx.x * NSLOT + slot, ns = (int64_t)gridDim.x * NSLOT;
    const int k0 = a.stash ? (int)(gs * a.ntiles / ns) : (int)gs, k1 = a.stash ? (int)((gs + 1) * a.ntiles / ns) : a.ntiles;
    const int kstep = a.stash ? 1 : (int)ns;
    for (int tile = (a.stash && k0 < k1) ? k0 - 1 : k0; tile < k1; tile += kstep) {
        const int64_t tl = (int64_t)tile * valid - (a.stash ? 0 : a.halo) + r;    // chunk-local time of this thread's row
        const bool dead = a.t0 + tl < 0;                          // before the stream start: zero at every layer input (A4)
        const bool store = (a.stash ? tile >= k0 : r >= a.halo) && tl >= 0 && tl < a.n;
        uint32_t uH[16];                                          // u of branch 0 (fp16 pairs), parked while branch 1 runs
#pragma unroll
        for (int b = 0; b < 2; b++) {
            // ---- lift (C.1 step 1): h0 = W_in x + b_in -> fp32 master in TMEM; skip sum starts at sum_i bs_i
            {
                float x = 0.f;
                if (tl >= 0) {
                    if (tl < a.n) x = __half2float(a.x[(int64_t)b * a.ldx + tl]);
                } else if (tl >= -a.halo) {
                    x = __half2float(a.xh[b * a.halo + a.halo + tl]);
                }
                uint32_t hv[16], pk[8];
#pragma unroll
                for (int c = 0; c < 16; c++) hv[c] = __float_as_uint(dead ? 0.f : fmaf(a.lift[b][c], x, a.lift[b][16 + c]));
#pragma unroll
                for (int c = 0; c < 8; c++) pk[c] = pack_half2(__uint_as_float(hv[2 * c]), __uint_as_float(hv[2 * c + 1]));
                tmem_st16(tlane + 32, hv);
                uint32_t sv[16];
#pragma unroll
                for (int c = 0; c < 16; c++) sv[c] = 0u;
                tmem_st16(tlane + 48, sv);                        // skip sum starts at 0; the bs_i arrive with GEMM2's bias step
                tmem_st16(tlane + 64, sv);
                put_operand(b * TT_MAX_L, pk);
                tc_wait_st();
                fence_proxy_async_smem();
                tc_fence_before();
            }
#pragma unroll
            for (int i = 0; i < (LT ? LT : L); i++) {
                const int d = a.dil[i];
                // ---- GEMM1: f | g/2 = [h(t-d) | h(t)] . Wfg^T                                  (C.1 step 2)
                mma_round([&] {
                    const uint64_t bw = dWfg + (uint64_t)(((b * L + i) * WFG_L) >> 4);
                    tc_mma_f16(tcol, dX - d, bw, idesc32, 0u);
                    tc_mma_f16(tcol, dX, bw + ((2 * 32 * 16) >> 4), idesc32, 1u);
                    tc_mma_f16(tcol, dOnes, bw + ((4 * 32 * 16) >> 4), idesc32, 1u);       // + bf | bg/2
                });
                // ---- gate: z' = tanh(f) (1 + tanh(g/2)) (biases already in the accumulators), fp16, over the g columns = A operand of GEMM2
                {
                    uint32_t f[16], g[16], z[8];
                    tmem_ld16(tlane, f);
                    tmem_ld16(tlane + 16, g);
                    tc_wait_ld();
                    TT_TRACE(5);
#pragma unroll
                    for (int c = 0; c < 8; c++) {
#ifdef GWI_TT_NOMUFU   // diagnostic only: the chain without the MUFU work
                        const float t0 = __uint_as_float(f[2 * c]) * 0.5f, t1 = __uint_as_float(f[2 * c + 1]) * 0.5f;
                        const float s0 = __uint_as_float(g[2 * c]) * 0.5f, s1 = __uint_as_float(g[2 * c + 1]) * 0.5f;
#else
                        const float t0 = tanh_approx(__uint_as_float(f[2 * c])), t1 = tanh_approx(__uint_as_float(f[2 * c + 1]));
                        const float s0 = tanh_approx(__uint_as_float(g[2 * c])), s1 = tanh_approx(__uint_as_float(g[2 * c + 1]));
#endif
                        z[c] = pack_half2(fmaf(t0, s0, t0), fmaf(t1, s1, t1));
                    }
                    TT_TRACE(6);
                    tmem_st8(tlane + 16, z);
                    tc_wait_st();
                    tc_fence_before();
                    TT_TRACE(7);
                }
                // ---- GEMM2: [h | skip] += z' . [Wr/2 | Ws/2]^T  (the last block's residual conv is dead, reading A8: its
                // contribution lands in h columns nobody reads again)
                mma_round([&] {
                    const uint64_t bw = dWrs + (uint64_t)(((b * L + i) * WRS_L) >> 4);
                    tc_mma_f16_ts(tcol + 32, tcol + 16, bw, idesc48, 1u);
                    tc_mma_f16(tcol + 32, dOnes, bw + ((2 * 48 * 16) >> 4), idesc48, 1u);   // + br | bs
                });
                if (i < L - 1) {
                    // ---- operand of the next block: fp16(h)
                    uint32_t hv[16], pk[8];
                    tmem_ld16(tlane + 32, hv);
                    tc_wait_ld();
                    TT_TRACE(8);
#pragma unroll
                    for (int c = 0; c < 8; c++) pk[c] = dead ? 0u : pack_half2(__uint_as_float(hv[2 * c]), __uint_as_float(hv[2 * c + 1]));
                    put_operand(b * TT_MAX_L + i + 1, pk);
                    TT_TRACE(9);
                    fence_proxy_async_smem();
                    tc_fence_before();
                    TT_TRACE(10);
                }
            }
            // ---- u_b = ReLU(skip sum)                                                         (C.1 step 3)
            uint32_t u[16];
            {
                uint32_t sv[32];
                tmem_ld32(tlane + 48, sv);
                tc_wait_ld();
#pragma unroll
                for (int c = 0; c < 16; c++)
                    u[c] = pack_half2(fmaxf(__uint_as_float(sv[2 * c]), 0.f), fmaxf(__uint_as_float(sv[2 * c + 1]), 0.f));
            }
            if (a.u16) {
                // ---- time-slide mode: the branch's half of the head's first layer, v_b = W1[:, 32 b : 32 b + 32] u_b (+ b1 for
                // b = 0).  W1 [u_H; u_L] + b1 = v_H[t] + v_L[t - lag] by linearity, so the per-lag work that follows
                // (gwi_heads.cu) is element-wise: no contraction per (sample, lag).
                tmem_st16(tlane + 32, u);
                tc_wait_st();
                tc_fence_before();
                mma_round([&] {
                    tc_mma_f16_ts(tcol, tcol + 32, dW1 + (uint64_t)(2 * b * 64), idesc32, 0u);
                    tc_mma_f16_ts(tcol, tcol + 40, dW1 + (uint64_t)((2 * b + 1) * 64), idesc32, 1u);
                    if (b == 0) tc_mma_f16(tcol, dOnes, dW1 + (uint64_t)(4 * 64), idesc32, 1u);
                });
                uint32_t v[32];
                tmem_ld32(tlane, v);
                tc_wait_ld();
                if (store) {
                    uint4* up = reinterpret_cast<uint4*>(a.u16 + ((size_t)b * a.lds + tl) * 32);
#pragma unroll
                    for (int c = 0; c < 4; c++)
                        up[c] = make_uint4(pack_half2(__uint_as_float(v[8 * c]), __uint_as_float(v[8 * c + 1])),
                                           pack_half2(__uint_as_float(v[8 * c + 2]), __uint_as_float(v[8 * c + 3])),
                                           pack_half2(__uint_as_float(v[8 * c + 4]), __uint_as_float(v[8 * c + 5])),
                                           pack_half2(__uint_as_float(v[8 * c + 6]), __uint_as_float(v[8 * c + 7])));
                }
                tc_fence_before();
            } else if (b == 0) {
#pragma unroll
                for (int c = 0; c < 16; c++) uH[c] = u[c];
            } else {
                // ---- head (C.1 steps 4, 5): [u_H | u_L] as the A operand in TMEM (h and skip columns), D over the f|g columns
                tmem_st16(tlane + 32, uH);
                tmem_st16(tlane + 48, u);
                tc_wait_st();
                tc_fence_before();
                mma_round([&] {
#pragma unroll
                    for (int kk = 0; kk < 4; kk++) tc_mma_f16_ts(tcol, tcol + 32 + 8 * kk, dW1 + (uint64_t)((kk * 2 * 32 * 16) >> 4), idesc32, kk > 0 ? 1u : 0u);
                    tc_mma_f16(tcol, dOnes, dW1 + (uint64_t)((8 * 32 * 16) >> 4), idesc32, 1u);   // + b1
                });
                uint32_t v[32];
                tmem_ld32(tlane, v);
                tc_wait_ld();
                float y0 = 0.f, y1 = 0.f, y2 = 0.f, y3 = 0.f;
#pragma unroll
                for (int c = 0; c < 32; c += 4) {
                    y0 = fmaf(a.head[c], fmaxf(__uint_as_float(v[c]), 0.f), y0);
                    y1 = fmaf(a.head[c + 1], fmaxf(__uint_as_float(v[c + 1]), 0.f), y1);
                    y2 = fmaf(a.head[c + 2], fmaxf(__uint_as_float(v[c + 2]), 0.f), y2);
                    y3 = fmaf(a.head[c + 3], fmaxf(__uint_as_float(v[c + 3]), 0.f), y3);
                }
                const float y = ((y0 + y1) + (y2 + y3)) + a.head[32];
                if (store) a.prob[tl] = 1.0f / (1.0f + __expf(-y));
                tc_fence_before();
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) tmem_dealloc(tmem, 512);
}

inline uint16_t h16(float v)
{
    __half h = __float2half_rn(v);
    uint16_t u;
    memcpy(&u, &h, 2);
    return u;
}

} // namespace

struct GwiTinyTcPack {
    uint8_t* d_w = nullptr;
    size_t w_bytes = 0;
    int smem = 0, num_sms = 148, halo = 16, stash = 0;
    float lift[2][32], head[33];
};

bool gwi_tiny_tc_supported(const GwiArch& a)
{
    if (a.n_branch != 2 || a.c_in != 1 || a.R != 16 || a.S != 32 || a.Hh != 32 || a.k != 2 || a.L > TT_MAX_L) return false;
    int s = 0;
    for (int i = 0; i < a.L; i++) {
        if (a.dil[i] > PADR) return false;
        s += a.dil[i];
    }
    return s <= 64;
}

int gwi_tiny_tc_halo(const gwi_model* m) { return m->tinytc ? m->tinytc->halo : 0; }

gwi_status gwi_tiny_tc_pack(gwi_model* m)
{
    const GwiArch& a = m->arch;
    const int L = a.L;
    GwiTinyTcPack* p = new GwiTinyTcPack();
    m->tinytc = p;
    int sum = 0;
    for (int i = 0; i < L; i++) sum += a.dil[i];
    p->halo = ((sum + 15) / 16) * 16;
    if (p->halo < 16) p->halo = 16;
    p->stash = 1;
    for (int i = 0; i < L; i++)
        if (a.dil[i] > SR) p->stash = 0;
    const float* W = m->host_blob.data();
    const size_t off_wrs = (size_t)2 * L * WFG_L, off_w1 = off_wrs + (size_t)2 * L * WRS_L;
    p->w_bytes = off_w1 + W1_B;
    std::vector<uint16_t> w(p->w_bytes / 2, 0);
    memset(p->lift, 0, sizeof(p->lift));
    // B operand, K-major, no swizzle: element (n, k) of an N x K block at (k / 8) * (N * 8) + n * 8 + k % 8 (halves)
    for (int b = 0; b < 2; b++) {
        for (int c = 0; c < 16; c++) p->lift[b][c] = W[m->off.W_in[b] + c], p->lift[b][16 + c] = W[m->off.b_in[b] + c];
        for (int i = 0; i < L; i++) {
            const GwiLayerOff& lo = m->off.layer[b][i];
            uint16_t* fg = w.data() + ((size_t)(b * L + i) * WFG_L) / 2;
            for (int n = 0; n < 32; n++) {
                for (int k = 0; k < 32; k++) {
                    const int tap = k < 16 ? 0 : 1, kin = k & 15;    // tap 0 = past sample, tap 1 = current (reading A5)
                    const float v = n < 16 ? W[lo.Wf + ((int64_t)n * 16 + kin) * 2 + tap] : 0.5f * W[lo.Wg + ((int64_t)(n - 16) * 16 + kin) * 2 + tap];
                    fg[(k / 8) * (32 * 8) + n * 8 + k % 8] = h16(v);
                }
                fg[4 * (32 * 8) + n * 8] = h16(n < 16 ? W[lo.bf + n] : 0.5f * W[lo.bg + n - 16]);   // k = 32: the bias step
            }
            uint16_t* rs = w.data() + (off_wrs + (size_t)(b * L + i) * WRS_L) / 2;
            for (int n = 0; n < 48; n++) {
                for (int k = 0; k < 16; k++) {
                    const float v = n < 16 ? 0.5f * W[lo.Wr + (int64_t)n * 16 + k] : 0.5f * W[lo.Ws + (int64_t)(n - 16) * 16 + k];
                    rs[(k / 8) * (48 * 8) + n * 8 + k % 8] = h16(v);
                }
                rs[2 * (48 * 8) + n * 8] = h16(n < 16 ? W[lo.br + n] : W[lo.bs + n - 16]);          // k = 16: the bias step
            }
        }
    }
    uint16_t* w1 = w.data() + off_w1 / 2;
    for (int n = 0; n < 32; n++) {
        for (int k = 0; k < 64; k++) w1[(k / 8) * (32 * 8) + n * 8 + k % 8] = h16(W[m->off.W1 + (int64_t)n * 64 + k]);
        w1[8 * (32 * 8) + n * 8] = h16(W[m->off.b1 + n]);                                           // k = 64: the bias step
    }
    for (int c = 0; c < 32; c++) p->head[c] = W[m->off.W2 + c];
    p->head[32] = W[m->off.b2];
    GWI_CUDA_CHECK(cudaMalloc((void**)&p->d_w, p->w_bytes));
    GWI_CUDA_CHECK(cudaMemcpy(p->d_w, w.data(), p->w_bytes, cudaMemcpyHostToDevice));
    p->smem = (int)(((off_w1 + W1_B + ONES_B + 1023) & ~(size_t)1023) + NSLOT * (X_SLOT + STASH_SLOT) + 8 * NSLOT + 16);
    cudaDeviceProp prop;
    GWI_CUDA_CHECK(cudaGetDeviceProperties(&prop, m->device));
    p->num_sms = prop.multiProcessorCount;
    GWI_CUDA_CHECK(cudaFuncSetAttribute(k_tiny_tc<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, p->smem));
    GWI_CUDA_CHECK(cudaFuncSetAttribute(k_tiny_tc<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, p->smem));
    return GWI_OK;
}

void gwi_tiny_tc_free(gwi_model* m)
{
    GwiTinyTcPack* p = m->tinytc;
    if (!p) return;
    cudaFree(p->d_w);
    delete p;
    m->tinytc = nullptr;
}

// One chunk of n samples of a planar fp16 stream through one model: probabilities (fused head) or, with d_prob == null,
// the branch features u as fp16 time-major rows at d_u16 (row of sample 0 inside a [2][lds][32] buffer).  xh_cur: the
// carried last halo samples of the previous chunk ([2][halo]).
gwi_status gwi_tiny_tc_stream(const gwi_model* m, const __half* d_x, int64_t ldx, int n, int64_t t0, const __half* xh_cur,
                              float* d_prob, __half* d_u16, int64_t lds, cudaStream_t st)
{
    const GwiTinyTcPack* p = m->tinytc;
    TtArgs a;
    a.w = p->d_w, a.x = d_x, a.xh = xh_cur, a.ldx = ldx, a.t0 = t0, a.n = n, a.L = m->arch.L, a.halo = p->halo;
    a.stash = p->stash;
    const int valid = a.stash ? 128 : 128 - p->halo;
    a.ntiles = (n + valid - 1) / valid;
    for (int i = 0; i < TT_MAX_L; i++) a.dil[i] = i < m->arch.L ? m->arch.dil[i] : 0;
    a.prob = d_prob, a.u16 = d_prob ? nullptr : d_u16, a.lds = lds;
    memcpy(a.lift, p->lift, sizeof(a.lift)), memcpy(a.head, p->head, sizeof(a.head));
    const int slots = (a.ntiles + NSLOT - 1) / NSLOT;
    const int grid = slots < p->num_sms ? slots : p->num_sms;
    if (a.L == 4) k_tiny_tc<4><<<grid, TT_THREADS, p->smem, st>>>(a);
    else k_tiny_tc<0><<<grid, TT_THREADS, p->smem, st>>>(a);
    gwi_count_launch(1);
    GWI_CUDA_CHECK(cudaGetLastError());
#ifdef GWI_TT_TRACE
    if (const char* tp = getenv("GWI_TT_TRACE_FILE")) {
        cudaStreamSynchronize(st);
        std::vector<unsigned long long> ev(8192);
        cudaMemcpyFromSymbol(ev.data(), g_tt_trace, ev.size() * 8);
        if (FILE* f = fopen(tp, "w")) {
            for (auto e : ev) fprintf(f, "%llu %llu\n", e >> 48, e & 0xffffffffffffull);
            fclose(f);
        }
    }
#endif
    return GWI_OK;
}
