// gwi_tc.cu -- FP16-mode tensor-core path for paper-scale models (R = 64, S = Hh = 128, k = 2, c_in = 1).
//
// Two kernels, both hand-written tcgen05 (sm_100a) with accumulators in TMEM:
//
//  k_stack  one persistent CTA per SM walks "jobs" = (pair of windows, branch).  For every 128-timestep tile it runs
//           the lift and all L gated residual blocks depth-first (DESIGN.md C.1 steps 1-3), so that
//           no activation of a block ever goes to HBM:
//             GEMM1  [128 x 128] = [h(t-d) | h(t)] [128 x 128] . [Wf|Wg/2]^T      (tcgen05.mma, fp32 accum in TMEM)
//             gate   z' = tanh(f) (1 + tanh(g/2)) = 2 tanh(f) sigmoid(g)           (epilogue warps, MUFU tanh.approx)
//             GEMM2  skip[128 x 128] += z' (Ws/2)^T ;  res[128 x 64] = z' (Wr/2)^T  (skip sum stays in TMEM for all L)
//             h     += res + br  (fp32 master in registers), fp16 copy -> shared memory = next block's operand
//           Time runs along M (TMEM lanes), channels along K/N.  The past tap of a dilated conv is the SAME shared
//           buffer addressed d rows earlier (no-swizzle K-major layout, rows 16 bytes apart), so a dilation costs no
//           data movement; the d rows that precede a tile come from a per-layer stash in shared memory (d <= 64) or,
//           for d = 128, 256, 512, from an L2-resident ring in global memory that the bulk-copy engine prefetches.
//           Two windows ("slots") are in flight per CTA so that the tensor pipe works on one while the epilogue
//           warps gate the other.  Output: u = ReLU(sum of skips) per branch, fp16, tile-major in the workspace.
//  k_head   [128 x 128] = [u_H | u_L] . W1^T on tcgen05, then ReLU, dot with W2, sigmoid (C.1 steps 4-5).
//
// Roles in k_stack (320 threads): warps 0-3 epilogue of slot 0, warps 4-7 epilogue of slot 1 (warp % 4 = TMEM lane
// quadrant), warp 8 lane 0 = bulk-copy producer (weights, ring tiles), warp 9 lane 0 = MMA issuer.
#include <cstring>
#include <vector>

#include "gwi_internal.h"
#include "gwi_tc_ptx.h"

using namespace tc;

namespace {

constexpr int TM = 128;                 // timesteps per tile = MMA M
constexpr int TC_MAX_L = 20;
constexpr int WFG_BYTES = 128 * 128 * 2;            // B operand of GEMM1: N = 128 (f|g) x K = 128 (past|current)
constexpr int WRS_BYTES = 192 * 64 * 2;             // B operand of GEMM2: N = 192 (skip|res) x K = 64
constexpr int X_CHUNK = 192 * 16;                   // chunk-column stride of the X buffer (64 pre rows + 128 rows)
constexpr int X_BYTES = 8 * X_CHUNK;                // 24576
constexpr int PST_BYTES = 8 * 128 * 16;             // 16384: one past tile, chunk stride 2048
constexpr int STASH_BYTES = 32768;                  // per slot: sum over layers with d <= 64 of d rows x 128 B
constexpr int BIAS_FLOATS = 192;                    // per layer: bf[64], bg/2[64], br[64]
constexpr int U_TILE_BYTES = 16 * 128 * 16;         // 32768: u tile, 16 chunks x 128 rows x 16 B
constexpr int NTHREADS = 320;

struct TcMeta {
    int L, n_branch;
    int dil[TC_MAX_L];
    int big[TC_MAX_L];        // 1: d is a multiple of 128 (history through the global ring), 0: d <= 64 (stash)
    int D[TC_MAX_L];          // d / 128 for big layers
    int stash_off[TC_MAX_L];  // byte offset of the layer's stash inside the slot's stash area
    int ring_off[TC_MAX_L];   // first ring entry (in tiles) of the layer
    int ring_tiles;           // ring entries per slot
};

struct StackArgs {
    const uint8_t* wfg;   // [n_branch][L][WFG_BYTES]
    const uint8_t* wrs;   // [n_branch][L][WRS_BYTES]
    const float* bias;    // [n_branch][L][192]
    const float* cst;     // [n_branch][256]: W_in[64], b_in[64], sum_i bs_i[128]
    const __half* strain; // [B][T][C]
    int64_t w0, nwin;     // windows [w0, w0 + nwin) of this launch
    int T, ntiles, C;
    uint8_t* ring;        // [gridDim.x][2][ring_tiles][PST_BYTES]
    uint8_t* u;           // [nwin][n_branch][ntiles][U_TILE_BYTES]
    TcMeta meta;
};

// ---- shared memory map of k_stack ----------------------------------------------------------------------------------
constexpr int SM_WFG = 0;
constexpr int SM_WRS = SM_WFG + WFG_BYTES;
constexpr int SM_X = SM_WRS + WRS_BYTES;                  // 2 slots
constexpr int SM_PST = SM_X + 2 * X_BYTES;                // 2 slots
constexpr int SM_STASH = SM_PST + 2 * PST_BYTES;          // 2 slots
constexpr int SM_BIAS = SM_STASH + 2 * STASH_BYTES;       // L x 192 floats
constexpr int SM_BAR = SM_BIAS + TC_MAX_L * BIAS_FLOATS * 4;
constexpr int SM_TOTAL = SM_BAR + 256;

enum { B_WFG_FULL = 0, B_WFG_FREE, B_WRS_FULL, B_WRS_FREE, B_FG_FULL, B_Z_READY = B_FG_FULL + 2, B_RS_FULL = B_Z_READY + 2,
       B_H_READY = B_RS_FULL + 2, B_PST_FULL = B_H_READY + 2, B_PST_FREE = B_PST_FULL + 2, B_COUNT = B_PST_FREE + 2 };

__global__ void __launch_bounds__(NTHREADS, 1) k_stack(const StackArgs a)
{
    extern __shared__ __align__(1024) uint8_t smem[];
    const uint32_t sbase = smem_u32(smem);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const TcMeta& M = a.meta;
    const int L = M.L, nb = M.n_branch;
    auto bar = [&](int i) { return sbase + SM_BAR + 8 * i; };
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + SM_BAR + 8 * B_COUNT);

    if (threadIdx.x == 0) {
        for (int i = 0; i < B_COUNT; i++) {
            uint32_t cnt = (i >= B_Z_READY && i < B_Z_READY + 2) || (i >= B_H_READY && i < B_H_READY + 2) ? 128u : 1u;
            mbar_init(bar(i), cnt);
        }
        mbar_fence_init();
    }
    if (warp == 8) tmem_alloc(smem_u32(tmem_slot), 512);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;
    // TMEM columns: slot s: f|g accumulator (res reuses its first 64 columns) at 128 s, skip sum at 256 + 128 s

    const int64_t npairs = (a.nwin + 1) / 2;
    const int64_t njobs = npairs * nb;
    // phase counters (each role keeps its own copy; the schedules are identical by construction)
    uint32_t n_it = 0;                 // (job, tile, layer) iterations done
    uint32_t n_pst[2] = {0, 0};        // ring-tile loads done per slot

    for (int64_t job = blockIdx.x; job < njobs; job += gridDim.x) {
        const int b = (int)(job % nb);
        const int64_t pair = job / nb;
        // ---- job prologue (all threads): bias table of this branch, zero the stashes and the X buffers --------------
        __syncthreads();
        {
            const float* bsrc = a.bias + (size_t)b * L * BIAS_FLOATS;
            float* bdst = reinterpret_cast<float*>(smem + SM_BIAS);
            for (int i = threadIdx.x; i < L * BIAS_FLOATS; i += NTHREADS) bdst[i] = bsrc[i];
            uint4 z4 = make_uint4(0, 0, 0, 0);
            uint4* zs = reinterpret_cast<uint4*>(smem + SM_STASH);
            for (int i = threadIdx.x; i < 2 * STASH_BYTES / 16; i += NTHREADS) zs[i] = z4;
            uint4* zx = reinterpret_cast<uint4*>(smem + SM_X);
            for (int i = threadIdx.x; i < 2 * X_BYTES / 16; i += NTHREADS) zx[i] = z4;
        }
        fence_proxy_async_smem();
        __syncthreads();

        if (warp == 8) {
            // =========================== producer: weights and ring tiles ===========================================
            if (lane == 0) {
                for (int j = 0; j < a.ntiles; j++)
                    for (int i = 0; i < L; i++, n_it++) {
                        mbar_wait(bar(B_WFG_FREE), (n_it & 1) ^ 1);
                        mbar_arrive_expect_tx(bar(B_WFG_FULL), WFG_BYTES);
                        bulk_g2s(sbase + SM_WFG, a.wfg + ((size_t)b * L + i) * WFG_BYTES, WFG_BYTES, bar(B_WFG_FULL));
                        if (M.big[i] && j >= M.D[i]) {
                            for (int s = 0; s < 2; s++) {
                                mbar_wait(bar(B_PST_FREE + s), (n_pst[s] & 1) ^ 1);
                                mbar_arrive_expect_tx(bar(B_PST_FULL + s), PST_BYTES);
                                const uint8_t* src = a.ring + (((size_t)blockIdx.x * 2 + s) * M.ring_tiles + M.ring_off[i] +
                                                               (j - M.D[i]) % (M.D[i] + 1)) * PST_BYTES;
                                bulk_g2s(sbase + SM_PST + s * PST_BYTES, src, PST_BYTES, bar(B_PST_FULL + s));
                                n_pst[s]++;
                            }
                        }
                        mbar_wait(bar(B_WRS_FREE), (n_it & 1) ^ 1);
                        mbar_arrive_expect_tx(bar(B_WRS_FULL), WRS_BYTES);
                        bulk_g2s(sbase + SM_WRS, a.wrs + ((size_t)b * L + i) * WRS_BYTES, WRS_BYTES, bar(B_WRS_FULL));
                    }
            }
            __syncwarp();
        } else if (warp == 9) {
            // =========================== MMA issuer ===================================================================
            if (lane == 0) {
                const uint32_t idesc128 = make_idesc_f16(128, 128), idesc64 = make_idesc_f16(128, 64);
                for (int j = 0; j < a.ntiles; j++)
                    for (int i = 0; i < L; i++, n_it++) {
                        const uint32_t ph = n_it & 1;
                        const int d = M.dil[i];
                        // ---- GEMM1: f|g = [h(t-d) | h(t)] . Wfg^T
                        mbar_wait(bar(B_WFG_FULL), ph);
                        for (int s = 0; s < 2; s++) {
                            mbar_wait(bar(B_H_READY + s), ph);
                            const uint32_t xs = sbase + SM_X + s * X_BYTES;
                            const uint32_t dt = tmem + 128 * s;
                            uint32_t acc = 0;
                            if (!M.big[i]) {
                                tc_fence_after();
                                for (int kk = 0; kk < 4; kk++, acc = 1)
                                    tc_mma_f16(dt, make_sdesc(xs + (64 - d) * 16 + 2 * kk * X_CHUNK, X_CHUNK, 128),
                                               make_sdesc(sbase + SM_WFG + 2 * kk * 2048, 2048, 128), idesc128, acc);
                            } else if (j >= M.D[i]) {
                                mbar_wait(bar(B_PST_FULL + s), n_pst[s] & 1);
                                n_pst[s]++;
                                tc_fence_after();
                                const uint32_t ps = sbase + SM_PST + s * PST_BYTES;
                                for (int kk = 0; kk < 4; kk++, acc = 1)
                                    tc_mma_f16(dt, make_sdesc(ps + 2 * kk * 2048, 2048, 128),
                                               make_sdesc(sbase + SM_WFG + 2 * kk * 2048, 2048, 128), idesc128, acc);
                            } else {
                                tc_fence_after();
                            }
                            for (int kk = 0; kk < 4; kk++, acc = 1)
                                tc_mma_f16(dt, make_sdesc(xs + 64 * 16 + 2 * kk * X_CHUNK, X_CHUNK, 128),
                                           make_sdesc(sbase + SM_WFG + (8 + 2 * kk) * 2048, 2048, 128), idesc128, acc);
                            tc_commit(bar(B_FG_FULL + s));
                            if (M.big[i] && j >= M.D[i]) tc_commit(bar(B_PST_FREE + s));
                        }
                        tc_commit(bar(B_WFG_FREE));
                        // ---- GEMM2: skip += z' Ws'^T ; res = z' Wr'^T
                        mbar_wait(bar(B_WRS_FULL), ph);
                        for (int s = 0; s < 2; s++) {
                            mbar_wait(bar(B_Z_READY + s), ph);
                            tc_fence_after();
                            const uint32_t zs = sbase + SM_X + s * X_BYTES + 64 * 16;
                            for (int kk = 0; kk < 4; kk++)
                                tc_mma_f16(tmem + 256 + 128 * s, make_sdesc(zs + 2 * kk * X_CHUNK, X_CHUNK, 128),
                                           make_sdesc(sbase + SM_WRS + 2 * kk * 3072, 3072, 128), idesc128,
                                           (i > 0 || kk > 0) ? 1u : 0u);
                            if (i < L - 1)   // reading A8: the last block's residual conv has no effect
                                for (int kk = 0; kk < 4; kk++)
                                    tc_mma_f16(tmem + 128 * s, make_sdesc(zs + 2 * kk * X_CHUNK, X_CHUNK, 128),
                                               make_sdesc(sbase + SM_WRS + 128 * 16 + 2 * kk * 3072, 3072, 128), idesc64,
                                               kk > 0 ? 1u : 0u);
                            tc_commit(bar(B_RS_FULL + s));
                        }
                        tc_commit(bar(B_WRS_FREE));
                    }
            }
            __syncwarp();
        } else {
            // =========================== epilogue warpgroup of slot s ==================================================
            const int s = warp >> 2;
            const int r = (warp & 3) * 32 + lane;                    // row of the tile = TMEM lane
            const int64_t wl = 2 * pair + s;                          // window index inside this launch
            const bool valid = wl < a.nwin;
            const int64_t w = a.w0 + (valid ? wl : a.nwin - 1);
            const uint32_t xs = sbase + SM_X + s * X_BYTES;
            const uint32_t st0 = sbase + SM_STASH + s * STASH_BYTES;
            const uint32_t lane_t = tmem + ((uint32_t)((warp & 3) * 32) << 16);
            uint8_t* ring_s = a.ring + ((size_t)blockIdx.x * 2 + s) * M.ring_tiles * PST_BYTES;
            const float* cst = a.cst + b * 256;
            const float* biasL = reinterpret_cast<const float*>(smem + SM_BIAS);
            float h[64];

            // writes the fp16 copy of h as the operand of layer `inext` for tile j, maintains stash / ring, signals MMA
            auto publish = [&](int inext, int j) {
                uint32_t pk[32];
#pragma unroll
                for (int c = 0; c < 32; c++) pk[c] = pack_half2(h[2 * c], h[2 * c + 1]);
#pragma unroll
                for (int c = 0; c < 8; c++)
                    st_shared_v4(xs + (64 + r) * 16 + c * X_CHUNK, pk[4 * c], pk[4 * c + 1], pk[4 * c + 2], pk[4 * c + 3]);
                const int d = M.dil[inext];
                if (!M.big[inext]) {
                    if (r >= 128 - d) {
                        const int rp = r - (128 - d);
                        const uint32_t sb = st0 + M.stash_off[inext] + rp * 16;
#pragma unroll
                        for (int c = 0; c < 8; c++) {
                            uint4 old = ld_shared_v4(sb + c * d * 16);
                            st_shared_v4(xs + (64 - d + rp) * 16 + c * X_CHUNK, old.x, old.y, old.z, old.w);
                            st_shared_v4(sb + c * d * 16, pk[4 * c], pk[4 * c + 1], pk[4 * c + 2], pk[4 * c + 3]);
                        }
                    }
                } else {
                    uint8_t* g = ring_s + (size_t)(M.ring_off[inext] + j % (M.D[inext] + 1)) * PST_BYTES + r * 16;
#pragma unroll
                    for (int c = 0; c < 8; c++)
                        *reinterpret_cast<uint4*>(g + c * 2048) = make_uint4(pk[4 * c], pk[4 * c + 1], pk[4 * c + 2], pk[4 * c + 3]);
                    __threadfence();
                    fence_proxy_async();
                }
                tc_fence_before();
                fence_proxy_async_smem();
                mbar_arrive(bar(B_H_READY + s));
            };

            for (int j = 0; j < a.ntiles; j++) {
                // ---- lift: h0 = W_in x + b_in                                                   (C.1 step 1)
                {
                    const int t = j * TM + r;
                    float x = 0.f;
                    if (t < a.T) x = __half2float(a.strain[((size_t)w * a.T + t) * a.C + b]);
#pragma unroll
                    for (int c = 0; c < 64; c++) h[c] = fmaf(__ldg(cst + c), x, __ldg(cst + 64 + c));
                    tc_wait_ld();   // the previous tile's TMEM reads of this thread are complete
                    publish(0, j);
                }
                for (int i = 0; i < L; i++, n_it++) {
                    const uint32_t ph = n_it & 1;
                    const float* bl = biasL + i * BIAS_FLOATS;
                    // ---- gate: z' = tanh(f + bf) * (1 + tanh(g/2 + bg/2))
                    mbar_wait(bar(B_FG_FULL + s), ph);
                    tc_fence_after();
#pragma unroll
                    for (int cc = 0; cc < 2; cc++) {
                        uint32_t f[32], g[32];
                        tmem_ld32(lane_t + 128 * s + 32 * cc, f);
                        tmem_ld32(lane_t + 128 * s + 64 + 32 * cc, g);
                        tc_wait_ld();
                        uint32_t pk[16];
#pragma unroll
                        for (int c = 0; c < 32; c += 2) {
                            float tf0 = tanh_approx(__uint_as_float(f[c]) + bl[32 * cc + c]);
                            float tg0 = tanh_approx(__uint_as_float(g[c]) + bl[64 + 32 * cc + c]);
                            float tf1 = tanh_approx(__uint_as_float(f[c + 1]) + bl[32 * cc + c + 1]);
                            float tg1 = tanh_approx(__uint_as_float(g[c + 1]) + bl[64 + 32 * cc + c + 1]);
                            pk[c >> 1] = pack_half2(fmaf(tf0, tg0, tf0), fmaf(tf1, tg1, tf1));
                        }
#pragma unroll
                        for (int c = 0; c < 4; c++)
                            st_shared_v4(xs + (64 + r) * 16 + (4 * cc + c) * X_CHUNK, pk[4 * c], pk[4 * c + 1], pk[4 * c + 2],
                                         pk[4 * c + 3]);
                    }
                    tc_fence_before();
                    fence_proxy_async_smem();
                    mbar_arrive(bar(B_Z_READY + s));
                    // ---- residual update (or, after the last block, the branch output)
                    mbar_wait(bar(B_RS_FULL + s), ph);
                    tc_fence_after();
                    if (i < L - 1) {
#pragma unroll
                        for (int cc = 0; cc < 2; cc++) {
                            uint32_t v[32];
                            tmem_ld32(lane_t + 128 * s + 32 * cc, v);
                            tc_wait_ld();
#pragma unroll
                            for (int c = 0; c < 32; c++) h[32 * cc + c] += __uint_as_float(v[c]) + bl[128 + 32 * cc + c];
                        }
                        publish(i + 1, j);
                    } else {
                        // u = ReLU(sum_i skip_i) -> fp16 tile in the workspace                       (C.1 step 3)
                        uint8_t* ut = a.u + (((size_t)wl * nb + b) * a.ntiles + j) * U_TILE_BYTES + r * 16;
#pragma unroll
                        for (int cc = 0; cc < 4; cc++) {
                            uint32_t v[32];
                            tmem_ld32(lane_t + 256 + 128 * s + 32 * cc, v);
                            tc_wait_ld();
                            if (valid) {
#pragma unroll
                                for (int c = 0; c < 4; c++) {
                                    uint32_t q[4];
#pragma unroll
                                    for (int e = 0; e < 4; e++) {
                                        int col = 8 * c + 2 * e;
                                        float u0 = fmaxf(__uint_as_float(v[col]) + __ldg(cst + 128 + 32 * cc + col), 0.f);
                                        float u1 = fmaxf(__uint_as_float(v[col + 1]) + __ldg(cst + 128 + 32 * cc + col + 1), 0.f);
                                        q[e] = pack_half2(u0, u1);
                                    }
                                    *reinterpret_cast<uint4*>(ut + (4 * cc + c) * 2048) = make_uint4(q[0], q[1], q[2], q[3]);
                                }
                            }
                        }
                    }
                }
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 8) tmem_dealloc(tmem, 512);
}

// ---- head kernel ---------------------------------------------------------------------------------------------------
struct HeadArgs {
    const uint8_t* w1;    // B operand: N = 128 x K = n_branch*128, chunk-column (chunk stride 2048)
    const float* hc;      // b1[128], W2[128], b2
    const uint8_t* u;     // [nwin][n_branch][ntiles][U_TILE_BYTES]
    float* prob;          // [B][T]
    int64_t w0, nwin;
    int T, ntiles, n_branch;
};
constexpr int HEAD_THREADS = 192;   // warps 0-3 epilogue, warp 4 producer, warp 5 MMA

__global__ void __launch_bounds__(HEAD_THREADS, 1) k_head_tc(const HeadArgs a)
{
    extern __shared__ __align__(1024) uint8_t smem[];
    const uint32_t sbase = smem_u32(smem);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int nb = a.n_branch;
    const int W1B = nb * U_TILE_BYTES;            // bytes of W1 blob == bytes of one u stage
    const int OFF_U = W1B, OFF_BAR = W1B + 2 * W1B;
    // barriers: 0 w1_full, 1-2 u_full[st], 3-4 u_free[st], 5-6 acc_full[st], 7-8 acc_free[st]
    auto bar = [&](int i) { return sbase + OFF_BAR + 8 * i; };
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + OFF_BAR + 8 * 9);
    if (threadIdx.x == 0) {
        for (int i = 0; i < 9; i++) mbar_init(bar(i), (i == 7 || i == 8) ? 128u : 1u);
        mbar_fence_init();
    }
    if (warp == 4) tmem_alloc(smem_u32(tmem_slot), 256);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;
    const int64_t nitems = a.nwin * a.ntiles;

    if (warp == 4) {
        if (lane == 0) {
            mbar_arrive_expect_tx(bar(0), W1B);
            bulk_g2s(sbase, a.w1, W1B, bar(0));
            uint32_t n = 0;
            for (int64_t it = blockIdx.x; it < nitems; it += gridDim.x, n++) {
                const int st = n & 1;
                const int64_t wl = it / a.ntiles, j = it % a.ntiles;
                mbar_wait(bar(3 + st), ((n >> 1) & 1) ^ 1);
                mbar_arrive_expect_tx(bar(1 + st), W1B);
                for (int b = 0; b < nb; b++)
                    bulk_g2s(sbase + OFF_U + st * W1B + b * U_TILE_BYTES,
                             a.u + (((size_t)wl * nb + b) * a.ntiles + j) * U_TILE_BYTES, U_TILE_BYTES, bar(1 + st));
            }
        }
        __syncwarp();
    } else if (warp == 5) {
        if (lane == 0) {
            const uint32_t idesc = make_idesc_f16(128, 128);
            mbar_wait(bar(0), 0);
            uint32_t n = 0;
            for (int64_t it = blockIdx.x; it < nitems; it += gridDim.x, n++) {
                const int st = n & 1;
                const uint32_t ph = (n >> 1) & 1;
                mbar_wait(bar(1 + st), ph);
                mbar_wait(bar(7 + st), ph ^ 1);
                tc_fence_after();
                for (int kk = 0; kk < nb * 8; kk++)
                    tc_mma_f16(tmem + 128 * st, make_sdesc(sbase + OFF_U + st * W1B + 2 * kk * 2048, 2048, 128),
                               make_sdesc(sbase + 2 * kk * 2048, 2048, 128), idesc, kk > 0 ? 1u : 0u);
                tc_commit(bar(5 + st));
                tc_commit(bar(3 + st));
            }
        }
        __syncwarp();
    } else {
        const int r = warp * 32 + lane;
        const uint32_t lane_t = tmem + ((uint32_t)(warp * 32) << 16);
        const float b2 = __ldg(a.hc + 256);
        uint32_t n = 0;
        for (int64_t it = blockIdx.x; it < nitems; it += gridDim.x, n++) {
            const int st = n & 1;
            const uint32_t ph = (n >> 1) & 1;
            const int64_t wl = it / a.ntiles, j = it % a.ntiles;
            mbar_wait(bar(5 + st), ph);
            tc_fence_after();
            float y = b2;
#pragma unroll
            for (int cc = 0; cc < 4; cc++) {
                uint32_t v[32];
                tmem_ld32(lane_t + 128 * st + 32 * cc, v);
                tc_wait_ld();
#pragma unroll
                for (int c = 0; c < 32; c++) {
                    float hv = fmaxf(__uint_as_float(v[c]) + __ldg(a.hc + 32 * cc + c), 0.f);
                    y = fmaf(__ldg(a.hc + 128 + 32 * cc + c), hv, y);
                }
            }
            tc_fence_before();
            mbar_arrive(bar(7 + st));
            const int t = (int)j * TM + r;
            if (t < a.T) a.prob[(size_t)(a.w0 + wl) * a.T + t] = 1.0f / (1.0f + __expf(-y));
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 4) tmem_dealloc(tmem, 256);
}

} // namespace

// ---- host side: packing and launch -----------------------------------------------------------------------------------
struct GwiTcPack {
    uint8_t *d_wfg = nullptr, *d_wrs = nullptr, *d_w1 = nullptr;
    float *d_bias = nullptr, *d_cst = nullptr, *d_hc = nullptr;
    TcMeta meta;
    int num_sms = 148;
};

bool gwi_tc_supported(const GwiArch& a)
{
    if (a.R != 64 || a.S != 128 || a.Hh != 128 || a.k != 2 || a.c_in != 1 || a.n_branch > 2 || a.L > TC_MAX_L) return false;
    int stash = 0;
    for (int i = 0; i < a.L; i++) {
        int d = a.dil[i];
        if (d <= 64) stash += d * 128;
        else if (d % 128 != 0) return false;
    }
    return stash <= STASH_BYTES;
}

static inline uint16_t h16(float v)
{
    __half h = __float2half_rn(v);
    uint16_t u;
    memcpy(&u, &h, 2);
    return u;
}

gwi_status gwi_tc_pack(gwi_model* m)
{
    const GwiArch& a = m->arch;
    const int L = a.L, nb = a.n_branch;
    GwiTcPack* p = new GwiTcPack();
    m->tc = p;
    TcMeta& M = p->meta;
    memset(&M, 0, sizeof(M));
    M.L = L, M.n_branch = nb;
    int so = 0, ro = 0;
    for (int i = 0; i < L; i++) {
        M.dil[i] = a.dil[i];
        M.big[i] = a.dil[i] > 64;
        M.D[i] = M.big[i] ? a.dil[i] / 128 : 0;
        M.stash_off[i] = so, M.ring_off[i] = ro;
        if (M.big[i]) ro += M.D[i] + 1;
        else so += a.dil[i] * 128;
    }
    M.ring_tiles = ro > 0 ? ro : 1;
    const float* W = m->host_blob.data();
    std::vector<uint16_t> wfg((size_t)nb * L * WFG_BYTES / 2), wrs((size_t)nb * L * WRS_BYTES / 2), w1((size_t)nb * U_TILE_BYTES / 2);
    std::vector<float> bias((size_t)nb * L * BIAS_FLOATS), cst((size_t)nb * 256, 0.f), hc(257);
    for (int b = 0; b < nb; b++) {
        for (int c = 0; c < 64; c++) {
            cst[b * 256 + c] = W[m->off.W_in[b] + c];      // c_in = 1
            cst[b * 256 + 64 + c] = W[m->off.b_in[b] + c];
        }
        for (int i = 0; i < L; i++) {
            const GwiLayerOff& lo = m->off.layer[b][i];
            uint16_t* fg = wfg.data() + ((size_t)b * L + i) * (WFG_BYTES / 2);
            for (int n = 0; n < 128; n++)
                for (int k = 0; k < 128; k++) {
                    int tap = k < 64 ? 0 : 1, kin = k & 63;   // tap 0 = past sample, tap 1 = current (reading A5)
                    float v = n < 64 ? W[lo.Wf + ((int64_t)n * 64 + kin) * 2 + tap]
                                     : 0.5f * W[lo.Wg + ((int64_t)(n - 64) * 64 + kin) * 2 + tap];
                    fg[(k / 8) * (128 * 8) + n * 8 + (k % 8)] = h16(v);
                }
            uint16_t* rs = wrs.data() + ((size_t)b * L + i) * (WRS_BYTES / 2);
            for (int n = 0; n < 192; n++)
                for (int k = 0; k < 64; k++) {
                    float v = n < 128 ? 0.5f * W[lo.Ws + (int64_t)n * 64 + k] : 0.5f * W[lo.Wr + (int64_t)(n - 128) * 64 + k];
                    rs[(k / 8) * (192 * 8) + n * 8 + (k % 8)] = h16(v);
                }
            float* bl = bias.data() + ((size_t)b * L + i) * BIAS_FLOATS;
            for (int c = 0; c < 64; c++) {
                bl[c] = W[lo.bf + c];
                bl[64 + c] = 0.5f * W[lo.bg + c];
                bl[128 + c] = W[lo.br + c];
            }
            for (int q = 0; q < 128; q++) cst[b * 256 + 128 + q] += W[lo.bs + q];
        }
    }
    for (int mm = 0; mm < 128; mm++)
        for (int q = 0; q < nb * 128; q++) w1[(q / 8) * (128 * 8) + mm * 8 + (q % 8)] = h16(W[m->off.W1 + (int64_t)mm * nb * 128 + q]);
    for (int c = 0; c < 128; c++) hc[c] = W[m->off.b1 + c], hc[128 + c] = W[m->off.W2 + c];
    hc[256] = W[m->off.b2];
    auto up = [&](void** dst, const void* src, size_t bytes) -> cudaError_t {
        cudaError_t e = cudaMalloc(dst, bytes);
        if (e != cudaSuccess) return e;
        return cudaMemcpy(*dst, src, bytes, cudaMemcpyHostToDevice);
    };
    GWI_CUDA_CHECK(up((void**)&p->d_wfg, wfg.data(), wfg.size() * 2));
    GWI_CUDA_CHECK(up((void**)&p->d_wrs, wrs.data(), wrs.size() * 2));
    GWI_CUDA_CHECK(up((void**)&p->d_w1, w1.data(), w1.size() * 2));
    GWI_CUDA_CHECK(up((void**)&p->d_bias, bias.data(), bias.size() * 4));
    GWI_CUDA_CHECK(up((void**)&p->d_cst, cst.data(), cst.size() * 4));
    GWI_CUDA_CHECK(up((void**)&p->d_hc, hc.data(), hc.size() * 4));
    cudaDeviceProp prop;
    GWI_CUDA_CHECK(cudaGetDeviceProperties(&prop, m->device));
    p->num_sms = prop.multiProcessorCount;
    GWI_CUDA_CHECK(cudaFuncSetAttribute(k_stack, cudaFuncAttributeMaxDynamicSharedMemorySize, SM_TOTAL));
    GWI_CUDA_CHECK(cudaFuncSetAttribute(k_head_tc, cudaFuncAttributeMaxDynamicSharedMemorySize, 3 * 2 * U_TILE_BYTES + 256));
    return GWI_OK;
}

void gwi_tc_free(gwi_model* m)
{
    GwiTcPack* p = m->tc;
    if (!p) return;
    cudaFree(p->d_wfg), cudaFree(p->d_wrs), cudaFree(p->d_w1), cudaFree(p->d_bias), cudaFree(p->d_cst), cudaFree(p->d_hc);
    delete p;
    m->tc = nullptr;
}

static int64_t tc_chunk(int64_t B) { return B < 1024 ? B : 1024; }

size_t gwi_tc_workspace_bytes(const gwi_model* m, int64_t B, int32_t T)
{
    const GwiTcPack* p = m->tc;
    int64_t ntiles = (T + TM - 1) / TM;
    size_t ring = (size_t)p->num_sms * 2 * p->meta.ring_tiles * PST_BYTES;
    size_t u = (size_t)tc_chunk(B) * m->arch.n_branch * ntiles * U_TILE_BYTES;
    return ring + u + 256;
}

gwi_status gwi_tc_infer(const gwi_model* m, const __half* d_strain, int64_t B, int32_t T, float* d_prob, void* d_ws,
                        size_t ws_bytes, cudaStream_t st)
{
    const GwiTcPack* p = m->tc;
    const int nb = m->arch.n_branch;
    const int ntiles = (T + TM - 1) / TM;
    size_t ring_bytes = ((size_t)p->num_sms * 2 * p->meta.ring_tiles * PST_BYTES + 255) & ~(size_t)255;
    uint8_t* ring = (uint8_t*)d_ws;
    uint8_t* u = ring + ring_bytes;
    const int64_t Bc = tc_chunk(B);
    for (int64_t w0 = 0; w0 < B; w0 += Bc) {
        const int64_t nwin = (B - w0 < Bc) ? B - w0 : Bc;
        StackArgs sa;
        sa.wfg = p->d_wfg, sa.wrs = p->d_wrs, sa.bias = p->d_bias, sa.cst = p->d_cst, sa.strain = d_strain;
        sa.w0 = w0, sa.nwin = nwin, sa.T = T, sa.ntiles = ntiles, sa.C = nb * m->arch.c_in;
        sa.ring = ring, sa.u = u, sa.meta = p->meta;
        int64_t njobs = ((nwin + 1) / 2) * nb;
        int grid = (int)(njobs < p->num_sms ? njobs : p->num_sms);
        k_stack<<<grid, NTHREADS, SM_TOTAL, st>>>(sa);
        HeadArgs ha;
        ha.w1 = p->d_w1, ha.hc = p->d_hc, ha.u = u, ha.prob = d_prob, ha.w0 = w0, ha.nwin = nwin, ha.T = T, ha.ntiles = ntiles,
        ha.n_branch = nb;
        int64_t nitems = nwin * ntiles;
        int hgrid = (int)(nitems < p->num_sms ? nitems : p->num_sms);
        k_head_tc<<<hgrid, HEAD_THREADS, 3 * nb * U_TILE_BYTES + 256, st>>>(ha);
        gwi_count_launch(2);
        GWI_CUDA_CHECK(cudaGetLastError());
    }
    return GWI_OK;
}
