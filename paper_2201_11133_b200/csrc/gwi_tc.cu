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
// Roles in k_stack (608 threads): warps 0-7 epilogue of slot 0, warps 8-15 of slot 1 (warp % 4 = TMEM lane quadrant,
// (warp / 4) % 2 = channel half), warp 16 lane 0 = bulk-copy producer (weights, ring tiles), warps 17 / 18: one elected
// lane each = MMA issuer of slot 0 / 1.
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <type_traits>
#include <vector>

#include "gwi_internal.h"
#include "gwi_tc_ptx.h"

// L2 residency hints: the history rings (66 MB for the whole grid, re-read 1-4 tile times after they are written) are
// stored and loaded evict-last, the u tiles (2 GB per launch, read by the next kernel) are stored evict-first
#ifndef GWI_TC_L2HINT
#define GWI_TC_L2HINT 1
#endif
#if GWI_TC_L2HINT
#define GWI_RING_G2S(dst, src, bytes, bar) bulk_g2s_hint(dst, src, bytes, bar, ring_pol)
#define GWI_RING_S2G(dst, src, bytes) bulk_s2g_hint(dst, src, bytes, ring_pol)
#define GWI_U_STORE(ptr, val) __stcs(ptr, val)
#else
#define GWI_RING_G2S(dst, src, bytes, bar) bulk_g2s(dst, src, bytes, bar)
#define GWI_RING_S2G(dst, src, bytes) bulk_s2g(dst, src, bytes)
#define GWI_U_STORE(ptr, val) (*(ptr) = (val))
#endif

using namespace tc;

namespace {

constexpr int TM = 128;                 // timesteps per tile = MMA M
constexpr int TC_MAX_L = 20;
constexpr int WFG_BYTES = 128 * 128 * 2;            // B operand of GEMM1: N = 128 (f|g) x K = 128 (past|current)
constexpr int WRS_BYTES = 192 * 64 * 2;             // B operand of GEMM2: N = 192 (skip|res) x K = 64
constexpr int BIAS_FLOATS = 192;                    // per layer: bf[64], bg/2[64], br[64]; streamed behind Wrs
constexpr int WRS_STRIDE = WRS_BYTES + BIAS_FLOATS * 4;   // 25344
constexpr int X_CHUNK = 192 * 16;                   // chunk-column stride of the X buffer (64 pre rows + 128 rows)
constexpr int X_BYTES = 8 * X_CHUNK;                // 24576
constexpr int PST_BYTES = 8 * 128 * 16;             // 16384: one past tile, chunk stride 2048
constexpr int PRE_BYTES = 8 * 64 * 16;              // 8192: the 64 rows that precede a tile (d = 64 layers)
constexpr int STASH_BYTES = 16384;                  // per slot: sum over layers with d <= 32 of d rows x 128 B
constexpr int U_TILE_BYTES = 16 * 128 * 16;         // 32768: u tile, 16 chunks x 128 rows x 16 B
constexpr int NEPI = 16;                            // epilogue warps: slot = w >> 3, column half = (w >> 2) & 1
constexpr int NTHREADS = (NEPI + 3) * 32;           // + producer warp + one MMA issuer warp per slot

struct TcMeta {
    int L, n_branch;
    int dil[TC_MAX_L];
    int kind[TC_MAX_L];       // 0: d <= 32 (stash in shared memory), 1: d == 64 (pre rows through the global ring64),
                              // 2: d multiple of 128 (whole past tiles through the global ring)
    int lay[TC_MAX_L];        // kind | d << 2 (one constant load per GEMM in the MMA thread)
    int D[TC_MAX_L];          // d / 128 for kind 2 (a power of two: the ring of a layer has D entries)
    int stash_off[TC_MAX_L];  // byte offset of the layer's stash inside the slot's stash area
    int ring_off[TC_MAX_L];   // kind 2: first ring entry (in tiles) of the layer; kind 1: index among the d = 64 layers
    int ring_tiles;           // ring entries per slot
    int n64;                  // number of d = 64 layers
};

#ifdef GWI_TC_TRACE
// debug build only (-DGWI_TC_TRACE): the MMA issuer, the producer and lane 0 of every epilogue warp of CTA 0 record
// (event, slot, iteration, clock) tuples, each into its own region (plain stores, no atomics)
#define TRACE_CAP 4096
__device__ uint4 g_trace[19 * TRACE_CAP];
#define TRACE(ev, slot, n)                                                                                   \
    do {                                                                                                     \
        if (blockIdx.x == 0 && trace_k < TRACE_CAP)                                                          \
            g_trace[trace_role * TRACE_CAP + trace_k++] = make_uint4((unsigned)(ev), (unsigned)(slot), (unsigned)(n), (unsigned)clock64()); \
    } while (0)
#else
#define TRACE(ev, slot, n)
#endif

#if !defined(GWI_TC_ALTERNATE) && !defined(GWI_TC_ONESLOT)
#define GWI_TC_ALTERNATE 0
#endif

struct StackArgs {
    const uint8_t* wfg;   // [n_branch][L][WFG_BYTES]
    const uint8_t* wrs;   // [n_branch][L][WRS_STRIDE]  (Wrs operand followed by the layer's 192 bias floats)
    const float* cst;     // [n_branch][256]: W_in[64], b_in[64], sum_i bs_i[128]
    const __half* strain; // [B][T][C]
    int64_t w0, nwin;     // windows [w0, w0 + nwin) of this launch
    int T, ntiles, C;
    uint8_t* ring;        // [gridDim.x][2][ring_tiles][PST_BYTES]
    uint8_t* ring64;      // [gridDim.x][2][n64][2][PRE_BYTES]
    uint8_t* u;           // [nwin][n_branch][ntiles][U_TILE_BYTES]
    TcMeta meta;
    // bf[64], bg/2[64], br[64] of every (branch, layer), passed by value: the epilogue warps read them as constant-bank
    // operands.  Through shared memory every such load queued behind the operand reads of the SS-mode MMAs, which take
    // all 128 B/clk the SM has: a gate running next to the other slot's GEMMs took 2950 clk instead of 1450 (measured
    // in isolation, _work micro-benchmark)
    float bias[2][TC_MAX_L][BIAS_FLOATS];
};
static_assert(sizeof(StackArgs) <= 32764, "kernel parameter space");

// ---- shared memory map of k_stack ----------------------------------------------------------------------------------
constexpr int SM_WFG = 0;                                 // 2 stages
constexpr int SM_WRS = SM_WFG + 2 * WFG_BYTES;            // 2 stages
constexpr int SM_X = SM_WRS + 2 * WRS_STRIDE;             // 2 slots
constexpr int SM_PST = SM_X + 2 * X_BYTES;                // 2 slots
constexpr int SM_STASH = SM_PST + 2 * PST_BYTES;          // 2 slots
constexpr int SM_BAR = SM_STASH + 2 * STASH_BYTES;
constexpr int SM_CST = SM_BAR + 256;                      // the branch's lift weights and skip-bias sum (256 floats)
constexpr int SM_TOTAL = SM_CST + 1024;
static_assert(SM_TOTAL <= 232448, "shared memory budget");

enum { B_WFG_FULL = 0, B_WFG_FREE = 2, B_WRS_FULL = 4, B_WRS_FREE = 6, B_FG_FULL = 8, B_Z_READY = 10, B_RS_FULL = 12,
       B_H_READY = 14, B_PST_FULL = 16, B_PST_FREE = 18, B_PRE_FULL = 20, B_SKD = 22, B_HALF = 24, B_COUNT = 26 };

__device__ __forceinline__ float2 add2(float2 a, float2 b)
{
    float2 r;
    asm("{\n\t.reg .b64 ra, rb, rc;\n\tmov.b64 ra, {%2, %3};\n\tmov.b64 rb, {%4, %5};\n\tadd.rn.f32x2 rc, ra, rb;\n\t"
        "mov.b64 {%0, %1}, rc;\n\t}"
        : "=f"(r.x), "=f"(r.y)
        : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y));
    return r;
}
__device__ __forceinline__ float2 fma2(float2 a, float2 b, float2 c)
{
    float2 r;
    asm("{\n\t.reg .b64 ra, rb, rc, rd;\n\tmov.b64 ra, {%2, %3};\n\tmov.b64 rb, {%4, %5};\n\tmov.b64 rc, {%6, %7};\n\t"
        "fma.rn.f32x2 rd, ra, rb, rc;\n\tmov.b64 {%0, %1}, rd;\n\t}"
        : "=f"(r.x), "=f"(r.y)
        : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y), "f"(c.x), "f"(c.y));
    return r;
}

// Schedule (one CTA per SM, persistent over jobs = (pair of windows, branch)).  The two windows of a job are two
// "slots" that run the same (tile, layer) sequence half a layer apart: the single MMA thread issues
//     G1(slot 0, n)  G2(slot 1, n-1)  G1(slot 1, n)  G2(slot 0, n)          n = (tile, layer) iteration
// so that while one slot's 8 epilogue warps gate (MUFU-bound), the tensor pipe and the other slot's warps work on the
// other slot.  Weights (and the layer's biases) are double-buffered and shared by the two slots.
__global__ void __launch_bounds__(NTHREADS, 1) k_stack(const __grid_constant__ StackArgs a)
{
    extern __shared__ __align__(1024) uint8_t smem[];
    const uint32_t sbase = smem_u32(smem);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const TcMeta& M = a.meta;
    const int L = M.L, nb = M.n_branch;
    auto bar = [&](int i) { return sbase + SM_BAR + 8 * i; };
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + SM_BAR + 8 * B_COUNT);
#if GWI_TC_L2HINT
    const uint64_t ring_pol = l2_policy_evict_last();
#endif

    if (threadIdx.x == 0) {
        for (int i = 0; i < B_COUNT; i++) {
            uint32_t cnt = (i >= B_Z_READY && i < B_Z_READY + 2) || (i >= B_H_READY && i < B_H_READY + 2) ? 256u : 1u;
            if (i >= B_HALF && i < B_HALF + 2) cnt = 256u;
#ifndef GWI_TC_ONESLOT
            if ((i >= B_WFG_FREE && i < B_WFG_FREE + 2) || (i >= B_WRS_FREE && i < B_WRS_FREE + 2)) cnt = 2u;   // both issuers
#endif
            mbar_init(bar(i), cnt);
        }
        mbar_fence_init();
    }
    if (warp == NEPI) tmem_alloc(smem_u32(tmem_slot), 512);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;
    // TMEM columns: slot s: f|g accumulator (res reuses its first 64 columns) at 128 s, skip sum at 256 + 128 s

    const int64_t npairs = (a.nwin + 1) / 2;
    const int64_t njobs = npairs * nb;
    const int NI = a.ntiles * L;
    // phase counters (each role keeps its own copy; the schedules are identical by construction)
    uint32_t n_it = 0;                 // (job, tile, layer) iterations done
    uint32_t n_pst[2] = {0, 0};        // ring-tile loads done per slot
    uint32_t n_pre[2] = {0, 0};        // pre-row loads done per slot
#ifdef GWI_TC_TRACE
    unsigned trace_k = 0;
    const int trace_role = warp == NEPI + 1 ? 0 : (warp == NEPI ? 17 : (warp == NEPI + 2 ? 18 : 1 + (warp & 15)));
#endif

    for (int64_t job = blockIdx.x; job < njobs; job += gridDim.x) {
        const int b = (int)(job % nb);
        const int64_t pair = job / nb;
        // ---- job prologue (all threads): zero the stashes and the X buffers (causal zero history, reading A4) --------
        __syncthreads();
        {
            uint4 z4 = make_uint4(0, 0, 0, 0);
            uint4* zs = reinterpret_cast<uint4*>(smem + SM_STASH);
            for (int i = threadIdx.x; i < 2 * STASH_BYTES / 16; i += NTHREADS) zs[i] = z4;
            uint4* zx = reinterpret_cast<uint4*>(smem + SM_X);
            for (int i = threadIdx.x; i < 2 * X_BYTES / 16; i += NTHREADS) zx[i] = z4;
            if (threadIdx.x < 256) reinterpret_cast<float*>(smem + SM_CST)[threadIdx.x] = a.cst[b * 256 + threadIdx.x];
        }
        fence_proxy_async_smem();
        __syncthreads();

        if (warp == NEPI) {
            // =========================== producer: weights and ring tiles ===========================================
            if (elect_one()) {
                for (int n = 0; n < NI; n++, n_it++) {
                    const int i = n % L, j = n / L;
                    const int st = n_it & 1;
                    const uint32_t wph = (n_it >> 1) & 1;
                    mbar_wait(bar(B_WFG_FREE + st), wph ^ 1);
                    mbar_arrive_expect_tx(bar(B_WFG_FULL + st), WFG_BYTES);
                    bulk_g2s(sbase + SM_WFG + st * WFG_BYTES, a.wfg + ((size_t)b * L + i) * WFG_BYTES, WFG_BYTES,
                             bar(B_WFG_FULL + st));
                    mbar_wait(bar(B_WRS_FREE + st), wph ^ 1);
                    mbar_arrive_expect_tx(bar(B_WRS_FULL + st), WRS_STRIDE);
                    bulk_g2s(sbase + SM_WRS + st * WRS_STRIDE, a.wrs + ((size_t)b * L + i) * WRS_STRIDE, WRS_STRIDE,
                             bar(B_WRS_FULL + st));
                    // the past tiles last: their waits (GEMM2 of the previous iteration of both slots) must not hold back
                    // the weights and biases of this iteration, which the gate needs first
                    if (M.kind[i] == 2 && j >= M.D[i]) {
#ifdef GWI_TC_ONESLOT
                        for (int s = 0; s < 1; s++) {
#else
                        for (int s = 0; s < 2; s++) {
#endif
                            // the tile was stored (j - D) tiles ago by the MMA thread, which waits for the completion
                            // of its bulk stores before it issues GEMM2 of the same iteration: GEMM2 of the previous
                            // iteration of this slot being done implies the tile is in L2
                            mbar_wait(bar(B_RS_FULL + s), (n_it - 1) & 1);
                            mbar_wait(bar(B_PST_FREE + s), (n_pst[s] & 1) ^ 1);
                            mbar_arrive_expect_tx(bar(B_PST_FULL + s), PST_BYTES);
                            const uint8_t* src = a.ring + (((size_t)blockIdx.x * 2 + s) * M.ring_tiles + M.ring_off[i] +
                                                           (j & (M.D[i] - 1))) * PST_BYTES;
                            GWI_RING_G2S(sbase + SM_PST + s * PST_BYTES, src, PST_BYTES, bar(B_PST_FULL + s));
                            n_pst[s]++;
                        }
                    }
                }
            }
            __syncwarp();
        } else if (warp == NEPI + 1 || warp == NEPI + 2) {
            // =========================== MMA issuers: one thread per slot ===============================================
            // Each slot has its own issuer (a single thread issues ~8 tcgen05.mma per GEMM in a dependent instruction
            // stream; with one thread for both slots that stream was the bottleneck).  The two threads only meet in
            // the tensor pipe and on the weight-stage barriers (WFG_FREE / WRS_FREE take one commit from each).
            if (elect_one()) {
                const uint32_t idesc128 = make_idesc_f16(128, 128), idesc64 = make_idesc_f16(128, 64);
                auto issuer = [&](auto SC) {
                    constexpr int s = decltype(SC)::value;
                    // descriptors built once; the address field is the low 14 bits (16-byte units)
                    const uint64_t ax = make_sdesc(sbase + SM_X + s * X_BYTES + 64 * 16, X_CHUNK, 128);   // current rows / z
                    const uint64_t apst = make_sdesc(sbase + SM_PST + s * PST_BYTES, 2048, 128);           // past tile
                    const uint64_t dWfg = make_sdesc(sbase + SM_WFG, 2048, 128);
                    const uint64_t dWrs = make_sdesc(sbase + SM_WRS, 3072, 128);
                    const uint32_t dt = tmem + 128 * s, dskip = tmem + 256 + 128 * s;
                    const uint32_t xrows = sbase + SM_X + s * X_BYTES + 64 * 16;
                    uint8_t* const ring_s = a.ring + ((size_t)blockIdx.x * 2 + s) * M.ring_tiles * PST_BYTES;
                    uint8_t* const ring64_s = a.ring64 + ((size_t)blockIdx.x * 2 + s) * M.n64 * 2 * PRE_BYTES;
                    uint32_t nit = n_it, npst = n_pst[s], npre = n_pre[s];
                    int i = 0, j = 0;
                    for (int n = 0; n < NI; n++, nit++) {
                        const uint32_t st = nit & 1, wpar = (nit >> 1) & 1, par = nit & 1;
                        // ---- GEMM1: f|g = [h(t-d) | h(t)] . Wfg^T
                        const int li = M.lay[i], kind = li & 3, d = li >> 2;
                        const bool past = kind < 2 || j >= (d >> 7);
                        mbar_wait(bar(B_WFG_FULL + st), wpar);
                        mbar_wait(bar(B_H_READY + s), par);
                        if (kind == 1 && j >= 1) {
                            mbar_wait(bar(B_PRE_FULL + s), npre & 1);
                            npre++;
                        }
                        if (kind == 2 && past) {
                            mbar_wait(bar(B_PST_FULL + s), npst & 1);
                            npst++;
                        }
                        tc_fence_after();
                        TRACE(1, s, n);
                        // history for later tiles: the freshly published operand rows go from shared memory to the
                        // L2-resident rings through the bulk-copy engine.  The ring entry of tile j is the one tile
                        // j - D was read from, and that read has landed (PST_FULL above).
                        bool stored = false;
                        if (kind == 2 && j + (d >> 7) < a.ntiles) {
                            uint8_t* dst = ring_s + (size_t)(M.ring_off[i] + (j & ((d >> 7) - 1))) * PST_BYTES;
#pragma unroll
                            for (int c = 0; c < 8; c++) GWI_RING_S2G(dst + c * 2048, xrows + c * X_CHUNK, 2048);
                            bulk_commit();
                            stored = true;
                        } else if (kind == 1 && j + 1 < a.ntiles) {
                            uint8_t* dst = ring64_s + (size_t)(M.ring_off[i] * 2 + (j & 1)) * PRE_BYTES;
#pragma unroll
                            for (int c = 0; c < 8; c++) GWI_RING_S2G(dst + c * 1024, xrows + 64 * 16 + c * X_CHUNK, 1024);
                            bulk_commit();
                            stored = true;
                        }
                        {
                            const uint64_t bw = dWfg + st * (WFG_BYTES >> 4);
                            uint32_t acc = 0;
                            if (past) {
                                const uint64_t ap = kind < 2 ? ax - d : apst;
                                const uint32_t ka = kind < 2 ? (2 * X_CHUNK) >> 4 : 4096 >> 4;
#pragma unroll
                                for (int kk = 0; kk < 4; kk++, acc = 1) tc_mma_f16(dt, ap + kk * ka, bw + kk * 256, idesc128, acc);
                            }
#pragma unroll
                            for (int kk = 0; kk < 4; kk++, acc = 1)
                                tc_mma_f16(dt, ax + kk * ((2 * X_CHUNK) >> 4), bw + 1024 + kk * 256, idesc128, acc);
                        }
                        tc_commit(bar(B_FG_FULL + s));
                        if (kind == 2 && past) tc_commit(bar(B_PST_FREE + s));
                        tc_commit(bar(B_WFG_FREE + st));          // one commit per slot frees the stage
                        TRACE(2, s, n);
                        // ---- GEMM2: skip += z' Ws'^T ; res = z' Wr'^T
                        mbar_wait(bar(B_WRS_FULL + st), wpar);
                        mbar_wait(bar(B_Z_READY + s), par);
                        tc_fence_after();
                        if (stored) bulk_wait_all();   // ring write complete before RS_FULL of this iteration (producer's cue)
                        TRACE(3, s, n);
                        {
                            // the residual GEMM is on the critical path (next layer's operand), the skip GEMM is not:
                            // residual first with its own commit, the skip sum runs under the residual epilogue
                            // A = z' in tensor memory (the gate wrote it over the g columns it had drained: channels
                            // 0-31 at columns 64..79, channels 32-63 at 96..111 of the slot's f|g accumulator)
                            const uint64_t bw = dWrs + st * (WRS_STRIDE >> 4);
                            const uint32_t az = dt + 64;
                            if (i < L - 1) {  // reading A8: the last block's residual conv has no effect
#pragma unroll
                                for (int kk = 0; kk < 4; kk++)
                                    tc_mma_f16_ts(dt, az + 32 * (kk >> 1) + 8 * (kk & 1), bw + 128 + kk * 384, idesc64, kk > 0 ? 1u : 0u);
                            }
                            tc_commit(bar(B_RS_FULL + s));
                            {
                                // pre rows of the next iteration (d = 64 layers): GEMM1 of this iteration is done with them
                                // (its gate has ended), and this thread's own bulk store of the entry (a tile ago) has
                                // completed (bulk_wait_all above, in that iteration)
                                const int inx = (i + 1 < L) ? i + 1 : 0, jnx = (i + 1 < L) ? j : j + 1;
                                if ((M.lay[inx] & 3) == 1 && jnx >= 1 && jnx < a.ntiles) {
                                    const uint8_t* src = ring64_s + (size_t)(M.ring_off[inx] * 2 + ((jnx - 1) & 1)) * PRE_BYTES;
                                    mbar_arrive_expect_tx(bar(B_PRE_FULL + s), PRE_BYTES);
#pragma unroll
                                    for (int c = 0; c < 8; c++)
                                        GWI_RING_G2S(xrows - 64 * 16 + c * X_CHUNK, src + c * 1024, 1024, bar(B_PRE_FULL + s));
                                }
                            }
#pragma unroll
                            for (int kk = 0; kk < 4; kk++)
                                tc_mma_f16_ts(dskip, az + 32 * (kk >> 1) + 8 * (kk & 1), bw + kk * 384, idesc128, (i > 0 || kk > 0) ? 1u : 0u);
                        }
                        tc_commit(bar(B_SKD + s));
                        tc_commit(bar(B_WRS_FREE + st));
                        TRACE(4, s, n);
                        if (++i == L) i = 0, j++;
                    }
                    n_pst[s] = npst, n_pre[s] = npre;
                };
                if (warp == NEPI + 1) issuer(std::integral_constant<int, 0>{});
#ifndef GWI_TC_ONESLOT
                else issuer(std::integral_constant<int, 1>{});
#endif
            }
            n_it += NI;
            __syncwarp();
        } else {
            // =========================== epilogue: slot s, column half wg, row r =======================================
            const int s = warp >> 3, wg = (warp >> 2) & 1;
#ifdef GWI_TC_ONESLOT
            if (s == 1) { n_it += NI; continue; }
#endif
            const int r = (warp & 3) * 32 + lane;                    // row of the tile = TMEM lane
            const int ch0 = 32 * wg, c0 = 4 * wg;                     // first channel / first 16-byte chunk of this half
            const int64_t wl = 2 * pair + s;                          // window index inside this launch
            const bool valid = wl < a.nwin;
            const int64_t w = a.w0 + (valid ? wl : a.nwin - 1);
            const uint32_t xs = sbase + SM_X + s * X_BYTES;
            const uint32_t st0 = sbase + SM_STASH + s * STASH_BYTES;
            const uint32_t lane_t = tmem + ((uint32_t)((warp & 3) * 32) << 16);
            const float* cst = reinterpret_cast<const float*>(smem + SM_CST);   // W_in[64], b_in[64], sum_i bs_i[128]
            float2 h[16];                                             // fp32 master of the residual stream, 32 channels

            // writes the fp16 copy of h as the operand of layer `inext` for tile j, maintains stash / rings, signals MMA
            auto publish = [&](int inext, int j) {
                uint32_t pk[16];
#pragma unroll
                for (int c = 0; c < 16; c++) pk[c] = pack_half2(h[c].x, h[c].y);
#pragma unroll
                for (int c = 0; c < 4; c++)
                    st_shared_v4(xs + (64 + r) * 16 + (c0 + c) * X_CHUNK, pk[4 * c], pk[4 * c + 1], pk[4 * c + 2], pk[4 * c + 3]);
                const int d = M.dil[inext], kind = M.kind[inext];
                if (kind == 0) {
                    if (r >= 128 - d) {
                        const int rp = r - (128 - d);
                        const uint32_t sb = st0 + M.stash_off[inext] + rp * 16;
#pragma unroll
                        for (int c = 0; c < 4; c++) {
                            uint4 old = ld_shared_v4(sb + (c0 + c) * d * 16);
                            st_shared_v4(xs + (64 - d + rp) * 16 + (c0 + c) * X_CHUNK, old.x, old.y, old.z, old.w);
                            st_shared_v4(sb + (c0 + c) * d * 16, pk[4 * c], pk[4 * c + 1], pk[4 * c + 2], pk[4 * c + 3]);
                        }
                    }
                } else if (kind == 1) {
                    if (j == 0 && r < 64) {
#pragma unroll
                        for (int c = 0; c < 4; c++) st_shared_v4(xs + r * 16 + (c0 + c) * X_CHUNK, 0u, 0u, 0u, 0u);
                    }
                }
#ifdef GWI_TC_TRACE
                if (lane == 0) TRACE(10, 10 * (warp & 7) + s, 0);
#endif
                tc_fence_before();
                fence_proxy_async_smem();
                mbar_arrive(bar(B_H_READY + s));
            };

            // ---- lift of tile j: h0 = W_in x + b_in, published as the operand of layer 0            (C.1 step 1)
            auto load_x = [&](int j) {
                const int t = j * TM + r;
                return t < a.T ? __half2float(a.strain[((size_t)w * a.T + t) * a.C + b]) : 0.f;
            };
            auto lift = [&](int j, float x) {
#pragma unroll
                for (int c = 0; c < 16; c++) {
                    float2 wi = *(reinterpret_cast<const float2*>(cst + ch0) + c);
                    float2 bi = *(reinterpret_cast<const float2*>(cst + 64 + ch0) + c);
                    h[c] = make_float2(fmaf(wi.x, x, bi.x), fmaf(wi.y, x, bi.y));
                }
                publish(0, j);
            };
            lift(0, load_x(0));
            float xnext = 0.f;
            for (int j = 0; j < a.ntiles; j++) {
                for (int i = 0; i < L; i++, n_it++) {
                    const uint32_t ph = n_it & 1;
                    const int st = n_it & 1;
                    if (i == L - 1 && j + 1 < a.ntiles) xnext = load_x(j + 1);   // strain of the next tile, a whole layer early
                    // ---- off the critical path, while GEMM1 runs: the residual bias into the fp32 master
                    const float* bl = a.bias[b][i];      // constant bank (kernel parameters)
                    if (i < L - 1) {
#pragma unroll
                        for (int c = 0; c < 16; c++) h[c] = add2(h[c], make_float2(bl[128 + ch0 + 2 * c], bl[128 + ch0 + 2 * c + 1]));
                    }
                    // ---- gate: z' = tanh(f + bf) * (1 + tanh(g/2 + bg/2))
                    mbar_wait(bar(B_FG_FULL + s), ph);
#ifdef GWI_TC_ALTERNATE
                    // The gates of the two slots are kept out of phase: a gate starts once the other slot's previous gate
                    // is through chunk GWI_TC_ALTERNATE of 4 (measured: lockstep 14.1 ms, strict alternation 14.0 ms,
                    // half-overlap 13.7 ms for configs[1]) instead of drifting into lockstep
                    if (s == 0) {
                        if (j + i > 0) mbar_wait(bar(B_HALF + 1), (n_it - 1) & 1);
                    } else {
                        mbar_wait(bar(B_HALF + 0), n_it & 1);
                    }
#endif
                    if (lane == 0) TRACE(5, 10 * (warp & 7) + s, j * L + i);
                    __syncwarp();
                    tc_fence_after();
                    {
                        // 4 chunks of 8 channels; the TMEM loads of chunk q+1 are in flight while chunk q is gated
                        uint32_t fb[2][8], gb[2][8];
                        const uint32_t tf0 = lane_t + 128 * s + ch0, tg0 = tf0 + 64;
                        tmem_ld8(tf0, fb[0]);
                        tmem_ld8(tg0, gb[0]);
#pragma unroll
                        for (int q = 0; q < 4; q++) {
                            tc_wait_ld();
                            if (q < 3) {
                                tmem_ld8(tf0 + 8 * (q + 1), fb[(q + 1) & 1]);
                                tmem_ld8(tg0 + 8 * (q + 1), gb[(q + 1) & 1]);
                            }
                            const uint32_t* f = fb[q & 1];
                            const uint32_t* g = gb[q & 1];
                            uint32_t pk[4];
#pragma unroll
                            for (int c = 0; c < 4; c++) {
                                float2 bf = make_float2(bl[ch0 + 8 * q + 2 * c], bl[ch0 + 8 * q + 2 * c + 1]);
                                float2 bg = make_float2(bl[64 + ch0 + 8 * q + 2 * c], bl[64 + ch0 + 8 * q + 2 * c + 1]);
                                float2 fa = add2(make_float2(__uint_as_float(f[2 * c]), __uint_as_float(f[2 * c + 1])), bf);
                                float2 ga = add2(make_float2(__uint_as_float(g[2 * c]), __uint_as_float(g[2 * c + 1])), bg);
                                float2 tf = make_float2(tanh_approx(fa.x), tanh_approx(fa.y));
                                float2 tg = make_float2(tanh_approx(ga.x), tanh_approx(ga.y));
                                float2 z = fma2(tf, tg, tf);
                                pk[c] = pack_half2(z.x, z.y);
                            }
                            // z' chunk q (8 channels = 4 packed columns) over the g columns already read: the A operand of GEMM2
                            tmem_st4(tg0 + 4 * q, pk[0], pk[1], pk[2], pk[3]);
#ifdef GWI_TC_ALTERNATE
                            if (q == GWI_TC_ALTERNATE) mbar_arrive(bar(B_HALF + s));
#endif
                        }
                    }
                    tc_wait_st();
                    tc_fence_before();
                    mbar_arrive(bar(B_Z_READY + s));
                    if (lane == 0) TRACE(6, 10 * (warp & 7) + s, j * L + i);
                    // ---- residual update (or, after the last block, the branch output)
                    mbar_wait(bar(B_RS_FULL + s), ph);
                    if (lane == 0) TRACE(7, 10 * (warp & 7) + s, j * L + i);
                    tc_fence_after();
                    if (i < L - 1) {
                        uint32_t v[32];
                        tmem_ld32(lane_t + 128 * s + ch0, v);
                        tc_wait_ld();
                        if (lane == 0) TRACE(9, 10 * (warp & 7) + s, j * L + i);
#pragma unroll
                        for (int c = 0; c < 16; c++)
                            h[c] = add2(h[c], make_float2(__uint_as_float(v[2 * c]), __uint_as_float(v[2 * c + 1])));
                        publish(i + 1, j);
                        if (lane == 0) TRACE(8, 10 * (warp & 7) + s, j * L + i);
                    } else {
                        // u = ReLU(sum_i skip_i) -> fp16 tile in the workspace                       (C.1 step 3)
                        mbar_wait(bar(B_SKD + s), ph);
                        tc_fence_after();
                        // the next tile starts first (its GEMM1 runs under the u output below; its first skip GEMM, which
                        // overwrites the skip sum, needs this warp's gate of layer 0, i.e. comes after the reads below)
                        if (j + 1 < a.ntiles) lift(j + 1, xnext);
                        uint8_t* ut = a.u + (((size_t)wl * nb + b) * a.ntiles + j) * U_TILE_BYTES + r * 16;
#pragma unroll
                        for (int cc = 0; cc < 2; cc++) {
                            uint32_t v[32];
                            tmem_ld32(lane_t + 256 + 128 * s + 64 * wg + 32 * cc, v);
                            tc_wait_ld();
                            if (valid) {
#pragma unroll
                                for (int c = 0; c < 4; c++) {
                                    uint32_t q[4];
#pragma unroll
                                    for (int e = 0; e < 4; e++) {
                                        int col = 8 * c + 2 * e;
                                        float2 bs = *reinterpret_cast<const float2*>(cst + 128 + 64 * wg + 32 * cc + col);
                                        float u0 = fmaxf(__uint_as_float(v[col]) + bs.x, 0.f);
                                        float u1 = fmaxf(__uint_as_float(v[col + 1]) + bs.y, 0.f);
                                        q[e] = pack_half2(u0, u1);
                                    }
                                    GWI_U_STORE(reinterpret_cast<uint4*>(ut + (8 * wg + 4 * cc + c) * 2048), make_uint4(q[0], q[1], q[2], q[3]));
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
    if (warp == NEPI) tmem_dealloc(tmem, 512);
}

// ---- head kernel ---------------------------------------------------------------------------------------------------
struct HeadArgs {
    const uint8_t* w1;    // B operand: N = 128 x K = n_branch*128, chunk-column (chunk stride 2048)
    float b1[128], w2[128], b2;   // head constants by value: read as constant-bank operands, not through shared memory
    const uint8_t* u;     // [nwin][n_branch][ntiles][U_TILE_BYTES]
    float* prob;          // [B][T]
    int64_t w0, nwin;
    int T, ntiles, n_branch;
    // stream mode (mode = 1, gwi_stream.cu tensor-core back end with time slides, reading A24): the items are the nq
    // output tiles of a block of segments; output tile q lives in window q / seg_tiles at tile q % seg_tiles +
    // warm_tiles (no warm-up in the first window of the stream).  Every lag of the list is evaluated while the H1 tile
    // of the item sits in shared memory: the L1 tile of lag k is taken lags[k] / 128 tiles earlier, from the block or,
    // before its start, from hist = the R L1 tiles that precede the block (those tiles were read by the items just
    // before, so they come from L2); probabilities of lag k go to prob + k * stride_k.
    int mode;
    const uint8_t* hist;
    const int64_t* lags;      // device, samples, multiples of 128
    int64_t nq, stride_k;
    int n_lags, R, seg_tiles, warm_tiles, stream_start, n_valid;
    // k_vhalf_tc: the two halves of the head's first layer per sample, fp16 rows of 128: v_H = W1[:, :128] u_H + b1 and
    // v_L = W1[:, 128:] u_L, at vout + (branch * vlds + row) * 128, row = sample index inside the block (warm-up tiles skipped)
    __half* vout;
    int64_t vlds;
};
constexpr int HEAD_SMEM_EXTRA = 2048;   // barriers, TMEM slot, b1 | W2 | b2
constexpr int HEAD_SMEM = 7 * U_TILE_BYTES + HEAD_SMEM_EXTRA;   // W1 (2 tiles) + 5 feature-tile buffers
constexpr int HEAD_THREADS = 320;   // warps 0-7 epilogue (warps 0-3: accumulator buffer 0, warps 4-7: buffer 1), warp 8 producer, warp 9 MMA

__global__ void __launch_bounds__(HEAD_THREADS, 1) k_head_tc(const HeadArgs a)
{
    extern __shared__ __align__(1024) uint8_t smem[];
    const uint32_t sbase = smem_u32(smem);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int nb = a.n_branch;
    const int W1B = nb * U_TILE_BYTES;            // bytes of W1 blob == bytes of one u stage
    const int OFF_U = W1B, OFF_BAR = 7 * U_TILE_BYTES;
    const int OFF_L = OFF_U + 2 * U_TILE_BYTES;   // stream mode: two H1 tile buffers at OFF_U, three L1 tile buffers at OFF_L
    // barriers: 0 w1_full, 1-2 u_full[st], 3-4 u_free[st], 5-6 acc_full[st], 7-8 acc_free[st]; stream mode: H1 tiles (one
    // per item) 9-10 h_full, 11-12 h_free; L1 tiles (one per lag, three buffers) l_full 1, 2, 13 and l_free 3, 4, 14;
    // the H1 half of the contraction (one per item, TMEM columns 0-255) 15-16 ah_full, 17-18 ah_free; the L1 halves
    // (one per lag, TMEM columns 256-511) use 5-8.
    // The SS-mode MMAs read 128 B/clk of shared memory, all there is: whatever else goes through shared memory (the
    // bulk copies of the tiles, epilogue constants) adds to the MMA time, so the H1 half W1[:, :128] u_H is contracted
    // once per item and only the K = 128 of the L1 half per lag, and the epilogue takes b1 and W2 from the constant bank.
    auto bar = [&](int i) { return sbase + OFF_BAR + 8 * i; };
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + OFF_BAR + 8 * 20);
    auto l_full = [&](int ls) { return bar(ls < 2 ? 1 + ls : 13); };
    auto l_free = [&](int ls) { return bar(ls < 2 ? 3 + ls : 14); };
    if (threadIdx.x == 0) {
        for (int i = 0; i < 19; i++) mbar_init(bar(i), (i == 7 || i == 8) ? 128u : (i == 17 || i == 18) ? 256u : 1u);
        mbar_fence_init();
    }
    if (warp == 8) tmem_alloc(smem_u32(tmem_slot), 512);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;
    const int64_t nitems = a.mode ? a.nq : a.nwin * a.ntiles;
    // stream mode: address of the u tile of branch b that holds block-local output tile q (q < 0: history)
    auto stream_tile = [&](int64_t q, int b) -> const uint8_t* {
        if (q < 0) return a.hist + (size_t)(a.R + q) * U_TILE_BYTES;
        const int64_t w = q / a.seg_tiles;
        const int64_t tl = q % a.seg_tiles + ((w == 0 && a.stream_start) ? 0 : a.warm_tiles);
        return a.u + (((size_t)w * nb + b) * a.ntiles + tl) * U_TILE_BYTES;
    };

    if (warp == 8) {
        if (lane == 0) {
            mbar_arrive_expect_tx(bar(0), W1B);
            bulk_g2s(sbase, a.w1, W1B, bar(0));
            // stream mode: an H1 tile is read once, an L1 tile by every lag of the next max-lag output tiles
            const uint64_t pol_once = l2_policy_evict_first(), pol_keep = l2_policy_evict_last();
            uint32_t n = 0, c = 0;
            for (int64_t it = blockIdx.x; it < nitems; it += gridDim.x, n++) {
                if (a.mode) {
                    const int hs = n & 1;
                    mbar_wait(bar(11 + hs), ((n >> 1) & 1) ^ 1);
                    mbar_arrive_expect_tx(bar(9 + hs), U_TILE_BYTES);
                    bulk_g2s_hint(sbase + OFF_U + hs * U_TILE_BYTES, stream_tile(it, 0), U_TILE_BYTES, bar(9 + hs), pol_once);
                    for (int k = 0; k < a.n_lags; k++, c++) {
                        const int ls = c % 3;
                        mbar_wait(l_free(ls), ((c / 3) & 1) ^ 1);
                        mbar_arrive_expect_tx(l_full(ls), U_TILE_BYTES);
                        bulk_g2s_hint(sbase + OFF_L + ls * U_TILE_BYTES, stream_tile(it - __ldg(a.lags + k) / TM, 1), U_TILE_BYTES,
                                      l_full(ls), pol_keep);
                    }
                    continue;
                }
                const int st = n & 1;
                const int64_t wl = it / a.ntiles, j = it % a.ntiles;
                mbar_wait(bar(3 + st), ((n >> 1) & 1) ^ 1);
                mbar_arrive_expect_tx(bar(1 + st), W1B);
                for (int b = 0; b < nb; b++)
                    bulk_g2s(sbase + OFF_U + st * W1B + b * U_TILE_BYTES, a.u + (((size_t)wl * nb + b) * a.ntiles + j) * U_TILE_BYTES,
                             U_TILE_BYTES, bar(1 + st));
            }
        }
        __syncwarp();
    } else if (warp == 9) {
        // one elected thread issues; under elect_one() the compiler keeps the descriptors in uniform registers and the
        // unrolled tcgen05.mma go out back to back (the address field of a descriptor counts 16-byte units)
        if (elect_one()) {
            const uint32_t idesc = make_idesc_f16(128, 128);
            const uint64_t dW = make_sdesc(sbase, 2048, 128);
            const uint64_t dU = make_sdesc(sbase + OFF_U, 2048, 128);
            const uint64_t dL = make_sdesc(sbase + OFF_L, 2048, 128);
            mbar_wait(bar(0), 0);
            uint32_t n = 0, c = 0;
            for (int64_t it = blockIdx.x; it < nitems; it += gridDim.x, n++) {
                if (a.mode) {
                    const int hs = n & 1;
                    const uint32_t hp = (n >> 1) & 1;
                    mbar_wait(bar(9 + hs), hp);
                    mbar_wait(bar(17 + hs), hp ^ 1);
                    tc_fence_after();
                    const uint64_t dh = dU + hs * (U_TILE_BYTES >> 4);
#pragma unroll
                    for (int kk = 0; kk < 8; kk++) tc_mma_f16(tmem + 128 * hs, dh + kk * 256, dW + kk * 256, idesc, kk > 0 ? 1u : 0u);
                    tc_commit(bar(15 + hs));
                    tc_commit(bar(11 + hs));
                    for (int k = 0; k < a.n_lags; k++, c++) {
                        const int ls = c % 3, as = c & 1;
                        mbar_wait(l_full(ls), (c / 3) & 1);
                        mbar_wait(bar(7 + as), ((c >> 1) & 1) ^ 1);
                        tc_fence_after();
                        const uint64_t dl = dL + ls * (U_TILE_BYTES >> 4);
                        const uint32_t dt = tmem + 256 + 128 * as;
#pragma unroll
                        for (int kk = 0; kk < 8; kk++) tc_mma_f16(dt, dl + kk * 256, dW + (8 + kk) * 256, idesc, kk > 0 ? 1u : 0u);
                        tc_commit(bar(5 + as));
                        tc_commit(l_free(ls));
                    }
                    continue;
                }
                const int st = n & 1;
                const uint32_t ph = (n >> 1) & 1;
                mbar_wait(bar(1 + st), ph);
                mbar_wait(bar(7 + st), ph ^ 1);
                tc_fence_after();
                const uint64_t du = dU + st * (W1B >> 4);
                const uint32_t dt = tmem + 128 * st;
#pragma unroll
                for (int kk = 0; kk < 8; kk++) tc_mma_f16(dt, du + kk * 256, dW + kk * 256, idesc, kk > 0 ? 1u : 0u);
                if (nb == 2) {
#pragma unroll
                    for (int kk = 8; kk < 16; kk++) tc_mma_f16(dt, du + kk * 256, dW + kk * 256, idesc, 1u);
                }
                tc_commit(bar(5 + st));
                tc_commit(bar(3 + st));
            }
        }
        __syncwarp();
    } else {
        // the two accumulator buffers alternate, each has its own four warps (one per TMEM lane quadrant), so that the
        // epilogue of one tile overlaps the whole MMA time of the next
        const int set = warp >> 2, r = (warp & 3) * 32 + lane;
        const uint32_t lane_t = tmem + ((uint32_t)((warp & 3) * 32) << 16);
        // y = W2 . ReLU(acc + b1) + b2 of this thread's row; acc = accumulator columns at `ta` (+ those at `tb` when
        // SPLIT: the H1 half of the contraction); four independent chains over the 128 channels
        auto finish = [&](uint32_t ta, uint32_t tb, auto SPLIT) {
            float y0 = 0.f, y1 = 0.f, y2 = 0.f, y3 = 0.f;
#pragma unroll
            for (int cc = 0; cc < 4; cc++) {
                uint32_t v[32], w[32];
                tmem_ld32(lane_t + ta + 32 * cc, v);
                if (decltype(SPLIT)::value) tmem_ld32(lane_t + tb + 32 * cc, w);
                tc_wait_ld();
#pragma unroll
                for (int c = 0; c < 32; c += 4) {
                    float x0 = __uint_as_float(v[c]), x1 = __uint_as_float(v[c + 1]), x2 = __uint_as_float(v[c + 2]),
                          x3 = __uint_as_float(v[c + 3]);
                    if (decltype(SPLIT)::value)
                        x0 += __uint_as_float(w[c]), x1 += __uint_as_float(w[c + 1]), x2 += __uint_as_float(w[c + 2]),
                            x3 += __uint_as_float(w[c + 3]);
                    y0 = fmaf(a.w2[32 * cc + c], fmaxf(x0 + a.b1[32 * cc + c], 0.f), y0);
                    y1 = fmaf(a.w2[32 * cc + c + 1], fmaxf(x1 + a.b1[32 * cc + c + 1], 0.f), y1);
                    y2 = fmaf(a.w2[32 * cc + c + 2], fmaxf(x2 + a.b1[32 * cc + c + 2], 0.f), y2);
                    y3 = fmaf(a.w2[32 * cc + c + 3], fmaxf(x3 + a.b1[32 * cc + c + 3], 0.f), y3);
                }
            }
            const float y = ((y0 + y1) + (y2 + y3)) + a.b2;
            return 1.0f / (1.0f + __expf(-y));
        };
        uint32_t n = 0, c = 0;
        for (int64_t it = blockIdx.x; it < nitems; it += gridDim.x, n++) {
            if (a.mode) {
                const int64_t t = it * TM + r;
                const int hs = n & 1;
                for (int k = 0; k < a.n_lags; k++, c++) {
                    if ((int)(c & 1) != set) continue;
                    mbar_wait(bar(15 + hs), (n >> 1) & 1);
                    mbar_wait(bar(5 + set), (c >> 1) & 1);
                    tc_fence_after();
                    const float pr = finish(256 + 128 * set, 128 * hs, std::true_type{});
                    tc_fence_before();
                    mbar_arrive(bar(7 + set));
                    if (t < a.n_valid) a.prob[(size_t)k * a.stride_k + t] = pr;
                }
                // both sets have read the H1 half of this item (n_lags >= 2: each set had at least one lag)
                tc_fence_before();
                mbar_arrive(bar(17 + hs));
                continue;
            }
            if ((int)(n & 1) != set) continue;
            const int64_t wl = it / a.ntiles, j = it % a.ntiles;
            mbar_wait(bar(5 + set), (n >> 1) & 1);
            tc_fence_after();
            const float pr = finish(128 * set, 0, std::false_type{});
            tc_fence_before();
            mbar_arrive(bar(7 + set));
            const int t = (int)j * TM + r;
            if (t < a.T) a.prob[(size_t)(a.w0 + wl) * a.T + t] = pr;
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 8) tmem_dealloc(tmem, 512);
}

// ---- half-heads for the element-wise time-slide evaluation (gwi_heads.cu) ---------------------------------------------
// Same roles as k_head_tc (warps 0-7 epilogue in two sets, warp 8 bulk-copy producer, warp 9 MMA issuer), items = (window,
// tile) of a block of segments; per item two accumulators: u_H . W1[:, :128]^T and u_L . W1[:, 128:]^T (8 K steps each),
// written as fp16 rows.  Warm-up tiles of a segment are skipped by all three roles alike.
__global__ void __launch_bounds__(HEAD_THREADS, 1) k_vhalf_tc(const HeadArgs a)
{
    extern __shared__ __align__(1024) uint8_t smem[];
    const uint32_t sbase = smem_u32(smem);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int W1B = 2 * U_TILE_BYTES, OFF_U = W1B, OFF_BAR = 7 * U_TILE_BYTES;
    auto bar = [&](int i) { return sbase + OFF_BAR + 8 * i; };   // 0 w1_full, 1-2 u_full, 3-4 u_free, 5-6 acc_full, 7-8 acc_free
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + OFF_BAR + 8 * 20);
    if (threadIdx.x == 0) {
        for (int i = 0; i < 9; i++) mbar_init(bar(i), (i == 7 || i == 8) ? 128u : 1u);
        mbar_fence_init();
    }
    if (warp == 8) tmem_alloc(smem_u32(tmem_slot), 512);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;
    const int64_t nitems = a.nwin * a.ntiles;
    auto skip = [&](int64_t it) { return (int)(it % a.ntiles) < (((it / a.ntiles) == 0 && a.stream_start) ? 0 : a.warm_tiles); };
    if (warp == 8) {
        if (lane == 0) {
            mbar_arrive_expect_tx(bar(0), W1B);
            bulk_g2s(sbase, a.w1, W1B, bar(0));
            uint32_t n = 0;
            for (int64_t it = blockIdx.x; it < nitems; it += gridDim.x) {
                if (skip(it)) continue;
                const int st = n & 1;
                const int64_t wl = it / a.ntiles, j = it % a.ntiles;
                mbar_wait(bar(3 + st), ((n >> 1) & 1) ^ 1);
                mbar_arrive_expect_tx(bar(1 + st), W1B);
                for (int b = 0; b < 2; b++)
                    bulk_g2s(sbase + OFF_U + st * W1B + b * U_TILE_BYTES, a.u + (((size_t)wl * 2 + b) * a.ntiles + j) * U_TILE_BYTES,
                             U_TILE_BYTES, bar(1 + st));
                n++;
            }
        }
        __syncwarp();
    } else if (warp == 9) {
        if (elect_one()) {
            const uint32_t idesc = make_idesc_f16(128, 128);
            const uint64_t dW = make_sdesc(sbase, 2048, 128);
            const uint64_t dU = make_sdesc(sbase + OFF_U, 2048, 128);
            mbar_wait(bar(0), 0);
            uint32_t n = 0;
            for (int64_t it = blockIdx.x; it < nitems; it += gridDim.x) {
                if (skip(it)) continue;
                const int st = n & 1;
                const uint32_t ph = (n >> 1) & 1;
                mbar_wait(bar(1 + st), ph);
                mbar_wait(bar(7 + st), ph ^ 1);
                tc_fence_after();
                const uint64_t du = dU + st * (W1B >> 4);
                const uint32_t dt = tmem + 256 * st;
#pragma unroll
                for (int kk = 0; kk < 8; kk++) tc_mma_f16(dt, du + kk * 256, dW + kk * 256, idesc, kk > 0 ? 1u : 0u);
#pragma unroll
                for (int kk = 8; kk < 16; kk++) tc_mma_f16(dt + 128, du + kk * 256, dW + kk * 256, idesc, kk > 8 ? 1u : 0u);
                tc_commit(bar(5 + st));
                tc_commit(bar(3 + st));
                n++;
            }
        }
        __syncwarp();
    } else {
        const int set = warp >> 2, r = (warp & 3) * 32 + lane;
        const uint32_t lane_t = tmem + ((uint32_t)((warp & 3) * 32) << 16);
        uint32_t n = 0;
        for (int64_t it = blockIdx.x; it < nitems; it += gridDim.x) {
            if (skip(it)) continue;
            const uint32_t my = n++;
            if ((int)(my & 1) != set) continue;
            const int64_t wl = it / a.ntiles, j = it % a.ntiles;
            const int warm = (wl == 0 && a.stream_start) ? 0 : a.warm_tiles;
            const int64_t row = (wl * a.seg_tiles + (j - warm)) * TM + r;
            mbar_wait(bar(5 + set), (my >> 1) & 1);
            tc_fence_after();
#pragma unroll
            for (int b = 0; b < 2; b++) {
                uint4* dst = reinterpret_cast<uint4*>(a.vout + ((size_t)b * a.vlds + row) * 128);
#pragma unroll
                for (int cc = 0; cc < 4; cc++) {
                    uint32_t v[32];
                    tmem_ld32(lane_t + 256 * set + 128 * b + 32 * cc, v);
                    tc_wait_ld();
                    if (row < a.n_valid) {
#pragma unroll
                        for (int c = 0; c < 4; c++) {
                            uint32_t q[4];
#pragma unroll
                            for (int e = 0; e < 4; e++) {
                                const int col = 8 * c + 2 * e;
                                float x0 = __uint_as_float(v[col]), x1 = __uint_as_float(v[col + 1]);
                                if (b == 0) x0 += a.b1[32 * cc + col], x1 += a.b1[32 * cc + col + 1];
                                q[e] = pack_half2(x0, x1);
                            }
                            dst[4 * cc + c] = make_uint4(q[0], q[1], q[2], q[3]);
                        }
                    }
                }
            }
            tc_fence_before();
            mbar_arrive(bar(7 + set));
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 8) tmem_dealloc(tmem, 512);
}

} // namespace

// ---- host side: packing and launch -----------------------------------------------------------------------------------
struct GwiTcPack {
    uint8_t *d_wfg = nullptr, *d_wrs = nullptr, *d_w1 = nullptr;
    float *d_cst = nullptr;
    float h_hc[257];        // b1[128], W2[128], b2 (passed to k_head_tc by value)
    float h_bias[2][TC_MAX_L][BIAS_FLOATS];   // bf, bg/2, br of every (branch, layer) (passed to k_stack by value)
    TcMeta meta;
    int num_sms = 148;
};

bool gwi_tc_supported(const GwiArch& a)
{
    if (a.R != 64 || a.S != 128 || a.Hh != 128 || a.k != 2 || a.c_in != 1 || a.n_branch > 2 || a.L > TC_MAX_L) return false;
    int stash = 0;
    for (int i = 0; i < a.L; i++) {
        int d = a.dil[i];
        if (d <= 32) stash += d * 128;
        else if (d == 64) continue;
        else if (d % 128 != 0 || ((d / 128) & (d / 128 - 1)) != 0) return false;   // whole tiles, power of two
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
    memset(p->h_bias, 0, sizeof(p->h_bias));
    int so = 0, ro = 0, n64 = 0;
    for (int i = 0; i < L; i++) {
        M.dil[i] = a.dil[i];
        M.kind[i] = a.dil[i] <= 32 ? 0 : (a.dil[i] == 64 ? 1 : 2);
        M.D[i] = M.kind[i] == 2 ? a.dil[i] / 128 : 0;
        M.stash_off[i] = so;
        M.lay[i] = M.kind[i] | (a.dil[i] << 2);
        if (M.kind[i] == 2) M.ring_off[i] = ro, ro += M.D[i];
        else if (M.kind[i] == 1) M.ring_off[i] = n64++;
        else M.ring_off[i] = 0, so += a.dil[i] * 128;
    }
    M.ring_tiles = ro > 0 ? ro : 1;
    M.n64 = n64 > 0 ? n64 : 1;
    const float* W = m->host_blob.data();
    std::vector<uint16_t> wfg((size_t)nb * L * WFG_BYTES / 2), wrs((size_t)nb * L * WRS_STRIDE / 2), w1((size_t)nb * U_TILE_BYTES / 2);
    std::vector<float> cst((size_t)nb * 256, 0.f), hc(257);
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
            uint16_t* rs = wrs.data() + ((size_t)b * L + i) * (WRS_STRIDE / 2);
            for (int n = 0; n < 192; n++)
                for (int k = 0; k < 64; k++) {
                    float v = n < 128 ? 0.5f * W[lo.Ws + (int64_t)n * 64 + k] : 0.5f * W[lo.Wr + (int64_t)(n - 128) * 64 + k];
                    rs[(k / 8) * (192 * 8) + n * 8 + (k % 8)] = h16(v);
                }
            float bl[BIAS_FLOATS];
            for (int c = 0; c < 64; c++) {
                bl[c] = W[lo.bf + c];
                bl[64 + c] = 0.5f * W[lo.bg + c];
                bl[128 + c] = W[lo.br + c];
            }
            memcpy(rs + WRS_BYTES / 2, bl, sizeof(bl));
            memcpy(p->h_bias[b][i], bl, sizeof(bl));
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
    GWI_CUDA_CHECK(up((void**)&p->d_cst, cst.data(), cst.size() * 4));
    memcpy(p->h_hc, hc.data(), sizeof(p->h_hc));
    cudaDeviceProp prop;
    GWI_CUDA_CHECK(cudaGetDeviceProperties(&prop, m->device));
    p->num_sms = prop.multiProcessorCount;
    GWI_CUDA_CHECK(cudaFuncSetAttribute(k_stack, cudaFuncAttributeMaxDynamicSharedMemorySize, SM_TOTAL));
    GWI_CUDA_CHECK(cudaFuncSetAttribute(k_head_tc, cudaFuncAttributeMaxDynamicSharedMemorySize, HEAD_SMEM));
    GWI_CUDA_CHECK(cudaFuncSetAttribute(k_vhalf_tc, cudaFuncAttributeMaxDynamicSharedMemorySize, HEAD_SMEM));
    return GWI_OK;
}

void gwi_tc_free(gwi_model* m)
{
    GwiTcPack* p = m->tc;
    if (!p) return;
    cudaFree(p->d_wfg), cudaFree(p->d_wrs), cudaFree(p->d_w1), cudaFree(p->d_cst);
    delete p;
    m->tc = nullptr;
}

// Windows per launch: the u workspace (32 KB per window-branch-tile) is bounded to ~16 GiB; a batch is cut into equal
// launches so that no launch is left with a handful of windows (one job is a whole window pair: a short launch would
// run on a few SMs for as long as a full one).
static int64_t tc_chunk(int64_t B, int nb, int64_t ntiles)
{
    int64_t cap = (16LL << 30) / ((int64_t)nb * ntiles * U_TILE_BYTES);
    if (cap < 296) cap = 296;
    if (B <= cap) return B;
    int64_t launches = (B + cap - 1) / cap;
    return (B + launches - 1) / launches;
}

size_t gwi_tc_workspace_bytes(const gwi_model* m, int64_t B, int32_t T)
{
    const GwiTcPack* p = m->tc;
    int64_t ntiles = (T + TM - 1) / TM;
    size_t ring = (size_t)p->num_sms * 2 * p->meta.ring_tiles * PST_BYTES;
    size_t ring64 = (size_t)p->num_sms * 2 * p->meta.n64 * 2 * PRE_BYTES;
    size_t u = (size_t)tc_chunk(B, m->arch.n_branch, ntiles) * m->arch.n_branch * ntiles * U_TILE_BYTES;
    return ring + ring64 + u + 512;
}

gwi_status gwi_tc_infer(const gwi_model* m, const __half* d_strain, int64_t B, int32_t T, float* d_prob, void* d_ws,
                        size_t ws_bytes, cudaStream_t st)
{
    const GwiTcPack* p = m->tc;
    const int nb = m->arch.n_branch;
    const int ntiles = (T + TM - 1) / TM;
    size_t ring_bytes = ((size_t)p->num_sms * 2 * p->meta.ring_tiles * PST_BYTES + 255) & ~(size_t)255;
    size_t ring64_bytes = ((size_t)p->num_sms * 2 * p->meta.n64 * 2 * PRE_BYTES + 255) & ~(size_t)255;
    uint8_t* ring = (uint8_t*)d_ws;
    uint8_t* ring64 = ring + ring_bytes;
    uint8_t* u = ring64 + ring64_bytes;
    const int64_t Bc = tc_chunk(B, nb, ntiles);
    for (int64_t w0 = 0; w0 < B; w0 += Bc) {
        const int64_t nwin = (B - w0 < Bc) ? B - w0 : Bc;
        StackArgs sa;
        sa.wfg = p->d_wfg, sa.wrs = p->d_wrs, sa.cst = p->d_cst, sa.strain = d_strain;
        sa.w0 = w0, sa.nwin = nwin, sa.T = T, sa.ntiles = ntiles, sa.C = nb * m->arch.c_in;
        sa.ring = ring, sa.ring64 = ring64, sa.u = u, sa.meta = p->meta;
        memcpy(sa.bias, p->h_bias, sizeof(sa.bias));
        int64_t njobs = ((nwin + 1) / 2) * nb;
        int grid = (int)(njobs < p->num_sms ? njobs : p->num_sms);
        k_stack<<<grid, NTHREADS, SM_TOTAL, st>>>(sa);
        HeadArgs ha;
        memcpy(ha.b1, p->h_hc, 128 * 4), memcpy(ha.w2, p->h_hc + 128, 128 * 4), ha.b2 = p->h_hc[256];
        ha.w1 = p->d_w1, ha.u = u, ha.prob = d_prob, ha.w0 = w0, ha.nwin = nwin, ha.T = T, ha.ntiles = ntiles,
        ha.n_branch = nb, ha.mode = 0, ha.hist = nullptr, ha.lags = nullptr, ha.nq = 0, ha.stride_k = 0, ha.n_lags = 0, ha.R = 0,
        ha.seg_tiles = 0, ha.warm_tiles = 0, ha.stream_start = 0, ha.n_valid = 0, ha.vout = nullptr, ha.vlds = 0;
        int64_t nitems = nwin * ntiles;
        int hgrid = (int)(nitems < p->num_sms ? nitems : p->num_sms);
        k_head_tc<<<hgrid, HEAD_THREADS, HEAD_SMEM, st>>>(ha);
        gwi_count_launch(2);
        GWI_CUDA_CHECK(cudaGetLastError());
#ifdef GWI_TC_TRACE
        if (const char* tp = getenv("GWI_TC_TRACE_FILE")) {
            cudaStreamSynchronize(st);
            std::vector<uint4> ev(19 * TRACE_CAP);
            cudaMemcpyFromSymbol(ev.data(), g_trace, ev.size() * 16);
            if (FILE* f = fopen(tp, "w")) {
                for (auto& e : ev) fprintf(f, "%u %u %u %u\n", e.x, e.y, e.z, e.w);
                fclose(f);
            }
        }
#endif
    }
    return GWI_OK;
}

// ---- pieces for the streaming back end with time slides (gwi_stream.cu) ---------------------------------------------
int64_t gwi_tc_max_windows(const gwi_model* m, int32_t T)
{
    const int64_t ntiles = (T + TM - 1) / TM;
    int64_t cap = (16LL << 30) / ((int64_t)m->arch.n_branch * ntiles * U_TILE_BYTES);
    return cap < 296 ? 296 : cap;
}

int gwi_tc_num_sms(const gwi_model* m) { return m->tc->num_sms; }

// Branch stacks only: B windows (B <= gwi_tc_max_windows) -> u tiles [B][n_branch][ntiles][U_TILE_BYTES] at *u_out
// inside the workspace (same layout as gwi_tc_infer uses between its two kernels).
gwi_status gwi_tc_stack(const gwi_model* m, const __half* d_strain, int64_t B, int32_t T, void* d_ws, size_t ws_bytes,
                        cudaStream_t st, const uint8_t** u_out)
{
    const GwiTcPack* p = m->tc;
    const int nb = m->arch.n_branch;
    const int ntiles = (T + TM - 1) / TM;
    if (B > gwi_tc_max_windows(m, T) || ws_bytes < gwi_tc_workspace_bytes(m, B, T)) {
        gwi_set_error("gwi_tc_stack: batch of %lld windows does not fit one launch / the workspace", (long long)B);
        return GWI_ERR_NOMEM;
    }
    size_t ring_bytes = ((size_t)p->num_sms * 2 * p->meta.ring_tiles * PST_BYTES + 255) & ~(size_t)255;
    size_t ring64_bytes = ((size_t)p->num_sms * 2 * p->meta.n64 * 2 * PRE_BYTES + 255) & ~(size_t)255;
    uint8_t* ring = (uint8_t*)d_ws;
    uint8_t* ring64 = ring + ring_bytes;
    uint8_t* u = ring64 + ring64_bytes;
    StackArgs sa;
    sa.wfg = p->d_wfg, sa.wrs = p->d_wrs, sa.cst = p->d_cst, sa.strain = d_strain;
    sa.w0 = 0, sa.nwin = B, sa.T = T, sa.ntiles = ntiles, sa.C = nb * m->arch.c_in;
    sa.ring = ring, sa.ring64 = ring64, sa.u = u, sa.meta = p->meta;
    memcpy(sa.bias, p->h_bias, sizeof(sa.bias));
    int64_t njobs = ((B + 1) / 2) * nb;
    int grid = (int)(njobs < p->num_sms ? njobs : p->num_sms);
    k_stack<<<grid, NTHREADS, SM_TOTAL, st>>>(sa);
    gwi_count_launch(1);
    GWI_CUDA_CHECK(cudaGetLastError());
    *u_out = u;
    return GWI_OK;
}

// Half-heads v_H, v_L of every output sample of a block of B windows whose u tiles gwi_tc_stack has just written (same
// segment layout): fp16 rows at d_v + (branch * lds + row) * 128, row = sample index inside the block.
gwi_status gwi_tc_vhalf(const gwi_model* m, const uint8_t* u, int64_t B, int ntiles, int seg_tiles, int warm_tiles, int stream_start,
                        int n_valid, __half* d_v, int64_t lds, cudaStream_t st)
{
    const GwiTcPack* p = m->tc;
    HeadArgs ha;
    memcpy(ha.b1, p->h_hc, 128 * 4), memcpy(ha.w2, p->h_hc + 128, 128 * 4), ha.b2 = p->h_hc[256];
    ha.w1 = p->d_w1, ha.u = u, ha.prob = nullptr, ha.w0 = 0, ha.nwin = B, ha.T = 0, ha.ntiles = ntiles;
    ha.n_branch = 2, ha.mode = 0, ha.hist = nullptr, ha.lags = nullptr, ha.nq = 0, ha.stride_k = 0, ha.n_lags = 0, ha.R = 0;
    ha.seg_tiles = seg_tiles, ha.warm_tiles = warm_tiles, ha.stream_start = stream_start, ha.n_valid = n_valid;
    ha.vout = d_v, ha.vlds = lds;
    const int64_t nitems = B * ntiles;
    int grid = (int)(nitems < p->num_sms ? nitems : p->num_sms);
    k_vhalf_tc<<<grid, HEAD_THREADS, HEAD_SMEM, st>>>(ha);
    gwi_count_launch(1);
    GWI_CUDA_CHECK(cudaGetLastError());
    return GWI_OK;
}

// Heads of all lags over the nq output tiles of a block (see HeadArgs, stream mode); d_lags: device array of n_lags lags
// in samples (multiples of 128); probabilities of lag k at d_prob + k * stride_k.
gwi_status gwi_tc_head_stream(const gwi_model* m, const uint8_t* u, int ntiles, const uint8_t* hist, int R, int64_t nq,
                              const int64_t* d_lags, int n_lags, int seg_tiles, int warm_tiles, int stream_start, int n_valid,
                              float* d_prob, int64_t stride_k, cudaStream_t st)
{
    const GwiTcPack* p = m->tc;
    if (m->arch.n_branch != 2 || n_lags < 2) {
        gwi_set_error("gwi_tc_head_stream: two branches and at least two slides (zero lag + one lag) expected");
        return GWI_ERR_UNSUPPORTED;
    }
    HeadArgs ha;
    memcpy(ha.b1, p->h_hc, 128 * 4), memcpy(ha.w2, p->h_hc + 128, 128 * 4), ha.b2 = p->h_hc[256];
    ha.w1 = p->d_w1, ha.u = u, ha.prob = d_prob, ha.w0 = 0, ha.nwin = 0, ha.T = 0, ha.ntiles = ntiles;
    ha.n_branch = 2, ha.mode = 1, ha.hist = hist, ha.lags = d_lags, ha.nq = nq, ha.stride_k = stride_k, ha.n_lags = n_lags, ha.R = R;
    ha.seg_tiles = seg_tiles, ha.warm_tiles = warm_tiles, ha.stream_start = stream_start, ha.n_valid = n_valid;
    ha.vout = nullptr, ha.vlds = 0;
    int hgrid = (int)(nq < p->num_sms ? nq : p->num_sms);
    k_head_tc<<<hgrid, HEAD_THREADS, HEAD_SMEM, st>>>(ha);
    gwi_count_launch(1);
    GWI_CUDA_CHECK(cudaGetLastError());
    return GWI_OK;
}
