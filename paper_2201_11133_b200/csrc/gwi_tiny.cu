// gwi_tiny.cu -- fused FP16-mode stream kernel for the narrow ("config-1") architecture: n_branch = 2, c_in = 1,
// R = 16, S = Hh = 32, k = 2, any dilation list whose receptive field fits the halo (sum d_i <= 64).
//
// The ensembles of BASELINE.json configs 3-5 are built from this architecture.  Its contractions are tiny (K = 32 and
// K = 16 per block), so the path is bound by MUFU (256 tanh per output sample) and plain ALU work, not by the tensor
// pipe.  One kernel evaluates lift -> L gated residual blocks -> skip sum -> ReLU ->
// head -> sigmoid (DESIGN.md C.1 steps 1-5) for a tile of 128 - 16*HT consecutive stream samples per
// CTA without writing any activation to global memory:
//
//   * time runs along the MMA M dimension, 16 rows per warp, 8 warps per CTA; the small channel contractions are
//     warp-level m16n8k16 MMAs (fp16 operands, fp32 accumulate, reading A14) whose accumulator fragments are gated
//     in registers and re-used directly as the A fragments of the next MMA (no shuffle, no shared-memory round trip);
//   * the past tap h(t - d) of a dilated conv is the only cross-row access: every layer's fp16 operand tile is
//     parked in shared memory (row stride 48 B: conflict-free fragment loads) and read back d rows earlier;
//   * overlap reuse (row a-2): the first 16*HT rows of a tile are a halo that is recomputed from the carried last
//     16*HT input samples of the previous chunk, so nothing but those samples is carried across chunks; rows at global
//     time t < 0 are forced to zero at every layer input, which is exactly the causal padding of reading A4.
//     Every output sample is an independent fixed-order computation, so chunked == unchunked bit for bit (reading A17).
//
// Output: either the per-sample probability (fused head, zero lag) or, for time slides (reading A24), the branch
// features u = ReLU(skip sum) as fp16 time-major rows, from which k_tiny_heads evaluates the head for every lag.
#include <cstdlib>
#include <cstring>
#include <vector>

#include "gwi_internal.h"

namespace {

constexpr int TW = 8;             // warps per CTA
constexpr int NT = 2;             // 16-row MMA tiles per warp: every weight / bias fragment load serves 32 rows
constexpr int ROWS = TW * NT * 16;   // rows (time steps) per CTA tile, halo included
constexpr int RS = 24;            // shared-memory row stride in halves (16 channels + 8 pad = 48 bytes)
constexpr int PADROWS = 64;       // zero rows in front of the tile (reads at row - d of the first rows)
constexpr int TINY_MAX_L = 8;

struct TinyArgs {
    const uint2* wfg;     // [nb][L][ks 2][nt 4][32]   B fragments of [past | current] x [f | g/2]
    const uint2* wrs;     // [nb][L][nt 6][32]         B fragments of z' x [res | skip], both halved
    const uint2* w1;      // [ks 4][nt 4][32]          B fragments of [u_H | u_L] x W1^T
    const float* bias;    // [nb][L][80]: bf[16], bg/2[16], br[16], bs[32]
    const float* cst;     // [nb][32]: W_in[16], b_in[16];  then head: b1[32], W2[32], b2
    const __half* x;      // planar strain chunk: channel c at x + c * ldx, n samples
    const __half* xh;     // [2][HALO] last HALO samples of the previous chunk (zeros at the stream start)
    int64_t ldx;
    int64_t t0;           // global index of sample 0 of this chunk
    int n, L, halo;       // halo = 16 * HT rows
    int dil[TINY_MAX_L];
    float* prob;          // fused head: [n] probabilities (null in skip mode)
    __half* u16;          // time-slide mode: [nb][lds][32] branch features u = ReLU(skip sum), fp16, time-major
    int64_t lds;          //   (null in fused mode); row 0 = sample 0 of this chunk
};

// D (+)= A B, accumulating in place
__device__ __forceinline__ void mma16816(float (&c)[4], const uint32_t (&a)[4], uint2 b)
{
    asm("mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
        : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
        : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b.x), "r"(b.y));
}
// D = A B + (c0, c1, c0, c1): the accumulator starts at the bias of its two columns without being initialised by moves
__device__ __forceinline__ void mma16816_bias(float (&d)[4], const uint32_t (&a)[4], uint2 b, float c0, float c1)
{
    asm("mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%10,%11,%10,%11};"
        : "=f"(d[0]), "=f"(d[1]), "=f"(d[2]), "=f"(d[3])
        : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b.x), "r"(b.y), "f"(c0), "f"(c1));
}
__device__ __forceinline__ uint32_t pack2(float lo, float hi)
{
    __half2 h = __floats2half2_rn(lo, hi);
    return *reinterpret_cast<uint32_t*>(&h);
}
__device__ __forceinline__ float tanh_fast(float x)
{
    float y;
    asm("tanh.approx.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

__global__ void __launch_bounds__(TW * 32, 2) k_tiny(const __grid_constant__ TinyArgs a)
{
    // two operand buffers (layer parity), each PADROWS zero rows + ROWS rows of 16 halves (+ pad)
    __shared__ __align__(16) __half sm[2][(PADROWS + ROWS) * RS];
    __shared__ uint4 sm_u[NT][2][TW * 32];                               // branch 0's head fragments, parked while branch 1 runs
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
    const int valid = ROWS - a.halo;                                    // output rows per CTA
    const int64_t tile0 = (int64_t)blockIdx.x * valid - a.halo;          // chunk-local time of row 0
    // this thread's rows: tile tl of the warp holds rows rbase + 16 tl + g and + 8
    const int rbase = warp * (16 * NT) + g;
    // rows before the stream start are zero at every layer input (reading A4)
    const bool premask = a.t0 + tile0 < 0;                               // CTA-uniform: only the first tile of a stream
    for (int i = threadIdx.x; i < 2 * PADROWS * RS / 2; i += TW * 32) {
        int buf = i / (PADROWS * RS / 2), k = i % (PADROWS * RS / 2);
        reinterpret_cast<uint32_t*>(sm[buf])[k] = 0u;
    }
    const float* hcst = a.cst + 2 * 32;
    uint32_t ua[NT][2][4];                                               // head A fragments of the current branch

#pragma unroll
    for (int b = 0; b < 2; b++) {
        // ---- lift (C.1 step 1): h0[r] = W_in[r] x + b_in[r]; fp32 master in accumulator-fragment layout
        float h[NT][2][4];                                               // [tile][n-tile (8 channels)][c0..c3]
        {
            const __half* xc = a.x + (int64_t)b * a.ldx;
            const __half* xp = a.xh + b * a.halo;
            const float* cb = a.cst + b * 32;
            float2 w[2], bi[2];
#pragma unroll
            for (int nt = 0; nt < 2; nt++) {
                w[nt] = __ldg(reinterpret_cast<const float2*>(cb + 8 * nt + 2 * t));
                bi[nt] = __ldg(reinterpret_cast<const float2*>(cb + 16 + 8 * nt + 2 * t));
            }
#pragma unroll
            for (int tl = 0; tl < NT; tl++) {
                const int64_t tl0 = tile0 + rbase + 16 * tl, tl1 = tl0 + 8;
                float x0 = 0.f, x1 = 0.f;
                if (tl0 >= 0) { if (tl0 < a.n) x0 = __half2float(xc[tl0]); } else x0 = __half2float(xp[a.halo + tl0]);
                if (tl1 >= 0) { if (tl1 < a.n) x1 = __half2float(xc[tl1]); } else x1 = __half2float(xp[a.halo + tl1]);
#pragma unroll
                for (int nt = 0; nt < 2; nt++) {
                    h[tl][nt][0] = fmaf(w[nt].x, x0, bi[nt].x), h[tl][nt][1] = fmaf(w[nt].y, x0, bi[nt].y);
                    h[tl][nt][2] = fmaf(w[nt].x, x1, bi[nt].x), h[tl][nt][3] = fmaf(w[nt].y, x1, bi[nt].y);
                }
                if (premask) {
                    if (a.t0 + tl0 < 0) h[tl][0][0] = h[tl][0][1] = h[tl][1][0] = h[tl][1][1] = 0.f;
                    if (a.t0 + tl1 < 0) h[tl][0][2] = h[tl][0][3] = h[tl][1][2] = h[tl][1][3] = 0.f;
                }
            }
        }
        float sk[NT][4][4];                                              // skip sum, 4 n-tiles of 8 channels
#pragma unroll
        for (int nt = 0; nt < 4; nt++) {                                 // starts at sum_i bs_i (summed on the host)
            float2 bb = __ldg(reinterpret_cast<const float2*>(a.cst + 2 * 32 + 66 + b * 32 + 8 * nt + 2 * t));
#pragma unroll
            for (int tl = 0; tl < NT; tl++) sk[tl][nt][0] = bb.x, sk[tl][nt][1] = bb.y, sk[tl][nt][2] = bb.x, sk[tl][nt][3] = bb.y;
        }

        const float* bl = a.bias + (size_t)b * a.L * 80 + 2 * t;
        const uint2* wf = a.wfg + (size_t)b * a.L * (2 * 4 * 32) + lane;
        const uint2* wr = a.wrs + (size_t)b * a.L * (6 * 32) + lane;
        for (int i = 0; i < a.L; i++, bl += 80, wf += 2 * 4 * 32, wr += 6 * 32) {
            const int d = a.dil[i];
            __half* buf = sm[i & 1] + (PADROWS + rbase) * RS + 2 * t;
            // ---- current-tap A fragment = this thread's own h values; parked in shared memory for the rows d later
            uint32_t ac[NT][4], ap[NT][4];
#pragma unroll
            for (int tl = 0; tl < NT; tl++) {
                ac[tl][0] = pack2(h[tl][0][0], h[tl][0][1]), ac[tl][1] = pack2(h[tl][0][2], h[tl][0][3]);
                ac[tl][2] = pack2(h[tl][1][0], h[tl][1][1]), ac[tl][3] = pack2(h[tl][1][2], h[tl][1][3]);
                __half* row = buf + 16 * tl * RS;
                *reinterpret_cast<uint32_t*>(row) = ac[tl][0];
                *reinterpret_cast<uint32_t*>(row + 8 * RS) = ac[tl][1];
                *reinterpret_cast<uint32_t*>(row + 8) = ac[tl][2];
                *reinterpret_cast<uint32_t*>(row + 8 * RS + 8) = ac[tl][3];
            }
            __syncthreads();   // one barrier per layer: the buffers alternate, so layer i+2 cannot overtake layer i readers
#pragma unroll
            for (int tl = 0; tl < NT; tl++) {
                const __half* row = buf + (16 * tl - d) * RS;
                ap[tl][0] = *reinterpret_cast<const uint32_t*>(row);
                ap[tl][1] = *reinterpret_cast<const uint32_t*>(row + 8 * RS);
                ap[tl][2] = *reinterpret_cast<const uint32_t*>(row + 8);
                ap[tl][3] = *reinterpret_cast<const uint32_t*>(row + 8 * RS + 8);
            }
            // ---- f | g/2 = [h(t-d) | h(t)] . W^T + bias                                      (C.1 step 2)
            float fg[NT][4][4];
#pragma unroll
            for (int nt = 0; nt < 4; nt++) {
                const float2 bb = __ldg(reinterpret_cast<const float2*>(bl + 8 * nt));
                const uint2 w0 = __ldg(wf + (0 * 4 + nt) * 32), w1 = __ldg(wf + (1 * 4 + nt) * 32);
#pragma unroll
                for (int tl = 0; tl < NT; tl++) {
                    mma16816_bias(fg[tl][nt], ap[tl], w0, bb.x, bb.y);
                    mma16816(fg[tl][nt], ac[tl], w1);
                }
            }
            // ---- z' = tanh(f) (1 + tanh(g/2)) = 2 tanh(f) sigmoid(g); the 2 is folded into Wr/2, Ws/2
            uint32_t az[NT][4];
#pragma unroll
            for (int tl = 0; tl < NT; tl++) {
                float z[2][4];
#pragma unroll
                for (int nt = 0; nt < 2; nt++)
#pragma unroll
                    for (int c = 0; c < 4; c++) {
                        float tf = tanh_fast(fg[tl][nt][c]), tg = tanh_fast(fg[tl][nt + 2][c]);
                        z[nt][c] = fmaf(tf, tg, tf);
                    }
                az[tl][0] = pack2(z[0][0], z[0][1]), az[tl][1] = pack2(z[0][2], z[0][3]);
                az[tl][2] = pack2(z[1][0], z[1][1]), az[tl][3] = pack2(z[1][2], z[1][3]);
            }
            // ---- h += br + z' . (Wr/2)^T ;  skip += z' . (Ws/2)^T
            if (i < a.L - 1) {                                           // reading A8: the last residual conv is dead
#pragma unroll
                for (int nt = 0; nt < 2; nt++) {
                    const float2 bb = __ldg(reinterpret_cast<const float2*>(bl + 32 + 8 * nt));
                    const uint2 w = __ldg(wr + nt * 32);
#pragma unroll
                    for (int tl = 0; tl < NT; tl++) {
                        float rr[4];
                        mma16816_bias(rr, az[tl], w, bb.x, bb.y);
                        h[tl][nt][0] += rr[0], h[tl][nt][1] += rr[1], h[tl][nt][2] += rr[2], h[tl][nt][3] += rr[3];
                    }
                }
                if (premask) {
#pragma unroll
                    for (int tl = 0; tl < NT; tl++) {
                        const int64_t tg0 = a.t0 + tile0 + rbase + 16 * tl;
                        if (tg0 < 0) h[tl][0][0] = h[tl][0][1] = h[tl][1][0] = h[tl][1][1] = 0.f;
                        if (tg0 + 8 < 0) h[tl][0][2] = h[tl][0][3] = h[tl][1][2] = h[tl][1][3] = 0.f;
                    }
                }
            }
#pragma unroll
            for (int nt = 0; nt < 4; nt++) {
                const uint2 w = __ldg(wr + (2 + nt) * 32);
#pragma unroll
                for (int tl = 0; tl < NT; tl++) mma16816(sk[tl][nt], az[tl], w);
            }
        }
#pragma unroll
        for (int tl = 0; tl < NT; tl++) {
            const int r0 = rbase + 16 * tl, r1 = r0 + 8;
            const int64_t tl0 = tile0 + r0, tl1 = tl0 + 8;
            if (a.u16) {
                // ---- time-slide mode: u_b = ReLU(skip sum) in fp16, time-major, for the per-lag heads (k_tiny_heads)
                __half* up = a.u16 + (size_t)b * a.lds * 32;
#pragma unroll
                for (int nt = 0; nt < 4; nt++) {
                    const int q = 8 * nt + 2 * t;
                    if (r0 >= a.halo && tl0 < a.n)
                        *reinterpret_cast<uint32_t*>(up + tl0 * 32 + q) = pack2(fmaxf(sk[tl][nt][0], 0.f), fmaxf(sk[tl][nt][1], 0.f));
                    if (r1 >= a.halo && tl1 < a.n)
                        *reinterpret_cast<uint32_t*>(up + tl1 * 32 + q) = pack2(fmaxf(sk[tl][nt][2], 0.f), fmaxf(sk[tl][nt][3], 0.f));
                }
            } else {
                // ---- u_b = ReLU(skip sum) as the A fragments of the head                        (C.1 steps 3, 4)
#pragma unroll
                for (int ks = 0; ks < 2; ks++) {
                    ua[tl][ks][0] = pack2(fmaxf(sk[tl][2 * ks][0], 0.f), fmaxf(sk[tl][2 * ks][1], 0.f));
                    ua[tl][ks][1] = pack2(fmaxf(sk[tl][2 * ks][2], 0.f), fmaxf(sk[tl][2 * ks][3], 0.f));
                    ua[tl][ks][2] = pack2(fmaxf(sk[tl][2 * ks + 1][0], 0.f), fmaxf(sk[tl][2 * ks + 1][1], 0.f));
                    ua[tl][ks][3] = pack2(fmaxf(sk[tl][2 * ks + 1][2], 0.f), fmaxf(sk[tl][2 * ks + 1][3], 0.f));
                    if (b == 0) sm_u[tl][ks][threadIdx.x] = make_uint4(ua[tl][ks][0], ua[tl][ks][1], ua[tl][ks][2], ua[tl][ks][3]);
                }
            }
        }
        __syncthreads();   // the next branch starts again with buffer 0
    }
    if (a.u16) return;
    // ---- head: v = ReLU(W1 [u_H; u_L] + b1), y = W2 . v + b2, p = sigmoid(y)                   (C.1 step 5)
    float y[NT][2];
#pragma unroll
    for (int tl = 0; tl < NT; tl++) y[tl][0] = y[tl][1] = 0.f;
#pragma unroll
    for (int nt = 0; nt < 4; nt++) {
        const float2 bb = __ldg(reinterpret_cast<const float2*>(hcst + 8 * nt + 2 * t));
        const float2 w2 = __ldg(reinterpret_cast<const float2*>(hcst + 32 + 8 * nt + 2 * t));
        uint2 w[4];
#pragma unroll
        for (int ks = 0; ks < 4; ks++) w[ks] = __ldg(a.w1 + (ks * 4 + nt) * 32 + lane);
#pragma unroll
        for (int tl = 0; tl < NT; tl++) {
            float v[4];
#pragma unroll
            for (int ks = 0; ks < 2; ks++) {                             // H1 half (parked), then L1 half
                uint4 p = sm_u[tl][ks][threadIdx.x];
                uint32_t ah[4] = {p.x, p.y, p.z, p.w};
                if (ks == 0) mma16816_bias(v, ah, w[0], bb.x, bb.y);
                else mma16816(v, ah, w[1]);
            }
#pragma unroll
            for (int ks = 0; ks < 2; ks++) mma16816(v, ua[tl][ks], w[2 + ks]);
            y[tl][0] = fmaf(w2.x, fmaxf(v[0], 0.f), y[tl][0]), y[tl][0] = fmaf(w2.y, fmaxf(v[1], 0.f), y[tl][0]);
            y[tl][1] = fmaf(w2.x, fmaxf(v[2], 0.f), y[tl][1]), y[tl][1] = fmaf(w2.y, fmaxf(v[3], 0.f), y[tl][1]);
        }
    }
    const float b2 = __ldg(hcst + 64);
#pragma unroll
    for (int tl = 0; tl < NT; tl++) {
        float y0 = y[tl][0], y1 = y[tl][1];
        y0 += __shfl_xor_sync(0xffffffffu, y0, 1), y1 += __shfl_xor_sync(0xffffffffu, y1, 1);
        y0 += __shfl_xor_sync(0xffffffffu, y0, 2), y1 += __shfl_xor_sync(0xffffffffu, y1, 2);
        if (t == 0) {
            const int r0 = rbase + 16 * tl, r1 = r0 + 8;
            const int64_t tl0 = tile0 + r0, tl1 = tl0 + 8;
            if (r0 >= a.halo && tl0 < a.n) a.prob[tl0] = 1.0f / (1.0f + __expf(-(y0 + b2)));
            if (r1 >= a.halo && tl1 < a.n) a.prob[tl1] = 1.0f / (1.0f + __expf(-(y1 + b2)));
        }
    }
}

// Time-slide heads (reading A24): p_k[t] = head(u_H1[t], u_L1[t - lag_k]) for every lag of the list, from the fp16
// time-major branch features.  W1 [u_H; u_L] is split by linearity: the H1 half of the contraction is done once per
// 16-row tile and re-used for every lag, each lag adds its L1 half.  u16 row 0 = sample 0 of the chunk; L1 rows at negative indices are the
// ring of the previous max-lag samples.
struct HeadsArgs {
    const uint4* w1t;       // [half 2][mt 2][kk 2][32] A fragments of W1 in the k order of the 16-byte row loads (see the kernel)
    const float* hcst;      // b1[32], W2[32], b2
    const __half* u16;      // [2][lds][32], pointing at row 0 of this chunk
    int64_t lds;
    int n, n_lags;
    const int64_t* lags;    // device array
    float* prob;            // [n_lags][stride_k] ; this model's slice starts at prob
    int64_t stride_k;
};

__global__ void __launch_bounds__(256) k_tiny_heads(const HeadsArgs a)
{
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
    const int64_t row0 = ((int64_t)blockIdx.x * 8 + warp) * 16;
    if (row0 >= a.n) return;
    // The contraction is done transposed, D[channel][time] = W1 . u^T: the weights are the A operand (two m-tiles of 16
    // hidden channels), eight feature rows the B operand.  A lane's B fragments of both k-steps are then the 16 bytes
    // at offset 16 t of feature row g, one load and no register shuffling (the k order of the packed weights w1t is
    // permuted to match).  The warp handles two groups of eight rows.
    const int64_t ra = row0 + g, rb = ra + 8;
    const int64_t ca = ra < a.n ? ra : a.n - 1, cb = rb < a.n ? rb : a.n - 1;   // clamp loads of the ragged tail
    const uint4* uH = reinterpret_cast<const uint4*>(a.u16);
    const uint4* uL = reinterpret_cast<const uint4*>(a.u16 + a.lds * 32);
    // H1 half: acc[group][m-tile] = b1 + W1[:, 0:32] u_H; c0, c1: channel 16 mt + g, c2, c3: channel 16 mt + g + 8
    float acc[2][2][4];
    {
        const uint4 ha = uH[ca * 4 + t], hb = uH[cb * 4 + t];
#pragma unroll
        for (int mt = 0; mt < 2; mt++) {
            const float b_lo = __ldg(a.hcst + 16 * mt + g), b_hi = __ldg(a.hcst + 16 * mt + g + 8);
            const uint4 w0 = __ldg(a.w1t + (mt * 2 + 0) * 32 + lane), w1 = __ldg(a.w1t + (mt * 2 + 1) * 32 + lane);
            const uint32_t a0[4] = {w0.x, w0.y, w0.z, w0.w}, a1[4] = {w1.x, w1.y, w1.z, w1.w};
#pragma unroll
            for (int gr = 0; gr < 2; gr++) {
                const uint4 h = gr ? hb : ha;
                acc[gr][mt][0] = b_lo, acc[gr][mt][1] = b_lo, acc[gr][mt][2] = b_hi, acc[gr][mt][3] = b_hi;
                mma16816(acc[gr][mt], a0, make_uint2(h.x, h.y));
                mma16816(acc[gr][mt], a1, make_uint2(h.z, h.w));
            }
        }
    }
    uint32_t wl[2][2][4];
    float w2lo[2], w2hi[2];
#pragma unroll
    for (int mt = 0; mt < 2; mt++) {
#pragma unroll
        for (int kk = 0; kk < 2; kk++) {
            const uint4 w = __ldg(a.w1t + ((2 + mt) * 2 + kk) * 32 + lane);
            wl[mt][kk][0] = w.x, wl[mt][kk][1] = w.y, wl[mt][kk][2] = w.z, wl[mt][kk][3] = w.w;
        }
        w2lo[mt] = __ldg(a.hcst + 32 + 16 * mt + g), w2hi[mt] = __ldg(a.hcst + 32 + 16 * mt + g + 8);
    }
    const float b2 = __ldg(a.hcst + 64);
    // after the reduction over the eight channel lanes, lane (g, t) holds the row 8 (g >> 2) + 2 t + ((g >> 1) & 1)
    const bool hi16 = lane & 16, hi8 = lane & 8;
    const int64_t rst = row0 + 8 * (g >> 2) + 2 * t + ((g >> 1) & 1);
    const bool store = !(g & 1) && rst < a.n;
#pragma unroll 2
    for (int k = 0; k < a.n_lags; k++) {
        const int64_t lag = __ldg(a.lags + k);
        const uint4 la = uL[(ca - lag) * 4 + t], lb = uL[(cb - lag) * 4 + t];
        float p[4];                                  // group A time 2t, 2t + 1; group B time 2t, 2t + 1
#pragma unroll
        for (int gr = 0; gr < 2; gr++) {
            const uint4 l = gr ? lb : la;
            float y0 = 0.f, y1 = 0.f;
#pragma unroll
            for (int mt = 0; mt < 2; mt++) {
                float v[4] = {acc[gr][mt][0], acc[gr][mt][1], acc[gr][mt][2], acc[gr][mt][3]};
                mma16816(v, wl[mt][0], make_uint2(l.x, l.y));
                mma16816(v, wl[mt][1], make_uint2(l.z, l.w));
                y0 = fmaf(w2lo[mt], fmaxf(v[0], 0.f), y0), y0 = fmaf(w2hi[mt], fmaxf(v[2], 0.f), y0);
                y1 = fmaf(w2lo[mt], fmaxf(v[1], 0.f), y1), y1 = fmaf(w2hi[mt], fmaxf(v[3], 0.f), y1);
            }
            p[2 * gr] = y0, p[2 * gr + 1] = y1;
        }
        // sum over the 8 channel lanes (lane bits 2-4), halving the number of values at each step
        const float r0 = __shfl_xor_sync(0xffffffffu, hi16 ? p[0] : p[2], 16);
        const float r1 = __shfl_xor_sync(0xffffffffu, hi16 ? p[1] : p[3], 16);
        const float k0 = (hi16 ? p[2] : p[0]) + r0, k1 = (hi16 ? p[3] : p[1]) + r1;
        const float r2 = __shfl_xor_sync(0xffffffffu, hi8 ? k0 : k1, 8);
        float y = (hi8 ? k1 : k0) + r2;
        y += __shfl_xor_sync(0xffffffffu, y, 4);
        const float pr = __fdividef(1.0f, 1.0f + __expf(-(y + b2)));
        if (store) a.prob[(size_t)k * a.stride_k + rst] = pr;
    }
}

// keeps the last `halo` samples of each detector for the next chunk (older history shifts when n < halo)
__global__ void k_tiny_xhist(const __half* x, int64_t ldx, int n, int halo, const __half* xh_old, __half* xh_new)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= 2 * halo) return;
    int c = i / halo, k = i % halo;
    int64_t p = (int64_t)n - halo + k;
    xh_new[i] = p >= 0 ? x[c * ldx + p] : xh_old[c * halo + (halo + p)];
}

inline uint16_t h16(float v)
{
    __half h = __float2half_rn(v);
    uint16_t u;
    memcpy(&u, &h, 2);
    return u;
}

} // namespace

struct GwiTinyPack {
    uint2 *d_wfg = nullptr, *d_wrs = nullptr, *d_w1 = nullptr;
    uint4* d_w1t = nullptr;
    float *d_bias = nullptr, *d_cst = nullptr;
    int halo = 16;
    bool force_mma_sync = false;
};

bool gwi_tiny_supported(const GwiArch& a)
{
    if (a.n_branch != 2 || a.c_in != 1 || a.R != 16 || a.S != 32 || a.Hh != 32 || a.k != 2 || a.L > TINY_MAX_L) return false;
    int s = 0;
    for (int i = 0; i < a.L; i++) {
        if (a.dil[i] > PADROWS) return false;
        s += a.dil[i];
    }
    return s <= 64;
}

int gwi_tiny_halo(const gwi_model* m) { return m->tiny ? m->tiny->halo : 0; }

// true: gwi_tiny_stream in time-slide mode writes the half-head pre-activations v (tcgen05 kernel) for gwi_heads_fused;
// false: it writes the branch features u for gwi_tiny_heads (warp-MMA reference kernel)
bool gwi_tiny_writes_v(const gwi_model* m) { return m->tiny && m->tinytc && !m->tiny->force_mma_sync; }

gwi_status gwi_tiny_pack(gwi_model* m)
{
    const GwiArch& a = m->arch;
    const int L = a.L, nb = 2;
    GwiTinyPack* p = new GwiTinyPack();
    m->tiny = p;
    int sum = 0;
    for (int i = 0; i < L; i++) sum += a.dil[i];
    p->halo = ((sum + 15) / 16) * 16;
    if (p->halo < 16) p->halo = 16;
    const float* W = m->host_blob.data();
    // B fragment of mma.m16n8k16 (col-major 16 x 8): lane (g = lane / 4, t = lane % 4) holds
    //   b0 = {B[k = 2t][n = g], B[2t + 1][g]},  b1 = {B[2t + 8][g], B[2t + 9][g]}
    auto frag = [&](auto&& B, int k0, int n0, int lane) {
        int g = lane >> 2, t = lane & 3;
        uint2 r;
        r.x = (uint32_t)h16(B(k0 + 2 * t, n0 + g)) | ((uint32_t)h16(B(k0 + 2 * t + 1, n0 + g)) << 16);
        r.y = (uint32_t)h16(B(k0 + 2 * t + 8, n0 + g)) | ((uint32_t)h16(B(k0 + 2 * t + 9, n0 + g)) << 16);
        return r;
    };
    std::vector<uint2> wfg((size_t)nb * L * 8 * 32), wrs((size_t)nb * L * 6 * 32), w1(16 * 32);
    std::vector<float> bias((size_t)nb * L * 80), cst(2 * 32 + 65 + 1 + 2 * 32, 0.f);   // + pad + sum_i bs_i per branch
    for (int b = 0; b < nb; b++) {
        for (int c = 0; c < 16; c++) cst[b * 32 + c] = W[m->off.W_in[b] + c], cst[b * 32 + 16 + c] = W[m->off.b_in[b] + c];
        for (int i = 0; i < L; i++) {
            const GwiLayerOff& lo = m->off.layer[b][i];
            // B[k][n]: k < 16 past tap (tap 0) of channel k, k >= 16 current tap (tap 1); n < 16: f, n >= 16: g / 2
            auto Bfg = [&](int k, int n) {
                int tap = k < 16 ? 0 : 1, kin = k & 15;
                return n < 16 ? W[lo.Wf + ((int64_t)n * 16 + kin) * 2 + tap] : 0.5f * W[lo.Wg + ((int64_t)(n - 16) * 16 + kin) * 2 + tap];
            };
            for (int ks = 0; ks < 2; ks++)
                for (int nt = 0; nt < 4; nt++)
                    for (int l = 0; l < 32; l++) wfg[(((size_t)b * L + i) * 8 + ks * 4 + nt) * 32 + l] = frag(Bfg, 16 * ks, 8 * nt, l);
            // B[k][n]: n < 16: Wr[n][k] / 2, n >= 16: Ws[n - 16][k] / 2
            auto Brs = [&](int k, int n) { return n < 16 ? 0.5f * W[lo.Wr + (int64_t)n * 16 + k] : 0.5f * W[lo.Ws + (int64_t)(n - 16) * 16 + k]; };
            for (int nt = 0; nt < 6; nt++)
                for (int l = 0; l < 32; l++) wrs[(((size_t)b * L + i) * 6 + nt) * 32 + l] = frag(Brs, 0, 8 * nt, l);
            float* bl = bias.data() + ((size_t)b * L + i) * 80;
            for (int c = 0; c < 16; c++) bl[c] = W[lo.bf + c], bl[16 + c] = 0.5f * W[lo.bg + c], bl[32 + c] = W[lo.br + c];
            for (int q = 0; q < 32; q++) bl[48 + q] = W[lo.bs + q], cst[2 * 32 + 66 + b * 32 + q] += W[lo.bs + q];
        }
    }
    auto B1 = [&](int k, int n) { return W[m->off.W1 + (int64_t)n * 64 + k]; };   // k over [u_H(32) | u_L(32)]
    for (int ks = 0; ks < 4; ks++)
        for (int nt = 0; nt < 4; nt++)
            for (int l = 0; l < 32; l++) w1[(ks * 4 + nt) * 32 + l] = frag(B1, 16 * ks, 8 * nt, l);
    // k_tiny_heads contracts transposed (weights = A operand, 8 feature rows = B operand, see the kernel): A fragment of
    // half hb (0: u_H, 1: u_L), m-tile mt, k-step kk; fragment position (2t, 2t+1) <-> input channels 8t + 4kk + (0, 1),
    // position (2t+8, 2t+9) <-> channels 8t + 4kk + (2, 3)
    std::vector<uint4> w1t(16 * 32);
    for (int hb = 0; hb < 2; hb++)
        for (int mt = 0; mt < 2; mt++)
            for (int kk = 0; kk < 2; kk++)
                for (int l = 0; l < 32; l++) {
                    const int g = l >> 2, t = l & 3, c0 = 32 * hb + 8 * t + 4 * kk, n0 = 16 * mt + g;
                    auto pk = [&](int k, int n) { return (uint32_t)h16(B1(k, n)) | ((uint32_t)h16(B1(k + 1, n)) << 16); };
                    w1t[((hb * 2 + mt) * 2 + kk) * 32 + l] = make_uint4(pk(c0, n0), pk(c0, n0 + 8), pk(c0 + 2, n0), pk(c0 + 2, n0 + 8));
                }
    for (int c = 0; c < 32; c++) cst[64 + c] = W[m->off.b1 + c], cst[96 + c] = W[m->off.W2 + c];
    cst[128] = W[m->off.b2];
    auto up = [&](void** dst, const void* src, size_t bytes) -> cudaError_t {
        cudaError_t e = cudaMalloc(dst, bytes);
        if (e != cudaSuccess) return e;
        return cudaMemcpy(*dst, src, bytes, cudaMemcpyHostToDevice);
    };
    GWI_CUDA_CHECK(up((void**)&p->d_wfg, wfg.data(), wfg.size() * 8));
    GWI_CUDA_CHECK(up((void**)&p->d_wrs, wrs.data(), wrs.size() * 8));
    GWI_CUDA_CHECK(up((void**)&p->d_w1, w1.data(), w1.size() * 8));
    GWI_CUDA_CHECK(up((void**)&p->d_w1t, w1t.data(), w1t.size() * 16));
    GWI_CUDA_CHECK(up((void**)&p->d_bias, bias.data(), bias.size() * 4));
    GWI_CUDA_CHECK(up((void**)&p->d_cst, cst.data(), cst.size() * 4));
    const char* env = getenv("GWI_TINY_MMASYNC");
    p->force_mma_sync = env && env[0] == '1';
    if (gwi_tiny_tc_supported(a)) return gwi_tiny_tc_pack(m);
    return GWI_OK;
}

void gwi_tiny_free(gwi_model* m)
{
    GwiTinyPack* p = m->tiny;
    if (!p) return;
    cudaFree(p->d_wfg), cudaFree(p->d_wrs), cudaFree(p->d_w1), cudaFree(p->d_w1t), cudaFree(p->d_bias), cudaFree(p->d_cst);
    delete p;
    m->tiny = nullptr;
}

// One chunk of n samples of a planar fp16 stream through one model.  xh_cur / xh_next: [2][halo] carried input samples
// (xh_next may be null: no update).  prob: fused-head output [n], or null with d_u16 != null (time-slide mode:
// d_u16 = row of sample 0 inside a [2][lds][32] fp16 buffer).
gwi_status gwi_tiny_stream(const gwi_model* m, const __half* d_x, int64_t ldx, int n, int64_t t0, const __half* xh_cur,
                           __half* xh_next, float* d_prob, __half* d_u16, int64_t lds, cudaStream_t st)
{
    const GwiTinyPack* p = m->tiny;
    if (m->tinytc && !p->force_mma_sync) {
        // the tcgen05 kernel (gwi_tiny_tc.cu); the warp-MMA kernel below stays as the A/B reference (GWI_TINY_MMASYNC=1)
        gwi_status rc = gwi_tiny_tc_stream(m, d_x, ldx, n, t0, xh_cur, d_prob, d_u16, lds, st);
        if (rc != GWI_OK) return rc;
        if (xh_next) {
            k_tiny_xhist<<<(2 * p->halo + 127) / 128, 128, 0, st>>>(d_x, ldx, n, p->halo, xh_cur, xh_next);
            gwi_count_launch(1);
            GWI_CUDA_CHECK(cudaGetLastError());
        }
        return GWI_OK;
    }
    TinyArgs a;
    a.wfg = p->d_wfg, a.wrs = p->d_wrs, a.w1 = p->d_w1, a.bias = p->d_bias, a.cst = p->d_cst;
    a.x = d_x, a.xh = xh_cur, a.ldx = ldx, a.t0 = t0, a.n = n, a.L = m->arch.L, a.halo = p->halo;
    for (int i = 0; i < m->arch.L; i++) a.dil[i] = m->arch.dil[i];
    a.prob = d_prob, a.u16 = d_prob ? nullptr : d_u16, a.lds = lds;
    const int valid = ROWS - p->halo;
    const int grid = (n + valid - 1) / valid;
    k_tiny<<<grid, TW * 32, 0, st>>>(a);
    gwi_count_launch(1);
    if (xh_next) {
        k_tiny_xhist<<<(2 * p->halo + 127) / 128, 128, 0, st>>>(d_x, ldx, n, p->halo, xh_cur, xh_next);
        gwi_count_launch(1);
    }
    GWI_CUDA_CHECK(cudaGetLastError());
    return GWI_OK;
}

// Heads of all lags for one model on one chunk (time-slide mode).  d_u16: row of sample 0; d_lags: device array.
gwi_status gwi_tiny_heads(const gwi_model* m, const __half* d_u16, int64_t lds, int n, const int64_t* d_lags, int n_lags,
                          float* d_prob, int64_t stride_k, cudaStream_t st)
{
    const GwiTinyPack* p = m->tiny;
    HeadsArgs a;
    a.w1t = p->d_w1t, a.hcst = p->d_cst + 64, a.u16 = d_u16, a.lds = lds, a.n = n, a.n_lags = n_lags, a.lags = d_lags;
    a.prob = d_prob, a.stride_k = stride_k;
    k_tiny_heads<<<(n + 127) / 128, 256, 0, st>>>(a);
    gwi_count_launch(1);
    GWI_CUDA_CHECK(cudaGetLastError());
    return GWI_OK;
}

// carried input samples, any halo length (used by the stream back ends that recompute their warm-up from the input)
gwi_status gwi_xhist_update(const __half* d_x, int64_t ldx, int n, int halo, const __half* xh_cur, __half* xh_next, cudaStream_t st)
{
    k_tiny_xhist<<<(2 * halo + 127) / 128, 128, 0, st>>>(d_x, ldx, n, halo, xh_cur, xh_next);
    gwi_count_launch(1);
    GWI_CUDA_CHECK(cudaGetLastError());
    return GWI_OK;
}
