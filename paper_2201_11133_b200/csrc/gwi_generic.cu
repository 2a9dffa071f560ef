// gwi_generic.cu -- generic CUDA-core (fp32 FMA) implementation of the network for ANY GWIM architecture.
//
// This is the FP32 mode of the library (parity bar 1e-5) and the FP16-mode path for architectures the tcgen05
// kernel does not cover (operands rounded to binary16, fp32 arithmetic).  One kernel per layer, activations in a
// caller-provided device workspace:  lift -> L x block -> head.   Network definition: DESIGN.md C.1
// (two WaveNet-style branches, one per detector, concatenated, two conv layers, per-timestep
// probability); readings A3 (1x1 lift), A4 (per-layer causal zero padding), A5 (tap k-1 = current sample),
// A6/A7 (gated tanh*sigmoid, 1x1 residual and skip convs with bias), A8 (last residual conv has no effect),
// A9-A11 (skip sum -> ReLU -> concat -> 1x1 -> ReLU -> 1x1 -> sigmoid).
//
// Accuracy: every accumulation is bias first, then input-channel-major / tap-minor fp32 FMAs; tanhf/expf are the
// accurate CUDA libm versions (no fast-math), so the result is within ~3e-7 of the fp64 oracle.
#include "gwi_internal.h"

namespace {

constexpr int TT = 32;     // timesteps per CTA in the block / head kernels (one warp = 32 consecutive timesteps)
constexpr int GROUPS = 8;  // channel groups per CTA in the block kernel
constexpr int HGROUPS = 4; // hidden-unit groups per CTA in the head kernel

// h0[r][t] = b_in[r] + sum_c W_in[r][c] x[c][t]                                        (C.1 step 1, reading A3)
// Window mode: strain is [B][T][C] channels-last.  Stream mode (ldx > 0): strain is planar, channel c of branch br at
// strain + (br * c_in + c) * ldx.  ldh = row stride (in floats) of the activation buffers.
template <typename XT>
__global__ void k_lift(GwiDevModel m, const GwiOffsets* __restrict__ off, const XT* __restrict__ strain, int64_t w0,
                       int T, float* __restrict__ h, int64_t ldh, int64_t ldx, int br0)
{
    int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= T) return;
    int br = br0 + blockIdx.y;
    int64_t w = blockIdx.z;
    int C = m.n_branch * m.c_in;
    float xv[8];
    if (ldx > 0) {
        for (int c = 0; c < m.c_in; c++) xv[c] = (float)strain[(int64_t)(br * m.c_in + c) * ldx + t];
    } else {
        const XT* x = strain + ((w0 + w) * T + t) * C + br * m.c_in;
        for (int c = 0; c < m.c_in; c++) xv[c] = (float)x[c];
    }
    const float* W = m.blob + off->W_in[br];
    const float* b = m.blob + off->b_in[br];
    float* ho = h + ((w * m.n_branch + br) * m.R) * ldh + t;
    for (int r = 0; r < m.R; r++) {
        float acc = b[r];
        for (int c = 0; c < m.c_in; c++) acc = fmaf(W[r * m.c_in + c], xv[c], acc);
        ho[(int64_t)r * ldh] = acc;
    }
}

// One gated residual block on a TT-timestep tile of one (window, branch)                    (C.1 step 2)
//   f,g = causal dilated conv of h_in;  z = tanh(f) * sigmoid(g);  skip (+)= bs + Ws z;  h_out = h_in + br + Wr z
// hist (stream mode, else null): [n_branch][R][(k-1) d] = the layer input over the (k-1) d samples that precede this
// chunk (zeros at the stream start == the causal zero padding of reading A4).  ldh / lds: row strides of h / skip.
__global__ void k_block(GwiDevModel m, const GwiOffsets* __restrict__ off, int layer, int d, int T,
                        const float* __restrict__ hin, float* __restrict__ hout, float* __restrict__ skip, int first,
                        int last, int64_t ldh, int64_t lds, const float* __restrict__ hist, int br0)
{
    extern __shared__ float sm[];
    const int R = m.R, S = m.S, k = m.k;
    float* in = sm;              // [k][R][TT]: tap j holds h_in[r][t - (k-1-j) d]
    float* z = sm + k * R * TT;  // [R][TT]
    int br = br0 + blockIdx.y;
    int64_t w = blockIdx.z;
    int t0 = blockIdx.x * TT;
    const float* hi = hin + ((w * m.n_branch + br) * R) * ldh;
    const int64_t Hd = (int64_t)(k - 1) * d;
    const float* hs = hist ? hist + (int64_t)br * R * Hd : nullptr;
    for (int idx = threadIdx.x; idx < k * R * TT; idx += blockDim.x) {
        int tt = idx % TT, r = (idx / TT) % R, j = idx / (TT * R);
        int64_t tg = (int64_t)t0 + tt - (int64_t)(k - 1 - j) * d;
        float v = 0.f;                                     // reads at t < 0 return 0 (reading A4) or the carried history
        if (t0 + tt < T) {
            if (tg >= 0) v = hi[(int64_t)r * ldh + tg];
            else if (hs) v = hs[(int64_t)r * Hd + (Hd + tg)];
        }
        in[idx] = v;
    }
    __syncthreads();
    const GwiLayerOff lo = off->layer[br][layer];
    const int tt = threadIdx.x % TT, g = threadIdx.x / TT;
    {
        const float* Wf = m.blob + lo.Wf;
        const float* Wg = m.blob + lo.Wg;
        const float* bf = m.blob + lo.bf;
        const float* bg = m.blob + lo.bg;
        for (int r = g; r < R; r += GROUPS) {
            float f = bf[r], gg = bg[r];
            const float* wf = Wf + (int64_t)r * R * k;
            const float* wg = Wg + (int64_t)r * R * k;
            for (int rp = 0; rp < R; rp++)
                for (int j = 0; j < k; j++) {
                    float x = in[(j * R + rp) * TT + tt];
                    f = fmaf(wf[rp * k + j], x, f);
                    gg = fmaf(wg[rp * k + j], x, gg);
                }
            z[r * TT + tt] = tanhf(f) * (1.0f / (1.0f + expf(-gg)));
        }
    }
    __syncthreads();
    const int t = t0 + tt;
    if (t >= T) return;
    {
        const float* Ws = m.blob + lo.Ws;
        const float* bs = m.blob + lo.bs;
        float* sk = skip + ((w * m.n_branch + br) * S) * lds + t;
        for (int q = g; q < S; q += GROUPS) {
            float acc = bs[q];
            const float* ws = Ws + (int64_t)q * R;
            for (int rp = 0; rp < R; rp++) acc = fmaf(ws[rp], z[rp * TT + tt], acc);
            sk[(int64_t)q * lds] = first ? acc : sk[(int64_t)q * lds] + acc;
        }
    }
    if (!last) {                                          // reading A8: the last block's residual conv is dead
        const float* Wr = m.blob + lo.Wr;
        const float* brs = m.blob + lo.br;
        float* ho = hout + ((w * m.n_branch + br) * R) * ldh + t;
        for (int r = g; r < R; r += GROUPS) {
            float acc = brs[r];
            const float* wr = Wr + (int64_t)r * R;
            for (int rp = 0; rp < R; rp++) acc = fmaf(wr[rp], z[rp * TT + tt], acc);
            ho[(int64_t)r * ldh] = in[((k - 1) * R + r) * TT + tt] + acc;
        }
    }
}

// u = ReLU(skip sum) per branch, concat (H1 first), v = ReLU(W1 c + b1), y = W2 v + b2, p = sigmoid(y)   (C.1 3-5)
// lds: row stride of skip.  lag (stream mode, reading A24): branches >= 1 are read `lag` samples earlier, i.e.
// p_k[t] = head(u_H1[t], u_L1[t - lag]); the caller's skip buffer holds those earlier columns (negative indices).
__global__ void k_head(GwiDevModel m, const GwiOffsets* __restrict__ off, int T, const float* __restrict__ skip,
                       float* __restrict__ prob, int64_t w0, int64_t lds, int64_t lag)
{
    extern __shared__ float sm[];
    const int S = m.S, nbS = m.n_branch * m.S, Hh = m.Hh;
    float* u = sm;                 // [nbS][TT]
    float* part = sm + nbS * TT;   // [HGROUPS][TT]
    int64_t w = blockIdx.y;
    int t0 = blockIdx.x * TT;
    const float* sk = skip + (w * m.n_branch * S) * lds;
    for (int idx = threadIdx.x; idx < nbS * TT; idx += blockDim.x) {
        int tt = idx % TT, q = idx / TT;
        float v = 0.f;
        if (t0 + tt < T) v = fmaxf(sk[(int64_t)q * lds + t0 + tt - (q >= S ? lag : 0)], 0.f);
        u[idx] = v;
    }
    __syncthreads();
    const int tt = threadIdx.x % TT, g = threadIdx.x / TT;
    const float* W1 = m.blob + off->W1;
    const float* b1 = m.blob + off->b1;
    const float* W2 = m.blob + off->W2;
    float ys = 0.f;
    for (int a = g; a < Hh; a += HGROUPS) {
        float v = b1[a];
        const float* w1 = W1 + (int64_t)a * nbS;
        for (int q = 0; q < nbS; q++) v = fmaf(w1[q], u[q * TT + tt], v);
        ys = fmaf(W2[a], fmaxf(v, 0.f), ys);
    }
    part[g * TT + tt] = ys;
    __syncthreads();
    if (g == 0 && t0 + tt < T) {
        float y = m.blob[off->b2];
        for (int i = 0; i < HGROUPS; i++) y += part[i * TT + tt];
        prob[(w0 + w) * T + t0 + tt] = 1.0f / (1.0f + expf(-y));
    }
}

int64_t chunk_windows(const gwi_model* m, int64_t B, int32_t T)
{
    // bound the workspace to ~1 GiB per call chunk
    const GwiArch& a = m->arch;
    int64_t per = (int64_t)a.n_branch * (2 * a.R + a.S) * (int64_t)T * 4;
    int64_t c = (1LL << 30) / (per > 0 ? per : 1);
    if (c < 1) c = 1;
    if (c > 32768) c = 32768; // gridDim.z / .y limit is 65535
    return c < B ? c : B;
}

} // namespace

size_t gwi_generic_workspace_bytes(const gwi_model* m, int64_t B, int32_t T)
{
    const GwiArch& a = m->arch;
    int64_t Bc = chunk_windows(m, B, T);
    return (size_t)(Bc * a.n_branch * (2 * a.R + a.S) * (int64_t)T * 4);
}

gwi_status gwi_generic_infer(const gwi_model* m, const void* d_strain, bool strain_is_half, int64_t B, int32_t T,
                             float* d_prob, void* d_ws, size_t ws_bytes, cudaStream_t st)
{
    const GwiArch& a = m->arch;
    GwiDevModel dm{m->d_blob, a.n_branch, a.c_in, a.R, a.S, a.k, a.L, a.Hh};
    int64_t Bc = chunk_windows(m, B, T);
    float* hA = (float*)d_ws;
    float* hB = hA + Bc * a.n_branch * a.R * (int64_t)T;
    float* skip = hB + Bc * a.n_branch * a.R * (int64_t)T;
    size_t smem_block = (size_t)(a.k + 1) * a.R * TT * sizeof(float);
    size_t smem_head = (size_t)(a.n_branch * a.S + HGROUPS) * TT * sizeof(float);
    static thread_local size_t set_block = 0, set_head = 0;
    if (smem_block > 48 * 1024 && smem_block > set_block) {
        GWI_CUDA_CHECK(cudaFuncSetAttribute(k_block, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_block));
        set_block = smem_block;
    }
    if (smem_head > 48 * 1024 && smem_head > set_head) {
        GWI_CUDA_CHECK(cudaFuncSetAttribute(k_head, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_head));
        set_head = smem_head;
    }
    for (int64_t w0 = 0; w0 < B; w0 += Bc) {
        int64_t nb = (B - w0 < Bc) ? B - w0 : Bc;
        dim3 gl((T + 255) / 256, a.n_branch, (unsigned)nb);
        if (strain_is_half)
            k_lift<__half><<<gl, 256, 0, st>>>(dm, m->d_off, (const __half*)d_strain, w0, T, hA, T, 0, 0);
        else
            k_lift<float><<<gl, 256, 0, st>>>(dm, m->d_off, (const float*)d_strain, w0, T, hA, T, 0, 0);
        float *hin = hA, *hout = hB;
        dim3 gb((T + TT - 1) / TT, a.n_branch, (unsigned)nb);
        for (int i = 0; i < a.L; i++) {
            k_block<<<gb, TT * GROUPS, smem_block, st>>>(dm, m->d_off, i, a.dil[i], T, hin, hout, skip, i == 0,
                                                          i == a.L - 1, T, T, nullptr, 0);
            float* tmp = hin;
            hin = hout, hout = tmp;
        }
        dim3 gh((T + TT - 1) / TT, (unsigned)nb);
        k_head<<<gh, TT * HGROUPS, smem_head, st>>>(dm, m->d_off, T, skip, d_prob, w0, T, 0);
        gwi_count_launch(2 + a.L);
        GWI_CUDA_CHECK(cudaGetLastError());
    }
    return GWI_OK;
}

// ---- stream mode (gwi_stream.cu): one causal pass over a long stream, per-layer history carried across chunks ---------
namespace {

// new[row][idx] = layer input at relative time n - Hd + idx: from this chunk if >= 0, else from the old history
__global__ void k_hist_update(const float* __restrict__ hin, int64_t ldh, int n, const float* __restrict__ hold,
                              float* __restrict__ hnew, int64_t Hd, int64_t rows, int64_t row0)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= rows * Hd) return;
    int64_t r = row0 + i / Hd, idx = i % Hd;
    int64_t p = (int64_t)n - Hd + idx;
    hnew[r * Hd + idx] = p >= 0 ? hin[r * ldh + p] : hold[r * Hd + (Hd + p)];
}

} // namespace

int64_t gwi_generic_hist_floats(const gwi_model* m)
{
    const GwiArch& a = m->arch;
    int64_t s = 0;
    for (int i = 0; i < a.L; i++) s += (int64_t)(a.k - 1) * a.dil[i];
    return s * a.n_branch * a.R;
}

gwi_status gwi_generic_stream_branches(const gwi_model* m, const void* d_strain, bool strain_is_half, int64_t ldx, int n,
                                       float* hA, float* hB, int64_t ldh, float* skip, int64_t lds,
                                       const float* hist_cur, float* hist_next, int br0, int nbr, cudaStream_t st)
{
    const GwiArch& a = m->arch;
    GwiDevModel dm{m->d_blob, a.n_branch, a.c_in, a.R, a.S, a.k, a.L, a.Hh};
    size_t smem_block = (size_t)(a.k + 1) * a.R * TT * sizeof(float);
    if (smem_block > 48 * 1024)
        GWI_CUDA_CHECK(cudaFuncSetAttribute(k_block, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_block));
    dim3 gl((n + 255) / 256, nbr, 1);
    if (strain_is_half)
        k_lift<__half><<<gl, 256, 0, st>>>(dm, m->d_off, (const __half*)d_strain, 0, n, hA, ldh, ldx, br0);
    else
        k_lift<float><<<gl, 256, 0, st>>>(dm, m->d_off, (const float*)d_strain, 0, n, hA, ldh, ldx, br0);
    float *hin = hA, *hout = hB;
    dim3 gb((n + TT - 1) / TT, nbr, 1);
    int64_t ho = 0;
    for (int i = 0; i < a.L; i++) {
        const int64_t Hd = (int64_t)(a.k - 1) * a.dil[i];
        k_block<<<gb, TT * GROUPS, smem_block, st>>>(dm, m->d_off, i, a.dil[i], n, hin, hout, skip, i == 0, i == a.L - 1,
                                                      ldh, lds, hist_cur + ho, br0);
        if (Hd > 0) {
            int64_t rows = (int64_t)nbr * a.R;
            k_hist_update<<<(unsigned)((rows * Hd + 255) / 256), 256, 0, st>>>(hin, ldh, n, hist_cur + ho, hist_next + ho, Hd,
                                                                               rows, (int64_t)br0 * a.R);
            gwi_count_launch(1);
        }
        ho += Hd * a.n_branch * a.R;
        float* tmp = hin;
        hin = hout, hout = tmp;
    }
    gwi_count_launch(1 + a.L);
    GWI_CUDA_CHECK(cudaGetLastError());
    return GWI_OK;
}

gwi_status gwi_generic_stream_head(const gwi_model* m, const float* skip, int64_t lds, int64_t lag, int n, float* d_prob,
                                   cudaStream_t st)
{
    const GwiArch& a = m->arch;
    GwiDevModel dm{m->d_blob, a.n_branch, a.c_in, a.R, a.S, a.k, a.L, a.Hh};
    size_t smem_head = (size_t)(a.n_branch * a.S + HGROUPS) * TT * sizeof(float);
    if (smem_head > 48 * 1024)
        GWI_CUDA_CHECK(cudaFuncSetAttribute(k_head, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_head));
    dim3 gh((n + TT - 1) / TT, 1);
    k_head<<<gh, TT * HGROUPS, smem_head, st>>>(dm, m->d_off, n, skip, d_prob, 0, lds, lag);
    gwi_count_launch(1);
    GWI_CUDA_CHECK(cudaGetLastError());
    return GWI_OK;
}
