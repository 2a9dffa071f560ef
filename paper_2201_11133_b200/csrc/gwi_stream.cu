// gwi_stream.cu -- streaming ensemble driver (gwi_stream_*): SURVEY.md section 8 rows a-1, a-2, a-7, a-8..a-11.
//
//   a-1  host -> device streaming of strain chunks from (pinned) host buffers on a side stream, double-buffered, so
//        that the copy of chunk c+1 overlaps the compute of chunk c
//   a-2  overlap reuse: the stream is evaluated by ONE causal pass (reading A15: stitched 1 s windows with 0.5 s
//        stride == one pass), every output sample computed once; the (k-1) d_i samples of each layer's input that
//        precede a chunk are carried in a per-layer history (reading A17: chunked == unchunked, bit for bit)
//   a-7  time slides on branch features (reading A24): p_k[t] = head(u_H1[t], u_L1[(t - lag_k) mod N]); the L1
//        features of the last max-lag samples are kept in a ring, primed with the features of the stream's tail so
//        that the circular wrap needs no second pass
//   a-8..a-10  per slide: ensemble mean, strict threshold, run clustering with the run carried across chunks
//   a-11 trigger records copied to the host at finish, sorted by (slide, start)
//
// Back ends (gwi_stream_backend): the fused narrow-architecture kernel (gwi_tiny_tc.cu; FP16 mode, config-1 widths: the
// ensembles of BASELINE.json configs 3-5; with slides followed by the fused element-wise heads of gwi_heads.cu), the
// tcgen05 kernel for paper-scale models over segments with recomputed warm-up (gwi_tc.cu; zero lag, or with slides on the
// 128-sample tile grid), and the generic CUDA-core kernels (gwi_generic.cu) for every other architecture and for FP32
// mode.  In all of them each output sample is an independent fixed-order computation, which is what makes
// chunked == unchunked exact.  Time-shard mode (gwi_stream_set_shard) runs one rank's span of a longer stream.
#include <algorithm>
#include <cstdlib>
#include <new>
#include <vector>

#include "gwi_internal.h"

struct gwi_stream {
    std::vector<const gwi_model*> models;
    int M = 0, device = 0;
    bool half_in = false;
    std::vector<int64_t> lags;     // lags[0] = 0 (zero lag), then the lags in samples as the heads use them: the caller's
                                   // lags mod n_total (circular slides, reading A24), the caller's own in shard mode
    std::vector<int64_t> lags_in;  // the caller's lags (lags_in[0] = 0)
    int64_t maxlag = 0, N_total = 0, min_len = 0, t_done = 0;
    float theta = 0.5f;
    int cap = 0, sub = 0;          // record capacity; internal sub-chunk length (samples)
    int R = 0, S = 0, nb = 0, Rf = 0;
    int64_t lds = 0;               // row stride of the skip buffers = maxlag + sub
    bool primed = false, finished = false;
    // device memory
    void* d_x[2] = {nullptr, nullptr};   // staging: planar [nb*c_in][xcap] strain, double-buffered
    int64_t xcap = 0;
    float *d_hA = nullptr, *d_hB = nullptr;
    std::vector<float*> d_skip;          // per model [nb][S][lds]; column maxlag = first sample of the sub-chunk
    float* d_tmp = nullptr;              // [S][maxlag] scratch for the ring shift
    std::vector<float*> d_hist[2];       // per model, ping-pong
    int hist_cur = 0;
    float* d_prob = nullptr;             // [n_slides][M][sub]
    void* d_carry = nullptr;             // [n_slides] carry blocks
    void* d_post_ws = nullptr;
    size_t post_ws_bytes = 0;
    gwi_trigger* d_trig = nullptr;
    int32_t* d_count = nullptr;
    float* d_pbar = nullptr;             // optional caller sink [n_slides][N_total]
    cudaStream_t copy_stream = nullptr;
    cudaEvent_t ev_copied[2] = {nullptr, nullptr}, ev_consumed[2] = {nullptr, nullptr};
    int stage = 0;
    int64_t launches = 0;
    // fused narrow-architecture kernel (FP16 mode, gwi_tiny.cu): carries only the last `halo` input samples
    bool tiny = false;
    int halo = 0;
    __half* d_xh[2] = {nullptr, nullptr};   // [2 detectors][halo], ping-pong
    int xh_cur = 0;
    std::vector<__half*> d_u16;             // time slides: per model [2][lds][32] fp16 branch features, time-major
    int64_t* d_lags = nullptr;              // device copy of the lag list
    int rule = 0;                           // GWI_RULE_MEAN / GWI_RULE_PER_MODEL
    // fused time-slide heads of the narrow architecture (gwi_heads.cu): per slide a bit mask, the mean and the model bytes
    bool fused = false;
    uint32_t* d_fbits = nullptr;
    float* d_fpbar = nullptr;
    uint8_t* d_fmm = nullptr;
    int64_t fbits_stride = 0;
    // time-shard mode (gwi_stream_set_shard): the first `warm` pushed samples are warm-up, the first kept sample has the
    // global index t_first
    bool shard = false;
    int64_t warm = 0, t_first = 0;
    void* d_carry_pm = nullptr;             // per-model rule: [n_slides][M] carry blocks
    // tensor-core back end (paper-scale models, FP16 mode, zero lag only)
    bool tcb = false;
    int seg = 0, segT = 0, segH = 0;        // outputs per segment, window length H + seg, warm-up H = R_f - 1 (seg, segT: of the
    int64_t segx_cap = 0;                   // samples d_segx and the stack workspace hold (time-slide back end)
    int segT0 = 0;                          // current block, chosen by pick_seg; segT0 = the shortest window length)
    __half2* d_segx = nullptr;              // [B][segT][2] channels-last batch
    float* d_segp = nullptr;                // [B][segT] probabilities of the batch
    void* d_tcws = nullptr;
    size_t tcws_bytes = 0;
    // ... with time slides (lags, n_total multiples of 128): incoming chunks are re-blocked into whole segments, the L1
    // feature tiles of the last max-lag samples are kept as history, one head launch per lag on the u tiles
    bool tcs = false;
    bool tcv = false;                       // ... with the element-wise heads on the half-head rows v (gwi_tc_vhalf + gwi_heads_fused)
                                            // instead of one tcgen05 GEMM per lag (GWI_TCS_GEMM_HEADS=1 keeps the latter)
    int Rt = 0;                             // history tiles = maxlag / 128
    __half* d_acc = nullptr;                // [2][acc_cap] samples received but not yet processed (+ the new chunk)
    int64_t acc_cap = 0, pend = 0, t_recv = 0;
    std::vector<uint8_t*> d_hist_t[2];      // per model [R][32 KB] L1 feature tiles that precede the next block, ping-pong
    int hist_t_cur = 0;
};

namespace {

// ---- tensor-core back end (paper-scale models, FP16 mode, zero lag): the chunk is cut into segments of SEG outputs;
// segment w > 0 is evaluated as a window of T = H + SEG samples whose first H = R_f - 1 samples are warm-up that is
// recomputed from the input (exact: no output after the warm-up sees the window's zero padding), segment 0 of the
// STREAM is a window without warm-up (its zero padding is the stream's, reading A4), segment 0 of a later chunk takes
// its warm-up from the carried last H samples of the previous chunk.  All segments of a chunk go through the fused
// tcgen05 kernel (gwi_tc.cu) as one batch of windows.
__global__ void k_seg_gather(const __half* __restrict__ x, int64_t ldx, const __half* __restrict__ xh, int n, int SEG, int H,
                             int T, int stream_start, __half2* __restrict__ out, int64_t total)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;   // (window, t)
    if (i >= total) return;
    int w = (int)(i / T), t = (int)(i % T);
    int64_t src = (w == 0 && stream_start) ? t : (int64_t)w * SEG - H + t;   // chunk-local sample
    __half a = __float2half(0.f), b = a;
    if (src >= n) {
    } else if (src >= 0) {
        a = x[src], b = x[ldx + src];
    } else {
        a = xh[H + src], b = xh[H + H + src];
    }
    out[i] = __halves2half2(a, b);
}
__global__ void k_seg_scatter(const float* __restrict__ pb, int n, int SEG, int H, int T, int stream_start,
                              float* __restrict__ prob)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;   // chunk-local output sample
    if (i >= n) return;
    int w = (int)(i / SEG), o = (int)(i % SEG);
    int t = (w == 0 && stream_start) ? o : H + o;
    prob[i] = pb[(int64_t)w * T + t];
}

// history of L1 feature tiles: new[i] = tile (nq - R + i) of the block just processed (branch 1, segment layout), or the
// old history when that index is negative
__global__ void k_hist_tiles(const uint8_t* __restrict__ u, int ntiles, int64_t nq, int R, int seg_tiles, int warm_tiles,
                             int stream_start, const uint8_t* __restrict__ hold, uint8_t* __restrict__ hnew)
{
    const int64_t i = blockIdx.x, q = nq - R + i;
    const uint8_t* src;
    if (q >= 0) {
        const int64_t w = q / seg_tiles, tl = q % seg_tiles + ((w == 0 && stream_start) ? 0 : warm_tiles);
        src = u + ((size_t)(w * 2 + 1) * ntiles + tl) * 32768;
    } else {
        src = hold + (size_t)(i + nq) * 32768;
    }
    const uint4* s4 = reinterpret_cast<const uint4*>(src);
    uint4* d4 = reinterpret_cast<uint4*>(hnew + (size_t)i * 32768);
    for (int k = threadIdx.x; k < 2048; k += blockDim.x) d4[k] = s4[k];
}

size_t elt(const gwi_stream* s) { return s->half_in ? 2 : 4; }

gwi_status post_block(gwi_stream* s, int n, bool last, cudaStream_t st);

constexpr int SEGT_MAX = 131072;   // longest segment window (samples)

// Segment length for a block of n samples (tensor-core back ends).  The persistent k_stack grid works through
// jobs = 2 branches x pairs of segments in ceil(jobs / SMs) rounds, each as long as one segment window, and every
// segment recomputes segH warm-up samples: the window length (whole tiles) with the smallest rounds x length wins,
// ties go to the shorter one.  An hour of 4096 Hz data gives 148 segments of 101 760 samples (one round, 2 % warm-up)
// instead of 1029 of 16 384 (seven rounds, 12.5 % warm-up).  Results do not depend on the segmentation: every output
// sees its whole receptive field either way.
void pick_seg(gwi_stream* s, int64_t n, int min_segT = 0)
{
    const int sms = gwi_tc_num_sms(s->models[0]);
    if (min_segT <= 0) min_segT = s->segT0;
    int best = min_segT;
    int64_t best_cost = INT64_MAX;
    for (int segT = min_segT; segT <= SEGT_MAX; segT += 128) {
        const int64_t seg = segT - s->segH;
        if (seg < 128) continue;
        const int64_t B = (n + seg - 1) / seg, jobs = ((B + 1) / 2) * 2, rounds = (jobs + sms - 1) / sms;
        if (s->segx_cap > 0 && B * segT > s->segx_cap) continue;
        if (rounds * segT < best_cost) best_cost = rounds * segT, best = segT;
    }
    s->segT = best, s->seg = best - s->segH;
}

// one sub-chunk of n <= sub samples, already in staging buffer `xb` at column `x0`
gwi_status run_sub(gwi_stream* s, int xb, int64_t x0, int n, bool last, cudaStream_t st)
{
    const int nslides = (int)s->lags.size();
    const char* x = (const char*)s->d_x[xb] + (size_t)x0 * elt(s);
    for (int m = 0; m < s->M; m++) {
        const gwi_model* gm = s->models[m];
        float* skip0 = (s->tiny || s->tcb || s->tcs) ? nullptr : s->d_skip[m] + s->maxlag;
        gwi_status rc;
        if (s->tcb) {
            if (m == 0) pick_seg(s, n);
            const int B = (n + s->seg - 1) / s->seg;
            const int start = s->t_done == 0 ? 1 : 0;
            if (m == 0) {
                int64_t total = (int64_t)B * s->segT;
                k_seg_gather<<<(unsigned)((total + 255) / 256), 256, 0, st>>>((const __half*)x, s->xcap, s->d_xh[s->xh_cur], n, s->seg,
                                                                             s->segH, s->segT, start, s->d_segx, total);
                rc = gwi_xhist_update((const __half*)x, s->xcap, n, s->segH, s->d_xh[s->xh_cur], s->d_xh[s->xh_cur ^ 1], st);
                if (rc != GWI_OK) return rc;
            }
            rc = gwi_tc_infer(gm, (const __half*)s->d_segx, B, s->segT, s->d_segp, s->d_tcws, s->tcws_bytes, st);
            if (rc != GWI_OK) return rc;
            k_seg_scatter<<<(n + 255) / 256, 256, 0, st>>>(s->d_segp, n, s->seg, s->segH, s->segT, start, s->d_prob + (size_t)m * s->sub);
            gwi_count_launch(m == 0 ? 2 : 1);
            GWI_CUDA_CHECK(cudaGetLastError());
            continue;
        }
        if (s->tiny) {
            // fused kernel: zero lag only -> probabilities straight out of the kernel; with slides -> skip sums, the
            // per-lag heads follow below
            __half* xh_next = (m == 0) ? s->d_xh[s->xh_cur ^ 1] : nullptr;
            __half* u0 = nslides > 1 ? s->d_u16[m] + (size_t)s->maxlag * 32 : nullptr;
            // global time of the chunk (rows before the stream start are zero at every layer input, reading A4); a time
            // shard that does not own t = 0 has no such rows
            rc = gwi_tiny_stream(gm, (const __half*)x, s->xcap, n, (s->shard && s->warm > 0 ? (int64_t)1 << 40 : 0) + s->t_done,
                                 s->d_xh[s->xh_cur], xh_next,
                                 nslides == 1 ? s->d_prob + (size_t)m * s->sub : nullptr, u0, s->lds, st);
            if (rc != GWI_OK) return rc;
            if (nslides == 1 || s->fused) continue;
            rc = gwi_tiny_heads(gm, u0, s->lds, n, s->d_lags, nslides, s->d_prob + (size_t)m * s->sub, (int64_t)s->M * s->sub, st);
            if (rc != GWI_OK) return rc;
            if (s->fused) continue;   // (shifted after the fused heads launch below)
            // ring shift: the last maxlag rows of the L1 features move to the front
            __half* base = s->d_u16[m] + (size_t)s->lds * 32;
            GWI_CUDA_CHECK(cudaMemcpyAsync(s->d_tmp, base + (size_t)n * 32, (size_t)s->maxlag * 64, cudaMemcpyDeviceToDevice, st));
            GWI_CUDA_CHECK(cudaMemcpyAsync(base, s->d_tmp, (size_t)s->maxlag * 64, cudaMemcpyDeviceToDevice, st));
            continue;
        } else {
            rc = gwi_generic_stream_branches(gm, x, s->half_in, s->xcap, n, s->d_hA, s->d_hB, s->sub, skip0, s->lds,
                                             s->d_hist[s->hist_cur][m], s->d_hist[s->hist_cur ^ 1][m], 0, s->nb, st);
            if (rc != GWI_OK) return rc;
        }
        for (int k = 0; k < nslides; k++) {
            rc = gwi_generic_stream_head(gm, skip0, s->lds, s->lags[k], n, s->d_prob + ((size_t)k * s->M + m) * s->sub, st);
            if (rc != GWI_OK) return rc;
        }
        if (s->maxlag > 0 && s->nb > 1) {
            // ring shift: the last maxlag columns of the L1 (and later) branches move to the front
            float* base = s->d_skip[m] + (size_t)s->S * s->lds;   // branch 1 onwards
            size_t rows = (size_t)(s->nb - 1) * s->S;
            GWI_CUDA_CHECK(cudaMemcpy2DAsync(s->d_tmp, s->maxlag * 4, base + n, s->lds * 4, s->maxlag * 4, rows,
                                             cudaMemcpyDeviceToDevice, st));
            GWI_CUDA_CHECK(cudaMemcpy2DAsync(base, s->lds * 4, s->d_tmp, s->maxlag * 4, s->maxlag * 4, rows,
                                             cudaMemcpyDeviceToDevice, st));
        }
    }
    if (s->fused) {
        // every lag, every model, mean and threshold in one launch on the kept samples of the block (a time shard's
        // warm-up samples produce no output); the rings shift afterwards
        const int64_t skip = (s->rule == GWI_RULE_PER_MODEL) ? 0 : (s->t_done < s->warm ? std::min<int64_t>(n, s->warm - s->t_done) : 0);
        if (skip < n) {
            const __half* vp[GWI_MAX_MODELS];
            for (int m = 0; m < s->M; m++) vp[m] = s->d_u16[m] + (size_t)(s->maxlag + skip) * 32;
            const bool pm = s->rule == GWI_RULE_PER_MODEL;
            gwi_status rc = gwi_heads_fused(s->models.data(), s->M, vp, s->lds, (int)(n - skip), s->d_lags, nslides, s->lags.data(), s->theta,
                                            s->d_fbits, s->fbits_stride, s->d_fpbar, s->d_fmm, s->sub, pm ? s->d_prob : nullptr, st);
            if (rc != GWI_OK) return rc;
        }
        for (int m = 0; m < s->M; m++) {
            __half* base = s->d_u16[m] + (size_t)s->lds * 32;
            GWI_CUDA_CHECK(cudaMemcpyAsync(s->d_tmp, base + (size_t)n * 32, (size_t)s->maxlag * 64, cudaMemcpyDeviceToDevice, st));
            GWI_CUDA_CHECK(cudaMemcpyAsync(base, s->d_tmp, (size_t)s->maxlag * 64, cudaMemcpyDeviceToDevice, st));
        }
    }
    s->hist_cur ^= 1;
    s->xh_cur ^= 1;
    return post_block(s, n, last, st);
}

// ensemble mean / per-model rule, threshold, clustering of one processed block for every slide; advances t_done
gwi_status post_block(gwi_stream* s, int n, bool last, cudaStream_t st)
{
    const int nslides = (int)s->lags.size();
    // time-shard mode: warm-up samples produce no output; times are global
    const int64_t skip = s->t_done < s->warm ? std::min<int64_t>(n, s->warm - s->t_done) : 0;
    if (skip == n) {
        s->t_done += n;
        return GWI_OK;
    }
    const int64_t nn = n - skip, kept = s->t_done + skip - s->warm;   // kept = index of the block's first kept sample
    const int64_t t0 = s->t_first + kept, Nk = s->N_total - s->warm;
    const int64_t sb = s->shard ? s->t_first : -1, se = s->shard ? s->t_first + Nk : -1;
    if (s->rule == GWI_RULE_PER_MODEL) {
        // the paper's rule: every model thresholded and clustered on its own; slide k and model m are
        // packed into the record's slide field (k | m << 20) and unpacked at finish
        for (int k = 0; k < nslides; k++)
            for (int m = 0; m < s->M; m++) {
                const float* ptr1[1] = {s->d_prob + ((size_t)k * s->M + m) * s->sub + skip};
                float* pb = s->d_pbar ? s->d_pbar + ((size_t)k * s->M + m) * Nk + kept : nullptr;
                gwi_status rc = gwi_post_run(ptr1, 1, nn, t0, s->theta, s->min_len, k | (m << 20), last ? 1 : 0,
                                             (char*)s->d_carry_pm + ((size_t)k * s->M + m) * gwi_carry_bytes(), s->d_trig, s->cap,
                                             s->d_count, 1, pb, s->d_post_ws, s->post_ws_bytes, st, sb, se);
                if (rc != GWI_OK) return rc;
            }
        s->t_done += n;
        return GWI_OK;
    }
    if (s->fused) {
        // the fused heads kernel has written mask, mean and model bytes of the kept samples, starting at index 0
        // ... of every slide: one batch of six launches clusters all of them (198 launches per block at 33 slides before)
        gwi_status rc = gwi_post_run_bits_batch(s->d_fbits, s->fbits_stride, s->d_fpbar, s->d_fmm, s->sub, nslides, nn, t0, s->theta,
                                                s->min_len, 0, last ? 1 : 0, s->d_carry, s->d_trig, s->cap, s->d_count, 1,
                                                s->d_post_ws, s->post_ws_bytes, st, sb, se);
        if (rc != GWI_OK) return rc;
        if (s->d_pbar)
            GWI_CUDA_CHECK(cudaMemcpy2DAsync(s->d_pbar + kept, (size_t)Nk * 4, s->d_fpbar, (size_t)s->sub * 4, (size_t)nn * 4, nslides,
                                             cudaMemcpyDeviceToDevice, st));
        s->t_done += n;
        return GWI_OK;
    }
    for (int k = 0; k < nslides; k++) {
        const float* ptrs[GWI_MAX_MODELS];
        for (int m = 0; m < s->M; m++) ptrs[m] = s->d_prob + ((size_t)k * s->M + m) * s->sub + skip;
        float* pb = s->d_pbar ? s->d_pbar + (size_t)k * Nk + kept : nullptr;
        gwi_status rc = gwi_post_run(ptrs, s->M, nn, t0, s->theta, s->min_len, k, last ? 1 : 0,
                                     (char*)s->d_carry + (size_t)k * gwi_carry_bytes(), s->d_trig, s->cap, s->d_count, 1, pb,
                                     s->d_post_ws, s->post_ws_bytes, st, sb, se);
        if (rc != GWI_OK) return rc;
    }
    s->t_done += n;
    return GWI_OK;
}

gwi_status run_chunk(gwi_stream* s, int xb, int64_t n, cudaStream_t st)
{
    for (int64_t o = 0; o < n; o += s->sub) {
        int nn = (int)std::min<int64_t>(s->sub, n - o);
        bool last = (s->t_done + nn == s->N_total);
        gwi_status rc = run_sub(s, xb, o, nn, last, st);
        if (rc != GWI_OK) return rc;
    }
    return GWI_OK;
}

// ---- tensor-core back end with time slides: one block of n samples (whole segments, or the stream's last samples) that
// sit at the front of d_acc
gwi_status tcs_block(gwi_stream* s, int n, bool last, cudaStream_t st)
{
    const int nslides = (int)s->lags.size();
    const int B = (n + s->seg - 1) / s->seg, start = (s->t_done == 0 && !(s->shard && s->warm > 0)) ? 1 : 0;
    const int ntiles = s->segT / 128, seg_tiles = s->seg / 128, warm_tiles = s->segH / 128;
    const int64_t nq = (n + 127) / 128, total = (int64_t)B * s->segT;
    k_seg_gather<<<(unsigned)((total + 255) / 256), 256, 0, st>>>(s->d_acc, s->acc_cap, s->d_xh[s->xh_cur], n, s->seg, s->segH, s->segT,
                                                                 start, s->d_segx, total);
    gwi_count_launch(1);
    gwi_status rc = gwi_xhist_update(s->d_acc, s->acc_cap, n, s->segH, s->d_xh[s->xh_cur], s->d_xh[s->xh_cur ^ 1], st);
    if (rc != GWI_OK) return rc;
    s->xh_cur ^= 1;
    for (int m = 0; m < s->M; m++) {
        const uint8_t* u = nullptr;
        rc = gwi_tc_stack(s->models[m], (const __half*)s->d_segx, B, s->segT, s->d_tcws, s->tcws_bytes, st, &u);
        if (rc != GWI_OK) return rc;
        if (s->tcv) {
            rc = gwi_tc_vhalf(s->models[m], u, B, ntiles, seg_tiles, warm_tiles, start, n, s->d_u16[m] + (size_t)s->maxlag * 128, s->lds, st);
            if (rc != GWI_OK) return rc;
            continue;
        }
        rc = gwi_tc_head_stream(s->models[m], u, ntiles, s->d_hist_t[s->hist_t_cur][m], s->Rt, nq, s->d_lags, nslides, seg_tiles,
                                warm_tiles, start, n, s->d_prob + (size_t)m * s->sub, (int64_t)s->M * s->sub, st);
        if (rc != GWI_OK) return rc;
        if (s->Rt > 0 && !s->tcv) {
            k_hist_tiles<<<s->Rt, 256, 0, st>>>(u, ntiles, nq, s->Rt, seg_tiles, warm_tiles, start, s->d_hist_t[s->hist_t_cur][m],
                                               s->d_hist_t[s->hist_t_cur ^ 1][m]);
            gwi_count_launch(1);
        }
    }
    if (s->tcv) {
        // every lag, every model, mean and threshold element-wise on the half-head rows; then the L1 rings shift
        const int64_t skip = (s->rule == GWI_RULE_PER_MODEL) ? 0 : (s->t_done < s->warm ? std::min<int64_t>(n, s->warm - s->t_done) : 0);
        if (skip < n) {
            const __half* vp[GWI_MAX_MODELS];
            for (int m = 0; m < s->M; m++) vp[m] = s->d_u16[m] + (size_t)(s->maxlag + skip) * 128;
            rc = gwi_heads_fused(s->models.data(), s->M, vp, s->lds, (int)(n - skip), s->d_lags, nslides, s->lags.data(), s->theta,
                                 s->d_fbits, s->fbits_stride, s->d_fpbar, s->d_fmm, s->sub,
                                 s->rule == GWI_RULE_PER_MODEL ? s->d_prob : nullptr, st);
            if (rc != GWI_OK) return rc;
        }
        for (int m = 0; m < s->M; m++) {
            __half* base = s->d_u16[m] + (size_t)s->lds * 128;
            GWI_CUDA_CHECK(cudaMemcpyAsync(s->d_tmp, base + (size_t)n * 128, (size_t)s->maxlag * 256, cudaMemcpyDeviceToDevice, st));
            GWI_CUDA_CHECK(cudaMemcpyAsync(base, s->d_tmp, (size_t)s->maxlag * 256, cudaMemcpyDeviceToDevice, st));
        }
    }
    s->hist_t_cur ^= 1;
    GWI_CUDA_CHECK(cudaGetLastError());
    return GWI_OK;
}

// appends the n samples of staging buffer xb to the pending ones and processes every whole segment (everything at the end
// of the stream); what is left moves to the front
gwi_status tcs_append_and_run(gwi_stream* s, int xb, int64_t x0, int64_t n, cudaStream_t st)
{
    const size_t rowb = (size_t)s->xcap * 2;
    GWI_CUDA_CHECK(cudaMemcpy2DAsync(s->d_acc + s->pend, (size_t)s->acc_cap * 2, (const __half*)s->d_x[xb] + x0, rowb, (size_t)n * 2, 2,
                                     cudaMemcpyDeviceToDevice, st));
    s->pend += n, s->t_recv += n;
    const bool final = s->t_recv == s->N_total;
    const int seg0 = s->segT0 - s->segH;
    // whole blocks only (a short block leaves most of the 148 SMs idle for a full segment time); what is left waits for
    // the next push, or for the end of the stream
    while (s->pend >= s->sub || (final && s->pend > 0)) {
        const int64_t avail = std::min<int64_t>(s->pend, s->sub);
        pick_seg(s, avail);
        int64_t proc = (final && avail == s->pend) ? avail : (avail / s->seg) * s->seg;
        if (proc == 0) s->segT = s->segT0, s->seg = seg0, proc = (avail / seg0) * seg0;
        const bool last = final && proc == s->pend;
        gwi_status rc = tcs_block(s, (int)proc, last, st);
        if (rc != GWI_OK) return rc;
        rc = post_block(s, (int)proc, last, st);
        if (rc != GWI_OK) return rc;
        const int64_t rest = s->pend - proc;
        if (rest > 0) {
            // the remainder moves to the front; staged through the (now free) segment batch buffer because the ranges can overlap
            GWI_CUDA_CHECK(cudaMemcpy2DAsync(s->d_segx, (size_t)rest * 2, s->d_acc + proc, (size_t)s->acc_cap * 2, (size_t)rest * 2, 2,
                                             cudaMemcpyDeviceToDevice, st));
            GWI_CUDA_CHECK(cudaMemcpy2DAsync(s->d_acc, (size_t)s->acc_cap * 2, s->d_segx, (size_t)rest * 2, (size_t)rest * 2, 2,
                                             cudaMemcpyDeviceToDevice, st));
        }
        s->pend = rest;
    }
    return GWI_OK;
}

// a push of any size: pieces of at most `sub` samples, so that the pending samples (< one segment window + one piece) and
// the remainder staged through d_segx stay inside their buffers whatever max_chunk is
gwi_status tcs_push(gwi_stream* s, int xb, int64_t n, cudaStream_t st)
{
    for (int64_t o = 0; o < n; o += s->sub) {
        gwi_status rc = tcs_append_and_run(s, xb, o, std::min<int64_t>(s->sub, n - o), st);
        if (rc != GWI_OK) return rc;
    }
    return GWI_OK;
}

gwi_status check_push(gwi_stream* s, const void* a, const void* b, int64_t n, const char* who)
{
    if (!s || !a || (s->nb > 1 && !b) || n < 1) {
        gwi_set_error("%s: bad argument", who);
        return GWI_ERR_ARG;
    }
    if (s->finished || (s->tcs ? s->t_recv : s->t_done) + n > s->N_total) {
        gwi_set_error("%s: %lld samples pushed + %lld > stream length %lld (or stream finished)", who, (long long)s->t_done,
                      (long long)n, (long long)s->N_total);
        return GWI_ERR_ARG;
    }
    if (n > s->xcap) {
        gwi_set_error("%s: chunk of %lld samples > max_chunk %lld", who, (long long)n, (long long)s->xcap);
        return GWI_ERR_ARG;
    }
    if (s->maxlag > 0 && !s->primed) {
        gwi_set_error("%s: a stream with time slides must be primed with gwi_stream_prime first", who);
        return GWI_ERR_ARG;
    }
    return GWI_OK;
}

} // namespace

extern "C" gwi_status gwi_stream_create(const gwi_model* const* models, int32_t n_models, const int64_t* lags,
                                        int32_t n_lags, int64_t n_total, int64_t max_chunk, float threshold,
                                        int64_t min_len, int32_t capacity, float* d_pbar, gwi_stream** out)
{
    if (!models || n_models < 1 || n_models > GWI_MAX_MODELS || n_lags < 0 || (n_lags > 0 && !lags) || n_total < 1 ||
        max_chunk < 1 || min_len < 1 || capacity < 1 || !out) {
        gwi_set_error("gwi_stream_create: bad argument");
        return GWI_ERR_ARG;
    }
    *out = nullptr;
    const gwi_model* m0 = models[0];
    for (int i = 0; i < n_models; i++) {
        const gwi_model* m = models[i];
        if (!m || m->device != m0->device || m->prec != m0->prec || m->arch.n_branch != m0->arch.n_branch ||
            m->arch.c_in != m0->arch.c_in || m->arch.R != m0->arch.R || m->arch.S != m0->arch.S || m->arch.k != m0->arch.k ||
            m->arch.L != m0->arch.L) {
            gwi_set_error("gwi_stream_create: the models of an ensemble must share device, precision and architecture");
            return GWI_ERR_ARG;
        }
        for (int l = 0; l < m->arch.L; l++)
            if (m->arch.dil[l] != m0->arch.dil[l]) {
                gwi_set_error("gwi_stream_create: the models of an ensemble must share the dilation schedule");
                return GWI_ERR_ARG;
            }
    }
    gwi_stream* s = new (std::nothrow) gwi_stream();
    if (!s) return GWI_ERR_NOMEM;
    s->models.assign(models, models + n_models);
    s->M = n_models, s->device = m0->device, s->half_in = (m0->prec == GWI_FP16);
    s->lags.push_back(0);
    s->lags_in.push_back(0);
    for (int i = 0; i < n_lags; i++) {
        if (lags[i] < 1) {
            gwi_set_error("gwi_stream_create: lag %lld < 1", (long long)lags[i]);
            delete s;
            return GWI_ERR_ARG;
        }
        if (m0->arch.n_branch < 2) {
            gwi_set_error("gwi_stream_create: time slides need a two-branch model (reading A24)");
            delete s;
            return GWI_ERR_UNSUPPORTED;
        }
        // the slides are circular over the stream: a lag >= n_total wraps (a multiple of n_total is the zero lag again).  The
        // ring of L1 features is sized by the largest lag as given, which is what a time shard needs (gwi_stream_set_shard)
        s->lags.push_back(lags[i] % n_total);
        s->lags_in.push_back(lags[i]);
        s->maxlag = std::max(s->maxlag, lags[i]);
    }
    s->N_total = n_total, s->min_len = min_len, s->theta = threshold, s->cap = capacity, s->d_pbar = d_pbar;
    s->R = m0->arch.R, s->S = m0->arch.S, s->nb = m0->arch.n_branch, s->Rf = m0->arch.receptive_field();
    s->tiny = true;
    for (int i = 0; i < n_models; i++) s->tiny = s->tiny && models[i]->tiny != nullptr;
    s->halo = s->tiny ? gwi_tiny_halo(m0) : 0;
    s->tcb = s->half_in && n_lags == 0 && !s->tiny && m0->arch.n_branch == 2 && m0->arch.c_in == 1;
    for (int i = 0; i < n_models; i++) s->tcb = s->tcb && models[i]->tc != nullptr;
    if (s->tcb) {
        s->segH = s->Rf - 1;
        s->segT = ((s->segH + 8192 + 127) / 128) * 128;    // >= 8192 outputs per segment, whole tiles
        if (s->segT < 16384) s->segT = 16384;
        s->segT0 = s->segT;
        s->seg = s->segT - s->segH;
        s->halo = s->segH;
    }
    // the same back end with time slides: everything on the 128-sample tile grid
    s->tcs = s->half_in && n_lags > 0 && !s->tiny && m0->arch.n_branch == 2 && m0->arch.c_in == 1 && n_total % 128 == 0 &&
             n_total >= s->maxlag + s->Rf - 1;
    for (int i = 0; i < n_models; i++) s->tcs = s->tcs && models[i]->tc != nullptr;
    for (int i = 0; i < n_lags; i++) s->tcs = s->tcs && lags[i] % 128 == 0;
    if (s->tcs) {
        s->segH = ((s->Rf - 1 + 127) / 128) * 128;
        s->segT = s->segH + 8192 < 16384 ? 16384 : s->segH + 8192;
        s->segT0 = s->segT;
        s->seg = s->segT - s->segH;
        s->halo = s->segH;
        s->Rt = (int)(s->maxlag / 128);
    }
    s->xcap = std::max<int64_t>(std::min(max_chunk, n_total), s->maxlag > 0 ? s->maxlag + s->Rf - 1 : 0);   // chunks and the primed tail
    // sub-chunk: bounds the activation workspace (2R floats per branch-sample) to ~2 GiB
    int64_t per = (int64_t)s->nb * 2 * s->R * 4;
    int64_t sub = std::max<int64_t>(4096, (2LL << 30) / per);
    if (s->tiny) sub = std::max<int64_t>(4096, (4LL << 30) / ((int64_t)(1 + n_lags) * n_models * 4));   // <= 4 GiB of probabilities
    {
        // the fused slide path keeps no per-lag, per-model probabilities (mean, model bytes and mask per slide, half-head
        // rows per model: ~0.7 KB per sample at 33 slides x 4 models): whole 2^24-sample blocks, half the launches per hour
        bool fused_ok = s->tiny && n_lags > 0 && n_models <= 8;
        for (int i = 0; i < n_models; i++) fused_ok = fused_ok && gwi_tiny_writes_v(models[i]);
        if (fused_ok && (int64_t)(1 + n_lags) * n_models <= 512) sub = 1 << 24;
    }
    if (s->tcb) sub = 1 << 24;
    if (s->tcs) {
        int64_t maxw = gwi_tc_max_windows(m0, s->segT);
        const char* env = getenv("GWI_TCS_GEMM_HEADS");
        s->tcv = n_models <= 8 && !(env && env[0] == '1');
        // v rows cost 512 B per sample and model: blocks of at most 2^23 samples
        sub = std::min<int64_t>(s->tcv ? 1 << 23 : 1 << 24, maxw * s->seg) / s->seg * s->seg;
        if (sub < s->maxlag) s->tcs = s->tcv = false;      // the priming pass runs the tail as one block
    }
    sub = std::min<int64_t>(sub, 1 << 24);
    if (!s->tcs) sub = std::min<int64_t>(sub, s->xcap);
    s->sub = (int)sub;
    s->lds = s->maxlag + s->sub;
    const int nslides = (int)s->lags.size();
    const int C = s->nb * m0->arch.c_in;
    auto fail = [&](cudaError_t e) {
        gwi_set_error("gwi_stream_create: %s", cudaGetErrorString(e));
        gwi_stream_destroy(s);
        return e == cudaErrorMemoryAllocation ? GWI_ERR_NOMEM : GWI_ERR_CUDA;
    };
    cudaError_t e;
    if ((e = cudaSetDevice(s->device)) != cudaSuccess) return fail(e);
    for (int b = 0; b < 2; b++)
        if ((e = cudaMalloc(&s->d_x[b], (size_t)C * s->xcap * elt(s))) != cudaSuccess) return fail(e);
    size_t hbytes = (size_t)s->nb * s->R * s->sub * 4;
    if (s->tcb) {
        // any segment length of pick_seg: B * segT <= n * segT0 / seg0 + SEGT_MAX samples
        const int64_t Bmax = ((int64_t)((double)s->sub * s->segT0 / s->seg) + 2 * SEGT_MAX) / s->segT0 + 1;
        if ((e = cudaMalloc(&s->d_segx, (size_t)Bmax * s->segT * 4)) != cudaSuccess) return fail(e);
        if ((e = cudaMalloc(&s->d_segp, (size_t)Bmax * s->segT * 4)) != cudaSuccess) return fail(e);
        s->tcws_bytes = gwi_tc_workspace_bytes(m0, Bmax, s->segT);
        if ((e = cudaMalloc(&s->d_tcws, s->tcws_bytes)) != cudaSuccess) return fail(e);
        for (int b = 0; b < 2; b++) {
            if ((e = cudaMalloc(&s->d_xh[b], (size_t)2 * s->segH * 2)) != cudaSuccess) return fail(e);
            if ((e = cudaMemset(s->d_xh[b], 0, (size_t)2 * s->segH * 2)) != cudaSuccess) return fail(e);
        }
    }
    if (s->tcs) {
        if ((e = cudaMalloc(&s->d_lags, (size_t)nslides * 8)) != cudaSuccess) return fail(e);
        if ((e = cudaMemcpy(s->d_lags, s->lags.data(), (size_t)nslides * 8, cudaMemcpyHostToDevice)) != cudaSuccess) return fail(e);
        const int64_t Bmax = ((int64_t)((double)s->sub * s->segT0 / s->seg) + 2 * SEGT_MAX) / s->segT0 + 1;
        // pending samples stay below one block (sub) and a piece of a push is at most one block
        s->acc_cap = (int64_t)2 * s->sub + SEGT_MAX;
        s->segx_cap = Bmax * s->segT;
        if ((e = cudaMalloc(&s->d_segx, (size_t)Bmax * s->segT * 4)) != cudaSuccess) return fail(e);
        s->tcws_bytes = gwi_tc_workspace_bytes(m0, Bmax, s->segT);
        if ((e = cudaMalloc(&s->d_tcws, s->tcws_bytes)) != cudaSuccess) return fail(e);
        if ((e = cudaMalloc(&s->d_acc, (size_t)2 * s->acc_cap * 2)) != cudaSuccess) return fail(e);
        if ((e = cudaMemset(s->d_acc, 0, (size_t)2 * s->acc_cap * 2)) != cudaSuccess) return fail(e);
        for (int b = 0; b < 2; b++) {
            if ((e = cudaMalloc(&s->d_xh[b], (size_t)2 * s->segH * 2)) != cudaSuccess) return fail(e);
            if ((e = cudaMemset(s->d_xh[b], 0, (size_t)2 * s->segH * 2)) != cudaSuccess) return fail(e);
            s->d_hist_t[b].assign(s->M, nullptr);
            for (int m = 0; m < s->M && !s->tcv; m++) {
                if ((e = cudaMalloc(&s->d_hist_t[b][m], (size_t)s->Rt * 32768)) != cudaSuccess) return fail(e);
                if ((e = cudaMemset(s->d_hist_t[b][m], 0, (size_t)s->Rt * 32768)) != cudaSuccess) return fail(e);
            }
        }
    }
    if (!s->tiny && !s->tcb && !s->tcs) {   // activation workspace of the generic per-layer kernels
        if ((e = cudaMalloc(&s->d_hA, hbytes)) != cudaSuccess) return fail(e);
        if ((e = cudaMalloc(&s->d_hB, hbytes)) != cudaSuccess) return fail(e);
    }
    size_t histb = (size_t)std::max<int64_t>(1, gwi_generic_hist_floats(m0)) * 4;
    s->d_skip.assign(s->M, nullptr);
    s->d_hist[0].assign(s->M, nullptr), s->d_hist[1].assign(s->M, nullptr);
    for (int m = 0; m < s->M && !s->tiny && !s->tcb && !s->tcs; m++) {
        size_t sb = (size_t)s->nb * s->S * s->lds * 4;
        if ((e = cudaMalloc(&s->d_skip[m], sb)) != cudaSuccess) return fail(e);
        if ((e = cudaMemset(s->d_skip[m], 0, sb)) != cudaSuccess) return fail(e);
        for (int b = 0; b < 2; b++) {
            if ((e = cudaMalloc(&s->d_hist[b][m], histb)) != cudaSuccess) return fail(e);
            if ((e = cudaMemset(s->d_hist[b][m], 0, histb)) != cudaSuccess) return fail(e);   // zero history == A4 padding
        }
    }
    s->fused = s->tiny && nslides > 1 && s->M <= 8;
    for (int i = 0; i < n_models; i++) s->fused = s->fused && gwi_tiny_writes_v(models[i]);
    if (s->tcv) {
        // half-head rows of every model: [2 branches][maxlag ring + sub][128] fp16
        s->fused = true;
        s->d_u16.assign(s->M, nullptr);
        for (int m = 0; m < s->M; m++) {
            size_t ub = (size_t)2 * s->lds * 128 * 2;
            if ((e = cudaMalloc(&s->d_u16[m], ub)) != cudaSuccess) return fail(e);
            if ((e = cudaMemset(s->d_u16[m], 0, ub)) != cudaSuccess) return fail(e);
        }
        if ((e = cudaMalloc(&s->d_tmp, (size_t)s->maxlag * 256)) != cudaSuccess) return fail(e);
    }
    if (s->fused) {
        s->fbits_stride = (s->sub + 31) / 32 + 8;
        if ((e = cudaMalloc(&s->d_fbits, (size_t)nslides * s->fbits_stride * 4)) != cudaSuccess) return fail(e);
        if ((e = cudaMemset(s->d_fbits, 0, (size_t)nslides * s->fbits_stride * 4)) != cudaSuccess) return fail(e);
        if ((e = cudaMalloc(&s->d_fpbar, (size_t)nslides * s->sub * 4)) != cudaSuccess) return fail(e);
        if ((e = cudaMalloc(&s->d_fmm, (size_t)nslides * s->sub)) != cudaSuccess) return fail(e);
    }
    if (s->maxlag > 0 && !s->tcs && (e = cudaMalloc(&s->d_tmp, (size_t)(s->nb - 1) * s->S * s->maxlag * 4)) != cudaSuccess) return fail(e);
    // (the fused slide path keeps no per-model probabilities; the per-model rule allocates them in gwi_stream_set_rule)
    if (!s->fused && (e = cudaMalloc(&s->d_prob, (size_t)nslides * s->M * s->sub * 4)) != cudaSuccess) return fail(e);
    if ((e = cudaMalloc(&s->d_carry, (size_t)nslides * gwi_carry_bytes())) != cudaSuccess) return fail(e);
    if ((e = cudaMemset(s->d_carry, 0, (size_t)nslides * gwi_carry_bytes())) != cudaSuccess) return fail(e);
    if ((e = cudaMalloc(&s->d_carry_pm, (size_t)nslides * s->M * gwi_carry_bytes())) != cudaSuccess) return fail(e);
    if ((e = cudaMemset(s->d_carry_pm, 0, (size_t)nslides * s->M * gwi_carry_bytes())) != cudaSuccess) return fail(e);
    s->post_ws_bytes = std::max(gwi_triggers_workspace_bytes(s->sub), gwi_post_batch_workspace_bytes(s->sub, nslides));
    if ((e = cudaMalloc(&s->d_post_ws, s->post_ws_bytes)) != cudaSuccess) return fail(e);
    if ((e = cudaMalloc(&s->d_trig, (size_t)capacity * sizeof(gwi_trigger))) != cudaSuccess) return fail(e);
    if ((e = cudaMalloc(&s->d_count, 4)) != cudaSuccess) return fail(e);
    if ((e = cudaMemset(s->d_count, 0, 4)) != cudaSuccess) return fail(e);
    if (s->tiny) {
        for (int b = 0; b < 2; b++) {
            if ((e = cudaMalloc(&s->d_xh[b], (size_t)2 * s->halo * 2)) != cudaSuccess) return fail(e);
            if ((e = cudaMemset(s->d_xh[b], 0, (size_t)2 * s->halo * 2)) != cudaSuccess) return fail(e);
        }
        if (nslides > 1) {
            s->d_u16.assign(s->M, nullptr);
            for (int m = 0; m < s->M; m++) {
                size_t ub = (size_t)2 * s->lds * 32 * 2;
                if ((e = cudaMalloc(&s->d_u16[m], ub)) != cudaSuccess) return fail(e);
                if ((e = cudaMemset(s->d_u16[m], 0, ub)) != cudaSuccess) return fail(e);
            }
            if ((e = cudaMalloc(&s->d_lags, (size_t)nslides * 8)) != cudaSuccess) return fail(e);
            if ((e = cudaMemcpy(s->d_lags, s->lags.data(), (size_t)nslides * 8, cudaMemcpyHostToDevice)) != cudaSuccess) return fail(e);
        }
    }
    if ((e = cudaStreamCreateWithFlags(&s->copy_stream, cudaStreamNonBlocking)) != cudaSuccess) return fail(e);
    for (int b = 0; b < 2; b++) {
        if ((e = cudaEventCreateWithFlags(&s->ev_copied[b], cudaEventDisableTiming)) != cudaSuccess) return fail(e);
        if ((e = cudaEventCreateWithFlags(&s->ev_consumed[b], cudaEventDisableTiming)) != cudaSuccess) return fail(e);
    }
    if ((e = cudaDeviceSynchronize()) != cudaSuccess) return fail(e);
    *out = s;
    return GWI_OK;
}

extern "C" void gwi_stream_destroy(gwi_stream* s)
{
    if (!s) return;
    cudaSetDevice(s->device);
    cudaDeviceSynchronize();
    for (int b = 0; b < 2; b++) {
        if (s->d_x[b]) cudaFree(s->d_x[b]);
        if (s->d_xh[b]) cudaFree(s->d_xh[b]);
        for (float* p : s->d_hist[b])
            if (p) cudaFree(p);
        if (s->ev_copied[b]) cudaEventDestroy(s->ev_copied[b]);
        if (s->ev_consumed[b]) cudaEventDestroy(s->ev_consumed[b]);
    }
    for (float* p : s->d_skip)
        if (p) cudaFree(p);
    for (__half* p : s->d_u16)
        if (p) cudaFree(p);
    if (s->d_lags) cudaFree(s->d_lags);
    if (s->d_segx) cudaFree(s->d_segx);
    if (s->d_segp) cudaFree(s->d_segp);
    if (s->d_tcws) cudaFree(s->d_tcws);
    if (s->d_acc) cudaFree(s->d_acc);
    for (int b = 0; b < 2; b++)
        for (uint8_t* p : s->d_hist_t[b])
            if (p) cudaFree(p);
    if (s->d_hA) cudaFree(s->d_hA);
    if (s->d_hB) cudaFree(s->d_hB);
    if (s->d_tmp) cudaFree(s->d_tmp);
    if (s->d_prob) cudaFree(s->d_prob);
    if (s->d_fbits) cudaFree(s->d_fbits);
    if (s->d_fpbar) cudaFree(s->d_fpbar);
    if (s->d_fmm) cudaFree(s->d_fmm);
    if (s->d_carry) cudaFree(s->d_carry);
    if (s->d_carry_pm) cudaFree(s->d_carry_pm);
    if (s->d_post_ws) cudaFree(s->d_post_ws);
    if (s->d_trig) cudaFree(s->d_trig);
    if (s->d_count) cudaFree(s->d_count);
    if (s->copy_stream) cudaStreamDestroy(s->copy_stream);
    delete s;
}

extern "C" int64_t gwi_stream_tail_samples(const gwi_stream* s)
{
    if (!s || s->maxlag == 0) return 0;
    // shard mode: the L1 samples that precede the first pushed sample in the global stream, as many as the largest lag
    // reaches back; otherwise the stream's own tail (at most the whole stream)
    return s->shard ? s->maxlag + s->Rf - 1 : std::min<int64_t>(s->N_total, s->maxlag + s->Rf - 1);
}

extern "C" gwi_status gwi_stream_prime(gwi_stream* s, const void* l1_tail, int64_t n_tail, void* cuda_stream)
{
    if (!s || !l1_tail || s->maxlag == 0 || n_tail != gwi_stream_tail_samples(s) || s->t_done != 0) {
        gwi_set_error("gwi_stream_prime: bad argument (n_tail must equal gwi_stream_tail_samples(), before the first push)");
        return GWI_ERR_ARG;
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    GWI_CUDA_CHECK(cudaSetDevice(s->device));
    if (s->tcs && s->shard && s->t_first - s->warm > 0 && n_tail > s->t_first - s->warm) {
        gwi_set_error("gwi_stream_prime: a time shard whose L1 prefix wraps around the global stream start is not supported by the "
                      "tensor-core slide back end (make the first shard longer than max lag + 2 R_f)");
        return GWI_ERR_UNSUPPORTED;
    }
    if (s->tcs) {
        // tail = L1[N - maxlag - (R_f - 1), N): the first R_f - 1 samples are the warm-up of the history tiles (the segment
        // warm-up is R_f - 1 rounded up to whole tiles, the front of it stays zero and is never looked at by an output)
        const int pre = s->Rf - 1, H = s->segH;
        const int64_t n = s->maxlag;
        GWI_CUDA_CHECK(cudaMemsetAsync(s->d_xh[0], 0, (size_t)2 * H * 2, st));
        GWI_CUDA_CHECK(cudaMemcpyAsync(s->d_xh[0] + H + (H - pre), l1_tail, (size_t)pre * 2, cudaMemcpyDefault, st));
        GWI_CUDA_CHECK(cudaMemsetAsync(s->d_acc, 0, (size_t)n * 2, st));
        GWI_CUDA_CHECK(cudaMemcpyAsync(s->d_acc + s->acc_cap, (const __half*)l1_tail + pre, (size_t)n * 2, cudaMemcpyDefault, st));
        pick_seg(s, n, H + 128);                             // any segment length: the tail is one small block, one round of the grid
        const int B = (int)((n + s->seg - 1) / s->seg);
        const int64_t total = (int64_t)B * s->segT;
        k_seg_gather<<<(unsigned)((total + 255) / 256), 256, 0, st>>>(s->d_acc, s->acc_cap, s->d_xh[0], (int)n, s->seg, H, s->segT, 0,
                                                                     s->d_segx, total);
        gwi_count_launch(1);
        for (int m = 0; m < s->M; m++) {
            const uint8_t* u = nullptr;
            gwi_status rc = gwi_tc_stack(s->models[m], (const __half*)s->d_segx, B, s->segT, s->d_tcws, s->tcws_bytes, st, &u);
            if (rc != GWI_OK) return rc;
            if (s->tcv) {
                // half-head rows of the tail (the H1 rows it produces are garbage and are overwritten by the first block),
                // then the same ring shift as after a block: the tail's maxlag rows land in front of row 0
                rc = gwi_tc_vhalf(s->models[m], u, B, s->segT / 128, s->seg / 128, H / 128, 0, (int)n, s->d_u16[m] + (size_t)s->maxlag * 128,
                                  s->lds, st);
                if (rc != GWI_OK) return rc;
                __half* base = s->d_u16[m] + (size_t)s->lds * 128;
                GWI_CUDA_CHECK(cudaMemcpyAsync(s->d_tmp, base + (size_t)n * 128, (size_t)s->maxlag * 256, cudaMemcpyDeviceToDevice, st));
                GWI_CUDA_CHECK(cudaMemcpyAsync(base, s->d_tmp, (size_t)s->maxlag * 256, cudaMemcpyDeviceToDevice, st));
                continue;
            }
            k_hist_tiles<<<s->Rt, 256, 0, st>>>(u, s->segT / 128, s->Rt, s->Rt, s->seg / 128, H / 128, 0, s->d_hist_t[1][m],
                                               s->d_hist_t[0][m]);
            gwi_count_launch(1);
        }
        GWI_CUDA_CHECK(cudaMemsetAsync(s->d_xh[0], 0, (size_t)2 * H * 2, st));
        GWI_CUDA_CHECK(cudaMemsetAsync(s->d_xh[1], 0, (size_t)2 * H * 2, st));
        if (s->shard && s->warm > 0 && n_tail >= H)   // time shard: the L1 warm-up of the first segment is the tail's end (see below)
            GWI_CUDA_CHECK(cudaMemcpyAsync(s->d_xh[0] + H, (const __half*)l1_tail + (n_tail - H), (size_t)H * 2, cudaMemcpyDefault, st));
        GWI_CUDA_CHECK(cudaGetLastError());
        s->xh_cur = 0, s->hist_t_cur = 0, s->pend = 0;
        s->primed = true;
        for (int b = 0; b < 2; b++) GWI_CUDA_CHECK(cudaEventRecord(s->ev_consumed[b], st));
        return GWI_OK;
    }
    const int c_in = s->models[0]->arch.c_in;
    // the tail goes to the branch-1 rows of staging buffer 0 (cudaMemcpyDefault: host or device source)
    GWI_CUDA_CHECK(cudaMemcpy2DAsync((char*)s->d_x[0] + (size_t)c_in * s->xcap * elt(s), s->xcap * elt(s), l1_tail,
                                     n_tail * elt(s), n_tail * elt(s), (size_t)c_in * (s->nb - 1), cudaMemcpyDefault, st));
    // features of the tail: zero history is exact for the last maxlag samples because either the tail starts at t = 0
    // or it starts R_f - 1 samples before them
    const bool keepL = s->shard && s->warm > 0;
    int tiny_xc = 0;
    // shard mode: the tail is the global samples [first_pushed - n_tail, first_pushed) taken circularly; position of the
    // global t = 0 inside it (0: no wrap inside the tail)
    const int64_t first_pushed = s->t_first - s->warm;
    const int64_t wrap_at = (s->shard && n_tail > first_pushed && first_pushed > 0) ? n_tail - first_pushed : 0;
    for (int m = 0; m < s->M; m++) {
        if (!s->tiny)
            GWI_CUDA_CHECK(cudaMemsetAsync(s->d_hist[0][m], 0, (size_t)std::max<int64_t>(1, gwi_generic_hist_floats(s->models[m])) * 4, st));
        if (s->tiny) {
            GWI_CUDA_CHECK(cudaMemsetAsync(s->d_xh[0], 0, (size_t)2 * s->halo * 2, st));
            GWI_CUDA_CHECK(cudaMemsetAsync(s->d_xh[1], 0, (size_t)2 * s->halo * 2, st));
        }
        int xc = 0;
        for (int64_t o = 0; o < n_tail;) {
            // a shard's tail may wrap around the global stream (.. N-1, 0, 1 ..): the part from global t = 0 on starts
            // from zero history again, as the stream itself does (reading A4), so that the features are the ones the
            // unsharded pass has
            const bool at_wrap = wrap_at > 0 && o == wrap_at;
            if (at_wrap) {
                if (s->tiny) {
                    GWI_CUDA_CHECK(cudaMemsetAsync(s->d_xh[0], 0, (size_t)2 * s->halo * 2, st));
                    GWI_CUDA_CHECK(cudaMemsetAsync(s->d_xh[1], 0, (size_t)2 * s->halo * 2, st));
                } else {
                    GWI_CUDA_CHECK(cudaMemsetAsync(s->d_hist[0][m], 0, (size_t)std::max<int64_t>(1, gwi_generic_hist_floats(s->models[m])) * 4, st));
                }
            }
            const int64_t lim = (wrap_at > 0 && o < wrap_at) ? wrap_at : n_tail;
            int nn = (int)std::min<int64_t>(s->sub, lim - o);
            const int64_t tail_t0 = !s->shard ? s->N_total - n_tail + o : (wrap_at > 0 && o >= wrap_at) ? o - wrap_at : ((int64_t)1 << 40) + o;
            gwi_status rc;
            if (s->tiny) {
                // both branches are evaluated; the H1 rows of the staging buffer hold nothing meaningful here and the
                // H1 skip rows they produce are overwritten by the first real chunk
                // global time of the tail's first sample: the stream's own tail, or (shard mode) samples somewhere inside
                // the global stream -- never the stream start, so no row is masked as "before t = 0"
                rc = gwi_tiny_stream(s->models[m], (const __half*)s->d_x[0] + o, s->xcap, nn, tail_t0,
                                     s->d_xh[xc], s->d_xh[xc ^ 1], nullptr, s->d_u16[m] + (size_t)s->maxlag * 32, s->lds, st);
                xc ^= 1;
                o += nn;
                if (rc != GWI_OK) return rc;
                __half* base16 = s->d_u16[m] + (size_t)s->lds * 32;
                GWI_CUDA_CHECK(cudaMemcpyAsync(s->d_tmp, base16 + (size_t)nn * 32, (size_t)s->maxlag * 64, cudaMemcpyDeviceToDevice, st));
                GWI_CUDA_CHECK(cudaMemcpyAsync(base16, s->d_tmp, (size_t)s->maxlag * 64, cudaMemcpyDeviceToDevice, st));
                continue;
            } else
            rc = gwi_generic_stream_branches(s->models[m], (const char*)s->d_x[0] + (size_t)o * elt(s), s->half_in,
                                                        s->xcap, nn, s->d_hA, s->d_hB, s->sub, s->d_skip[m] + s->maxlag,
                                                        s->lds, s->d_hist[0][m], s->d_hist[1][m], 1, s->nb - 1, st);
            if (rc != GWI_OK) return rc;
            // keep the last maxlag columns seen so far at the front of the ring, exactly as run_sub does
            float* base = s->d_skip[m] + (size_t)s->S * s->lds;
            size_t rows = (size_t)(s->nb - 1) * s->S;
            GWI_CUDA_CHECK(cudaMemcpy2DAsync(s->d_tmp, s->maxlag * 4, base + nn, s->lds * 4, s->maxlag * 4, rows,
                                             cudaMemcpyDeviceToDevice, st));
            GWI_CUDA_CHECK(cudaMemcpy2DAsync(base, s->lds * 4, s->d_tmp, s->maxlag * 4, s->maxlag * 4, rows,
                                             cudaMemcpyDeviceToDevice, st));
            // history ping-pong inside the tail pass
            std::swap(s->d_hist[0][m], s->d_hist[1][m]);
            o += nn;
        }
        // the real pass starts from zero history again -- except for the L1 branch of a time shard that does not start at
        // t = 0: its tail ends where the first pushed sample begins, so the L1 state carries over and the L1 features of
        // the warm-up samples, which the slides read max-lag later, are exact (the H1 branch starts from zero: its
        // warm-up outputs are discarded)
        if (s->tiny) {
            tiny_xc = xc;
            continue;
        }
        if (keepL) continue;
        GWI_CUDA_CHECK(cudaMemsetAsync(s->d_hist[0][m], 0, (size_t)std::max<int64_t>(1, gwi_generic_hist_floats(s->models[m])) * 4, st));
        GWI_CUDA_CHECK(cudaMemsetAsync(s->d_hist[1][m], 0, (size_t)std::max<int64_t>(1, gwi_generic_hist_floats(s->models[m])) * 4, st));
    }
    if (s->tiny) {
        if (keepL) {
            // carried input samples: L1 = the tail's last `halo` samples, H1 = zero
            GWI_CUDA_CHECK(cudaMemsetAsync(s->d_xh[tiny_xc], 0, (size_t)s->halo * 2, st));
            s->xh_cur = tiny_xc;
        } else {
            GWI_CUDA_CHECK(cudaMemsetAsync(s->d_xh[0], 0, (size_t)2 * s->halo * 2, st));
            GWI_CUDA_CHECK(cudaMemsetAsync(s->d_xh[1], 0, (size_t)2 * s->halo * 2, st));
            s->xh_cur = 0;
        }
    }
    s->hist_cur = 0;
    s->primed = true;
    // the first gwi_stream_push_host copies into staging buffer 0 on the side stream: it must wait for the kernels above,
    // which read the tail out of that buffer
    for (int b = 0; b < 2; b++) GWI_CUDA_CHECK(cudaEventRecord(s->ev_consumed[b], st));
    return GWI_OK;
}

extern "C" gwi_status gwi_stream_push(gwi_stream* s, const void* d_h1, const void* d_l1, int64_t n, void* cuda_stream)
{
    gwi_status rc = check_push(s, d_h1, d_l1, n, "gwi_stream_push");
    if (rc != GWI_OK) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    GWI_CUDA_CHECK(cudaSetDevice(s->device));
    const int c_in = s->models[0]->arch.c_in;
    const int b = s->stage;
    // staging buffer b may still be read by work enqueued on another caller stream
    GWI_CUDA_CHECK(cudaStreamWaitEvent(st, s->ev_consumed[b], 0));
    size_t rowb = (size_t)s->xcap * elt(s);
    GWI_CUDA_CHECK(cudaMemcpy2DAsync(s->d_x[b], rowb, d_h1, n * elt(s), n * elt(s), c_in, cudaMemcpyDeviceToDevice, st));
    if (s->nb > 1)
        GWI_CUDA_CHECK(cudaMemcpy2DAsync((char*)s->d_x[b] + c_in * rowb, rowb, d_l1, n * elt(s), n * elt(s),
                                         (size_t)c_in * (s->nb - 1), cudaMemcpyDeviceToDevice, st));
    rc = s->tcs ? tcs_push(s, b, n, st) : run_chunk(s, b, n, st);
    if (rc != GWI_OK) return rc;
    GWI_CUDA_CHECK(cudaEventRecord(s->ev_consumed[b], st));
    s->stage ^= 1;
    return GWI_OK;
}

extern "C" gwi_status gwi_stream_push_host(gwi_stream* s, const void* h_h1, const void* h_l1, int64_t n, void* cuda_stream)
{
    gwi_status rc = check_push(s, h_h1, h_l1, n, "gwi_stream_push_host");
    if (rc != GWI_OK) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    GWI_CUDA_CHECK(cudaSetDevice(s->device));
    const int c_in = s->models[0]->arch.c_in;
    const int b = s->stage;
    size_t rowb = (size_t)s->xcap * elt(s);
    // H2D on the side stream, as soon as the compute that last read staging buffer b has finished; the compute of
    // the previous chunk (other buffer) keeps running meanwhile
    GWI_CUDA_CHECK(cudaStreamWaitEvent(s->copy_stream, s->ev_consumed[b], 0));
    GWI_CUDA_CHECK(cudaMemcpy2DAsync(s->d_x[b], rowb, h_h1, n * elt(s), n * elt(s), c_in, cudaMemcpyHostToDevice, s->copy_stream));
    if (s->nb > 1)
        GWI_CUDA_CHECK(cudaMemcpy2DAsync((char*)s->d_x[b] + c_in * rowb, rowb, h_l1, n * elt(s), n * elt(s),
                                         (size_t)c_in * (s->nb - 1), cudaMemcpyHostToDevice, s->copy_stream));
    GWI_CUDA_CHECK(cudaEventRecord(s->ev_copied[b], s->copy_stream));
    GWI_CUDA_CHECK(cudaStreamWaitEvent(st, s->ev_copied[b], 0));
    rc = s->tcs ? tcs_push(s, b, n, st) : run_chunk(s, b, n, st);
    if (rc != GWI_OK) return rc;
    GWI_CUDA_CHECK(cudaEventRecord(s->ev_consumed[b], st));
    s->stage ^= 1;
    return GWI_OK;
}

extern "C" gwi_status gwi_stream_finish(gwi_stream* s, gwi_trigger* h_triggers, int32_t capacity, int32_t* h_count,
                                        void* cuda_stream)
{
    if (!s || !h_count || capacity < 0 || (capacity > 0 && !h_triggers)) {
        gwi_set_error("gwi_stream_finish: bad argument");
        return GWI_ERR_ARG;
    }
    if (s->t_done != s->N_total) {
        gwi_set_error("gwi_stream_finish: %lld of %lld samples pushed", (long long)s->t_done, (long long)s->N_total);
        return GWI_ERR_ARG;
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    GWI_CUDA_CHECK(cudaSetDevice(s->device));
    int32_t n = 0;
    GWI_CUDA_CHECK(cudaMemcpyAsync(&n, s->d_count, 4, cudaMemcpyDeviceToHost, st));
    GWI_CUDA_CHECK(cudaStreamSynchronize(st));
    int have = std::min(n, s->cap);
    std::vector<gwi_trigger> recs((size_t)have);
    if (have > 0) {
        GWI_CUDA_CHECK(cudaMemcpyAsync(recs.data(), s->d_trig, (size_t)have * sizeof(gwi_trigger), cudaMemcpyDeviceToHost, st));
        GWI_CUDA_CHECK(cudaStreamSynchronize(st));
    }
    if (s->rule == GWI_RULE_PER_MODEL)
        for (auto& r : recs) {
            r.model_mask = (1 << (r.slide >> 20)) | (r.model_mask & (GWI_EDGE_LEFT | GWI_EDGE_RIGHT));
            r.slide &= (1 << 20) - 1;
        }
    // records arrive grouped by sub-chunk; the list is sorted by (slide, start)
    std::stable_sort(recs.begin(), recs.end(), [](const gwi_trigger& a, const gwi_trigger& b) {
        return a.slide != b.slide ? a.slide < b.slide : a.start < b.start;
    });
    int give = std::min(have, capacity);
    for (int i = 0; i < give; i++) h_triggers[i] = recs[i];
    *h_count = n;
    s->finished = true;
    if (n > s->cap || n > capacity) {
        gwi_set_error("gwi_stream_finish: %d triggers, stream capacity %d, caller capacity %d", n, s->cap, capacity);
        return GWI_ERR_CAPACITY;
    }
    return GWI_OK;
}

extern "C" int64_t gwi_stream_samples_done(const gwi_stream* s) { return s ? s->t_done : -1; }

extern "C" gwi_status gwi_stream_set_shard(gwi_stream* s, int64_t t_first, int64_t warmup)
{
    if (!s || warmup < 0 || warmup >= s->N_total || t_first < 0 || s->t_done != 0 || s->t_recv != 0 || s->primed) {
        gwi_set_error("gwi_stream_set_shard: bad argument (before the first push and before gwi_stream_prime; 0 <= warmup < n_total)");
        return GWI_ERR_ARG;
    }
    s->shard = true, s->warm = warmup, s->t_first = t_first;
    s->lags = s->lags_in;      // no wrap inside a shard: the primed L1 prefix is the global stream's
    if (s->d_lags) {
        GWI_CUDA_CHECK(cudaSetDevice(s->device));
        GWI_CUDA_CHECK(cudaMemcpy(s->d_lags, s->lags.data(), s->lags.size() * 8, cudaMemcpyHostToDevice));
    }
    return GWI_OK;
}

extern "C" int gwi_stream_backend(const gwi_stream* s)
{
    if (!s) return -1;
    return s->tiny ? GWI_BACKEND_NARROW : s->tcb ? GWI_BACKEND_TENSOR : s->tcs ? GWI_BACKEND_TENSOR_SLIDES : GWI_BACKEND_GENERIC;
}

extern "C" gwi_status gwi_stream_set_rule(gwi_stream* s, gwi_rule rule)
{
    if (!s || (rule != GWI_RULE_MEAN && rule != GWI_RULE_PER_MODEL) || s->t_done != 0) {
        gwi_set_error("gwi_stream_set_rule: bad argument (must be called before the first push)");
        return GWI_ERR_ARG;
    }
    s->rule = (int)rule;
    if (rule == GWI_RULE_PER_MODEL && s->fused && !s->d_prob) {
        GWI_CUDA_CHECK(cudaSetDevice(s->device));
        if (cudaMalloc(&s->d_prob, s->lags.size() * s->M * (size_t)s->sub * 4) != cudaSuccess) {
            cudaGetLastError();
            gwi_set_error("gwi_stream_set_rule: out of device memory for the per-model probabilities");
            return GWI_ERR_NOMEM;
        }
    }
    return GWI_OK;
}

// Host-side coincidence of per-model triggers (include/gwi.h; reading A34).  Two-pointer sweeps over the per-model end
// lists, O(n log n) for the sorts.
extern "C" gwi_status gwi_coincidence(const gwi_trigger* h_triggers, int32_t n_triggers, int32_t n_models, int64_t window,
                                      gwi_event* h_events, int32_t capacity, int32_t* n_events)
{
    if (n_triggers < 0 || (n_triggers > 0 && !h_triggers) || n_models < 1 || n_models > GWI_MAX_MODELS || window < 0 ||
        capacity < 0 || (capacity > 0 && !h_events) || !n_events) {
        gwi_set_error("gwi_coincidence: bad argument");
        return GWI_ERR_ARG;
    }
    std::vector<int32_t> slides;
    for (int i = 0; i < n_triggers; i++) slides.push_back(h_triggers[i].slide);
    std::sort(slides.begin(), slides.end());
    slides.erase(std::unique(slides.begin(), slides.end()), slides.end());
    int64_t total = 0;
    for (int32_t sl : slides) {
        std::vector<std::vector<int64_t>> ends(n_models);
        std::vector<int64_t> all;
        for (int i = 0; i < n_triggers; i++) {
            const gwi_trigger& t = h_triggers[i];
            if (t.slide != sl) continue;
            for (int m = 0; m < n_models; m++)
                if (t.model_mask & (1 << m)) ends[m].push_back(t.end);
            all.push_back(t.end);
        }
        for (auto& e : ends) std::sort(e.begin(), e.end());
        std::sort(all.begin(), all.end());
        // anchors: ends a such that every model has an end in [a, a + window]
        std::vector<int64_t> anchors;
        for (int64_t a : all) {
            bool ok = true;
            for (int m = 0; m < n_models && ok; m++) {
                auto it = std::lower_bound(ends[m].begin(), ends[m].end(), a);
                ok = it != ends[m].end() && *it <= a + window;
            }
            if (ok && (anchors.empty() || anchors.back() != a)) anchors.push_back(a);
        }
        size_t i = 0;
        while (i < anchors.size()) {
            int64_t first = anchors[i], last = anchors[i];
            while (i + 1 < anchors.size() && anchors[i + 1] - last <= window) last = anchors[++i];
            i++;
            auto lo = std::lower_bound(all.begin(), all.end(), first);
            auto hi = std::upper_bound(all.begin(), all.end(), last + window);
            if (total < capacity) {
                gwi_event ev;
                ev.t_first = first, ev.t_last = *(hi - 1), ev.n_triggers = (int32_t)(hi - lo), ev.slide = sl;
                h_events[total] = ev;
            }
            total++;
        }
    }
    *n_events = (int32_t)total;
    if (total > capacity) {
        gwi_set_error("gwi_coincidence: %lld events > capacity %d", (long long)total, capacity);
        return GWI_ERR_CAPACITY;
    }
    return GWI_OK;
}
