/* gwi.h -- C-ABI of the B200-native hot path of arXiv 2201.11133
 * ("Inference-optimized AI and high performance computing for gravitational wave detection at scale").
 *
 * What the library computes (citations are PAPER.md lines; readings A1..A31 are listed in DESIGN.md):
 *   - batched inference of one detection model over 1 s windows of two-detector whitened strain,
 *     tensor contract (B,4096,2) -> (B,4096,1), one probability per time step
 *   - the same model run as ONE causal pass over a long stream (overlap reuse, reading A15)
 *   - ensemble averaging of the models' probabilities, strict threshold, clustering of supra-threshold
 *     runs of >= min_len samples into triggers
 *   - time slides of L1 against H1 for background estimation
 *
 * Conventions
 *   - Every entry point returns gwi_status; nothing throws or aborts across the ABI.  gwi_last_error()
 *     returns a thread-local message for the last non-OK status on the calling thread.
 *   - Pointers named d_* are DEVICE pointers on the model's device, everything else is a HOST pointer.
 *   - The caller owns every buffer it passes in (inputs, outputs, workspace, carry).  The library owns only
 *     what it returns through an opaque handle (gwi_model, gwi_stream) until the matching free/destroy.
 *   - `cuda_stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  All work is
 *     enqueued asynchronously on it; results are valid after the caller synchronises that stream.
 *   - There is no CPU fallback: without a usable CUDA device the calls fail with GWI_ERR_CUDA.
 */
#ifndef GWI_H
#define GWI_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct gwi_model gwi_model;   /* opaque; owns the packed device weights of ONE network */
typedef struct gwi_stream gwi_stream; /* opaque; streaming ensemble + slides + triggers state  */

typedef enum {
    GWI_OK = 0,
    GWI_ERR_ARG = 1,         /* null / misaligned / out-of-range argument                         */
    GWI_ERR_IO = 2,          /* model file cannot be opened or is truncated                       */
    GWI_ERR_FORMAT = 3,      /* model file is not GWIM v1 or has inconsistent fields               */
    GWI_ERR_UNSUPPORTED = 4, /* architecture outside what the kernels cover                       */
    GWI_ERR_CUDA = 5,        /* a CUDA runtime call failed (message in gwi_last_error())          */
    GWI_ERR_NOMEM = 6,       /* workspace / carry / capacity buffer too small                     */
    GWI_ERR_CAPACITY = 7     /* more triggers than `capacity`; the first `capacity` are valid     */
} gwi_status;

/* GWI_FP32: fp32 weights, inputs and arithmetic (CUDA-core FMA; parity bar 1e-5 on probabilities).
 * GWI_FP16: weights rounded to binary16 (RNE) at load, inputs binary16, fp32 accumulation (reading A14);
 *           paper-scale models (R=64,S=128,k=2) run on the tcgen05 tensor-core kernel (parity bar 2e-3). */
typedef enum { GWI_FP32 = 0, GWI_FP16 = 1 } gwi_precision;

/* One trigger (readings A19-A22): a maximal run [start,end) of samples with mean probability > threshold
 * and end-start >= min_len.  start/end are global sample indices (t0 added).  `end` is the merger-time
 * estimate.  model_mask bit j: model j alone exceeded the threshold somewhere in the run.
 * Exactly compared with the oracle: slide, start, end.  peak_p / mean_p are fp32 statistics of the mean
 * probability over the run. */
#define GWI_EDGE_LEFT (1 << 30)  /* time-shard mode only: the run starts at the shard's first sample */
#define GWI_EDGE_RIGHT (1 << 29) /* time-shard mode only: the run ends at the shard's last sample    */
typedef struct {
    int32_t slide;
    int32_t model_mask;
    int64_t start;
    int64_t end;
    float peak_p;
    float mean_p;
} gwi_trigger;

/* ---- model ------------------------------------------------------------------------------------------- */

/* Load a GWIM v1 model file (layout: DESIGN.md "Model file"; network: DESIGN.md C.1 = PAPER.md:45, 49) and
 * upload its weights to CUDA device `device`, packed for the kernels of precision `prec`.
 * path: host C string.  out: receives the handle (owned by the caller until gwi_free_model).
 * Errors: GWI_ERR_ARG (null), GWI_ERR_IO, GWI_ERR_FORMAT, GWI_ERR_UNSUPPORTED (k > 8, R or S > 256,
 * Hh > 512), GWI_ERR_CUDA. */
gwi_status gwi_load_model(const char* path, gwi_precision prec, int device, gwi_model** out);

/* Free the handle and its device memory.  NULL is a no-op. */
void gwi_free_model(gwi_model* m);

/* Architecture of a loaded model.  Any out pointer may be NULL.  receptive_field = 1 + (k-1) * sum(d_i). */
gwi_status gwi_model_info(const gwi_model* m, int32_t* n_branch, int32_t* c_in, int32_t* R, int32_t* S,
                          int32_t* k, int32_t* n_blocks, int32_t* Hh, int32_t* receptive_field);

/* 1 if FP16-mode gwi_infer on this model runs the tcgen05 tensor-core kernel, 0 if it runs the generic
 * CUDA-core kernel on fp16-rounded operands. */
int gwi_model_uses_tensor_cores(const gwi_model* m);

/* ---- window inference (the paper's tensor contract) --------------------------------------- */

/* Bytes of device workspace gwi_infer needs for B windows of T samples (0 on bad arguments). */
size_t gwi_infer_workspace_bytes(const gwi_model* m, int64_t B, int32_t T);

/* p[b][t] for B independent windows, each evaluated with zero history at t < 0 of every layer (reading A4).
 * d_strain: [B][T][C] channels-last, C = n_branch*c_in (H1 first); float in FP32 mode, __half in FP16 mode;
 *           16-byte aligned.   d_prob: [B][T] float.   d_workspace: >= gwi_infer_workspace_bytes, 256 B aligned.
 * T: any length >= 1 (not only 4096).  B >= 0 (B == 0 is a no-op).
 * Errors: GWI_ERR_ARG, GWI_ERR_NOMEM (workspace too small), GWI_ERR_CUDA. */
gwi_status gwi_infer(const gwi_model* m, const void* d_strain, int64_t B, int32_t T, float* d_prob,
                     void* d_workspace, size_t workspace_bytes, void* cuda_stream);

/* ---- ensemble mean + threshold + trigger clustering (readings A18-A22) ------------------- */

/* Bytes of the opaque device carry block / of the device scratch needed for N samples. */
size_t gwi_carry_bytes(void);
size_t gwi_triggers_workspace_bytes(int64_t N);

/* Post-processing on materialised probabilities.
 * d_prob: HOST array of n_models DEVICE pointers; d_prob[j] is model j's [N] float stream chunk.
 * The mean is the fixed fp32 expression (((p0+p1)+p2)+...)/(float)n_models, IEEE round-to-nearest adds and one
 * correctly rounded division; a sample is supra-threshold iff mean > threshold (strict).
 * t0: global sample index of element 0.  slide_id: copied into every record.
 * d_carry: NULL (the chunk is a whole stream) or a device block of gwi_carry_bytes() that the caller zeroes
 *          before the first chunk; it carries the open run across calls on consecutive chunks.
 * last_chunk != 0: a run still open at the end of this chunk is closed there (reading A21).
 * d_triggers / d_count: device; records sorted by start; *d_count = number of qualifying runs closed by this
 *          call (may exceed capacity; then only the first `capacity` are written: the call itself is asynchronous and
 *          returns GWI_OK, the caller compares *d_count with capacity after synchronising the stream).
 * d_pbar: optional device [N] float, receives the mean probability (NULL: not written).
 * 1 <= n_models <= 16, N >= 1.  Errors: GWI_ERR_ARG, GWI_ERR_NOMEM, GWI_ERR_CUDA. */
gwi_status gwi_ensemble_triggers(const float* const* d_prob, int32_t n_models, int64_t N, int64_t t0,
                                 float threshold, int64_t min_len, int32_t slide_id, int last_chunk,
                                 void* d_carry, gwi_trigger* d_triggers, int32_t capacity, int32_t* d_count,
                                 float* d_pbar, void* d_workspace, size_t workspace_bytes, void* cuda_stream);

/* The same call for callers that cannot allocate device memory (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): no workspace argument, the scratch is a file-scope device array inside the library,
 * sized for N <= GWI_TRIGGERS_STATIC_MAX_N samples (2^24 = 68 min at 4096 Hz: 2.1 MB, held by every GPU that loads the
 * library until the process exits).  The call allocates nothing: no cudaMalloc / cudaFree, no allocating library
 * routine; inputs and outputs are the caller's, exactly as above, and so are the results (same kernels).
 * The device that holds the buffers must be the CURRENT device (the scratch address is looked up per device, once).
 * Every call on a device shares the one array: calls that overlap on the GPU (different streams, or graph branches
 * without a dependency) race; serialise them.  Nothing is kept between calls (the scratch header is cleared by each call).
 * Errors: as above, plus GWI_ERR_CAPACITY when N > GWI_TRIGGERS_STATIC_MAX_N (the message says so). */
#define GWI_TRIGGERS_STATIC_MAX_N (1 << 24)
gwi_status gwi_ensemble_triggers_static(const float* const* d_prob, int32_t n_models, int64_t N, int64_t t0,
                                        float threshold, int64_t min_len, int32_t slide_id, int last_chunk,
                                        void* d_carry, gwi_trigger* d_triggers, int32_t capacity, int32_t* d_count,
                                        float* d_pbar, void* cuda_stream);

/* ---- streaming ensemble: one causal pass over a long two-detector stream ---
 *
 * What it computes (DESIGN.md C.1 "Stream", "Ensemble", "Slide k", "Triggers"):
 *   p_m[t], t in [0, n_total): model m evaluated ONCE over the whole stream with zero history only at t = 0 (by
 *   reading A15 / pin P8 this equals stitching 1 s windows taken every 0.5 s); for slide j with lag_j samples
 *   p_{m,j}[t] = head_m(u_{m,H1}[t], u_{m,L1}[(t - lag_j) mod n_total]) (reading A24; slide 0 is the zero lag);
 *   pbar_j = fp32 mean over models; triggers = maximal runs of pbar_j > threshold with length >= min_len, runs
 *   carried across chunk boundaries; records sorted by (slide, start).  Pushing the stream in chunks of any sizes
 *   gives bit-identical results to pushing it whole (reading A17).
 *
 * Back ends (chosen at create, same results contract; gwi_stream_backend tells which): FP16-mode ensembles of the narrow
 * config-1 architecture run on a fused tcgen05 kernel (with slides: the head's first layer is split by linearity into
 * per-sample halves, and every (sample, lag, model) is evaluated element-wise, fused with the mean and the threshold -- no
 * per-lag probability array exists unless d_pbar or the per-model rule asks for one); FP16-mode paper-scale models run on
 * the tcgen05 kernel over segments with recomputed warm-up (with slides when the lags and n_total are multiples of 128
 * samples and n_total >= max lag + R_f - 1: the same split of the head, its halves contracted per sample on the tensor
 * cores; this back end works in whole blocks of up to 2^23 samples, so the outputs of the last pushed samples may be
 * produced by a later push, or by the push that completes n_total -- gwi_stream_samples_done tells how far it is);
 * everything else (FP32 mode, other architectures) runs on the generic kernels.
 *
 * gwi_stream_create   models: HOST array of n_models loaded models sharing device, precision and architecture
 *                     (1..16).  lags: HOST array of n_lags lags in SAMPLES, each >= 1; a lag >= n_total wraps (lag mod n_total: the slides are
 *                     circular, so a multiple of n_total is the zero lag again) (n_lags = 0: zero lag
 *                     only; slides need a two-branch model).  max_chunk: largest n a push will carry.  capacity:
 *                     records the stream can hold.  d_pbar: NULL, or a DEVICE array [1 + n_lags][n_total] float that
 *                     receives pbar_j (for parity tests; ~4 B x n_total per slide).  The handle owns all its device
 *                     memory (staging, per-layer histories, L1 feature ring, probabilities, records).
 *                     Errors: GWI_ERR_ARG, GWI_ERR_UNSUPPORTED (slides on a one-branch model), GWI_ERR_NOMEM, GWI_ERR_CUDA.
 * gwi_stream_tail_samples / gwi_stream_prime   (only when n_lags > 0, before the first push) the circular wrap of the
 *                     slides needs the L1 features of the last max-lag samples at the START: the caller passes the last
 *                     gwi_stream_tail_samples() samples of the L1 strain (HOST or DEVICE pointer; __half in FP16 mode,
 *                     float in FP32 mode; for c_in > 1 planar [c_in][n_tail]).  The tail is max-lag + R_f - 1 samples
 *                     (or the whole stream if shorter), which makes its features exact.
 * gwi_stream_push     d_h1, d_l1: DEVICE pointers to the next n samples of each detector (planar; d_l1 ignored for a
 *                     one-branch model).  Enqueued on cuda_stream; the buffers may be reused once that work is done.
 * gwi_stream_push_host  same from HOST buffers (pinned for real overlap): the H2D copy runs on the handle's side
 *                     stream into a double-buffered staging area while the previous chunk computes on cuda_stream.
 *                     The host buffers must stay valid until the copy has completed (synchronise cuda_stream).
 * gwi_stream_finish   after exactly n_total samples: waits for cuda_stream, copies the records to the HOST array
 *                     h_triggers (up to `capacity`, sorted by (slide, start)) and the total to *h_count.
 *                     GWI_ERR_CAPACITY if the total exceeds either capacity (the returned prefix is then not guaranteed
 *                     to be the globally first records).
 * gwi_stream_destroy  frees the handle (NULL is a no-op).  The models must outlive the stream. */
gwi_status gwi_stream_create(const gwi_model* const* models, int32_t n_models, const int64_t* lags, int32_t n_lags,
                             int64_t n_total, int64_t max_chunk, float threshold, int64_t min_len, int32_t capacity,
                             float* d_pbar, gwi_stream** out);
int64_t gwi_stream_tail_samples(const gwi_stream* s);
gwi_status gwi_stream_prime(gwi_stream* s, const void* l1_tail, int64_t n_tail, void* cuda_stream);
gwi_status gwi_stream_push(gwi_stream* s, const void* d_h1, const void* d_l1, int64_t n, void* cuda_stream);
gwi_status gwi_stream_push_host(gwi_stream* s, const void* h_h1, const void* h_l1, int64_t n, void* cuda_stream);
gwi_status gwi_stream_finish(gwi_stream* s, gwi_trigger* h_triggers, int32_t capacity, int32_t* h_count,
                             void* cuda_stream);
/* samples whose outputs have been produced (enqueued) so far; n_total once the last push has been made */
int64_t gwi_stream_samples_done(const gwi_stream* s);
/* ---- time shards (one rank per GPU, the data sharded across ranks) -------------------------
 * A rank that owns the global samples [t_first, t_first + n) of a longer stream creates its handle with
 * n_total = warmup + n and pushes the `warmup` samples that precede its span (R_f - 1 of them make every kept output
 * exact, pin P8; 0 for the rank that owns t = 0) followed by its own samples.  gwi_stream_set_shard (before the first
 * push and before gwi_stream_prime) makes the handle
 *   - discard the outputs of the first `warmup` pushed samples (d_pbar, if given, is then [1 + n_lags][n_total - warmup]),
 *   - report global sample indices (t_first = index of the first kept sample),
 *   - emit a run that touches the shard's first or last sample whatever its length, flagged GWI_EDGE_LEFT / GWI_EDGE_RIGHT
 *     in model_mask: it may continue in the neighbouring shard; the caller joins such runs across ranks and applies
 *     min_len to the joined run (paper_2201_11133_b200/shard.py: merge_edge_records).
 * Time slides: the caller primes the handle with the L1 samples that precede its first PUSHED sample in the GLOBAL stream
 * (circularly), i.e. the global samples [t_first - warmup - tail, t_first - warmup) mod the global length, so that
 * every slide sees L1[(t - lag) mod N_global].  No collective is involved; the only exchange is the record gather.
 * Errors: GWI_ERR_ARG (after the first push, warmup < 0 or >= n_total). */
gwi_status gwi_stream_set_shard(gwi_stream* s, int64_t t_first, int64_t warmup);
/* which back end gwi_stream_create chose (parity tests assert that the kernel they mean to check is the one that ran) */
typedef enum { GWI_BACKEND_GENERIC = 0, GWI_BACKEND_NARROW = 1, GWI_BACKEND_TENSOR = 2, GWI_BACKEND_TENSOR_SLIDES = 3 } gwi_backend;
int gwi_stream_backend(const gwi_stream* s);

/* ---- the paper's decision rule: per-model triggers + all-model coincidence (reading A34) ------
 *
 * gwi_stream_set_rule   before the first push.  GWI_RULE_MEAN (default): triggers of the ensemble-mean probability
 *                     (BASELINE.json configs 3-5).  GWI_RULE_PER_MODEL: every model's own probability is thresholded
 *                     and clustered separately (same threshold, min_len, run carry); each record carries its slide and
 *                     model_mask = 1 << model.  In this mode d_pbar, if given at create, is [1 + n_lags][n_models][n_total]
 *                     and receives every model's probabilities.
 * gwi_coincidence     HOST function on HOST records (as gwi_stream_finish returns them in GWI_RULE_PER_MODEL mode, any
 *                     order).  Per slide: an end time a of some trigger is an anchor iff every one of the n_models
 *                     models has a trigger whose end lies in [a, a + window]; anchors more than `window` apart start
 *                     a new event; an event reports t_first = its first anchor, t_last = the largest trigger end in
 *                     [t_first, last anchor + window], n_triggers = the number of trigger ends in that span.
 *                     Events sorted by (slide, t_first); *n_events = total (GWI_ERR_CAPACITY if > capacity, the first
 *                     `capacity` are valid).  `end` is the merger-time estimate of a trigger.       */
typedef enum { GWI_RULE_MEAN = 0, GWI_RULE_PER_MODEL = 1 } gwi_rule;
typedef struct {
    int64_t t_first;
    int64_t t_last;
    int32_t n_triggers;
    int32_t slide;
} gwi_event;
gwi_status gwi_stream_set_rule(gwi_stream* s, gwi_rule rule);
gwi_status gwi_coincidence(const gwi_trigger* h_triggers, int32_t n_triggers, int32_t n_models, int64_t window,
                           gwi_event* h_events, int32_t capacity, int32_t* n_events);
void gwi_stream_destroy(gwi_stream* s);

/* ---- trigger counts at many thresholds in one pass (ROC sweep) ---------------
 * counts[j] = number of maximal runs of the ensemble mean (same fixed fp32 expression as gwi_ensemble_triggers) that are
 * strictly above thresholds[j] for at least min_len samples, for a WHOLE stream of N samples (no chunk carry).
 * d_prob: HOST array of n_models DEVICE pointers to [N] float.  d_thresholds: DEVICE [n_thresholds] float, ascending,
 * 1 <= n_thresholds <= 1024.  d_counts: DEVICE [n_thresholds] int64.  1 <= min_len <= 16384.
 * d_workspace: DEVICE, >= gwi_sweep_workspace_bytes(n_thresholds), 256 B aligned.
 * Method: one sliding-window minimum m[t] over min_len samples; count(theta) = rising edges of (m > theta).
 * Errors: GWI_ERR_ARG, GWI_ERR_NOMEM, GWI_ERR_UNSUPPORTED (min_len > 16384), GWI_ERR_CUDA. */
size_t gwi_sweep_workspace_bytes(int32_t n_thresholds);
gwi_status gwi_threshold_sweep(const float* const* d_prob, int32_t n_models, int64_t N, const float* d_thresholds,
                               int32_t n_thresholds, int64_t min_len, int64_t* d_counts, void* d_workspace,
                               size_t workspace_bytes, void* cuda_stream);

/* ---- the paper's peak rule: SciPy find_peaks(height, width) on one model's probabilities (NEXT-1) ------
 * "post-processed it with the find_peaks algorithm, a SciPy's off-the-shelve tool"; "peaks whose width is at
 * least 0.5 seconds long ... height in our find_peaks algorithms".  On the device array d_x[N] (one model's
 * per-timestep probabilities of a whole segment; the search for a peak's prominence is not local, so there is no chunk
 * carry) the call finds, exactly as scipy.signal.find_peaks(x, height=height, width=min_width) does:
 *   local maxima (a flat top counts once, at the floor of its middle; the first and last sample never),  x[p] >= height,
 *   prominence = x[p] - max(lowest sample between p and the nearest higher sample on the left, same on the right),
 *   width between the linearly interpolated crossings of x[p] - prominence / 2,  width >= min_width (in samples).
 * d_peaks: DEVICE [capacity], sorted by index; *d_count (DEVICE) = number of peaks found; if it exceeds capacity the
 * records are not valid (the call is asynchronous and returns GWI_OK; compare after synchronising).
 * d_workspace: DEVICE, >= gwi_find_peaks_workspace_bytes(N, capacity), 256 B aligned.  Peak positions, prominences and
 * widths equal the fp64 oracle's on the same fp32 samples (decisions are taken in fp64 on exact differences).
 * A peak's position is the model's trigger time for gwi_coincidence (pass index as `end`).
 * Errors: GWI_ERR_ARG, GWI_ERR_NOMEM, GWI_ERR_CUDA. */
typedef struct {
    int64_t index;
    float height;
    float prominence;
    double width;
    double left_ip;
    double right_ip;
} gwi_peak;
size_t gwi_find_peaks_workspace_bytes(int64_t N, int32_t capacity);
gwi_status gwi_find_peaks(const float* d_x, int64_t N, float height, double min_width, gwi_peak* d_peaks, int32_t capacity,
                          int32_t* d_count, void* d_workspace, size_t workspace_bytes, void* cuda_stream);

/* ---- whitening front end (reading A35) ----------------------------------------
 * One segment of n raw strain samples of one detector -> whitened, unit-variance samples (what gwi_infer / gwi_stream_*
 * take as input): Welch estimate of the segment's own PSD (frames of nper samples every nper/2, symmetric Hann window,
 * mean of the squared magnitudes), linear interpolation of it to the segment's frequencies, division of the spectrum
 * by its square root, inverse transform, division by the population standard deviation.
 * d_raw: DEVICE [n] float (not modified; any 4-byte alignment is accepted, 16 bytes is the fast path -- other pointers
 * cost one staging copy).  d_out: DEVICE [n], float, or __half when out_is_half != 0 (may not alias d_raw).  n, nper even, 4 <= nper <= n <= 2^30.  d_workspace: DEVICE, >= gwi_whiten_workspace_bytes(n, nper), 256 B
 * aligned.  The FFTs are cuFFT transforms; the library is loaded on first use (GWI_ERR_UNSUPPORTED if it cannot be).
 * The call enqueues on cuda_stream and returns; the FFT plans are cached per (device, n, nper, stream) for the life of the
 * process, so successive segments of one length re-use them.
 * Errors: GWI_ERR_ARG, GWI_ERR_NOMEM, GWI_ERR_UNSUPPORTED, GWI_ERR_CUDA. */
size_t gwi_whiten_workspace_bytes(int64_t n, int32_t nper);
gwi_status gwi_whiten(const float* d_raw, int64_t n, int32_t nper, void* d_out, int out_is_half, void* d_workspace,
                      size_t workspace_bytes, void* cuda_stream);

/* ---- misc ---------------------------------------------------------------------------------------------- */
const char* gwi_last_error(void);
int gwi_version(void);
/* number of kernels this library has launched since load (all threads); bench.py reports it */
int64_t gwi_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* GWI_H */
