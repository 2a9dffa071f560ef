// gwi_internal.h -- shared declarations of the library's translation units (NOT part of the C-ABI).
#pragma once
#include <cuda_runtime.h>
#include <cuda_fp16.h>
#include <stdint.h>
#include <string>
#include <vector>

#include "../../include/gwi.h"

#define GWI_MAX_LAYERS 64
#define GWI_MAX_MODELS 16

// ---- error plumbing ---------------------------------------------------------------------------------------
void gwi_set_error(const char* fmt, ...);
#define GWI_CUDA_CHECK(expr)                                                                     \
    do {                                                                                         \
        cudaError_t e__ = (expr);                                                                \
        if (e__ != cudaSuccess) {                                                                \
            gwi_set_error("%s:%d: %s -> %s", __FILE__, __LINE__, #expr, cudaGetErrorString(e__)); \
            return GWI_ERR_CUDA;                                                                 \
        }                                                                                        \
    } while (0)
void gwi_count_launch(int n = 1);

// ---- architecture (GWIM v1 header) -------------------------------------------------
struct GwiArch {
    int n_branch, c_in, R, S, k, L, Hh;
    int dil[GWI_MAX_LAYERS];
    int receptive_field() const {
        long s = 0;
        for (int i = 0; i < L; i++) s += dil[i];
        return (int)(1 + (long)(k - 1) * s);
    }
};

// Offsets (in floats) of every tensor inside the fp32 weight blob, which is the file's tensor section verbatim
// (FP16 mode: every value rounded to binary16 and widened again).
struct GwiLayerOff {
    int64_t Wf, bf, Wg, bg, Wr, br, Ws, bs;
};
struct GwiOffsets {
    int64_t W_in[4], b_in[4];             // per branch (n_branch <= 4)
    GwiLayerOff layer[4][GWI_MAX_LAYERS]; // [branch][block]
    int64_t W1, b1, W2, b2;
};

// Device-side view used by the generic fp32 kernels (passed by value to kernels: small).
struct GwiDevModel {
    const float* blob;
    int n_branch, c_in, R, S, k, L, Hh;
};

// Packed fp16 weights of the tcgen05 kernel (gwi_tc.cu); null when the architecture is not covered.
struct GwiTcPack;
// Packed fragments of the fused narrow-architecture stream kernel (gwi_tiny.cu); null when not covered / not FP16.
struct GwiTinyPack;
// Packed operands of the tcgen05 narrow-architecture stream kernel (gwi_tiny_tc.cu); null when not covered / not FP16.
struct GwiTinyTcPack;

struct gwi_model {
    GwiArch arch;
    gwi_precision prec;
    int device;
    std::vector<float> host_blob; // weights as the kernels see them (rounded to fp16 and widened in FP16 mode)
    GwiOffsets off;
    float* d_blob = nullptr;
    GwiOffsets* d_off = nullptr; // copy of `off` in device memory
    GwiTcPack* tc = nullptr;
    GwiTinyPack* tiny = nullptr;
    GwiTinyTcPack* tinytc = nullptr;
};

// ---- generic CUDA-core path (gwi_generic.cu) ---------------------------------------------------------------
size_t gwi_generic_workspace_bytes(const gwi_model* m, int64_t B, int32_t T);
gwi_status gwi_generic_infer(const gwi_model* m, const void* d_strain, bool strain_is_half, int64_t B, int32_t T,
                             float* d_prob, void* d_ws, size_t ws_bytes, cudaStream_t st);

// stream mode (gwi_stream.cu): branch stacks with per-layer history carried across chunks, head with an L1 lag
int64_t gwi_generic_hist_floats(const gwi_model* m);
gwi_status gwi_generic_stream_branches(const gwi_model* m, const void* d_strain, bool strain_is_half, int64_t ldx, int n,
                                       float* hA, float* hB, int64_t ldh, float* skip, int64_t lds,
                                       const float* hist_cur, float* hist_next, int br0, int nbr, cudaStream_t st);
gwi_status gwi_generic_stream_head(const gwi_model* m, const float* skip, int64_t lds, int64_t lag, int n, float* d_prob,
                                   cudaStream_t st);

int64_t gwi_tc_max_windows(const gwi_model* m, int32_t T);
int gwi_tc_num_sms(const gwi_model* m);
gwi_status gwi_tc_stack(const gwi_model* m, const __half* d_strain, int64_t B, int32_t T, void* d_ws, size_t ws_bytes,
                        cudaStream_t st, const uint8_t** u_out);
gwi_status gwi_tc_vhalf(const gwi_model* m, const uint8_t* u, int64_t B, int ntiles, int seg_tiles, int warm_tiles, int stream_start,
                        int n_valid, __half* d_v, int64_t lds, cudaStream_t st);
gwi_status gwi_tc_head_stream(const gwi_model* m, const uint8_t* u, int ntiles, const uint8_t* hist, int R, int64_t nq,
                              const int64_t* d_lags, int n_lags, int seg_tiles, int warm_tiles, int stream_start, int n_valid,
                              float* d_prob, int64_t stride_k, cudaStream_t st);

// ---- post-processing (gwi_post.cu) ---------------------------------------------------------------------------
gwi_status gwi_post_run(const float* const* d_prob, int32_t n_models, int64_t N, int64_t t0, float threshold,
                        int64_t min_len, int32_t slide_id, int last_chunk, void* d_carry, gwi_trigger* d_triggers,
                        int32_t capacity, int32_t* d_count, int append, float* d_pbar, void* d_workspace,
                        size_t workspace_bytes, cudaStream_t st, int64_t shard_begin = -1, int64_t shard_end = -1);

size_t gwi_post_batch_workspace_bytes(int64_t N, int nslides);
gwi_status gwi_post_run_bits_batch(const uint32_t* d_bits, int64_t bits_stride, const float* d_pbar, const uint8_t* d_mm, int64_t row_stride,
                                   int nslides, int64_t N, int64_t t0, float threshold, int64_t min_len, int32_t slide0, int last_chunk,
                                   void* d_carry, gwi_trigger* d_triggers, int32_t capacity, int32_t* d_count, int append,
                                   void* d_workspace, size_t workspace_bytes, cudaStream_t st, int64_t shard_begin, int64_t shard_end);
gwi_status gwi_post_run_bits(const uint32_t* d_bits, const float* d_pbar, const uint8_t* d_mm, int64_t N, int64_t t0, float threshold,
                             int64_t min_len, int32_t slide_id, int last_chunk, void* d_carry, gwi_trigger* d_triggers,
                             int32_t capacity, int32_t* d_count, int append, void* d_workspace, size_t workspace_bytes,
                             cudaStream_t st, int64_t shard_begin = -1, int64_t shard_end = -1);
// fused time-slide heads of the narrow architecture (gwi_heads.cu): all lags, all models, mean, threshold
gwi_status gwi_heads_fused(const gwi_model* const* models, int M, const __half* const* d_v, int64_t lds, int n, const int64_t* d_lags,
                           int n_lags, const int64_t* h_lags, float theta, uint32_t* d_bits, int64_t bits_stride, float* d_pbar,
                           uint8_t* d_mm, int64_t row_stride, float* d_prob, cudaStream_t st);
bool gwi_tiny_writes_v(const gwi_model* m);

// ---- tcgen05 path (gwi_tc.cu) -------------------------------------------------------------------------------
bool gwi_tc_supported(const GwiArch& a);
gwi_status gwi_tc_pack(gwi_model* m);
void gwi_tc_free(gwi_model* m);
size_t gwi_tc_workspace_bytes(const gwi_model* m, int64_t B, int32_t T);
gwi_status gwi_tc_infer(const gwi_model* m, const __half* d_strain, int64_t B, int32_t T, float* d_prob, void* d_ws,
                        size_t ws_bytes, cudaStream_t st);

// ---- fused narrow-architecture stream kernel (gwi_tiny.cu) ----------------------------------------------------
bool gwi_tiny_supported(const GwiArch& a);
gwi_status gwi_tiny_pack(gwi_model* m);
void gwi_tiny_free(gwi_model* m);
int gwi_tiny_halo(const gwi_model* m);
gwi_status gwi_tiny_stream(const gwi_model* m, const __half* d_x, int64_t ldx, int n, int64_t t0, const __half* xh_cur,
                           __half* xh_next, float* d_prob, __half* d_u16, int64_t lds, cudaStream_t st);
gwi_status gwi_tiny_heads(const gwi_model* m, const __half* d_u16, int64_t lds, int n, const int64_t* d_lags, int n_lags,
                          float* d_prob, int64_t stride_k, cudaStream_t st);
// tcgen05 version of the same kernel (gwi_tiny_tc.cu); gwi_tiny_stream dispatches to it
bool gwi_tiny_tc_supported(const GwiArch& a);
gwi_status gwi_tiny_tc_pack(gwi_model* m);
void gwi_tiny_tc_free(gwi_model* m);
gwi_status gwi_tiny_tc_stream(const gwi_model* m, const __half* d_x, int64_t ldx, int n, int64_t t0, const __half* xh_cur,
                              float* d_prob, __half* d_u16, int64_t lds, cudaStream_t st);
gwi_status gwi_xhist_update(const __half* d_x, int64_t ldx, int n, int halo, const __half* xh_cur, __half* xh_next, cudaStream_t st);
