// gwi_api.cu -- C-ABI entry points, model-file parser (GWIM v1) and dispatch.  See include/gwi.h.
#include <atomic>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>

#include "gwi_internal.h"

static thread_local char g_err[512] = "";
static std::atomic<long long> g_launches{0};

void gwi_set_error(const char* fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
}
void gwi_count_launch(int n) { g_launches += n; }

extern "C" const char* gwi_last_error(void) { return g_err; }
extern "C" int gwi_version(void) { return 100; }
extern "C" int64_t gwi_launch_count(void) { return (int64_t)g_launches.load(); }

// ---- GWIM v1 parser (own code; the oracle and gwsynth have their own) ---------------------------------------
// bytes 0..3 "GWIM"; int32 version=1, n_branch, c_in, R, S, k, L, Hh, dtype=0; int32 dil[L]; then fp32 tensors:
// per branch: W_in[R][c_in], b_in[R], per block Wf[R][R][k], bf[R], Wg[R][R][k], bg[R], Wr[R][R], br[R],
// Ws[S][R], bs[S]; head: W1[Hh][n_branch*S], b1[Hh], W2[Hh], b2[1].
static gwi_status parse_model(const char* path, gwi_model* m)
{
    FILE* f = fopen(path, "rb");
    if (!f) {
        gwi_set_error("cannot open %s", path);
        return GWI_ERR_IO;
    }
    struct Closer {
        FILE* f;
        ~Closer() { fclose(f); }
    } closer{f};
    unsigned char head[40];
    if (fread(head, 1, 40, f) != 40) {
        gwi_set_error("%s: truncated header", path);
        return GWI_ERR_IO;
    }
    int32_t h[9];
    memcpy(h, head + 4, 36);
    if (memcmp(head, "GWIM", 4) != 0 || h[0] != 1 || h[8] != 0) {
        gwi_set_error("%s: not a GWIM v1 fp32 file", path);
        return GWI_ERR_FORMAT;
    }
    GwiArch& a = m->arch;
    a.n_branch = h[1], a.c_in = h[2], a.R = h[3], a.S = h[4], a.k = h[5], a.L = h[6], a.Hh = h[7];
    if (a.n_branch < 1 || a.c_in < 1 || a.R < 1 || a.S < 1 || a.k < 1 || a.L < 1 || a.Hh < 1) {
        gwi_set_error("%s: non-positive architecture field", path);
        return GWI_ERR_FORMAT;
    }
    if (a.n_branch > 4 || a.c_in > 8 || a.R > 256 || a.S > 256 || a.k > 8 || a.L > GWI_MAX_LAYERS || a.Hh > 512) {
        gwi_set_error("%s: architecture outside kernel limits (n_branch<=4,c_in<=8,R,S<=256,k<=8,L<=%d,Hh<=512)", path,
                      GWI_MAX_LAYERS);
        return GWI_ERR_UNSUPPORTED;
    }
    int32_t dil[GWI_MAX_LAYERS];
    if (fread(dil, 4, a.L, f) != (size_t)a.L) {
        gwi_set_error("%s: truncated dilation list", path);
        return GWI_ERR_IO;
    }
    for (int i = 0; i < a.L; i++) {
        if (dil[i] < 1) {
            gwi_set_error("%s: dilation %d < 1", path, dil[i]);
            return GWI_ERR_FORMAT;
        }
        a.dil[i] = dil[i];
    }
    // offsets in file order
    int64_t o = 0;
    const int64_t R = a.R, S = a.S, k = a.k;
    for (int b = 0; b < a.n_branch; b++) {
        m->off.W_in[b] = o, o += R * a.c_in;
        m->off.b_in[b] = o, o += R;
        for (int i = 0; i < a.L; i++) {
            GwiLayerOff& l = m->off.layer[b][i];
            l.Wf = o, o += R * R * k;
            l.bf = o, o += R;
            l.Wg = o, o += R * R * k;
            l.bg = o, o += R;
            l.Wr = o, o += R * R;
            l.br = o, o += R;
            l.Ws = o, o += S * R;
            l.bs = o, o += S;
        }
    }
    m->off.W1 = o, o += (int64_t)a.Hh * a.n_branch * S;
    m->off.b1 = o, o += a.Hh;
    m->off.W2 = o, o += a.Hh;
    m->off.b2 = o, o += 1;
    m->host_blob.resize((size_t)o);
    if (fread(m->host_blob.data(), 4, (size_t)o, f) != (size_t)o) {
        gwi_set_error("%s: truncated tensor section (%lld floats expected)", path, (long long)o);
        return GWI_ERR_IO;
    }
    if (fgetc(f) != EOF) {
        gwi_set_error("%s: trailing bytes after the last tensor", path);
        return GWI_ERR_FORMAT;
    }
    return GWI_OK;
}

extern "C" gwi_status gwi_load_model(const char* path, gwi_precision prec, int device, gwi_model** out)
{
    if (!path || !out || (prec != GWI_FP32 && prec != GWI_FP16) || device < 0) {
        gwi_set_error("gwi_load_model: bad argument");
        return GWI_ERR_ARG;
    }
    *out = nullptr;
    gwi_model* m = new (std::nothrow) gwi_model();
    if (!m) return GWI_ERR_NOMEM;
    m->prec = prec;
    m->device = device;
    gwi_status st = parse_model(path, m);
    if (st != GWI_OK) {
        delete m;
        return st;
    }
    if (prec == GWI_FP16)  // reading A14 / C.2: weights are rounded to binary16 (RNE) at load
        for (float& v : m->host_blob) v = __half2float(__float2half_rn(v));
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || device >= ndev) {
        gwi_set_error("gwi_load_model: CUDA device %d not available (%s); there is no CPU fallback", device,
                      e != cudaSuccess ? cudaGetErrorString(e) : "device index out of range");
        delete m;
        return GWI_ERR_CUDA;
    }
    auto fail = [&](cudaError_t ce) {
        gwi_set_error("gwi_load_model: %s", cudaGetErrorString(ce));
        gwi_free_model(m);
        return GWI_ERR_CUDA;
    };
    if ((e = cudaSetDevice(device)) != cudaSuccess) return fail(e);
    size_t bytes = m->host_blob.size() * sizeof(float);
    if ((e = cudaMalloc(&m->d_blob, bytes)) != cudaSuccess) return fail(e);
    if ((e = cudaMemcpy(m->d_blob, m->host_blob.data(), bytes, cudaMemcpyHostToDevice)) != cudaSuccess) return fail(e);
    if ((e = cudaMalloc(&m->d_off, sizeof(GwiOffsets))) != cudaSuccess) return fail(e);
    if ((e = cudaMemcpy(m->d_off, &m->off, sizeof(GwiOffsets), cudaMemcpyHostToDevice)) != cudaSuccess) return fail(e);
    if (prec == GWI_FP16 && gwi_tc_supported(m->arch)) {
        st = gwi_tc_pack(m);
        if (st != GWI_OK) {
            gwi_free_model(m);
            return st;
        }
    }
    if (prec == GWI_FP16 && gwi_tiny_supported(m->arch)) {
        st = gwi_tiny_pack(m);
        if (st != GWI_OK) {
            gwi_free_model(m);
            return st;
        }
    }
    *out = m;
    return GWI_OK;
}

extern "C" void gwi_free_model(gwi_model* m)
{
    if (!m) return;
    gwi_tc_free(m);
    gwi_tiny_free(m);
    gwi_tiny_tc_free(m);
    if (m->d_blob) cudaFree(m->d_blob);
    if (m->d_off) cudaFree(m->d_off);
    delete m;
}

extern "C" gwi_status gwi_model_info(const gwi_model* m, int32_t* n_branch, int32_t* c_in, int32_t* R, int32_t* S,
                                     int32_t* k, int32_t* n_blocks, int32_t* Hh, int32_t* receptive_field)
{
    if (!m) {
        gwi_set_error("gwi_model_info: null model");
        return GWI_ERR_ARG;
    }
    const GwiArch& a = m->arch;
    if (n_branch) *n_branch = a.n_branch;
    if (c_in) *c_in = a.c_in;
    if (R) *R = a.R;
    if (S) *S = a.S;
    if (k) *k = a.k;
    if (n_blocks) *n_blocks = a.L;
    if (Hh) *Hh = a.Hh;
    if (receptive_field) *receptive_field = a.receptive_field();
    return GWI_OK;
}

extern "C" int gwi_model_uses_tensor_cores(const gwi_model* m) { return m && m->tc ? 1 : 0; }

extern "C" size_t gwi_infer_workspace_bytes(const gwi_model* m, int64_t B, int32_t T)
{
    if (!m || B < 0 || T < 1) return 0;
    if (m->tc) return gwi_tc_workspace_bytes(m, B, T);
    return gwi_generic_workspace_bytes(m, B, T);
}

extern "C" gwi_status gwi_infer(const gwi_model* m, const void* d_strain, int64_t B, int32_t T, float* d_prob,
                                void* d_workspace, size_t workspace_bytes, void* cuda_stream)
{
    if (!m || B < 0 || T < 1) {
        gwi_set_error("gwi_infer: bad argument (model=%p B=%lld T=%d)", (const void*)m, (long long)B, T);
        return GWI_ERR_ARG;
    }
    if (B == 0) return GWI_OK;
    if (!d_strain || !d_prob || ((uintptr_t)d_strain & 15) || ((uintptr_t)d_prob & 3) || ((uintptr_t)d_workspace & 255)) {
        gwi_set_error("gwi_infer: null or misaligned pointer");
        return GWI_ERR_ARG;
    }
    cudaPointerAttributes pa;
    if (cudaPointerGetAttributes(&pa, d_strain) != cudaSuccess || pa.type != cudaMemoryTypeDevice || pa.device != m->device) {
        cudaGetLastError();
        gwi_set_error("gwi_infer: d_strain is not a device pointer on device %d", m->device);
        return GWI_ERR_ARG;
    }
    if (cudaPointerGetAttributes(&pa, d_prob) != cudaSuccess || pa.type != cudaMemoryTypeDevice || pa.device != m->device) {
        cudaGetLastError();
        gwi_set_error("gwi_infer: d_prob is not a device pointer on device %d", m->device);
        return GWI_ERR_ARG;
    }
    size_t need = gwi_infer_workspace_bytes(m, B, T);
    if (workspace_bytes < need || (need && !d_workspace)) {
        gwi_set_error("gwi_infer: workspace %zu < %zu bytes", workspace_bytes, need);
        return GWI_ERR_NOMEM;
    }
    GWI_CUDA_CHECK(cudaSetDevice(m->device));
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (m->tc) return gwi_tc_infer(m, (const __half*)d_strain, B, T, d_prob, d_workspace, workspace_bytes, st);
    return gwi_generic_infer(m, d_strain, m->prec == GWI_FP16, B, T, d_prob, d_workspace, workspace_bytes, st);
}
