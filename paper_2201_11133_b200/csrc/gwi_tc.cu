// gwi_tc.cu -- tcgen05 tensor-core path (placeholder until the fused kernel lands; reports "not supported"
// so that FP16 mode runs the generic kernel on fp16-rounded operands).
#include "gwi_internal.h"

bool gwi_tc_supported(const GwiArch&) { return false; }
gwi_status gwi_tc_pack(gwi_model*) { return GWI_OK; }
void gwi_tc_free(gwi_model*) {}
size_t gwi_tc_workspace_bytes(const gwi_model*, int64_t, int32_t) { return 0; }
gwi_status gwi_tc_infer(const gwi_model*, const __half*, int64_t, int32_t, float*, void*, size_t, cudaStream_t)
{
    gwi_set_error("tcgen05 path not built");
    return GWI_ERR_UNSUPPORTED;
}
