// gemm_tc.cu — placeholder until the tcgen05 kernels land: reports "unsupported" so ffn.cu routes to
// the FP32-ALU kernels.
#include "piper_internal.cuh"
namespace piper {
size_t tc_scratch_bytes(const piper_moe_desc*) { return 256; }
int tc_init(piper_ctx*) { return PIPER_OK; }
bool tc_supported(const piper_ctx*, const FfnProblem&) { return false; }
int tc_ffn_fwd1(piper_ctx*, Lane, const FfnProblem&) { return PIPER_ERR_UNSUPPORTED; }
int tc_ffn_fwd2(piper_ctx*, Lane, const FfnProblem&) { return PIPER_ERR_UNSUPPORTED; }
int tc_ffn_dgrad1(piper_ctx*, Lane, const FfnProblem&) { return PIPER_ERR_UNSUPPORTED; }
int tc_ffn_dgrad2(piper_ctx*, Lane, const FfnProblem&) { return PIPER_ERR_UNSUPPORTED; }
int tc_ffn_wgrad(piper_ctx*, Lane, const FfnProblem&) { return PIPER_ERR_UNSUPPORTED; }
}  // namespace piper
