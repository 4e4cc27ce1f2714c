// tcgen05 implicit-GEMM convolution -- placeholder until the tensor-core kernel lands (next commit).
#include "ufnvc_internal.h"
namespace ufnvc {
cudaError_t launch_conv_tc(const ConvLayer &, const ConvProblem &, const CUtensorMap &, int, int, const EpiParams &, int, cudaStream_t)
{
    return cudaErrorNotSupported;
}
bool tc_make_weight_tmap(ConvLayer &, std::string &err) { err = "tcgen05 path not built"; return false; }
bool tc_make_act_tmap(CUtensorMap *, const bf16 *, int, int, int, int, int, int, std::string &err) { err = "tcgen05 path not built"; return false; }
}  // namespace ufnvc
