// gemm_tc.cu — BF16 tensor-core GEMMs (placeholder until the tcgen05 path lands: reports UNSUPPORTED).
#include "gemm_tc.cuh"

namespace pnn {
struct TcModel { int dummy; };
struct TcWorkspace { int dummy; };
int tc_model_create(const pnn_config*, const double*, TcModel**) { return PNN_ERR_UNSUPPORTED; }
void tc_model_destroy(TcModel*) {}
int tc_workspace_create(const TcModel*, int64_t, TcWorkspace**) { return PNN_ERR_UNSUPPORTED; }
void tc_workspace_destroy(TcWorkspace*) {}
int64_t tc_workspace_bytes(const TcWorkspace*) { return 0; }
} // namespace pnn
