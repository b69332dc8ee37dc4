// gemm_tc.cuh — BF16 tensor-core (tcgen05 + TMA + TMEM) side of the library: declarations.
#pragma once
#include <stdint.h>

#include "../../include/pnn.h"

namespace pnn {

struct TcModel;      // BF16 copies of the GEMM weights + their TMA descriptors
struct TcWorkspace;  // BF16 activation buffers + their TMA descriptors

int tc_model_create(const pnn_config* cfg, const double* weights_host, TcModel** out);
void tc_model_destroy(TcModel* m);
int tc_workspace_create(const TcModel* m, int64_t max_atoms, TcWorkspace** out);
void tc_workspace_destroy(TcWorkspace* ws);
int64_t tc_workspace_bytes(const TcWorkspace* ws);

} // namespace pnn
