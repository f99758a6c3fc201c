// mlp_tc.cu -- K5/K6 on the tcgen05 tensor cores (placeholder until the tensor-core tile kernel lands:
// reports "no tensor-core image", so workspaces start in NNP_MLP_FP32_SIMT).
#include "nnp_internal.h"
namespace nnp {
int tc_model_create(nnp_model* m, const nnp_mlp_desc*) { m->tc = nullptr; return NNP_OK; }
void tc_model_destroy(nnp_model*) {}
int tc_workspace_create(nnp_workspace* ws) { ws->tc_ws = nullptr; return NNP_OK; }
void tc_workspace_destroy(nnp_workspace*) {}
int launch_mlp_tc(nnp_workspace* ws, int64_t n_ml) { return launch_mlp_simt(ws, n_ml); }
}  // namespace nnp
