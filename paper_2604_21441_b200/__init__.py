"""paper_2604_21441_b200 -- B200-native NNP energy+force evaluation (the hot path behind the ML/MM interface
of arxiv/paper_2604_21441).  Thin ctypes binding over the C-ABI library declared in include/nnp.h; every step
of the path runs in the library's sm_100a kernels.  There is no CPU fallback: importing the binding raises if
libnnp_b200.so is missing, and every compute call returns NNP_ERR_CUDA without a device."""
from .binding import (  # noqa: F401
    NNPError, Model, Workspace, lib, lib_path,
    nnp_model_create, nnp_model_create_ensemble, nnp_model_destroy, nnp_model_aev_length, nnp_model_default_mlp_mode, nnp_workspace_create, nnp_workspace_destroy,
    nnp_workspace_set_mlp_mode, nnp_workspace_set_dense_k, nnp_workspace_set_virial_output, nnp_workspace_set_units, nnp_workspace_set_pair_list, nnp_workspace_set_small_path, nnp_workspace_set_bin_reuse, nnp_eval, nnp_eval_host, nnp_status, nnp_strerror,
    nnp_debug_neighbors, nnp_debug_aev, nnp_debug_daev, nnp_debug_mlp_timeline, nnp_link_place, nnp_link_spread,
    nnp_debug_atomic_energies, nnp_debug_counters, nnp_workspace_set_profiling, nnp_debug_stage_times, nnp_debug_fp32_peak,
    nnp_energy_sum_static, NNP_ERR_STATIC_LIMIT, NNP_STATIC_MAX_ATOMS,
    NNP_OK, NNP_MLP_FP32_SIMT, NNP_MLP_F16X3, NNP_MLP_F16X1,
)
