"""B200-native CoS / SB-CoS DAG evaluator (arxiv 2507.12349): thin Python binding of the C-ABI
declared in include/cos.h.  Argument marshalling only -- every step of the path runs in the CUDA
kernels of libcos_b200.so.  There is no CPU fallback and this package never imports oracle/.
"""
from ._binding import (  # noqa: F401
    COS_OK, COS_EINVAL, COS_ENOMEM, COS_ECUDA, COS_EUNSUPPORTED,
    COS_LATTICE_SQUARE, COS_LATTICE_HONEYCOMB, COS_BUILD_HOST_ONLY, COS_BUILD_NO_FUSED, COS_BUILD_UNIFORM_SHIFT,
    COS_DET_FP64, COS_DET_DD, INFO, TUNE, cos_reserve, cos_set_tuning, cos_debug_check_failures, cos_equivalence_stats,
    CosError, lib_path, load_library,
    cos_build, cos_build_ex, cos_eval, cos_free, cos_info, cos_last_error, cos_set_workspace_limit,
    cos_tab_build, cos_tabulate, cos_tab_free, cos_measure_fp64_fma_peak,
    cos_eval_host, cos_set_profiling, cos_get_layer_times, cos_build_orders, cos_flux_weights, EXPORTS,
    cos_det_workspace_bytes, cos_det_eval, cos_det_eval_static, COS_DET_STATIC_SCRATCH_BYTES,
    dag_summary,
)
