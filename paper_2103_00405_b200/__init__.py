"""paper_2103_00405_b200 -- B200-native hot path of the next-reaction random-time algorithm
(Liu & Wang, arXiv 2103.00405): thin Python binding over the C ABI of include/rt.h.

Every step of the simulation runs in the CUDA kernels of csrc/; this package only marshals
arguments.  There is no CPU fallback: if librt_b200.so is missing the import fails, and on a
machine without a CUDA device rt_create returns RT_ERR_CUDA.
"""
from .binding import (  # noqa: F401
    RT_OK, RT_ERR_NULL, RT_ERR_BAD_NETWORK, RT_ERR_BAD_ARG, RT_ERR_UNSUPPORTED, RT_ERR_OVERFLOW,
    RT_ERR_CUDA, RT_ERR_OOM, RT_ERR_SCRATCH, RT_NOALLOC_SCRATCH_BYTES, RT_STOP_T_END, RT_STOP_MAX_FIRINGS, RT_STOP_ABSORBED,
    RESULT_DTYPE, RtError, Model, lib, library_path,
    rt_validate_network, rt_create, rt_run, rt_run_resume, rt_run_dev, rt_noalloc_prepare, rt_run_dev_noalloc, rt_ensemble, rt_ensemble_dev, rt_sync,
    rt_set_option, rt_set_rate_schedule, rt_set_rate_exponent, rt_get_info, rt_destroy, rt_strerror,
)
from .dist import shard_range, ensemble_sharded  # noqa: F401
from .model_file import parse_model, load_model, ModelFileError  # noqa: F401
from .rewrite import rewrite_trimolecular, RewriteError  # noqa: F401
