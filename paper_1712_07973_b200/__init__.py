"""paper_1712_07973_b200 -- B200-native exact-exchange operator application (arXiv:1712.07973 hot path).

Thin Python binding of the C-ABI library libexx_b200.so (include/exx.h): argument marshalling only, every step
of the path runs in the library's CUDA kernels.  PyTorch is used for device memory and streams.
"""
from .binding import (  # noqa: F401
    EXX_BLOCK_ACCUMULATE_RESIDENT,
    EXX_BLOCK_ACCUMULATE_STREAMED,
    ExxError,
    ExxPlan,
    exx_apply,
    exx_diag_fp64,
    exx_diag_shfl,
    exx_exchange_energy_noalloc,
    exx_plan_create,
    exx_plan_destroy,
    exx_round_robin_step,
    exx_schedule_list,
    exx_schedule_list_block,
    exx_schedule_pairs,
    exx_version,
    library_path,
    load_library,
)
from .build import build  # noqa: F401
