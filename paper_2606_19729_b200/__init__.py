"""paper_2606_19729_b200 -- B200-native hot path of VOiLA's online planner (arxiv/paper_2606_19729):
vectorised Monte-Carlo rollout evaluation and the SIR belief update, as hand-written sm_100a CUDA
behind a C ABI (include/voila.h).  See DESIGN.md."""
from .voila import (EXPORTS, KERNEL_AUTO, KERNEL_FFMA, KERNEL_TCGEN05, KERNEL_TCGEN05_PAIR, PREC_BF16, PREC_FP32,
                    STATIC_MAX_N, Voila, VoilaError, lib_path, load_library, voila_resample_systematic_static)

__all__ = ["Voila", "VoilaError", "load_library", "lib_path", "EXPORTS", "KERNEL_AUTO",
           "KERNEL_FFMA", "KERNEL_TCGEN05", "KERNEL_TCGEN05_PAIR", "PREC_FP32", "PREC_BF16", "STATIC_MAX_N",
           "voila_resample_systematic_static"]
