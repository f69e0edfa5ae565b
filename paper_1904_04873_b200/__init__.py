"""B200-native BinarySkyHough hot path (arXiv:1904.04873): thin Python binding over the C-ABI CUDA library libbsh.so.

Every step of the path (peakgram, track generation, Hough accumulation, per-patch top-k, stage-2 power) runs in the
hand-written sm_100a kernels of csrc/; this package only marshals arguments.  PyTorch supplies device memory and the
CUDA stream.  There is no CPU fallback: importing works without a GPU (so the library and its symbols can be checked),
but creating a Context without a CUDA device raises.
"""
from . import binding
from .binding import (BSH_FAMILY_AUTO, BSH_FAMILY_PIXEL_LANE, BSH_FAMILY_TEMPLATE_LANE, BSH_FAMILY_WINDOW, BSH_NAIVE,
                      BSH_OPT_FORCE_CLAMP, BSH_OPT_KERNEL_FAMILY, BSH_OPT_PIXELS_PER_THREAD, BSH_UNWEIGHTED, BSH_WEIGHTED,
                      CAND_DTYPE, BshError, Context, Stats, library, post_coincidences_static, template_decode,
                      template_index)

__all__ = ["Context", "BshError", "Stats", "library", "CAND_DTYPE", "BSH_UNWEIGHTED", "BSH_WEIGHTED", "BSH_NAIVE",
           "template_index", "template_decode", "post_coincidences_static"]
