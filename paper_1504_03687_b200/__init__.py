"""paper_1504_03687_b200 -- B200-native regular-force step of the Hermite / Ahmad-Cohen scheme.

Thin Python binding over the C-ABI library ``libnbreg`` (include/nbreg.h).  Argument marshalling
only: every step of the path runs in the sm_100a kernels under ``csrc/``.  PyTorch supplies device
memory and streams.  There is no CPU fallback: if the library cannot be built/loaded, or no
sm_100 device is present, the calls raise.
"""
from .binding import (  # noqa: F401
    NbregError,
    NbContext,
    load_library,
    exported_symbols,
    nb_open,
    nb_close,
    nb_set_j,
    nb_predict_all,
    nb_regular,
    nb_regular_all,
    nb_step_host,
    nb_plan_regular,
    nb_plan_chunks,
    nb_update_j,
    nb_irregular,
    nb_next_block_static,
    NB_ELIMIT, NB_STATIC_MAX_N,
    NB_OK, NB_EINVAL, NB_ESTATE, NB_ENOMEM, NB_ECUDA, NB_EOVERFLOW,
)
from .build import build_lib  # noqa: F401
