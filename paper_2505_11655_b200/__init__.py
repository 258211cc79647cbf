"""B200-native ILE hot path of arxiv/paper_2505_11655: Python binding over libile.so.

The product is the C-ABI library declared in include/ile.h (hand-written CUDA for sm_100a);
this package only marshals arguments.  It never imports oracle/.
"""
from .binding import (Ile, IleError, Integrator, Integrand, Result, IntegratorOpts, RESULT_DTYPE, KINDS, load_library,  # noqa: F401
                      result_from_device, parse_state, pack_state, LIB_PATH)
