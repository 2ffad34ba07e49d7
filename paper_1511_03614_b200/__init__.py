"""B200-native integration hot path of FIESTA 4 (arXiv:1511.03614): thin Python binding.

Argument marshalling only -- every step of the path runs in the CUDA kernels behind the C ABI of
`include/fiesta_b200.h` (libfiesta_b200.so, built in-tree by `paper_1511_03614_b200.build`).
There is no CPU fallback: if the library is missing or no sm_100 device is present the calls
raise.
"""
from .binding import (  # noqa: F401
    Context, Program, Rule, FiestaError, LIB_PATH, load_library, exported_symbols, native_assemble,
    RULE_LATTICE, RULE_MC, RULE_VEGAS, MODE_EVAL, N_MODES, TIER_ANY, TIER_INTERPRETER, TIER_NATIVE,
    RESULT_DTYPE, INFO_DTYPE,
)

from .pool import IntegrationPool, ResultStore  # noqa: F401,E402
from .bisection import bisect_sector, bisect_text  # noqa: F401,E402

load = load_library
