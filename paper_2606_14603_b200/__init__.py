"""B200-native molecule-agent step engine (hot path of arxiv/paper_2606_14603).

`Sim` is a thin ctypes binding of the C-ABI library `libmolsim.so` (include/molsim.h): argument
marshalling only; every step of the path runs in the hand-written sm_100a kernels.  PyTorch is
used for device memory and the stream.  There is no CPU fallback: loading fails loudly when the
library has not been built.
"""
from .binding import Sim, SimError, check_config, load_library  # noqa: F401
