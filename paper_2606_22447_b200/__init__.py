"""paper_2606_22447_b200 — B200-native batched Atari 2600 VCS (hard-mode vcs_step hot path).

The product is libvcsb200.so (CUDA, sm_100a) behind include/vcs.h; this package is its thin binding."""
from .binding import VCS, VcsError, REGS_DTYPE, EXPORTS, load_library, optable, issue_peak  # noqa: F401
from .ale import AleVecEnv  # noqa: F401,E402
