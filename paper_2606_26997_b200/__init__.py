"""B200 (sm_100a) fused GRPO policy-loss step behind a C ABI (include/grpo.h).

The product is libgrpo_b200.so (hand-written CUDA: tcgen05 / TMEM / TMA); this package is a thin
ctypes binding.  Importing the package does not load the library; using it without the built
library raises (no CPU / PyTorch fallback exists).
"""
from .binding import (GrpoConfig, GrpoContext, GrpoError, GroupDesc, EXPORTS, grpo_cgp_plan,  # noqa: F401
                      grpo_loss_from_partials_static, load_library)
from .build import build, LIB_PATH  # noqa: F401
