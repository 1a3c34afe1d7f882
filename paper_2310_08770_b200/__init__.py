"""B200-native (sm_100a) hot path of the real-time cross-correlation tracker
of arxiv 2310.08770: a C-ABI CUDA library (``include/cc.h``) and this thin
binding.  See DESIGN.md."""
from .binding import CC_U8, CC_U16, CcError, Plan, RtSession, drift_correct, fp32_peak_probe, fp32_tile_probe, load_library, tc_gemm_probe  # noqa: F401
