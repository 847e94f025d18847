"""crownb200: B200-native IBP / CROWN / alpha-CROWN bound propagation (C-ABI library + thin binding)."""
from .binding import CrownContext, CrownError, load_library, gemm_noalloc, LIB_PATH, EXPORTS  # noqa: F401
