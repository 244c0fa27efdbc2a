"""cfgms — B200-native (sm_100a) CFG multi-stream audio decode head.

The product is the C-ABI library `libcfgms.so` (include/cfgms.h, sources under csrc/); this
package is its thin Python binding.  Build it in-tree with `python -m paper_2607_02119_b200.build`.
"""
from .binding import (CFGMS_BF16, CFGMS_ERR_LIMIT, CFGMS_F32, CFGMS_STATIC_SCRATCH_BYTES, CfgmsError, Context, EXPORTS,
                      LIB_PATH, deinterleave_host_static, library, version)

__all__ = ["Context", "CfgmsError", "library", "version", "EXPORTS", "LIB_PATH", "CFGMS_BF16", "CFGMS_F32",
           "deinterleave_host_static", "CFGMS_ERR_LIMIT", "CFGMS_STATIC_SCRATCH_BYTES"]
