"""paper_2109_05339_b200: B200-native M-TIP slicing + orientation matching (libspf).

The package is a thin binding over the C-ABI library in csrc/ (include/spf.h).  Importing the
package does not load the library; `binding.load_library()` / `SpfContext` do, and fail loudly
when libspf.so has not been built or no CUDA device is present.
"""
from .binding import (SpfContext, SpfError, SPF_OUT_COMPLEX, SPF_OUT_INTENSITY, load_library,  # noqa: F401
                      spf_plan_kernel_width, spf_plan_n_fine, spf_match_workspace_bytes, EXPORTS, LIB_PATH)
