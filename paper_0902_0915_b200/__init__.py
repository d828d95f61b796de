"""B200-native convolutional visibility gridding (arXiv 0902.0915) behind a C ABI.

`binding` mirrors include/mwa_grid.h one to one; `Plan` is a convenience holder for a plan handle.
There is no CPU path.  Without the built CUDA library only `_build` (the nvcc build step) is importable;
touching anything else raises ImportError.
"""
import os as _os

from . import _build

if _os.path.exists(_build.LIB) and not _build.needs_build():
    from .binding import *  # noqa: F401,F403
    from .binding import Plan, MwaGridError, DESIGNS, EXPORTS  # noqa: F401
else:
    def __getattr__(name):
        if _os.path.exists(_build.LIB) and not _build.needs_build():      # built since the package was imported
            from . import binding
            globals().update({k: getattr(binding, k) for k in dir(binding) if not k.startswith("__")})
            return globals()[name]
        raise ImportError(f"{_build.LIB} is missing or older than its sources: the CUDA library has not been built "
                          "(run `python -m paper_0902_0915_b200._build`); there is no CPU fallback")
