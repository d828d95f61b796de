"""B200-native convolutional visibility gridding (arXiv 0902.0915) behind a C ABI.

`binding` mirrors include/mwa_grid.h one to one; `Plan` is a convenience holder for a plan handle.
There is no CPU path.  Importing the package builds the CUDA library in-tree when it is missing or older
than its sources (nvcc, sm_100a only - `_build.py`); if that fails the import fails: nothing here works
without the built library.
"""
from . import _build

try:
    _build.build()
except Exception as _e:  # no nvcc, compile error, ...
    raise ImportError(f"{_build.LIB} could not be built ({_e!r}); there is no CPU fallback") from _e

from .binding import *  # noqa: F401,F403,E402
from .binding import Plan, MwaGridError, DESIGNS, EXPORTS  # noqa: F401,E402
