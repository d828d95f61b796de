"""B200-native convolutional visibility gridding (arXiv 0902.0915) behind a C ABI.

`binding` mirrors include/mwa_grid.h one to one; `Plan` is a convenience holder for a plan handle.
There is no CPU path: importing the binding without the built CUDA library raises ImportError.
"""
from .binding import *  # noqa: F401,F403
from .binding import Plan, MwaGridError, DESIGNS, EXPORTS  # noqa: F401
