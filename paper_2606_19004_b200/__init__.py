"""B200-native SPOTLIGHT seed-exploration rollout: Python binding over libspot.so.

The product is the C-ABI library (include/spot.h); this package only marshals arguments.
"""
from .binding import *  # noqa: F401,F403
from .binding import Context, Planner, SpotError, load_library, library_path  # noqa: F401
