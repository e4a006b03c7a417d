"""B200-native FARM mapping hot path (arxiv/paper_2606_15476): C-ABI library + thin binding.

    from paper_2606_15476_b200 import FarmMap          # binding of include/farm.h
    from paper_2606_15476_b200 import scenes           # seeded synthetic inputs (no method arithmetic)
"""
from . import scenes  # noqa: F401
from .binding import FarmMap, FarmError, load_library  # noqa: F401
