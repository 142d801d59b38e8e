"""B200-native LO event reweighting hot path (arXiv 2312.07440, eq. 3)."""
from . import events  # noqa: F401
