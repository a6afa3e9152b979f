"""B200-native TPC sector tracker (arxiv 1709.00618, section 2): C-ABI CUDA library + thin Python binding."""
from .tracker import Tracker, TrackResult, TpcError, load_library, LIB_PATH  # noqa: F401
