"""B200-native CKF track finding (arxiv 2505.22822 §2) behind the C ABI of include/ckf.h."""
from .binding import CKF, TrackArrays, EventBatch, concat_events, load_library, measure_alu_peak, resolve_static, EXPORTS, LIB_PATH

__all__ = ["CKF", "TrackArrays", "EventBatch", "concat_events", "load_library", "measure_alu_peak", "resolve_static", "EXPORTS", "LIB_PATH"]
