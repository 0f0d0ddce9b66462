"""B200-native HDC hot path of arxiv/paper_2606_26547 (ApproxHDC): encode -> similarity -> argmax /
class update, as hand-written CUDA for sm_100a behind the C ABI of include/hdc.h.

`binding` is a thin ctypes layer over lib/libhdc.so (built by `python -m paper_2606_26547_b200.build`).
"""
from .binding import *  # noqa: F401,F403
from .binding import Handle, HdcError, Model, hdc_adc_t, hdc_knobs_t, hdc_model_t, knobs, lib  # noqa: F401
