"""CPU oracle (test infrastructure only -- see hdc_oracle.py header)."""
from . import hdc_oracle  # noqa: F401
