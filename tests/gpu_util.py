"""Helpers of the `-m gpu` parity tests: numpy <-> device marshalling and the agreement rules of
DESIGN.md ("Agreement rules").  No arithmetic of the method lives here: expected values always come
from `oracle/`, actual values always come through the C ABI (paper_2606_26547_b200.binding)."""
from __future__ import annotations

import numpy as np
import torch

from oracle import hdc_oracle as O
from workloads import gen


def dev(a: np.ndarray) -> torch.Tensor:
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def dev_bits(bits: np.ndarray, ld_words: int | None = None) -> torch.Tensor:
    """[R][D] 0/1 array -> device int32 [R][ld] packed LSB-first (interface layout)."""
    return dev(gen.pack_bits_lsb(bits, ld_words).view(np.int32))


def host_bits(t: torch.Tensor, D: int) -> np.ndarray:
    """device packed int32 [R][>=W] -> [R][D] 0/1 uint8"""
    w = t.cpu().numpy().view(np.uint32)
    return O.unpack_bits(w, D)


def host_words(t: torch.Tensor) -> np.ndarray:
    return t.cpu().numpy().view(np.uint32)


def check_sign_band(bits_gpu, bits_or, acc_or, absum, F):
    """Sign after a float contraction: every differing bit must sit inside the band
    |acc| <= tau * sum|x p| with tau = 4*F*2^-24 (S4).  Returns the mismatch count."""
    diff = bits_gpu != bits_or
    n = int(diff.sum())
    if n:
        tau = 4.0 * F * 2.0 ** -24
        bad = diff & (np.abs(acc_or) > tau * absum)
        assert not bad.any(), f"{int(bad.sum())} sign mismatches outside the rounding band"
    return n


def check_scores(S_gpu, S_or, floor):
    """|s - s*| <= 1e-3 |s*| + floor (north_star: within 1e-3 relative, fp32 accumulate)."""
    err = np.abs(S_gpu.astype(np.float64) - S_or)
    tol = 1e-3 * np.abs(S_or) + floor
    assert (err <= tol).all(), f"max score error {err.max()}, worst excess {(err - tol).max()}"


def check_labels_float(lab_gpu, S_or, sim):
    """Labels identical except where the oracle's top-2 relative margin is below 1e-3."""
    lab_or, best, second = O.classify(S_or, sim)
    diff = np.nonzero(lab_gpu != lab_or)[0]
    if diff.size:
        margin = np.abs(best - second) / np.maximum(np.abs(best), 1e-30)
        assert (margin[diff] < 1e-3).all(), f"label mismatch with margin {margin[diff].max()}"
        # the GPU's choice must then be the runner-up class (score within the margin of the best)
        n = diff
        s_pick = S_or[n, lab_gpu[n]]
        assert (np.abs(s_pick - best[n]) <= 1e-3 * np.maximum(np.abs(best[n]), 1e-30)).all()
    return int(diff.size)
