"""hdc_classify_hamming_static: the entry point that allocates nothing and takes no workspace (its scratch is a fixed
`static __device__` array inside libhdc.so, include/hdc.h).  Checked against hdc_classify -- same labels, best and
runner-up distances bit for bit (integer path) -- and against the oracle, on calls in a row that leave stale contents
of different shapes in the shared array.  Collected last on purpose (file name): the suite runs with pytest -x."""
from __future__ import annotations

import numpy as np
import pytest
import torch

from oracle import hdc_oracle as O

from gpu_util import dev, dev_bits

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def hd():
    import paper_2606_26547_b200 as pkg
    return pkg


@pytest.fixture(scope="module")
def h(hd):
    hh = hd.Handle(0)
    yield hh
    hh.close()


def _case(key, N, K, D):
    r = np.random.default_rng([977, key])
    hb = r.integers(0, 2, size=(N, D), dtype=np.uint8)
    C = (r.standard_normal((K, D)) * 30).astype(np.float32)
    C[r.random((K, D)) < 0.03] = 0.0                       # sgn(0) = +1
    if K > 2:
        C[2] = C[1]                                        # exact tie -> lowest index
    return hb, C


def test_static_scratch_classify_equals_hdc_classify_on_calls_in_a_row(hd, h):
    # (N, K, D, D_eff, perforation): the second call is smaller than the first (stale class bits and a stale mask stay
    # behind it in the array), the third larger again and unperforated, the fourth repeats the second
    calls = [(700, 26, 10000, 10000, (3, 8)), (333, 6, 2100, 2049, (0, 1)), (1500, 64, 4099, 4099, (0, 1)),
             (333, 6, 2100, 2049, (0, 1)), (257, 10, 10000, 8400, (5, 2))]
    for i, (N, K, D, D_eff, perf) in enumerate(calls):
        hb, C = _case(i, N, K, D)
        kn = hd.knobs(D_eff, hv_bits=1, sim=hd.HDC_SIM_HAMMING, perf_begin=perf[0], perf_stride=perf[1])
        Hd, Cd = dev_bits(hb), dev(C)
        lab0, best0, sec0 = h.hdc_classify(Hd, Cd, kn, want_scores=True)
        lab = torch.full((N,), -1, dtype=torch.int32, device="cuda")
        best = torch.full((N,), -1.0, dtype=torch.float32, device="cuda")
        sec = torch.full((N,), -1.0, dtype=torch.float32, device="cuda")
        h.hdc_classify_hamming_static(Hd, Cd, kn, want_scores=True, labels=lab, best=best, second=sec)
        assert torch.equal(lab, lab0) and torch.equal(best, best0) and torch.equal(sec, sec0), i
        S_or = O.similarity(hb, C, D_eff, O.SIM_HAMMING, 1, perf[0], perf[1])
        lab_or, best_or, sec_or = O.classify(S_or, O.SIM_HAMMING)
        assert np.array_equal(lab.cpu().numpy(), lab_or), i
        assert np.array_equal(best.cpu().numpy(), best_or.astype(np.float32)), i
        assert np.array_equal(sec.cpu().numpy(), sec_or.astype(np.float32)), i


def test_static_scratch_call_allocates_nothing_and_rejects_what_does_not_fit(hd, h):
    N, K, D = 400, 10, 4096
    hb, C = _case(100, N, K, D)
    kn = hd.knobs(D, hv_bits=1, sim=hd.HDC_SIM_HAMMING)
    Hd, Cd = dev_bits(hb), dev(C)
    lab = torch.empty(N, dtype=torch.int32, device="cuda")
    ref = h.hdc_classify(Hd, Cd, kn)
    h.hdc_classify_hamming_static(Hd, Cd, kn, labels=lab)          # (first use of these kernels loads their modules)
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    alloc0 = torch.cuda.memory_allocated()
    for _ in range(3):
        h.hdc_classify_hamming_static(Hd, Cd, kn, labels=lab)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0 and torch.cuda.memory_allocated() == alloc0
    assert torch.equal(lab, ref)
    # beyond the stated limits: K > 64, (K + 1) * W * 4 > 1 MiB, another similarity / class width
    l0 = h.launch_count()
    big = torch.zeros((65, 64), dtype=torch.float32, device="cuda")
    Hs = torch.zeros((4, 2), dtype=torch.int32, device="cuda")
    with pytest.raises(hd.HdcError) as e:
        h.hdc_classify_hamming_static(Hs, big, hd.knobs(64, hv_bits=1, sim=hd.HDC_SIM_HAMMING))
    assert e.value.code == hd.HDC_ERR_UNSUPPORTED
    wide = torch.zeros((40, 262144), dtype=torch.float32, device="cuda")     # 41 * 8192 words * 4 B > 1 MiB
    Hw = torch.zeros((4, 8192), dtype=torch.int32, device="cuda")
    with pytest.raises(hd.HdcError) as e:
        h.hdc_classify_hamming_static(Hw, wide, hd.knobs(262144, hv_bits=1, sim=hd.HDC_SIM_HAMMING))
    assert e.value.code == hd.HDC_ERR_UNSUPPORTED and "HDC_STATIC_SCRATCH_BYTES" in str(e.value)
    with pytest.raises(hd.HdcError) as e:
        h.hdc_classify_hamming_static(Hd, Cd, hd.knobs(D, hv_bits=8, sim=hd.HDC_SIM_COS))
    assert e.value.code == hd.HDC_ERR_INVALID_ARG
    assert h.launch_count() == l0                                              # nothing was launched
    # a second handle on the same device shares the array; one call after the other is fine
    h2 = hd.Handle(0)
    assert torch.equal(h2.hdc_classify_hamming_static(Hd, Cd, kn), ref)
    h2.close()
