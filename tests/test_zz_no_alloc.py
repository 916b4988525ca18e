"""-m gpu: closure_compact_static, the no-allocation variant of the compaction (include/closure.h), against the
existing path closure_compact -- bit for bit, as for every other compaction test (integer / byte / index work),
on two calls in a row (the static scratch keeps the first call's contents and must be cleared by the second).

In a file of its own that pytest collects last: the suite runs with `pytest -x`, so a failure here hides nothing.
Passes alone in a fresh process (the first call on the device resolves the scratch's address) and after the other tests."""
import numpy as np
import pytest

from paper_2403_09990_b200 import binding as B
from paper_2403_09990_b200 import instances as I

pytestmark = pytest.mark.gpu


def _both(h, smp, flg):
    import torch
    n = int(flg.shape[0])
    ref_out, ref_cnt = h.closure_compact(smp, flg)
    out = torch.full((max(n, 1), 12), -7.0, dtype=torch.float64, device=smp.device)   # caller-allocated outputs
    cnt = torch.full((1,), -1, dtype=torch.int64, device=smp.device)
    B.closure_compact_static(smp, flg, out, cnt)
    torch.cuda.synchronize()
    c = int(cnt.item())
    assert c == int(ref_cnt.item()) == int((flg != 0).sum().item())
    assert np.array_equal(out[:c].cpu().numpy(), ref_out[:c].cpu().numpy())
    assert bool((out[c:] == -7.0).all())                      # nothing written past the kept records
    return c


def test_static_compaction_equals_existing_path_on_two_calls_in_a_row():
    import torch
    inst = I.make_instance(1)
    h = B.Closure.closure_create(inst)
    try:
        g = torch.Generator(device="cuda").manual_seed(5)
        # first call: many tiles and a ragged tail, about 70 % kept
        n1 = 300001
        smp1 = torch.rand((n1, 12), dtype=torch.float64, device="cuda", generator=g)
        flg1 = (torch.rand((n1,), device="cuda", generator=g) < 0.7).to(torch.uint8) * 3      # any non-zero byte keeps
        c1 = _both(h, smp1, flg1)
        assert 0 < c1 < n1
        # second call straight after it: fewer tiles than the first left behind, other flags, every record of some tiles kept
        n2 = 6145
        smp2 = torch.rand((n2, 12), dtype=torch.float64, device="cuda", generator=g)
        flg2 = torch.ones((n2,), dtype=torch.uint8, device="cuda")
        flg2[2048:4096:3] = 0
        c2 = _both(h, smp2, flg2)
        assert c2 == n2 - len(range(2048, 4096, 3))
        # and the first input again: same result as before
        assert _both(h, smp1, flg1) == c1
        # edge sizes
        for n in (0, 1, 2047, 2048, 2049):
            s = torch.rand((max(n, 1), 12), dtype=torch.float64, device="cuda", generator=g)[:n]
            f = (torch.rand((n,), device="cuda", generator=g) < 0.5).to(torch.uint8)
            _both(h, s, f)
    finally:
        h.closure_destroy()


def test_static_compaction_rejects_sizes_beyond_its_scratch():
    import torch
    n = B.COMPACT_STATIC_MAX + 1
    flg = torch.zeros((n,), dtype=torch.uint8, device="cuda")
    dummy = torch.zeros((1, 12), dtype=torch.float64, device="cuda")       # never dereferenced: rejected before any launch
    cnt = torch.full((1,), -1, dtype=torch.int64, device="cuda")
    with pytest.raises(B.ClosureError) as e:
        B.closure_compact_static(dummy, flg, dummy, cnt)
    assert e.value.status == B.ETOOLARGE and "CLOSURE_COMPACT_STATIC_MAX" in str(e.value)
    torch.cuda.synchronize()
    assert int(cnt.item()) == -1
