"""Helpers of the -m gpu parity tests: run the CUDA path through the C ABI binding, run the
oracle on the same seeded inputs, and apply DESIGN.md's parity protocol."""
import numpy as np

import oracle
from paper_2403_09990_b200 import binding as B

RTOL = 1e-9          # north_star: 1e-9 relative error in every sample coordinate / MEGB radius
TIE = 1e-9           # decisions may differ only where the oracle's decision slack is below this


def gpu_walk(inst, P, S0, num_walkers, steps, seed, *, walker_begin=0, trace=True):
    import torch
    h = B.Closure.closure_create(inst, P)
    try:
        if any(getattr(P, "pivot", (0.0, 0.0, 0.0))):
            h.closure_set_pivot(P.pivot)
        h.closure_set_init(S0)
        out = h.closure_sample(num_walkers, steps, seed, walker_begin=walker_begin, trace=trace)
        torch.cuda.synchronize()
        res = [o.cpu().numpy() for o in out]
    finally:
        h.closure_destroy()
    return res


def assert_parity(inst, P, S0, num_walkers, steps, seed, *, walker_ids=None, gpu=None, min_ok=0.98,
                  n_threads=8):
    """GPU vs oracle, walker by walker.  Returns (n_compared, n_near_tie_diverged)."""
    if gpu is None:
        gpu = gpu_walk(inst, P, S0, num_walkers, steps, seed)
    g_smp, g_flag, g_tr = gpu
    ids = np.arange(num_walkers) if walker_ids is None else np.asarray(walker_ids)
    o_smp, o_flag, o_tr, o_sl = oracle.walk(inst, P, S0, ids, steps, seed, trace=True, n_threads=n_threads)
    diverged = 0
    for q, w in enumerate(ids):
        gt = g_tr[w]
        if not np.array_equal(gt, o_tr[q]):
            first = int(np.argmax(gt != o_tr[q]))
            assert o_sl[q, first] < TIE, (
                f"walker {w}: decision differs at iteration {first + 1} (gpu {gt[first]:#x}, oracle "
                f"{o_tr[q, first]:#x}) with oracle slack {o_sl[q, first]:.3e} >= {TIE}")
            diverged += 1
            continue
        assert g_flag[w] == o_flag[q], f"walker {w}: on_boundary differs"
        err = np.abs(g_smp[w] - o_smp[q])
        tol = RTOL * np.abs(o_smp[q]) + 1e-13
        assert np.all(err <= tol), f"walker {w}: sample differs by {err.max():.3e}"
    assert diverged <= (1.0 - min_ok) * len(ids), f"{diverged} of {len(ids)} walkers diverged by near-ties"
    return len(ids), diverged
