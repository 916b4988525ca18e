"""-m gpu: BASELINE.json configs 2-5 at their FULL sizes, in the launch configuration bench.py times
(one closure_sample launch per instance, closure_sample_batch for C5), checked on sampled walkers
the oracle replays one by one (Philox is keyed by the walker id, so any walker can be replayed alone).

Protocol as in tests/gpu_common.py: final sample within 1e-9 relative and identical on_boundary flag;
a sampled walker that differs is replayed on the GPU alone with the decision trace (bit-identical to
its run inside the full launch) and must then fall under the near-tie exemption (oracle decision slack
< 1e-9 at the first differing decision); anything else fails.  Properties that hold at any size are
checked on the whole output: every flag is 0/1, every rotation block is orthonormal, and a strided
subset of the emitted poses passes the oracle's own PURSE test.
"""
import numpy as np
import pytest

import oracle
from paper_2403_09990_b200 import binding as B
from paper_2403_09990_b200 import instances as I
from tests.gpu_common import RTOL, TIE

pytestmark = pytest.mark.gpu

SEED = 42
N_SAMPLED = 512          # oracle-replayed walkers per config (0.7 - 2 s of oracle time on 16 cores each)


def _check_sampled(inst, S0, seed, ids, g_smp, g_flag, handle):
    """Oracle replay of walkers `ids`; g_smp/g_flag are the GPU's rows for those ids."""
    import torch
    P, S = inst.params, inst.num_steps
    o_smp, o_flag, o_tr, o_sl = oracle.walk(inst, P, S0, ids, S, seed, trace=True, n_threads=16)
    near_tie = 0
    for q, w in enumerate(ids):
        ok = g_flag[q] == o_flag[q] and np.all(np.abs(g_smp[q] - o_smp[q]) <= RTOL * np.abs(o_smp[q]) + 1e-13)
        if ok:
            continue
        smp1, flag1, tr1 = handle.closure_sample(1, S, seed, walker_begin=int(w), trace=True)
        torch.cuda.synchronize()
        assert np.array_equal(smp1.cpu().numpy()[0], g_smp[q]), f"walker {w}: replay differs from the full launch"
        tr1 = tr1.cpu().numpy()[0]
        diff = np.nonzero(tr1 != o_tr[q])[0]
        assert diff.size > 0, f"walker {w}: same decisions but a different sample"
        first = int(diff[0])
        assert o_sl[q, first] < TIE, (f"walker {w}: decision differs at iteration {first + 1} with oracle slack "
                                      f"{o_sl[q, first]:.3e}")
        near_tie += 1
    assert near_tie <= max(1, len(ids) // 20), f"{near_tie} of {len(ids)} sampled walkers diverged by near-ties"


def _check_global(inst, smp, flag):
    assert np.all((flag == 0) | (flag == 1))
    R = smp[:, :9].reshape(-1, 3, 3)
    err = np.abs(np.einsum("nij,nkj->nik", R, R) - np.eye(3)).max()
    assert err < 1e-11, f"rotation blocks drifted from orthonormal by {err:.2e}"
    assert np.all(np.isfinite(smp))
    for s in smp[:: max(1, smp.shape[0] // 256)]:
        assert oracle.margin(inst, s[:9], s[9:]) >= -1e-12      # still in S
    assert flag.mean() > 0.9


@pytest.mark.parametrize("config", [2, 3, 4])
def test_single_instance_configs_full_size(config):
    import torch
    inst = I.make_instance(config)
    S0 = I.make_init_poses(inst, 128)
    W, S = inst.num_walkers, inst.num_steps
    h = B.Closure.closure_create(inst)
    try:
        h.closure_set_init(S0)
        smp, flag = h.closure_sample(W, S, SEED)
        torch.cuda.synchronize()
        smp, flag = smp.cpu().numpy(), flag.cpu().numpy()
        rng = np.random.default_rng(config)
        ids = np.unique(np.concatenate([[0, 127, 128, W - 1], rng.integers(0, W, N_SAMPLED)]))
        _check_sampled(inst, S0, SEED, ids, smp[ids], flag[ids], h)
        _check_global(inst, smp, flag)
    finally:
        h.closure_destroy()


def test_c5_batch_of_64_instances_full_size():
    """Config 5: 64 independent instances x 65,536 walkers x 2,000 iterations in the batch launch."""
    import torch
    nb = I.make_instance(5).batch
    insts = [I.make_instance(5, b) for b in range(nb)]
    S0s = [I.make_init_poses(it, 128) for it in insts]
    W, S = insts[0].num_walkers, insts[0].num_steps
    hs = []
    try:
        for it, s0 in zip(insts, S0s):
            h = B.Closure.closure_create(it)
            h.closure_set_init(s0)
            hs.append(h)
        seeds = [SEED + 1000 * b for b in range(nb)]
        smp, flag = B.closure_sample_batch(hs, W, S, seeds)
        torch.cuda.synchronize()
        rng = np.random.default_rng(5)
        for b in (0, 9, 17, 26, 35, 44, 53, nb - 1):          # 8 instances x 64 + 2 walkers
            s_b, f_b = smp[b].cpu().numpy(), flag[b].cpu().numpy()
            ids = np.unique(np.concatenate([[0, W - 1], rng.integers(0, W, 64)]))
            _check_sampled(insts[b], S0s[b], seeds[b], ids, s_b[ids], f_b[ids], hs[b])
            _check_global(insts[b], s_b, f_b)
    finally:
        for h in hs:
            h.closure_destroy()


@pytest.mark.parametrize("config,walkers,steps", [(1, 65536, 200), (2, 65536, 400), (3, 65536, 400), (4, 65536, 400),
                                                  (5, 65536, 400)])
def test_certified_kernels_equal_plain_fp64_kernel_at_scale(config, walkers, steps):
    """The certificates of the cooperative kernels under load: ~2.6e7 walker-iterations per config, every sample
    and flag bit-identical to the one-walker-per-thread fp64 kernel (CLOSURE_FLAG_EXACT_ONLY).  One wrong
    certificate anywhere (a ranking accepted although fp64 ranks differently, a candidate classified against
    fp64) sends that walker down another path and shows up here."""
    import copy
    import torch
    inst = I.make_instance(config)
    S0 = I.make_init_poses(inst, 128)
    out = []
    for flags in (0, 1):
        P = copy.copy(inst.params)
        P.flags = flags
        h = B.Closure.closure_create(inst, P)
        try:
            h.closure_set_init(S0)
            smp, flag = h.closure_sample(walkers, steps, 2024 + config)
            torch.cuda.synchronize()
            out.append((smp.cpu().numpy(), flag.cpu().numpy()))
        finally:
            h.closure_destroy()
    assert np.array_equal(out[0][1], out[1][1])
    diff = np.nonzero((out[0][0] != out[1][0]).any(axis=1))[0]
    assert diff.size == 0, f"{diff.size} walkers differ from the fp64 kernel, first {diff[:5]}"
