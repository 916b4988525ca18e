"""-m gpu: randomised comparison of the certified kernels with the plain fp64 kernel (CLOSURE_FLAG_EXACT_ONLY).

Random config, instance, walk parameters, |S_0|, mode and seed per run; samples and flags must agree bit for bit.
(The same loop ran for 15 minutes twice in round 1, the second time on the final build with random bound runs and
body pivots as below: 8,349 + 8,080 runs, 68 M + 66 M walkers, and for 10 minutes on the last build of the round: 9,720
runs; no mismatch -- DESIGN.md 8.  Round 2 added streams 3 and 4 for the branch-and-bound kernel, N_P <= 32, and stream 5 for
the ellipsoid / ellipse norms, and ran the loop again on the final build; after the last two changes of the
translation sampler a loop of the same kind over config 3 in TRANS mode alone ran for 8 + 9 minutes: 14,340 + 16,119 runs.)"""
import copy

import numpy as np
import pytest

from paper_2403_09990_b200 import instances as I
from tests.gpu_common import gpu_walk

pytestmark = pytest.mark.gpu


def _n_p_choices(stream):
    # streams 3 and 4: N_P <= 32, the branch-and-bound kernel (best-first on one run of equal bounds, batched otherwise)
    if stream == 5:
        return [3, 20, 32, 33, 64, 150, 200]
    return [1, 3, 8, 20, 27, 32] if stream >= 3 else [20, 33, 64, 100, 150, 160, 200, 256]


@pytest.mark.parametrize("stream", [0, 1, 2, 3, 4, 5])
def test_random_parameters_bit_identical_to_plain_kernel(stream):
    rng = np.random.default_rng(1000 + stream)
    for _ in range(12):
        # stream 5: the ellipsoid / ellipse norms of eq. (6) (CLOSURE_REG_3D3D_ELL, CLOSURE_REPROJ_2D3D_ELL) on their certified kernels
        cfg = int(rng.choice([1, 2, 3, 5])) if stream == 5 else int(rng.integers(1, 6))
        inst = I.make_instance(cfg, int(rng.integers(0, 50)))
        if cfg == 4 and rng.random() < 0.3:
            inst = I.to_split(inst)
        P = copy.copy(inst.params)
        P.n_p = int(rng.choice(_n_p_choices(stream)))
        P.n_p_star = int(min(P.n_p, rng.choice([1, 2, 5, 10, 16, 20])))
        P.n_t = int(rng.choice([1, 5, 10, 15, 17, 40]))
        P.t_p = float(P.t_p * rng.choice([0.1, 0.5, 1.0, 2.0]))
        P.omega0 = float(P.omega0 * rng.choice([0.2, 1.0, 3.0]))
        P.gamma = float(rng.choice([0.3, 0.5, 0.8]))
        if cfg == 3 and rng.random() < 0.4:
            P.mode = I.MODE_TRANS
            P.theta_p = float(rng.choice([0.02, 0.1, 0.2, 0.35]))
            P.v0 = float(rng.choice([0.01, 0.05, 0.3, 2.0]))
            P.flags = int(rng.choice([0, 64]))
        if cfg in (1, 2, 5) and rng.random() < 0.5:          # several runs of equal bounds, odd lengths
            k = int(rng.integers(1, 5))
            inst.betas = inst.betas * rng.choice([1.0, 1.2, 1.5, 1.9][:k], size=inst.n)
        if stream == 5:
            inst = I.to_ellipsoidal(inst, int(rng.integers(0, 100)))
        if P.mode != I.MODE_TRANS and cfg in (1, 2, 3, 5) and rng.random() < 0.3:
            P.pivot = tuple(float(x) for x in rng.uniform(-0.5, 0.5, 3))      # closure_set_pivot (gpu_walk applies it)
        S0 = I.make_init_poses(inst, int(rng.choice([1, 16, 128])))
        # 1,024 walkers: the dense kernel's two-warps-per-walker form (launches of at most 1,184 walkers); 2,048: one warp per walker
        W, S, seed = int(rng.choice([1024, 2048])), int(rng.choice([50, 150])), int(rng.integers(0, 1 << 40))
        a = gpu_walk(inst, P, S0, W, S, seed, trace=False)
        b = gpu_walk(inst, copy.copy(P).__class__(**{**vars(P), "flags": P.flags | 1}), S0, W, S, seed, trace=False)
        assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1]), (cfg, inst.name, vars(P), S0.shape[0], S, seed)
