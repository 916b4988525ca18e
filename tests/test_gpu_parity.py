"""-m gpu: the CUDA walker kernel against the oracle, through the C ABI.

Protocol: identical per-iteration decisions (m_0, j_{k_0}) and on_boundary
flags, final samples within 1e-9 relative, except walkers whose first differing decision has an
oracle decision slack below 1e-9 (excluded, counted, bounded).
"""
import copy

import numpy as np
import pytest

from paper_2403_09990_b200 import binding as B
from paper_2403_09990_b200 import instances as I
from tests.gpu_common import assert_parity, gpu_walk

pytestmark = pytest.mark.gpu


def _small(P, **kw):
    P = copy.copy(P)
    for k, v in kw.items():
        setattr(P, k, v)
    return P


def test_c1_full_size_every_walker():
    """BASELINE config 1 at its full size: 1024 walkers x 200 iterations, all compared."""
    inst = I.make_instance(1)
    S0 = I.make_init_poses(inst, 128)
    n, div = assert_parity(inst, inst.params, S0, inst.num_walkers, inst.num_steps, 42)
    assert n == 1024


@pytest.mark.parametrize("config,walkers,steps", [(2, 384, 60), (3, 300, 60), (4, 300, 60), (5, 515, 120)])
def test_configs_reduced(config, walkers, steps):
    """Configs 2-5 with every walker compared; sizes span several CTAs and a ragged tail."""
    inst = I.make_instance(config)
    S0 = I.make_init_poses(inst, 128)
    assert_parity(inst, inst.params, S0, walkers, steps, 42)


def test_c3_translation_boundary_sampler():
    """Alg. A8 (TRANS mode) on the reprojection residual: C3's second number."""
    inst = I.make_instance(3)
    P = _small(inst.params, mode=I.MODE_TRANS, v0=0.05, theta_p=0.02, n_p=40, n_p_star=5, n_t=10)
    assert_parity(inst, P, I.make_init_poses(inst, 64), 200, 40, 7)


@pytest.mark.parametrize("kind", ["reg", "posereg", "split"])
def test_translation_boundary_sampler_other_residuals(kind):
    if kind == "reg":
        inst = I.make_instance(1)
        P = _small(inst.params, mode=I.MODE_TRANS, v0=0.1, theta_p=0.02, n_p=30, n_p_star=4, n_t=8)
    else:
        inst = I.make_instance(4)
        if kind == "split":
            inst = I.to_split(inst)
        P = _small(inst.params, mode=I.MODE_TRANS, v0=0.02, theta_p=0.02, n_p=20, n_p_star=3, n_t=8)
    assert_parity(inst, P, I.make_init_poses(inst, 32), 160, 30, 11)


def test_split_pose_regression_rot_mode():
    inst = I.to_split(I.make_instance(4))
    assert_parity(inst, inst.params, I.make_init_poses(inst, 64), 260, 50, 3)


@pytest.mark.parametrize("n_p,n_p_star,n_t", [(1, 1, 1), (7, 1, 3), (37, 3, 5), (150, 10, 15), (23, 15, 4),
                                              (64, 20, 6), (10, 10, 2), (40, 4, 33), (33, 2, 64), (200, 10, 8),
                                              (256, 20, 17), (300, 5, 6)])
def test_parameter_edges(n_p, n_p_star, n_t):
    """Ragged perturbation tiles, every top-k capacity, degenerate N_P = N_P* = N_T = 1, ladders longer than one
    screening block (N_T > 16), every NQ of the cooperative kernel, and N_P > 256 (plain kernel)."""
    inst = I.make_instance(1)
    P = _small(inst.params, n_p=n_p, n_p_star=n_p_star, n_t=n_t)
    assert_parity(inst, P, I.make_init_poses(inst, 16), 130, 25, 5)


@pytest.mark.parametrize("n,distinct", [(1, False), (2, True), (7, True), (33, True), (200, False), (1500, False)])
def test_constraint_count_edges(n, distinct):
    """N = 1, odd N, every beta different (one sqrt per constraint), the maximum config size, and an N whose
    per-warp tables do not fit the cooperative kernel (the one-walker-per-thread kernel takes over)."""
    inst = I.make_custom_reg(n, 100 + n, distinct_betas=distinct)
    P = _small(inst.params, n_p=30, n_p_star=4, n_t=8, t_p=0.05)
    assert_parity(inst, P, I.make_init_poses(inst, 8), 96, 20, 9)


def _three_bounds(n, seed, counts):
    inst = I.make_custom_reg(n, seed)
    scale = np.concatenate([np.full(c, f) for c, f in zip(counts, (1.0, 1.25, 1.6))])
    inst.betas = inst.betas * np.random.default_rng(seed).permutation(scale)
    return inst


@pytest.mark.parametrize("n,counts,n_p", [(200, (51, 67, 82), 24), (200, None, 20), (300, (1, 290, 9), 32), (130, (129, 1, 0), 9)])
def test_constraint_major_loop_with_several_runs(n, counts, n_p):
    """N_P <= 32 with a long table: the constraint-major eq. (14) loop, on runs of odd length, a run longer than 128
    pair-entries (the perturbation-major loop takes over), runs of one constraint, and every bound different."""
    inst = _three_bounds(n, 300 + n, counts) if counts else I.make_custom_reg(n, 300 + n, distinct_betas=True)
    P = _small(inst.params, n_p=n_p, n_p_star=3, n_t=6, t_p=0.05)
    S0 = I.make_init_poses(inst, 8)
    assert_parity(inst, P, S0, 64, 16, 11)
    fast = gpu_walk(inst, P, S0, 2048, 60, 77)
    plain = gpu_walk(inst, _small(P, flags=1), S0, 2048, 60, 77)
    for a, b in zip(fast, plain):
        assert np.array_equal(a, b)


def test_batch_members_with_different_tables():
    """closure_sample_batch over instances whose fp32 tables differ in size and run structure: the launch sizes
    shared memory for the largest, every member equals its own single-instance launch bit for bit."""
    import torch
    insts = [I.make_custom_reg(200, 41), _three_bounds(120, 42, (31, 40, 49)), I.make_custom_reg(9, 43, distinct_betas=True)]
    P = _small(insts[0].params, n_p=20, n_p_star=2, n_t=5, t_p=0.05)
    hs, single = [], []
    try:
        for it in insts:
            h = B.Closure.closure_create(it, P)
            h.closure_set_init(I.make_init_poses(it, 8))
            hs.append(h)
        smp, flag = B.closure_sample_batch(hs, 512, 40, [5, 6, 7])
        torch.cuda.synchronize()
        for b, h in enumerate(hs):
            s1, f1 = h.closure_sample(512, 40, 5 + b)
            torch.cuda.synchronize()
            assert np.array_equal(s1.cpu().numpy(), smp[b].cpu().numpy())
            assert np.array_equal(f1.cpu().numpy(), flag[b].cpu().numpy())
    finally:
        for h in hs:
            h.closure_destroy()


FLAG_ONE_WARP = 128      # CLOSURE_FLAG_ONE_WARP (include/closure.h)


@pytest.mark.parametrize("config,walkers,steps,extra", [
    (1, 1024, 200, {}),                        # BASELINE config 1 at full size
    (1, 1, 30, {}), (1, 3, 30, {}), (2, 5, 1, {}), (2, 7, 2, {}),          # partly filled CTAs, one and two iterations
    (2, 1184, 40, {}), (2, 1185, 40, {}),      # the largest launch on the two-warp kernel, the first one on the one-warp kernel
    (4, 1000, 120, {}),                        # pose regression
    (2, 600, 60, dict(flags=2)), (2, 600, 60, dict(flags=4)), (1, 600, 60, dict(flags=20)),      # forced fp64 fall-backs
    (2, 512, 80, dict(precision=32)),          # fp32 mode
    (2, 700, 50, dict(n_p=40, n_p_star=4, n_t=8)), (1, 700, 50, dict(n_p=200, n_p_star=10, n_t=17)),   # NQ = 2 and 8
    (2, 400, 60, dict(omega0=2.0, t_p=0.2)),   # many accepted moves: the producer's speculation is discarded often
])
def test_two_warps_per_walker_kernel_is_bit_identical_to_one_warp_kernel(config, walkers, steps, extra):
    """Launches of at most 1,184 walkers run walker_dense_pipe_kernel (a pair of warps per walker, one iteration apart:
    DESIGN.md 6.1b); CLOSURE_FLAG_ONE_WARP keeps walker_dense_kernel.  Samples, flags and per-iteration traces must agree
    bit for bit, and with the plain fp64 kernel where that applies."""
    inst = I.make_instance(config)
    S0 = I.make_init_poses(inst, 32)
    P = _small(inst.params, **extra)
    pipe = gpu_walk(inst, P, S0, walkers, steps, 909)
    one = gpu_walk(inst, _small(P, flags=P.flags | FLAG_ONE_WARP), S0, walkers, steps, 909)
    for a, b in zip(pipe, one):
        assert np.array_equal(a, b)
    if getattr(P, "precision", 64) == 64:
        plain = gpu_walk(inst, _small(P, flags=1), S0, walkers, steps, 909)
        for a, b in zip(pipe, plain):
            assert np.array_equal(a, b)


def test_two_warps_per_walker_kernel_in_a_batch_and_on_the_ellipsoid_norm():
    """closure_sample_batch with 3 x 300 walkers in all (one launch of the two-warp kernel with blockIdx.y = instance) equals the
    members' single launches; the ellipsoid norm of Ex.2 on the two-warp kernel equals its one-warp kernel."""
    import torch
    insts = [I.make_instance(1, k) for k in range(3)]
    hs = []
    try:
        for it in insts:
            h = B.Closure.closure_create(it, it.params)
            h.closure_set_init(I.make_init_poses(it, 16))
            hs.append(h)
        smp, flag = B.closure_sample_batch(hs, 300, 60, [11, 12, 13])
        torch.cuda.synchronize()
        for b, h in enumerate(hs):
            h.closure_set_params(_small(insts[b].params, flags=FLAG_ONE_WARP))
            s1, f1 = h.closure_sample(300, 60, 11 + b)
            torch.cuda.synchronize()
            assert np.array_equal(s1.cpu().numpy(), smp[b].cpu().numpy())
            assert np.array_equal(f1.cpu().numpy(), flag[b].cpu().numpy())
    finally:
        for h in hs:
            h.closure_destroy()
    inst = I.to_ellipsoidal(I.make_instance(2), 4)
    S0 = I.make_init_poses(inst, 32)
    pipe = gpu_walk(inst, inst.params, S0, 900, 80, 31)
    one = gpu_walk(inst, _small(inst.params, flags=FLAG_ONE_WARP), S0, 900, 80, 31)
    for a, b in zip(pipe, one):
        assert np.array_equal(a, b)


@pytest.mark.parametrize("walkers", [1, 31, 127, 128, 129])
def test_walker_count_edges(walkers):
    inst = I.make_instance(1)
    P = _small(inst.params, n_p=20, n_p_star=2, n_t=6)
    assert_parity(inst, P, I.make_init_poses(inst, 5), walkers, 15, 2)


def test_single_initial_pose_and_zero_velocity():
    """|S_0| = 1 (direction term undefined -> zero, R-3) and omega_0 = 0 (pure perturbation walk)."""
    inst = I.make_instance(1)
    S0 = I.make_init_poses(inst, 1)
    assert_parity(inst, _small(inst.params, n_p=30, n_p_star=3, n_t=6), S0, 64, 20, 8)
    assert_parity(inst, _small(inst.params, omega0=0.0, n_p=30, n_p_star=3, n_t=6), S0, 64, 20, 8)


def test_zero_steps_returns_initial_poses():
    inst = I.make_instance(1)
    S0 = I.make_init_poses(inst, 16)
    smp, flag = gpu_walk(inst, inst.params, S0, 40, 0, 1, trace=False)
    assert np.array_equal(smp, S0[np.arange(40) % 16]) and not flag.any()


def test_walker_range_and_replay_are_bit_identical():
    """Philox keyed by walker id: a sub-range, a re-run and a high walker id reproduce exactly."""
    inst = I.make_instance(1)
    S0 = I.make_init_poses(inst, 32)
    P = _small(inst.params, n_p=40, n_p_star=4, n_t=8)
    full = gpu_walk(inst, P, S0, 300, 20, 77)
    again = gpu_walk(inst, P, S0, 300, 20, 77)
    part = gpu_walk(inst, P, S0, 100, 20, 77, walker_begin=150)
    for a, b in zip(full, again):
        assert np.array_equal(a, b)
    for a, b in zip(full, part):
        assert np.array_equal(a[150:250], b)
    other = gpu_walk(inst, P, S0, 300, 20, 78)
    assert not np.array_equal(full[0], other[0])
    # walker ids beyond 2^32 use the high counter word
    big = (1 << 32) + 5
    hi = gpu_walk(inst, P, S0, 4, 20, 77, walker_begin=big)
    import oracle
    o_smp, o_flag = oracle.walk(inst, P, S0, big + np.arange(4), 20, 77)
    assert np.allclose(hi[0], o_smp, rtol=1e-9, atol=1e-13)
    assert not np.array_equal(hi[0][0], full[0][5])


def test_samples_are_feasible_and_orthonormal():
    """Invariant: every emitted pose is still in S (checked with the oracle's test)."""
    import oracle
    for config in (1, 3, 4):
        inst = I.make_instance(config)
        smp, flag, _ = gpu_walk(inst, inst.params, I.make_init_poses(inst, 64), 256, 40, 21)
        for s in smp:
            assert oracle.margin(inst, s[:9], s[9:]) >= -1e-12
            R = s[:9].reshape(3, 3)
            assert np.allclose(R.T @ R, np.eye(3), atol=1e-12)
        assert flag.mean() > 0.9


@pytest.mark.parametrize("config,walkers,steps", [(2, 4096, 150), (1, 1024, 200), (4, 2048, 120), (5, 2048, 150), (3, 4096, 150)])
def test_screened_kernel_is_bit_identical_to_exact_kernel(config, walkers, steps):
    """The fp32-screened kernel takes every decision on fp64 values: outputs and traces must equal the
    plain fp64 kernel's (CLOSURE_FLAG_EXACT_ONLY) bit for bit, on far more walkers than the oracle replays."""
    inst = I.make_instance(config)
    S0 = I.make_init_poses(inst, 128)
    fast = gpu_walk(inst, inst.params, S0, walkers, steps, 4242)
    plain = gpu_walk(inst, _small(inst.params, flags=1), S0, walkers, steps, 4242)
    for a, b in zip(fast, plain):
        assert np.array_equal(a, b)


def test_screened_kernel_falls_back_on_ties():
    """t_p = 0 makes all N_P distances equal: the candidate list cannot be proven complete, the warp must
    take the exact path, and results still match the oracle."""
    inst = I.make_instance(1)
    P = _small(inst.params, t_p=0.0, n_p=40, n_p_star=4, n_t=10)
    assert_parity(inst, P, I.make_init_poses(inst, 16), 96, 20, 13)
    sp = I.to_split(I.make_instance(4))
    fast = gpu_walk(sp, sp.params, I.make_init_poses(sp, 32), 512, 60, 5)
    plain = gpu_walk(sp, _small(sp.params, flags=1), I.make_init_poses(sp, 32), 512, 60, 5)
    for a, b in zip(fast, plain):
        assert np.array_equal(a, b)


@pytest.mark.parametrize("config", [1, 3, 4])
def test_all_perturbations_kept_stays_on_the_certified_path(config):
    """N_P = N_P*: the (N_P*+1)-th extraction finds an empty slot.  It must read as -inf ("none left"), not as a
    NaN that fails the certificate: the fp32 ranking stays certified for most iterations and the results equal
    the plain fp64 kernel's."""
    inst = I.make_instance(config)
    S0 = I.make_init_poses(inst, 64)
    P = _small(inst.params, n_p=10, n_p_star=10, n_t=8)
    h = B.Closure.closure_create(inst, P)
    try:
        h.closure_set_init(S0)
        h.closure_enable_stats(True)
        h.closure_sample(512, 60, 31)
        st = h.closure_get_stats()
    finally:
        h.closure_destroy()
    assert st["walker_steps"] == 512 * 60
    assert st["fallback_steps"] < 0.25 * st["walker_steps"], st
    a = gpu_walk(inst, P, S0, 512, 60, 31)
    b = gpu_walk(inst, _small(P, flags=1), S0, 512, 60, 31)
    for x, y in zip(a, b):
        assert np.array_equal(x, y)


@pytest.mark.parametrize("flags", [2, 4, 6, 20])
@pytest.mark.parametrize("config,walkers,steps", [(2, 1024, 80), (4, 512, 80), (5, 512, 100), (3, 1024, 80)])
def test_cooperative_kernel_forced_fp64_paths(config, walkers, steps, flags):
    """Debug switches of the warp-cooperative kernel: 2 = every ladder candidate goes to the fp64 test,
    4 = every iteration takes the fp64 top-k fallback (16: on all N_P perturbations).
    All of them must reproduce the plain fp64 kernel bit for bit."""
    inst = I.make_instance(config)
    S0 = I.make_init_poses(inst, 128)
    a = gpu_walk(inst, _small(inst.params, flags=flags), S0, walkers, steps, 99)
    b = gpu_walk(inst, _small(inst.params, flags=1), S0, walkers, steps, 99)
    for x, y in zip(a, b):
        assert np.array_equal(x, y)


@pytest.mark.parametrize("config", [1, 2, 3, 4, 5])
def test_fp32_mode_measured_difference(config):
    """precision = 32 takes the decisions on the fp32 values as they are (no certificate, no fp64 fall-back).
    It may differ from the fp64 path only where an fp32 error bound straddles a threshold: most walkers
    take identical decisions (then the fp64 poses are bit-identical).  A ladder candidate the fp32 bound cannot
    decide counts as violated, so every emitted pose is inside S (Prop. 4) as on the fp64 path."""
    import oracle
    inst = I.make_instance(config)
    S0 = I.make_init_poses(inst, 128)
    W, S = 2048, 100
    f32 = gpu_walk(inst, _small(inst.params, precision=32), S0, W, S, 7)
    f64 = gpu_walk(inst, inst.params, S0, W, S, 7)
    same = (f32[2] == f64[2]).all(axis=1)
    assert same.mean() > 0.9, f"only {same.mean():.3f} of the walkers take the fp64 decisions"
    assert np.array_equal(f32[0][same], f64[0][same]) and np.array_equal(f32[1][same], f64[1][same])
    scale = float(np.max(inst.betas))
    worst = min(oracle.margin(inst, s[:9], s[9:]) for s in f32[0][::8])
    assert worst >= -1e-12 * scale, f"fp32-mode sample violates a constraint by {-worst:.3e}"


def test_fp32_mode_is_refused_where_it_does_not_exist():
    from paper_2403_09990_b200 import binding as B
    inst = I.make_instance(3)
    with pytest.raises(B.ClosureError) as e:
        B.Closure.closure_create(inst, _small(inst.params, precision=32, mode=I.MODE_TRANS, v0=0.05, theta_p=0.02))
    assert e.value.status == B.EUNSUPPORTED


@pytest.mark.parametrize("kind", ["reproj", "reg", "posereg", "split", "reproj_ell", "reg_ell"])
def test_cooperative_translation_sampler_is_bit_identical_to_plain_kernel(kind):
    """Alg. A8 on the warp-cooperative fp64 kernel against the one-walker-per-thread kernel
    (CLOSURE_FLAG_EXACT_ONLY): same fp64 functions, so samples, flags and traces must be identical."""
    if kind in ("reproj", "reproj_ell"):
        inst = I.make_instance(3)
        if kind == "reproj_ell":
            inst = I.to_ellipsoidal(inst, 1)
        P = _small(inst.params, mode=I.MODE_TRANS, v0=0.05, theta_p=0.02)
    elif kind in ("reg", "reg_ell"):
        inst = I.make_instance(2)
        if kind == "reg_ell":
            inst = I.to_ellipsoidal(inst, 1)
        P = _small(inst.params, mode=I.MODE_TRANS, v0=0.1, theta_p=0.02, n_p=70, n_p_star=7)
    else:
        inst = I.make_instance(4)
        if kind == "split":
            inst = I.to_split(inst)
        P = _small(inst.params, mode=I.MODE_TRANS, v0=0.02, theta_p=0.02, n_p=33, n_p_star=20, n_t=12)
    S0 = I.make_init_poses(inst, 64)
    a = gpu_walk(inst, P, S0, 1500, 60, 17)
    b = gpu_walk(inst, _small(P, flags=1), S0, 1500, 60, 17)
    for x, y in zip(a, b):
        assert np.array_equal(x, y)
    assert (a[2] & 0xff).max() >= 1          # some moves were accepted


@pytest.mark.parametrize("config", [3, 4])
@pytest.mark.parametrize("n_p,n_p_star,n_t", [(33, 2, 40), (200, 10, 8), (64, 20, 6), (5, 5, 1)])
def test_parameter_edges_other_residuals(config, n_p, n_p_star, n_t):
    """The same edges on the reprojection kernel and on the stacked pose-regression residual."""
    inst = I.make_instance(config)
    P = _small(inst.params, n_p=n_p, n_p_star=n_p_star, n_t=n_t)
    assert_parity(inst, P, I.make_init_poses(inst, 16), 100, 25, 5)


@pytest.mark.parametrize("flags,theta_p,v0", [(0, 0.2, 2.0), (0, 0.05, 0.02), (4, 0.2, 0.05), (20, 0.05, 0.02), (0, 0.5, 0.02),
                                              (2, 0.05, 0.02), (0, 0.02, 0.005), (0, 0.2, 0.3)])
def test_certified_translation_sampler_on_reprojection(flags, theta_p, v0):
    """Alg. A8 on the reprojection residual: eq. (14) runs in certified fp32 (series of Exp, error bound unc,
    fp64 re-ranking of near-ties).  Bit-identical to the plain fp64 kernel at the paper's theta_p = 0.2 and v0 = 2,
    at small steps where walkers keep moving, with the fp64 ranking forced (4, 20) or every ladder candidate sent
    to fp64 (2), and beyond the range of the
    series (theta_p = 0.5: the fp64 evaluation takes over)."""
    inst = I.make_instance(3)
    P = _small(inst.params, mode=I.MODE_TRANS, v0=v0, theta_p=theta_p, flags=flags)
    S0 = I.make_init_poses(inst, 128)
    a = gpu_walk(inst, P, S0, 4096, 100, 23)
    b = gpu_walk(inst, _small(P, flags=1), S0, 4096, 100, 23)
    for x, y in zip(a, b):
        assert np.array_equal(x, y)


@pytest.mark.parametrize("config,flags", [(3, 64), (3, 65), (1, 64)])
def test_pca_normalised_centre_velocity(config, flags):
    """CLOSURE_FLAG_PCA_VELOCITY (R-23): closure_set_init rescales the centre velocity by
    sqrtm(Cov(S_t0)) / sqrt(lambda_max) (host Jacobi) -- against the oracle (numpy eigh), on the cooperative and on
    the plain kernel, with an anisotropic S_0."""
    inst = I.make_instance(config)
    S0 = I.make_init_poses(inst, 64)
    S0[:, 10] = inst.t_gt[1] + (S0[:, 10] - inst.t_gt[1]) * 0.1                  # squeeze the cloud along y
    P = _small(inst.params, mode=I.MODE_TRANS, v0=0.05 if config == 3 else 0.1, theta_p=0.02, n_p=40, n_p_star=5,
               n_t=10, flags=flags)
    assert_parity(inst, P, S0, 200, 40, 7)
    # the flag changes the walk
    a = gpu_walk(inst, P, S0, 64, 10, 7)
    b = gpu_walk(inst, _small(P, flags=flags & 1), S0, 64, 10, 7)
    assert not np.array_equal(a[0], b[0])


@pytest.mark.parametrize("config,flags", [(2, 0), (2, 1), (3, 0), (1, 0)])
def test_body_pivot_of_update_rotation(config, flags):
    """closure_set_pivot (R-1): the oracle applies t' = t + (R - R')c at every rotation step, the CUDA
    path walks the problem re-centred at c and maps the output back; inputs and outputs stay in (R, t)."""
    inst = I.make_instance(config)
    P = _small(inst.params, pivot=(0.3, -0.2, 0.45), flags=flags)
    S0 = I.make_init_poses(inst, 32)
    assert_parity(inst, P, S0, 192, 30, 17)
    plain = gpu_walk(inst, _small(P, pivot=(0.0, 0.0, 0.0)), S0, 192, 30, 17)
    piv = gpu_walk(inst, P, S0, 192, 30, 17)
    assert np.abs(plain[0] - piv[0]).max() > 1e-4                       # a different walk, not a no-op


def test_body_pivot_api_edges():
    import torch
    inst = I.make_instance(2)
    S0 = I.make_init_poses(inst, 16)
    h = B.Closure.closure_create(inst)
    try:
        h.closure_set_init(S0)
        ref = [o.cpu().numpy() for o in h.closure_sample(256, 20, 3)]
        h.closure_set_pivot((0.5, 0.1, -0.3))
        with pytest.raises(B.ClosureError) as e:                        # S_0 has to be given again
            h.closure_sample(16, 2, 3)
        assert e.value.status == B.ENOINIT
        poses, ok = h.closure_init_sample(500, 4)                       # Step I does not depend on the pivot
        h.closure_set_pivot((0.0, 0.0, 0.0))
        poses0, ok0 = h.closure_init_sample(500, 4)
        torch.cuda.synchronize()
        assert np.array_equal(ok.cpu().numpy(), ok0.cpu().numpy())
        assert np.abs(poses.cpu().numpy() - poses0.cpu().numpy()).max() < 1e-12
        h.closure_set_init(S0)                                          # pivot cleared: the default walk again
        again = [o.cpu().numpy() for o in h.closure_sample(256, 20, 3)]
        assert np.array_equal(ref[0], again[0]) and np.array_equal(ref[1], again[1])
        h.closure_set_pivot((0.5, 0.1, -0.3))
        Pt = _small(inst.params, mode=I.MODE_TRANS, v0=0.05, theta_p=0.05)
        with pytest.raises(B.ClosureError) as e:                        # Alg. A8 has no update_rotation
            h.closure_set_params(Pt)
        assert e.value.status == B.EUNSUPPORTED
        with pytest.raises(B.ClosureError) as e:
            h.closure_set_pivot((np.nan, 0.0, 0.0))
        assert e.value.status == B.EINVAL
    finally:
        h.closure_destroy()
    h = B.Closure.closure_create(I.make_instance(4))
    try:
        h.closure_set_pivot((0.0, 0.0, 0.0))
        with pytest.raises(B.ClosureError) as e:                        # no source points in Ex.3
            h.closure_set_pivot((0.1, 0.0, 0.0))
        assert e.value.status == B.EUNSUPPORTED
    finally:
        h.closure_destroy()
    # batch members with different pivots; closure_run end to end
    insts = [I.make_instance(1), I.make_instance(1, 1)]
    P = _small(insts[0].params, n_p=20, n_p_star=2, n_t=5)
    hs = []
    try:
        for b, it in enumerate(insts):
            hb = B.Closure.closure_create(it, P)
            if b == 1:
                hb.closure_set_pivot((0.2, 0.2, -0.1))
            hb.closure_set_init(I.make_init_poses(it, 8))
            hs.append(hb)
        smp, flag = B.closure_sample_batch(hs, 300, 25, [8, 9])
        torch.cuda.synchronize()
        for b, hb in enumerate(hs):
            s1, f1 = hb.closure_sample(300, 25, 8 + b)
            torch.cuda.synchronize()
            assert np.array_equal(s1.cpu().numpy(), smp[b].cpu().numpy())
        res = hs[1].closure_run(1024, 30, 5)
        assert res["count"] > 900 and res["trans_radius"] > 0
    finally:
        for hb in hs:
            hb.closure_destroy()


@pytest.mark.parametrize("config,mode", [(2, "rot"), (3, "rot"), (1, "rot"), (3, "trans"), (2, "trans")])
def test_ellipsoidal_noise_bounds(config, mode):
    """Lambda_i != I (eq. (6)): ellipsoids for Ex.2, ellipses for Ex.1, both
    samplers, on the fp64 kernels."""
    inst = I.to_ellipsoidal(I.make_instance(config), 3)
    P = _small(inst.params, n_p=40, n_p_star=4, n_t=8)
    if mode == "trans":
        P = _small(P, mode=I.MODE_TRANS, v0=0.05 if config == 2 else P.v0, theta_p=0.03 if config == 2 else P.theta_p)
    S0 = I.make_init_poses(inst, 32)
    assert_parity(inst, P, S0, 160, 25, 23)
    if mode == "rot":                                                  # and with a body pivot
        assert_parity(inst, _small(P, pivot=(0.2, 0.1, -0.3)), S0, 96, 20, 24)


@pytest.mark.parametrize("flags", [0, 2, 4, 6, 20])
@pytest.mark.parametrize("config,n_p,n_p_star,n_t,walkers,steps", [(2, 150, 10, 15, 2048, 100), (1, 150, 10, 15, 1024, 120),
                                                                   (5, 20, 2, 5, 1024, 100), (2, 33, 20, 17, 512, 60)])
def test_ellipsoid_certified_kernel_is_bit_identical_to_plain_kernel(config, n_p, n_p_star, n_t, walkers, steps, flags):
    """Ex.2 with the ellipsoid norm on the certified fp32 kernel (walker_dense_kernel<REG_3D3D_ELL>: the pair carries the
    quadratic form d^T Lambda_i d): outputs and traces equal the plain fp64 kernel's bit for bit -- on a long and a short table,
    with few perturbations, a ladder longer than one screening block, and with every fp64 fall-back forced (flags 2, 4, 16)."""
    inst = I.to_ellipsoidal(I.make_instance(config), 7)
    S0 = I.make_init_poses(inst, 64)
    P = _small(inst.params, n_p=n_p, n_p_star=n_p_star, n_t=n_t)
    fast = gpu_walk(inst, _small(P, flags=flags), S0, walkers, steps, 4343)
    plain = gpu_walk(inst, _small(P, flags=1), S0, walkers, steps, 4343)
    for a, b in zip(fast, plain):
        assert np.array_equal(a, b)
    if flags == 0:                                                      # the certificates carry most iterations
        h = B.Closure.closure_create(inst, P)
        try:
            h.closure_set_init(S0)
            h.closure_enable_stats(True)
            h.closure_sample(walkers, steps, 4343)
            st = h.closure_get_stats()
        finally:
            h.closure_destroy()
        assert st["perturb_pairs_f32"] > 0 and st["fallback_steps"] < 0.2 * st["walker_steps"], st


@pytest.mark.parametrize("flags", [0, 2, 4, 6, 20])
@pytest.mark.parametrize("n,n_p,n_p_star,n_t,walkers,steps", [(8, 150, 10, 10, 2048, 100), (8, 40, 4, 8, 1024, 60),
                                                              (24, 150, 10, 17, 512, 60), (8, 20, 2, 5, 1024, 80)])
def test_ellipse_certified_reprojection_kernel_is_bit_identical_to_plain_kernel(n, n_p, n_p_star, n_t, walkers, steps, flags):
    """Ex.1 with the ellipse norm (CLOSURE_REPROJ_2D3D_ELL) on the certified fp32 kernel (walker_coop_reproj_kernel<NQ, true>:
    rows whitened by the Cholesky factor of Lambda_i): outputs and traces equal the plain fp64 kernel's bit for bit -- C3's
    table and a longer one (the set-up's loop over constraints, a ladder longer than one screening block), few
    perturbations, and every fp64 fall-back forced (flags 2, 4, 16)."""
    inst = I.to_ellipsoidal(I.make_instance(3) if n == 8 else I.make_custom_reproj(n, 977), 7)
    S0 = I.make_init_poses(inst, 64)
    P = _small(inst.params, n_p=n_p, n_p_star=n_p_star, n_t=n_t)
    fast = gpu_walk(inst, _small(P, flags=flags), S0, walkers, steps, 4747)
    plain = gpu_walk(inst, _small(P, flags=1), S0, walkers, steps, 4747)
    for a, b in zip(fast, plain):
        assert np.array_equal(a, b)
    if flags == 0:                                                      # the certificates carry most iterations
        h = B.Closure.closure_create(inst, P)
        try:
            h.closure_set_init(S0)
            h.closure_enable_stats(True)
            h.closure_sample(walkers, steps, 4747)
            st = h.closure_get_stats()
        finally:
            h.closure_destroy()
        assert st["perturb_pairs_f32"] > 0 and st["fallback_steps"] < 0.2 * st["walker_steps"], st


def test_ellipsoid_with_several_bounds_and_a_pivot():
    """Runs of equal bounds of odd length and a body pivot on the ellipsoid kernel, against the oracle and the plain kernel."""
    inst = I.to_ellipsoidal(_three_bounds(77, 901, (25, 31, 21)), 8)
    P = _small(inst.params, n_p=64, n_p_star=5, n_t=9, t_p=0.05)
    S0 = I.make_init_poses(inst, 16)
    assert_parity(inst, P, S0, 96, 20, 31)
    assert_parity(inst, _small(P, pivot=(0.3, -0.2, 0.1)), S0, 64, 16, 32)
    fast = gpu_walk(inst, P, S0, 2048, 80, 55)
    plain = gpu_walk(inst, _small(P, flags=1), S0, 2048, 80, 55)
    for a, b in zip(fast, plain):
        assert np.array_equal(a, b)


def test_ellipsoidal_api_edges():
    import torch
    from oracle import step1
    inst = I.to_ellipsoidal(I.make_instance(2), 5)
    h = B.Closure.closure_create(inst)
    try:
        poses, ok = h.closure_init_sample(600, 13)                     # Step I: Arun, ellipsoid PURSE test
        torch.cuda.synchronize()
        o_poses, o_ok = step1.init_sample(inst, 600, 13)
        assert np.array_equal(ok.cpu().numpy(), o_ok)
        assert np.abs(poses.cpu().numpy() - o_poses).max() < 1e-9
        assert o_ok.mean() > 0.2
        n0 = h.closure_init_from_trials(600, 13, max_poses=64)
        res = h.closure_run(2048, 40, 3)
        assert n0 == 64 and res["count"] > 1500 and res["rot_radius"] > 0
        with pytest.raises(B.ClosureError) as e:                       # no fp32 kernel for the ellipsoid norm
            h.closure_set_params(_small(inst.params, precision=32))
            h.closure_sample(64, 2, 1)
        assert e.value.status in (B.EUNSUPPORTED, B.ECUDA, B.EINVAL)
    finally:
        h.closure_destroy()
    for bad in ("asym", "indef"):
        broken = I.to_ellipsoidal(I.make_instance(1), 6)
        broken.measurements = broken.measurements.copy()
        if bad == "asym":
            broken.measurements[0, 7] += 1e-3                          # Lambda[0][1] != Lambda[1][0]
        else:
            broken.measurements[0, 6:15] = np.diag([1.0, -0.5, 1.0]).reshape(-1)
        with pytest.raises(B.ClosureError) as e:
            B.Closure.closure_create(broken)
        assert e.value.status == B.EINVAL


def test_trans_batch_members_with_different_reprojection_tables():
    """Translation sampler, closure_sample_batch over reprojection instances whose tables differ in length: the launch sizes
    the certified ladder's row buffer (N_P* x N rows) for the largest table, every member lays its own out from its own N.
    60 constraints x N_P* = 10 exceeds the buffer's 512 rows, so that member takes the fp64 ladder inside the same launch.
    Every member equals its own single-instance launch, and the plain fp64 kernel, bit for bit."""
    import torch
    insts = [I.make_custom_reproj(5, 311), I.make_instance(3, 2), I.make_custom_reproj(23, 312), I.make_custom_reproj(60, 313)]
    P = _small(insts[1].params, mode=I.MODE_TRANS, n_p=150, n_p_star=10, n_t=10)
    hs, hx = [], []
    try:
        for it in insts:
            for flags, lst in ((0, hs), (1, hx)):
                h = B.Closure.closure_create(it, _small(P, flags=flags))
                h.closure_set_init(I.make_init_poses(it, 8))
                lst.append(h)
        smp, flag = B.closure_sample_batch(hs, 256, 30, [21, 22, 23, 24])
        torch.cuda.synchronize()
        for b, (h, x) in enumerate(zip(hs, hx)):
            s1, f1 = h.closure_sample(256, 30, 21 + b)
            s2, f2 = x.closure_sample(256, 30, 21 + b)
            torch.cuda.synchronize()
            assert np.array_equal(s1.cpu().numpy(), smp[b].cpu().numpy()), b
            assert np.array_equal(f1.cpu().numpy(), flag[b].cpu().numpy()), b
            assert np.array_equal(s2.cpu().numpy(), smp[b].cpu().numpy()), b
            assert np.array_equal(f2.cpu().numpy(), flag[b].cpu().numpy()), b
    finally:
        for h in hs + hx:
            h.closure_destroy()
