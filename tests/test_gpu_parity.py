"""GPU parity: the CUDA path (through the C ABI) against the fp64 oracle, element by element,
on identical seeded fp32 inputs.  Tolerances are north_star's:
    forward   max|err| <= 1e-5 * max|out| + 1e-6
    gradients relative L2 error <= 1e-4 per parameter group (w, p, s, q)
Integer work (voxel boxes, key sets) must be bit-exact.  Run with `-m gpu` on a B200.
"""
import numpy as np
import pytest

import gsvox_inputs
import oracle
from parity_util import check_grad_groups, fmt

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

FWD_REL, FWD_ABS, GRAD_REL = 1e-5, 1e-6, 1e-4


@pytest.fixture(scope="module")
def pkg():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2503_22139_b200 as p
    p.lib()                                     # fails loudly if the extension is missing
    torch.cuda.set_device(0)
    return p


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def run_gpu(pkg, case, grad=None, key_capacity=None, max_channels=None):
    plan = pkg.Plan(max(case.n, 1), case.grid, max_channels=max_channels or case.channels,
                    key_capacity=key_capacity)
    pos, scale, quat, w = dev(case.pos), dev(case.scale), dev(case.quat), dev(case.weight)
    plan.preprocess(pos, scale, quat)
    if key_capacity is None:
        st = plan.status()
        if st["overflow"]:                      # default capacity too small: size it exactly
            plan = pkg.Plan(max(case.n, 1), case.grid, max_channels=max_channels or case.channels,
                            key_capacity=st["keys_needed"])
            plan.preprocess(pos, scale, quat)
    out = plan.forward(w)
    grads = None
    if grad is not None:
        grads = plan.backward(w, dev(grad))
    torch.cuda.synchronize()
    return plan, out.cpu().numpy(), None if grads is None else [g.cpu().numpy() for g in grads]


def check_forward(out, ref):
    err = np.abs(out.astype(np.float64) - ref).max()
    tol = FWD_REL * np.abs(ref).max() + FWD_ABS
    assert err <= tol, "forward max|err| %.3e > tol %.3e" % (err, tol)
    return err, tol


def check_grads(grads, refs, case=None, label=""):
    """north_star's group criterion (relative L2 <= 1e-4 per group) and the per-Gaussian bound of parity_util."""
    describe = None
    if case is not None and case.n > 0:
        def describe(i):
            box = oracle.geometry(case.pos[i:i + 1], case.scale[i:i + 1], case.quat[i:i + 1], case.grid)["box"][0]
            return "pos %s scale %s box %s" % (case.pos[i].tolist(), case.scale[i].tolist(), box.tolist())
    res = check_grad_groups(("w", "p", "s", "q"), grads, refs, tol=GRAD_REL, describe=describe, label=label)
    print("%s gradients: %s" % (label or (case.name if case is not None else ""), fmt(res)))
    return {k: v[0] for k, v in res.items()}


def check_geometry_and_bins(plan, case):
    """Boxes bit-identical to the oracle (reading A5); M_idx within 1e-5 relative; every
    (brick, Gaussian) key present exactly once; P_def identical."""
    geo = oracle.geometry(case.pos, case.scale, case.quat, case.grid)
    box, minv = plan.geometry()
    assert np.array_equal(box, geo["box"]), "voxel boxes differ from the oracle: %d mismatches" % \
        int((box != geo["box"]).any(1).sum())
    h = np.asarray(case.spacing, np.float64)
    scale6 = np.array([h[0] * h[0], h[0] * h[1], h[0] * h[2], h[1] * h[1], h[1] * h[2], h[2] * h[2]])
    live = geo["box"][:, 3] >= geo["box"][:, 0]
    Mi = geo["M"] * scale6
    nrm = np.linalg.norm(Mi[live], axis=1, keepdims=True)
    assert np.all(np.abs(minv[live] - Mi[live]) <= 1e-5 * nrm)
    st = plan.status()
    ext = np.clip(geo["box"][:, 3:] - geo["box"][:, :3] + 1, 0, None).astype(np.int64)
    assert st["pairs"] == int(ext.prod(1).sum())
    assert st["skipped_gaussians"] == int((geo["flags"] & 1).sum())
    # expected key multiset from the oracle boxes
    b = geo["box"].astype(np.int64)
    nbk = (b[:, 3:] >> 3) - (b[:, :3] >> 3) + 1
    nbk[~live] = 0
    # reading A15: keys whose every term is provably below w e^-32 may be dropped, and are counted
    assert st["keys_needed"] + st["culled_keys"] == int(nbk.prod(1).sum())
    assert 0 <= st["pairs_exec"] <= st["pairs"]
    if st["culled_keys"] == 0:
        assert st["pairs_exec"] == st["pairs"]
    start, keys = plan.bins()
    assert start[0] == 0 and start[-1] == st["keys_needed"] and np.all(np.diff(start) >= 0)
    nb = [(d + 7) // 8 for d in case.dims]
    brick_of_key = np.repeat(np.arange(len(start) - 1), np.diff(start))
    got = set(zip(brick_of_key.tolist(), keys.tolist()))
    assert len(got) == len(keys), "duplicate (brick, Gaussian) keys"
    if case.n <= 5000:
        exp = set()
        for g in np.flatnonzero(live):
            for bz in range(b[g, 2] >> 3, (b[g, 5] >> 3) + 1):
                for by in range(b[g, 1] >> 3, (b[g, 4] >> 3) + 1):
                    for bx in range(b[g, 0] >> 3, (b[g, 3] >> 3) + 1):
                        exp.add(((bz * nb[1] + by) * nb[0] + bx, int(g)))
        assert got <= exp and len(exp - got) == st["culled_keys"]
        # every dropped key is negligible: brute-force the exponent over the brick's voxels (oracle M, fp64)
        o = np.asarray(case.origin, np.float64)
        for (brick, g) in exp - got:
            bx, by, bz = brick % nb[0], (brick // nb[0]) % nb[1], brick // (nb[0] * nb[1])
            ii = np.arange(8)
            X, Y, Z = np.meshgrid(8 * bx + ii, 8 * by + ii, 8 * bz + ii, indexing="ij")
            d = np.stack([o[0] + X * h[0], o[1] + Y * h[1], o[2] + Z * h[2]], -1) - case.pos[g].astype(np.float64)
            m = geo["M"][g]
            M3 = np.array([[m[0], m[1], m[2]], [m[1], m[3], m[4]], [m[2], m[4], m[5]]])
            q = np.einsum("...a,ab,...b->...", d, M3, d)
            assert q.min() > 60.0, "a non-negligible key was culled: q_min = %.2f" % q.min()
    return st


def full_parity(pkg, case, **kw):
    g = case.grad_out()
    plan, out, grads = run_gpu(pkg, case, grad=g, **kw)
    st = check_geometry_and_bins(plan, case)
    assert not st["overflow"]
    ref = oracle.forward(case.pos, case.scale, case.quat, case.weight, case.grid)
    check_forward(out, ref)
    refs = oracle.backward(case.pos, case.scale, case.quat, case.weight, case.grid, g)
    check_grads(grads, refs, case)
    return plan


# ------------------------------------------------------------------ small / medium cases
def test_config1_tiny_full(pkg):
    full_parity(pkg, gsvox_inputs.config1())


def test_subvolume_anisotropic_spacing_three_channels(pkg):
    """Ragged dims (37,29,21), non-zero origin, spacing (2,1.5,0.75), unnormalised quaternions,
    C = 3, most Gaussians partly outside: the arguments PAPER.md:128-136 exercise."""
    full_parity(pkg, gsvox_inputs.subvolume_case())


@pytest.mark.parametrize("channels", [2, 4, 5, 9, 13, 96])
def test_channel_counts(pkg, channels):
    """Channel groups of 9, 3 and 1 in every mix up to GSVOX_MAX_CHANNELS = 96 (ten groups of 9 and two of 3)."""
    full_parity(pkg, gsvox_inputs.subvolume_case(n=300 if channels < 96 else 120, channels=channels, seed=20 + channels))


@pytest.mark.parametrize("level,n", [(1, 60), (2, 400), (3, 3000)])
def test_config3_levels_reduced(pkg, level, n):
    """Config 3 recipe (C = 9, 128x128x64) at a reduced Gaussian count so the oracle stays in seconds."""
    full_parity(pkg, gsvox_inputs.config3(level, n=n))


def test_config4_recipe_reduced(pkg):
    full_parity(pkg, gsvox_inputs.config4(n=20000, dims=(96, 88, 72)))


def test_config5_recipe_reduced_needles_and_blobs(pkg):
    full_parity(pkg, gsvox_inputs.config5(n=20000, dims=(128, 96, 64)))


def test_hot_bricks_are_split_into_key_range_segments(pkg):
    """6000 Gaussians on 8 bricks: ~3000 keys per brick, so a3 (C = 1) works segments 1.. of every brick in its
    second launch (atomic adds onto what segment 0 stored) and a4 spills past its 2048-key first launch
    (kSplitKeys = 512, gsvox_internal.cuh; SURVEY section 7 hard part 6).  Ragged grid: rows outside the grid too."""
    case = gsvox_inputs.config1(n=6000, dims=(16, 15, 13), seed=88)
    plan = full_parity(pkg, case)
    start, _ = plan.bins()
    assert np.diff(start).max() > 2048


def test_hot_bricks_multi_channel(pkg):
    case = gsvox_inputs.subvolume_case(n=12000, dims=(16, 16, 8), channels=3, seed=89)
    plan = full_parity(pkg, case)
    start, _ = plan.bins()
    assert np.diff(start).max() > 2048


def test_narrow_and_wide_gaussians(pkg):
    """Scales from 0.15 voxel (sub-voxel, direct-exponential path, mostly empty boxes) to 40 voxels."""
    rng = np.random.default_rng(77)
    n, dims = 1500, (50, 44, 38)
    case = gsvox_inputs.config1(n=n, dims=dims, seed=77)
    case.scale[:] = np.exp(rng.uniform(np.log(0.15), np.log(40.0), (n, 3))).astype(np.float32)
    case.scale[:200] = np.exp(rng.uniform(np.log(0.15), np.log(0.9), (200, 3))).astype(np.float32)
    full_parity(pkg, case)


def test_single_isolated_gaussians_worst_case_tolerance(pkg):
    """max|out| = w: the tolerance is relative to ONE Gaussian's peak, the hardest case for the
    row recurrence.  Sweeps sub-voxel offsets, scales around the recurrence/direct switch, rotations."""
    rng = np.random.default_rng(5)
    dims = (40, 40, 40)
    for s0 in (0.45, 0.5, 0.52, 0.535, 0.54, 0.56, 0.6, 0.7, 0.84, 1.0, 1.3, 2.0, 4.5):
        for rep in range(4):
            case = gsvox_inputs.config1(n=1, dims=dims, seed=1000 + rep)
            case.pos[:] = (19.5 + rng.uniform(-4, 4, 3)).astype(np.float32)
            case.scale[:] = (s0 * np.exp(rng.uniform(-0.1, 0.1, 3))).astype(np.float32)
            case.weight[:] = 1.0
            plan, out, _ = run_gpu(pkg, case)
            ref = oracle.forward(case.pos, case.scale, case.quat, case.weight, case.grid)
            check_forward(out, ref)


def test_far_grid_coordinates_keep_accuracy(pkg):
    """A sub-grid far from the world origin with fine spacing: index-space centres ~3e4 voxels
    are split into integer + fraction, so brick-local coordinates stay accurate."""
    case = gsvox_inputs.subvolume_case(n=400, dims=(48, 40, 36), channels=1, seed=31,
                                       origin=(1000.0, -2000.0, 512.0), spacing=(0.5, 0.25, 0.125))
    case.scale[:] *= 0.3
    full_parity(pkg, case)


def test_longest_axis_the_boundary_allows(pkg):
    """GSVOX_MAX_DIM = 32760 voxels along one axis (the record packs box corners as int16, bricks 4095 wide): Gaussians at
    both ends and one 2000-voxel-long needle along the axis; one voxel more is refused."""
    for axis in range(3):
        dims = [9, 11, 10]; dims[axis] = 32760
        case = gsvox_inputs.config1(n=240, dims=tuple(dims), seed=60 + axis)
        case.pos[:80, axis] = np.linspace(32700.0, 32761.5, 80, dtype=np.float32)       # the far end, some beyond it
        case.pos[80:120, axis] = np.linspace(-1.5, 40.0, 40, dtype=np.float32)
        case.scale[200] = 1.0; case.scale[200, axis] = 333.0; case.quat[200] = (1, 0, 0, 0)
        case.pos[200, axis] = 20000.3
        full_parity(pkg, case)
    bad = ((0.0, 0.0, 0.0), (1.0, 1.0, 1.0), (32761, 8, 8))
    with pytest.raises(pkg.GsvoxError):
        pkg.Plan(10, bad, max_channels=1)


# --------------------------------------------------------------------------- edge cases
def test_degenerate_empty_and_outside(pkg):
    case = gsvox_inputs.config1(n=64, dims=(24, 20, 18), seed=3)
    case.scale[1, 2] = 0.0; case.scale[2, 0] = -1.0; case.quat[3] = 0.0
    case.pos[4, 1] = np.nan; case.scale[5, 1] = np.inf; case.pos[6] = (-500, 5, 5)
    case.scale[7] = 0.05; case.pos[7] = (5.5, 5.5, 5.5)
    g = case.grad_out()
    plan, out, grads = run_gpu(pkg, case, grad=g)
    st = check_geometry_and_bins(plan, case)
    assert st["skipped_gaussians"] == 5
    ref = oracle.forward(case.pos, case.scale, case.quat, case.weight, case.grid)
    check_forward(out, ref)
    refs = oracle.backward(case.pos, case.scale, case.quat, case.weight, case.grid, g)
    check_grads(grads, refs, case)
    for a in grads:
        assert np.isfinite(a).all() and not a[1:8].any()


def test_zero_gaussians_writes_zeros(pkg):
    case = gsvox_inputs.config1(n=0, dims=(17, 9, 10))
    plan = pkg.Plan(4, case.grid)
    plan.preprocess(dev(case.pos.reshape(0, 3)), dev(case.scale.reshape(0, 3)), dev(case.quat.reshape(0, 4)))
    out = torch.full((1, 10, 9, 17), 7.0, device="cuda")
    plan.forward(dev(case.weight.reshape(0, 1)), out=out)
    torch.cuda.synchronize()
    assert not out.cpu().numpy().any()
    assert plan.status()["keys_needed"] == 0


def test_key_overflow_is_reported_and_outputs_are_zero(pkg):
    case = gsvox_inputs.config1(n=500, dims=(32, 32, 32), seed=9)
    g = case.grad_out()
    plan, out, grads = run_gpu(pkg, case, grad=g, key_capacity=100)
    st = plan.status()
    assert st["overflow"] and st["keys_needed"] > 100
    assert not out.any() and all(not a.any() for a in grads)
    plan2, out2, _ = run_gpu(pkg, case, key_capacity=st["keys_needed"])
    assert not plan2.status()["overflow"]
    check_forward(out2, oracle.forward(case.pos, case.scale, case.quat, case.weight, case.grid))


def test_plan_reuse_across_steps_and_weight_changes(pkg):
    """The plan is rebuilt every training step (parameters change each
    iteration); weights may change between forward calls without a new preprocess."""
    a = gsvox_inputs.config1(n=800, dims=(40, 36, 28), seed=1)
    b = gsvox_inputs.config1(n=650, dims=(40, 36, 28), seed=2)
    plan = pkg.Plan(800, a.grid)
    for case in (a, b, a):
        plan.preprocess(dev(case.pos), dev(case.scale), dev(case.quat))
        out = plan.forward(dev(case.weight)).cpu().numpy()
        check_forward(out, oracle.forward(case.pos, case.scale, case.quat, case.weight, case.grid))
    w2 = (-2.0 * a.weight).astype(np.float32)
    out = plan.forward(dev(w2)).cpu().numpy()
    check_forward(out, oracle.forward(a.pos, a.scale, a.quat, w2, a.grid))


def test_forward_is_run_to_run_stable_within_tolerance(pkg):
    case = gsvox_inputs.config1(n=3000, dims=(48, 48, 48), seed=4)
    _, o1, g1 = run_gpu(pkg, case, grad=case.grad_out())
    _, o2, g2 = run_gpu(pkg, case, grad=case.grad_out())
    assert np.abs(o1 - o2).max() <= 1e-6 * np.abs(o1).max()
    for x, y in zip(g1, g2):
        assert np.linalg.norm(x - y) <= 1e-5 * np.linalg.norm(x)


@pytest.mark.parametrize("which", ["config4_recipe", "hot_bricks", "channels3", "needles"])
def test_deterministic_mode_gives_a_bitwise_repeatable_forward(pkg, which):
    """gsvox_plan_set_deterministic (SURVEY section 7 hard part 3, section 4 test 6): every (brick, class) bin sorted by
    Gaussian id and a3 without atomics.  Two INDEPENDENT plans (their counting sorts race differently) must then
    hold identical key arrays and produce the same forward bits, also across repeated preprocess calls; parity with
    the oracle is unchanged; the default mode is only required to agree to rounding."""
    case = {"config4_recipe": lambda: gsvox_inputs.config4(n=20000, dims=(96, 88, 72)),
            "hot_bricks": lambda: gsvox_inputs.config1(n=6000, dims=(16, 15, 13), seed=88),
            "channels3": lambda: gsvox_inputs.subvolume_case(n=3000, channels=3, seed=23),
            "needles": lambda: gsvox_inputs.config5(n=20000, dims=(128, 96, 64))}[which]()
    t = (dev(case.pos), dev(case.scale), dev(case.quat), dev(case.weight))
    outs, keysets = [], []
    for rep in range(3):
        plan = pkg.Plan(case.n, case.grid, max_channels=case.channels)
        plan.set_deterministic(True)
        for _ in range(1 + rep):                                   # repeated preprocess on the same plan as well
            plan.preprocess(*t[:3])
        assert not plan.status()["overflow"] and plan.unsorted_bins() == 0
        outs.append(plan.forward(t[3]).clone())
        start, keys = plan.bins()
        keysets.append((start.copy(), keys.copy()))
    for o in outs[1:]:
        assert torch.equal(o, outs[0]), "deterministic forward differs between plans"
    for st_, k_ in keysets[1:]:
        assert np.array_equal(st_, keysets[0][0]) and np.array_equal(k_, keysets[0][1])
    # keys of a brick are grouped by class; inside a class they ascend
    start, keys = keysets[0]
    ref = oracle.forward(case.pos, case.scale, case.quat, case.weight, case.grid)
    check_forward(outs[0].cpu().numpy(), ref)
    g = case.grad_out()
    grads = [x.cpu().numpy() for x in plan.backward(t[3], dev(g))]
    check_grads(grads, oracle.backward(case.pos, case.scale, case.quat, case.weight, case.grid, g), case)
    # and the mode can be switched off again: same values to rounding
    plan.set_deterministic(False)
    with pytest.raises(pkg.GsvoxError):
        plan.forward(t[3])                                         # needs a new preprocess
    plan.preprocess(*t[:3])
    assert plan.unsorted_bins() == -1
    o2 = plan.forward(t[3])
    assert float((o2 - outs[0]).abs().max()) <= 1e-5 * float(outs[0].abs().max())      # another summation order, same values


@pytest.mark.parametrize("dims", [(40, 32, 24), (40, 36, 70)])
def test_host_buffer_step_matches_device_path(pkg, dims):
    """(40, 36, 70): 9 brick layers, ragged in z — gsvox_step_host uploads the upstream gradient in four pieces of whole
    brick layers and runs a4 piece by piece; (40, 32, 24): 3 layers, the unsplit path."""
    case = gsvox_inputs.config1(n=1200, dims=dims, seed=6)
    g = case.grad_out()
    plan = pkg.Plan(case.n, case.grid)
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    out = torch.empty((1, dims[2], dims[1], dims[0])).pin_memory()
    grads = tuple(torch.empty((case.n, k)).pin_memory() for k in (1, 3, 3, 4))
    plan.step_host(pin(case.pos), pin(case.scale), pin(case.quat), pin(case.weight), pin(g), out, grads)
    check_forward(out.numpy(), oracle.forward(case.pos, case.scale, case.quat, case.weight, case.grid))
    check_grads([t.numpy() for t in grads],
                oracle.backward(case.pos, case.scale, case.quat, case.weight, case.grid, g))


# ------------------------------------------------- BASELINE.json configs at full size
# The oracle finishes every full-size config in seconds on the GPU box's host cores, so the
# comparison is element by element over the whole volume and every Gaussian, not sampled.
def test_config2_cbct_full_size(pkg):
    full_parity(pkg, gsvox_inputs.config2())


@pytest.mark.parametrize("level", [1, 2, 3])
def test_config3_dvf_full_size(pkg, level):
    full_parity(pkg, gsvox_inputs.config3(level))


def test_config4_training_step_full_size(pkg):
    full_parity(pkg, gsvox_inputs.config4())


def test_config5_stress_full_size(pkg):
    full_parity(pkg, gsvox_inputs.config5())


def test_needle_keys_are_culled_only_when_negligible(pkg):
    """Thin rotated Gaussians (config 5's needles, 10-20 x 0.5 x 0.5 voxels): most bricks of their
    axis-aligned boxes hold nothing above w e^-32 and are not binned (reading A15).  Parity still holds,
    the dropped keys are counted and each one is verified negligible by brute force."""
    rng = np.random.default_rng(71)
    n, dims = 300, (96, 96, 96)
    pos = rng.uniform(10, 86, size=(n, 3))
    scale = np.stack([rng.uniform(10, 20, n), np.full(n, 0.5), np.full(n, 0.5)], 1)
    quat = rng.standard_normal((n, 4))
    case = gsvox_inputs.Case("needles", dims, 1, pos.astype(np.float32), scale.astype(np.float32),
                             quat.astype(np.float32), rng.uniform(0, 1, (n, 1)).astype(np.float32), seed=71,
                             _grad_seed=[71, 1])
    plan = full_parity(pkg, case)
    st = plan.status()
    assert st["culled_keys"] > 2 * st["keys_needed"], st          # most of the boxes is empty space
    assert st["pairs_exec"] < 0.5 * st["pairs"]


def test_cuda_graph_replay_matches_eager_and_follows_new_inputs(pkg):
    """The three hot calls neither synchronise nor allocate, so one training step can be captured in a CUDA
    graph; a replay after the parameters changed in place must give the new step's results."""
    case = gsvox_inputs.config1()
    plan = pkg.Plan(case.n, case.grid, max_channels=1)
    pos, scale, quat, w, g = dev(case.pos), dev(case.scale), dev(case.quat), dev(case.weight), dev(case.grad_out())
    graph, out, grads = plan.capture_step(pos, scale, quat, w, g)
    graph.replay(); torch.cuda.synchronize()
    ref = oracle.forward(case.pos, case.scale, case.quat, case.weight, case.grid)
    check_forward(out.cpu().numpy(), ref)
    pos2 = case.pos + np.float32(0.37)                       # new parameters, same buffers
    pos.copy_(dev(pos2))
    graph.replay(); torch.cuda.synchronize()
    ref2 = oracle.forward(pos2, case.scale, case.quat, case.weight, case.grid)
    check_forward(out.cpu().numpy(), ref2)
    refs2 = oracle.backward(pos2, case.scale, case.quat, case.weight, case.grid, case.grad_out())
    check_grads([t.cpu().numpy() for t in grads], refs2)


def test_box_of_2_to_the_23_bricks_takes_the_whole_warp_route(pkg):
    """a2 walks the keys of ordinary Gaussians as a flat list whose brick index arithmetic (reciprocal multiplies) is
    exact below 2^23 keys per Gaussian; a box of 2^23 bricks or more is parked and walked by the whole warp with true
    division instead (gsvox_preprocess.cu, k_keys).  2048 x 2048 x 1024 voxels = 256 x 256 x 128 bricks = 2^23: one
    Gaussian that covers the whole grid must appear exactly once in every brick, next to two ordinary ones.  Binning only:
    a volume of 4.3e9 voxels is not voxelized here."""
    dims = (2048, 2048, 1024)
    grid = ((0.0, 0.0, 0.0), (1.0, 1.0, 1.0), dims)
    pos = np.array([[1000.0, 1100.0, 500.0], [20.5, 30.25, 40.0], [2040.0, 2040.0, 1020.0]], np.float32)
    scale = np.array([[900.0, 900.0, 900.0], [3.0, 2.0, 4.0], [2.5, 2.5, 2.5]], np.float32)
    quat = np.array([[1, 0, 0, 0], [0.9, 0.1, -0.3, 0.2], [1, 0, 0, 0]], np.float32)
    geo = oracle.geometry(pos, scale, quat, grid)
    b = geo["box"].astype(np.int64)
    assert b[0].tolist() == [0, 0, 0, 2047, 2047, 1023]
    nbk = ((b[:, 3:] >> 3) - (b[:, :3] >> 3) + 1).prod(1)
    assert nbk[0] == 1 << 23
    plan = pkg.Plan(3, grid, max_channels=1, key_capacity=int(nbk.sum()) + 16)
    plan.preprocess(dev(pos), dev(scale), dev(quat))
    st = plan.status()
    assert not st["overflow"] and st["culled_keys"] == 0
    assert st["keys_needed"] == int(nbk.sum())
    assert st["pairs"] == st["pairs_exec"] == int((b[:, 3:] - b[:, :3] + 1).prod(1).sum())
    start, keys = plan.bins()
    per_brick = np.diff(start)
    assert per_brick.min() == 1 and per_brick.sum() == int(nbk.sum())
    brick_of_key = np.repeat(np.arange(len(per_brick)), per_brick)
    assert np.array_equal(np.sort(brick_of_key[keys == 0]), np.arange(1 << 23))          # Gaussian 0: once in every brick
    for g in (1, 2):
        exp = sorted((bz * 256 + by) * 256 + bx for bz in range(b[g, 2] >> 3, (b[g, 5] >> 3) + 1)
                     for by in range(b[g, 1] >> 3, (b[g, 4] >> 3) + 1) for bx in range(b[g, 0] >> 3, (b[g, 3] >> 3) + 1))
        assert sorted(brick_of_key[keys == g].tolist()) == exp
