"""z-slab sharding on ONE GPU: W virtual ranks, each a plan
restricted to its brick layers, run one after another; their accumulators are summed where the
NCCL all-reduce would sit.  The assembled volume and the gradients must match the fp64 oracle to the
usual tolerances, and the key counts of the slabs must add up to the unsharded count.  `-m gpu`.
"""
import numpy as np
import pytest

import gsvox_inputs
import oracle

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def pkg():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2503_22139_b200 as p
    p.lib()
    torch.cuda.set_device(0)
    return p


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def sharded_run(pkg, case, world):
    from paper_2503_22139_b200.dist import slab_bounds
    nx, ny, nz = case.dims
    nbz = (nz + 7) // 8
    C = case.channels
    pos, scale, quat, w = dev(case.pos), dev(case.scale), dev(case.quat), dev(case.weight)
    g = dev(case.grad_out())
    out = torch.full((C, nz, ny, nx), float("nan"), device="cuda")       # every voxel must be written by exactly one slab
    plans, keys = [], 0
    for r in range(world):
        lo, hi = slab_bounds(nbz, r, world)
        plan = pkg.Plan(case.n, case.grid, max_channels=C)
        plan.set_slab(lo, hi)
        plan.preprocess(pos, scale, quat)
        st = plan.status()
        assert not st["overflow"]
        keys += st["keys_needed"]
        plan.forward(w, out=out)                                         # writes its slab only
        plan.backward_accumulate(w, g)
        plans.append(plan)
    total = sum(p.accumulators(C).clone() for p in plans)                 # <- the all-reduce
    grads = None
    for p in plans:
        p.accumulators(C).copy_(total)
        grads = p.backward_finish(C)                                     # identical on every rank
    torch.cuda.synchronize()
    return out.cpu().numpy(), [t.cpu().numpy() for t in grads], keys


@pytest.mark.parametrize("world", [2, 3, 8])
def test_sharded_matches_oracle_and_unsharded_key_count(pkg, world):
    case = gsvox_inputs.config3(3, n=1500, dims=(48, 40, 44), channels=3)   # nz = 44: ragged last brick layer
    out, grads, keys = sharded_run(pkg, case, world)
    ref = oracle.forward(case.pos, case.scale, case.quat, case.weight, case.grid)
    assert np.isfinite(out).all()
    assert np.abs(out - ref).max() <= 1e-5 * np.abs(ref).max() + 1e-6
    refs = oracle.backward(case.pos, case.scale, case.quat, case.weight, case.grid, case.grad_out())
    for name, a, b in zip("wpsq", grads, refs):
        assert np.linalg.norm(a - b) / np.linalg.norm(b) <= 1e-4, name
    plan = pkg.Plan(case.n, case.grid, max_channels=case.channels)
    plan.preprocess(dev(case.pos), dev(case.scale), dev(case.quat))
    assert keys == plan.status()["keys_needed"]


def test_sharded_config4_recipe_two_ranks(pkg):
    case = gsvox_inputs.config4(n=40_000, dims=(128, 128, 128))
    out, grads, _ = sharded_run(pkg, case, 2)
    ref = oracle.forward(case.pos, case.scale, case.quat, case.weight, case.grid)
    assert np.abs(out - ref).max() <= 1e-5 * np.abs(ref).max() + 1e-6
    refs = oracle.backward(case.pos, case.scale, case.quat, case.weight, case.grid, case.grad_out())
    for name, a, b in zip("wpsq", grads, refs):
        assert np.linalg.norm(a - b) / np.linalg.norm(b) <= 1e-4, name


def test_empty_slab_and_argument_checks(pkg):
    case = gsvox_inputs.config1(n=200, dims=(16, 16, 16))
    plan = pkg.Plan(case.n, case.grid, max_channels=1)
    with pytest.raises(pkg.GsvoxError):
        plan.set_slab(1, 3)                                               # only 2 brick layers
    plan.set_slab(1, 1)                                                   # empty: nothing written, zero accumulators
    plan.preprocess(dev(case.pos), dev(case.scale), dev(case.quat))
    out = torch.full((1, 16, 16, 16), 7.0, device="cuda")
    plan.forward(dev(case.weight), out=out)
    plan.backward_accumulate(dev(case.weight), dev(case.grad_out()))
    torch.cuda.synchronize()
    assert plan.status()["keys_needed"] == 0
    assert float(out.min()) == 7.0 and float(plan.accumulators(1).abs().max()) == 0.0


@pytest.mark.parametrize("world", [2, 8])
def test_sharded_config4_full_size_virtual_ranks(pkg, world):
    """The benched workload itself (256^3, 500 k Gaussians): 2 and 8 virtual ranks, whole volume and every gradient
    against the oracle."""
    from parity_util import check_grad_groups, fmt
    case = gsvox_inputs.config4()
    out, grads, keys = sharded_run(pkg, case, world)
    ref = oracle.forward(case.pos, case.scale, case.quat, case.weight, case.grid)
    assert np.isfinite(out).all()
    assert np.abs(out - ref).max() <= 1e-5 * np.abs(ref).max() + 1e-6
    refs = oracle.backward(case.pos, case.scale, case.quat, case.weight, case.grid, case.grad_out())
    res = check_grad_groups(("w", "p", "s", "q"), grads, refs, label="config4 %d slabs" % world)
    print("config 4, %d z-slabs: %s, keys %d" % (world, fmt(res), keys))


def test_key_balanced_slabs_on_the_blob_recipe(pkg):
    """Config 5's recipe (blobs): slabs cut on Plan.layer_keys() carry far more even key counts than equal-layer slabs,
    and the sharded result still matches the oracle."""
    from paper_2503_22139_b200.dist import slab_bounds, slab_bounds_by_keys
    case = gsvox_inputs.config5(n=60_000, dims=(128, 128, 128))
    t = (dev(case.pos), dev(case.scale), dev(case.quat))
    plan = pkg.Plan(case.n, case.grid)
    plan.preprocess(*t)
    lk = plan.layer_keys()
    assert sum(lk) == plan.status()["keys_needed"] and len(lk) == 16
    world = 4
    load = lambda f: [sum(lk[lo:hi]) for lo, hi in (f(r) for r in range(world))]
    eq = load(lambda r: slab_bounds(16, r, world)); kb = load(lambda r: slab_bounds_by_keys(lk, r, world))
    assert max(kb) <= max(eq) and max(kb) <= sum(lk) / world + max(lk)
    print("keys per rank, equal layers %s, key-balanced %s" % (eq, kb))
    # run the key-balanced slabs through the same virtual-rank emulation
    import paper_2503_22139_b200.dist as d
    orig = d.slab_bounds
    try:
        d.slab_bounds = lambda nbz, r, w: slab_bounds_by_keys(lk, r, w)
        out, grads, keys = sharded_run(pkg, case, world)
    finally:
        d.slab_bounds = orig
    ref = oracle.forward(case.pos, case.scale, case.quat, case.weight, case.grid)
    assert np.isfinite(out).all() and np.abs(out - ref).max() <= 1e-5 * np.abs(ref).max() + 1e-6
    assert keys == sum(lk)


def test_sharded_backward_through_a_real_nccl_group_of_one(pkg):
    """dist.sharded_backward with torch.distributed's NCCL backend actually initialised (world size 1: the only size
    one GPU allows): accumulate -> dist.all_reduce on the plan's accumulator view -> finish, against the oracle."""
    import socket
    import torch.distributed as dist
    from paper_2503_22139_b200.dist import sharded_backward
    if dist.is_initialized():
        pytest.skip("a process group already exists in this process")
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    dist.init_process_group("nccl", init_method="tcp://127.0.0.1:%d" % port, rank=0, world_size=1,
                            device_id=torch.device("cuda", 0))
    try:
        class R:                                   # a Ranks stand-in that forces the collective
            on, rank, world = True, 0, 1
        case = gsvox_inputs.config1()
        plan = pkg.Plan(case.n, case.grid)
        plan.preprocess(dev(case.pos), dev(case.scale), dev(case.quat))
        called = []

        def ar(t):
            called.append(t.numel()); dist.all_reduce(t)
        grads = sharded_backward(plan, dev(case.weight), dev(case.grad_out()), R, all_reduce=ar)
        torch.cuda.synchronize()
        assert called == [case.n * 12]                             # round4(9 + 1) floats per Gaussian
        refs = oracle.backward(case.pos, case.scale, case.quat, case.weight, case.grid, case.grad_out())
        for name, a, b in zip("wpsq", grads, refs):
            assert np.linalg.norm(a.cpu().numpy() - b) / np.linalg.norm(b) <= 1e-4, name
    finally:
        dist.destroy_process_group()
