"""GPU parity of the fused MBC -> DVF op (gsvox_dvf_forward / gsvox_dvf_backward, SURVEY.md 8(f)
rank 1) against oracle.dvf_forward / dvf_backward, which voxelize the nine MBC volumes and then
combine them (Eq. 3) — the CUDA path never forms those volumes.  Same tolerances as the
voxelizer: forward max|err| <= 1e-5 max|d| + 1e-6; gradients relative L2 <= 1e-4 per group
(feat, coef, pos, scale, quat).  Run with `-m gpu` on a B200.
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
    p.lib()
    torch.cuda.set_device(0)
    return p


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def run_gpu(pkg, case, backward=True):
    plan = pkg.Plan(max(case.n, 1), case.grid, max_channels=3 * case.batch)
    pos, scale, quat = dev(case.pos), dev(case.scale), dev(case.quat)
    plan.preprocess(pos, scale, quat)
    st = plan.status()
    if st["overflow"]:
        plan = pkg.Plan(max(case.n, 1), case.grid, max_channels=3 * case.batch, key_capacity=st["keys_needed"])
        plan.preprocess(pos, scale, quat)
    feat, level, coef = dev(case.feat), dev(case.level), dev(case.coef)
    d = plan.dvf_forward(feat, level, coef)
    grads = None
    if backward:
        grads = plan.dvf_backward(feat, level, coef, dev(case.grad_dvf()))
    torch.cuda.synchronize()
    assert not plan.status()["overflow"]
    return d.cpu().numpy(), None if grads is None else [g.cpu().numpy() for g in grads]


def rel_l2(a, b):
    nb = np.linalg.norm(b)
    return np.linalg.norm(a.astype(np.float64) - b) / nb if nb > 0 else float(np.abs(a).max())


def parity(pkg, case):
    d, grads = run_gpu(pkg, case)
    lv, ids = case.levels()
    ref = oracle.dvf_forward(lv, case.coef, case.grid)
    err = np.abs(d.astype(np.float64) - ref).max()
    tol = FWD_REL * np.abs(ref).max() + FWD_ABS
    assert err <= tol, "dvf forward max|err| %.3e > tol %.3e" % (err, tol)
    gc_ref, per = oracle.dvf_backward(lv, case.coef, case.grid, case.grad_dvf())
    gf, gc, gp, gs, gq = grads
    refs = [np.zeros((case.n, k)) for k in (3, 3, 3, 4)]
    for sel, (rf, rp, rs, rq) in zip(ids, per):          # scatter the per-level oracle gradients back
        refs[0][sel], refs[1][sel], refs[2][sel], refs[3][sel] = rf, rp, rs, rq
    rels = {"coef": rel_l2(gc, gc_ref)}
    assert rels["coef"] <= GRAD_REL, "dvf grad coef rel L2 %.3e > %.1e" % (rels["coef"], GRAD_REL)
    res = check_grad_groups(("feat", "pos", "scale", "quat"), (gf, gp, gs, gq), refs, tol=GRAD_REL, label="dvf " + case.name)
    print("dvf %s gradients: %s" % (case.name, fmt(res)))
    rels.update({k: v[0] for k, v in res.items()})
    return err / tol, rels


def test_dvf_small_ragged_grid(pkg):
    parity(pkg, gsvox_inputs.dvf_case(batch=3, counts=(6, 40, 300), dims=(37, 29, 21), seed=31,
                                      scales=((5.0, 9.0), (2.5, 5.0), (0.6, 2.0))))


def test_dvf_single_projection_single_level(pkg):
    parity(pkg, gsvox_inputs.dvf_case(batch=1, counts=(200,), dims=(40, 24, 16), seed=32, scales=((0.5, 4.0),)))


@pytest.mark.parametrize("batch", [2, 5, 8])
def test_dvf_reduced_config3_levels(pkg, batch):
    parity(pkg, gsvox_inputs.dvf_case(batch=batch, counts=(60, 400, 3000), dims=(64, 64, 32), seed=33))


def test_dvf_stage2_batch_32(pkg):
    """N_batch = 32 (Stage 2) = 96 channels, the library maximum."""
    parity(pkg, gsvox_inputs.dvf_case(batch=32, counts=(20, 120, 800), dims=(32, 32, 16), seed=34,
                                      scales=((8.0, 16.0), (3.0, 6.0), (1.0, 2.5))))


def test_dvf_out_of_range_level_contributes_nothing(pkg):
    case = gsvox_inputs.dvf_case(batch=2, counts=(10, 50, 200), dims=(32, 24, 16), seed=35,
                                 scales=((5.0, 9.0), (2.5, 5.0), (0.8, 2.0)))
    base, _ = run_gpu(pkg, case, backward=False)
    bad = np.flatnonzero(case.level == 1)
    case2 = gsvox_inputs.dvf_case(batch=2, counts=(10, 50, 200), dims=(32, 24, 16), seed=35,
                                  scales=((5.0, 9.0), (2.5, 5.0), (0.8, 2.0)))
    case2.level[bad] = 7                                   # not a level: those Gaussians drop out
    d2, grads = run_gpu(pkg, case2)
    coef0 = case.coef.copy(); coef0[:, 1, :] = 0.0
    lv, _ = case.levels()
    ref = oracle.dvf_forward(lv, coef0, case.grid)
    assert np.abs(d2 - ref).max() <= FWD_REL * np.abs(ref).max() + FWD_ABS
    assert np.all(grads[0][bad] == 0.0) and np.all(grads[1][:, 1, :] == 0.0)
    assert np.abs(base - d2).max() > 0


def test_dvf_argument_checks(pkg):
    case = gsvox_inputs.dvf_case(batch=2, counts=(4, 4, 4), dims=(16, 16, 16), seed=36)
    plan = pkg.Plan(case.n, case.grid, max_channels=3)          # too few channels for B = 2
    plan.preprocess(dev(case.pos), dev(case.scale), dev(case.quat))
    with pytest.raises(pkg.GsvoxError):
        plan.dvf_forward(dev(case.feat), dev(case.level), dev(case.coef))


def test_dvf_full_size_config3_batch8(pkg):
    """All three config-3 levels (1k + 8k + 64k Gaussians) on the 128x128x64 grid, B = 8."""
    ratio, rels = parity(pkg, gsvox_inputs.dvf_case(batch=8))
    print("dvf full size: forward err/tol %.3f, grad rel L2 %s" % (ratio, rels))


# ------------------------------------------------------------------ two-stage (HBM-bound combine)
@pytest.mark.parametrize("B,L,shape", [(1, 1, (3, 5, 7)), (3, 3, (21, 29, 37)), (8, 3, (16, 32, 64)),
                                       (32, 4, (9, 10, 11)), (11, 2, (4, 4, 4))])
def test_mbc_combine_against_definition(pkg, B, L, shape):
    """gsvox_mbc_combine_* against oracle.mbc_combine(_backward) on random volumes, including
    voxel counts that are not multiples of 4 (scalar tail) and every B tile."""
    rng = np.random.default_rng([B, L])
    e = rng.standard_normal((L, 3) + shape).astype(np.float32)
    coef = rng.standard_normal((B, L, 3)).astype(np.float32)
    g = rng.standard_normal((B, 3) + shape).astype(np.float32)
    d = pkg.mbc_combine_forward(dev(e), dev(coef)).cpu().numpy()
    ref = oracle.mbc_combine(e, coef)
    assert np.abs(d - ref).max() <= FWD_REL * np.abs(ref).max() + FWD_ABS
    ge, gc = pkg.mbc_combine_backward(dev(e), dev(coef), dev(g))
    ge_ref, gc_ref = oracle.mbc_combine_backward(e, coef, g)
    assert rel_l2(ge.cpu().numpy(), ge_ref) <= GRAD_REL
    assert rel_l2(gc.cpu().numpy(), gc_ref) <= GRAD_REL


def two_stage_gpu(pkg, case):
    """Per-level plans with C = 3, then the combine; backward in the reverse order."""
    lv, ids = case.levels()
    nx, ny, nz = case.dims
    L, B = case.nlevels, case.batch
    e = torch.empty((L, 3, nz, ny, nx), dtype=torch.float32, device="cuda")
    plans, params = [], []
    for i, (p, s, q, f) in enumerate(lv):
        plan = pkg.Plan(max(len(p), 1), case.grid, max_channels=3)
        dp, ds, dq, df = dev(p), dev(s), dev(q), dev(f)
        plan.preprocess(dp, ds, dq)
        st = plan.status()
        if st["overflow"]:
            plan = pkg.Plan(max(len(p), 1), case.grid, max_channels=3, key_capacity=st["keys_needed"])
            plan.preprocess(dp, ds, dq)
        plan.forward(df, out=e[i])
        plans.append(plan); params.append(df)
    coef = dev(case.coef)
    d = pkg.mbc_combine_forward(e, coef)
    ge, gc = pkg.mbc_combine_backward(e, coef, dev(case.grad_dvf()))
    per = [plans[i].backward(params[i], ge[i]) for i in range(L)]
    torch.cuda.synchronize()
    return d.cpu().numpy(), gc.cpu().numpy(), [[t.cpu().numpy() for t in g4] for g4 in per], ids


@pytest.mark.parametrize("full", [False, True])
def test_two_stage_dvf_matches_oracle(pkg, full):
    case = gsvox_inputs.dvf_case(batch=8) if full else \
        gsvox_inputs.dvf_case(batch=4, counts=(60, 400, 3000), dims=(64, 64, 32), seed=37)
    d, gc, per, ids = two_stage_gpu(pkg, case)
    lv, _ = case.levels()
    ref = oracle.dvf_forward(lv, case.coef, case.grid)
    assert np.abs(d - ref).max() <= FWD_REL * np.abs(ref).max() + FWD_ABS
    gc_ref, per_ref = oracle.dvf_backward(lv, case.coef, case.grid, case.grad_dvf())
    assert rel_l2(gc, gc_ref) <= GRAD_REL
    for i in range(case.nlevels):
        res = check_grad_groups(("feat", "pos", "scale", "quat"), per[i], per_ref[i], tol=GRAD_REL, label="two-stage level %d" % i)
        print("two-stage dvf level %d gradients: %s" % (i, fmt(res)))
