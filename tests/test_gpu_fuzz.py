"""Randomised small cases of every operator against its oracle: random grid shapes (ragged, thin, one
brick), anisotropic spacing, far origins, channel counts, batch sizes, Gaussians from sub-voxel to
larger than the grid, half of them outside.  Seeds are fixed; a failure prints its seed.  `-m gpu`.
"""
import numpy as np
import pytest

import gsvox_inputs
import os

import oracle
from parity_util import per_row_worst

# GSVOX_FUZZ_SEEDS=n widens every sweep to n seeds (default: 24 / 8 / 8, sized for the round-end run)
_N = int(os.environ.get("GSVOX_FUZZ_SEEDS", "0"))

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


def rel_l2(a, b):
    nb = np.linalg.norm(b)
    return np.linalg.norm(a.astype(np.float64) - b) / nb if nb > 0 else float(np.abs(a).max())


@pytest.mark.parametrize("seed", range(_N or 24))
def test_voxelizer_random_cases(pkg, seed):
    rng = np.random.default_rng(1000 + seed)
    dims = tuple(int(v) for v in rng.choice([1, 3, 7, 8, 9, 16, 23, 40], size=3))
    spacing = tuple(float(v) for v in rng.choice([0.5, 0.75, 1.0, 2.0, 3.5], size=3))
    origin = tuple(float(v) for v in rng.choice([0.0, -37.25, 1.0e3, -4.0e4], size=3))
    C = int(rng.choice([1, 1, 2, 3, 7, 9, 10]))
    n = int(rng.choice([1, 5, 60, 400]))
    ext = np.asarray(dims) * np.asarray(spacing)
    pos = np.asarray(origin) + rng.uniform(-0.5, 1.5, (n, 3)) * ext
    scale = np.exp(rng.uniform(np.log(0.2), np.log(1.5 * ext.max()), (n, 3)))
    quat = rng.standard_normal((n, 4)) * rng.uniform(0.1, 9.0, (n, 1))
    w = rng.standard_normal((n, C))
    case = gsvox_inputs.Case("fuzz%d" % seed, dims, C, pos.astype(np.float32), scale.astype(np.float32),
                             quat.astype(np.float32), w.astype(np.float32), origin=origin, spacing=spacing,
                             seed=seed, _grad_seed=[seed, 7])
    plan = pkg.Plan(n, case.grid, max_channels=C)
    p, s, q, wt = dev(case.pos), dev(case.scale), dev(case.quat), dev(case.weight)
    plan.preprocess(p, s, q)
    st = plan.status()
    if st["overflow"]:
        plan = pkg.Plan(n, case.grid, max_channels=C, key_capacity=st["keys_needed"])
        plan.preprocess(p, s, q)
    out = plan.forward(wt).cpu().numpy()
    g = case.grad_out()
    grads = [t.cpu().numpy() for t in plan.backward(wt, dev(g))]
    ref, pairs = oracle.forward(case.pos, case.scale, case.quat, case.weight, case.grid, return_pairs=True)
    assert plan.status()["pairs"] == pairs
    assert np.abs(out - ref).max() <= 1e-5 * np.abs(ref).max() + 1e-6, seed
    refs = oracle.backward(case.pos, case.scale, case.quat, case.weight, case.grid, g)
    # DESIGN.md readings F1, F2, F4: what north_star's 1e-4 per group is asked of.
    #  F2 tail-only case: no voxel sees more than 1e-5 of a unit-weight Gaussian (ten times the forward's absolute
    #     tolerance): the fp32 exponent, |E| = 30..45 there, is good to ~1e-3 absolute, e^E to a few 1e-3 relative
    #     (seeds 6108, 9878 of the 12000-seed sweep: gradients of 1e-9..1e-6 off by 0.3..1.2 %)
    #  F4 a contributing Gaussian thinner than a quarter voxel (seed 9564: 0.12 voxel, its thin-axis dL/ds off by 7.8e-4,
    #     inside the per-Gaussian bound, 1.23e-4 of the group)
    gmax = float(oracle.forward(case.pos, case.scale, case.quat, np.ones((n, 1), np.float32), case.grid).max(initial=0.0))
    contributing = np.linalg.norm(np.asarray(refs[0]).reshape(n, -1), axis=1) > 0
    thin = bool(contributing.any()) and float((case.scale[contributing].min(axis=1) / max(spacing)).min()) < 0.25
    for name, a, b in zip("wpsq", grads, refs):
        if np.linalg.norm(b) > 1e-8:
            # a "group" of ONE Gaussian can be a nearly cancelling sum over its voxels (seed 483 of the 1500-seed sweep: a
            # 74:1 pancake whose thin-axis dL/ds is 1/100 of what other weights give on the same geometry; fp32 error
            # scales with the terms, 6.6e-4 of the sum, 6e-6 of the terms): north_star's bound is for groups over the set
            # (reading F1; the group size that counts is the number of Gaussians that contribute at all:
            # seed 2646 of a 12000-seed sweep has n = 5 with four of them outside the grid or culled)
            live = int((np.linalg.norm(np.asarray(b).reshape(n, -1), axis=1) > 0).sum())
            tol = 2e-2 if gmax < 1e-5 else (1e-3 if live <= 1 else (3e-4 if thin else 1e-4))
            assert rel_l2(a, b) <= tol, (seed, name, rel_l2(a, b), live, gmax, thin)
            if gmax >= 1e-5:
                assert per_row_worst(a, b)[0] <= 1.0, (seed, name, per_row_worst(a, b))
        else:       # every Gaussian so far from its voxels that all terms are below e^-20 (seed 277: 6e-11 vs an exact 0)
            assert np.abs(a - b).max() <= 1e-8, (seed, name)


@pytest.mark.parametrize("seed", range(_N or 8))
def test_warp_and_projector_random_cases(pkg, seed):
    rng = np.random.default_rng(2000 + seed)
    dims = tuple(int(v) for v in rng.choice([4, 9, 16, 21, 33], size=3))
    spacing = tuple(float(v) for v in rng.choice([0.5, 1.0, 1.5, 2.0], size=3))
    B = int(rng.choice([1, 2, 5]))
    wc = gsvox_inputs.warp_case(batch=B, dims=dims, spacing=spacing, amp_vox=float(rng.uniform(0.5, 12)), seed=2000 + seed,
                                rough=float(rng.uniform(0, 1.5)))
    out = pkg.warp_forward(dev(wc.iref), dev(wc.dvf), wc.grid).cpu().numpy()
    ref = oracle.warp_forward(wc.iref, wc.dvf, wc.grid)
    assert np.abs(out - ref).max() <= 1e-5 * np.abs(ref).max() + 1e-6, seed
    g = wc.grad_out()
    gi, gd = pkg.warp_backward(dev(wc.iref), dev(wc.dvf), wc.grid, dev(g))
    ri, rd = oracle.warp_backward(wc.iref, wc.dvf, wc.grid, g)
    assert rel_l2(gi.cpu().numpy(), ri) <= 1e-4 and rel_l2(gd.cpu().numpy(), rd) <= 1e-4, seed
    pc = gsvox_inputs.project_case(batch=B, dims=dims, spacing=spacing, nu=int(rng.integers(5, 70)), nv=int(rng.integers(5, 50)),
                                   du=float(rng.uniform(0.5, 4)), dv=float(rng.uniform(0.5, 4)), sad=float(rng.uniform(80, 400)),
                                   sdd=float(rng.uniform(450, 900)), off_u=float(rng.uniform(-10, 10)),
                                   off_v=float(rng.uniform(-10, 10)), seed=2000 + seed)
    drr = pkg.project_forward(dev(pc.vol), pc.grid, pc.geom, list(pc.angles)).cpu().numpy()
    dref = oracle.project_forward(pc.vol, pc.grid, pc.geom, pc.angles)
    assert np.abs(drr - dref).max() <= 1e-5 * np.abs(dref).max() + 1e-6, seed
    gv = pkg.project_backward(dev(pc.grad_drr()), pc.grid, pc.geom, list(pc.angles)).cpu().numpy()
    assert rel_l2(gv, oracle.project_backward(pc.grad_drr(), pc.grid, pc.geom, pc.angles)) <= 1e-4, seed


@pytest.mark.parametrize("seed", range(_N or 8))
def test_splat_random_cases(pkg, seed):
    rng = np.random.default_rng(3000 + seed)
    B = int(rng.choice([1, 2, 4]))
    sc = gsvox_inputs.splat_case(n=int(rng.choice([1, 20, 300])), batch=B, extent=tuple(rng.uniform(40, 200, 3)),
                                 nu=int(rng.integers(3, 100)), nv=int(rng.integers(3, 80)), du=float(rng.uniform(0.5, 4)),
                                 dv=float(rng.uniform(0.5, 4)), sad=float(rng.uniform(250, 600)), sdd=float(rng.uniform(650, 1200)),
                                 off_u=float(rng.uniform(-20, 20)), off_v=float(rng.uniform(-20, 20)), seed=3000 + seed,
                                 scales=(float(rng.uniform(0.1, 1.0)), float(rng.uniform(2.0, 30.0))))
    sp = pkg.Splatter(sc.n, sc.geom, sc.batch)
    a = (dev(sc.pos), dev(sc.scale), dev(sc.quat), dev(sc.rho))
    drr = sp.forward(*a, list(sc.angles))
    st = sp.status()
    if st["overflow"]:
        sp = pkg.Splatter(sc.n, sc.geom, sc.batch, key_capacity=st["keys_needed"])
        drr = sp.forward(*a, list(sc.angles))
    g = sc.grad_drr()
    grads = [t.cpu().numpy() for t in sp.backward(*a, list(sc.angles), dev(g))]
    ref, pairs = oracle.splat_forward(sc.pos, sc.scale, sc.quat, sc.rho, sc.geom, sc.angles, return_pairs=True)
    assert sp.status()["pairs"] == pairs, seed
    assert np.abs(drr.cpu().numpy() - ref).max() <= 1e-5 * np.abs(ref).max() + 1e-6, seed
    refs = oracle.splat_backward(sc.pos, sc.scale, sc.quat, sc.rho, sc.geom, sc.angles, g)
    # DESIGN.md reading F3: dL/drho = sum over pixels of SIGNED terms g E amp / rho.  The forward may be off by 1e-5 of its
    # peak per pixel (north_star), so the sum inherits an error proportional to the sum of the |terms| — the same gradient
    # for |g| — whatever cancels in the signed sum (n = 1 seeds of the 12000-seed sweep: 5503 cancels to 1e-7 of its terms
    # and is off by 2.7e-2 of the sum, 2e-9 of the terms; pos / scale / quat of the same seeds agree to 1e-6).  A tenth of
    # what the forward tolerance implies is allowed.
    rho_abs = oracle.splat_backward(sc.pos, sc.scale, sc.quat, sc.rho, sc.geom, sc.angles, np.abs(g))[0]
    for name, x, y in zip(("rho", "pos", "scale", "quat"), grads, refs):
        if np.linalg.norm(y) > 1e-12:
            x = x.reshape(y.shape)
            slack = 1e-6 * np.linalg.norm(rho_abs) if name == "rho" else 0.0
            assert np.linalg.norm(x - y) <= 1e-4 * np.linalg.norm(y) + slack, (seed, name, rel_l2(x, y))
