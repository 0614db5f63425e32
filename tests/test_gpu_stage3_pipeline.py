"""The operators chained into one Stage-2/3 step (paper_2503_22139_b200/pipeline.py)
against the SAME chain of oracle functions: voxelize I_ref and the MBC volumes (Eq. 5), combine
(Eq. 3), warp (Eq. 2), project (Eq. 12 / Eq. 6), and back.  Each oracle stage is fed the fp32-rounded
output of the previous oracle stage.  Checks that the operators compose (layouts, units of the DVF,
gradient conventions), not only that each one is right alone.  Tolerances: three fp32 stages in a
row — forward 3e-5 max|DRR| + 1e-6, gradients relative L2 2e-4.  `-m gpu`, B200.
"""
import numpy as np
import pytest

import gsvox_inputs
import oracle
from parity_util import check_grad_groups, fmt

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


def oracle_chain(case, g_drr):
    f32 = lambda a: np.asarray(a, dtype=np.float32)
    grid = case.grid
    iref = oracle.forward(*case.ref, grid)[0]
    e = oracle.mbc_volumes(case.levels, grid)
    dvf = oracle.mbc_combine(f32(e), case.coef)
    warped = oracle.warp_forward(f32(iref), f32(dvf), grid)
    drr = oracle.project_forward(f32(warped), grid, case.geom, case.angles)
    # backward, stage by stage
    g_warped = oracle.project_backward(g_drr, grid, case.geom, case.angles)
    g_iref, g_dvf = oracle.warp_backward(f32(iref), f32(dvf), grid, f32(g_warped))
    g_e, g_coef = oracle.mbc_combine_backward(f32(e), case.coef, f32(g_dvf))

    def vox_backward(params, g):                       # exact hi + lo split of the fp64 upstream gradient
        hi = g.astype(np.float32); lo = (g - hi.astype(np.float64)).astype(np.float32)
        a = oracle.backward(*params, grid, hi); c = oracle.backward(*params, grid, lo)
        return tuple(x + y for x, y in zip(a, c))
    g_levels = [vox_backward(lv, g_e[i]) for i, lv in enumerate(case.levels)]
    g_ref = vox_backward(case.ref, g_iref[None])
    return drr, g_ref, g_levels, g_coef


def test_stage3_step_matches_the_chained_oracles(pkg):
    case = gsvox_inputs.stage3_case(batch=3, dims=(40, 36, 20), n_ref=600, n_levels=(12, 40, 150), nu=56, nv=44,
                                    du=3.0, dv=3.0, sad=300.0, sdd=450.0, seed=91, dvf_mm=5.0)
    step = pkg.Stage3Step(case.grid, case.geom, len(case.ref[0]), [len(l[0]) for l in case.levels], case.batch)
    ref = tuple(dev(a) for a in case.ref)
    levels = [tuple(dev(a) for a in lv) for lv in case.levels]
    g = case.grad_drr()
    drr = step.forward(ref, levels, dev(case.coef), list(case.angles)).cpu().numpy()
    grads = step.backward(dev(g))
    torch.cuda.synchronize()
    o_drr, o_ref, o_levels, o_coef = oracle_chain(case, g)
    assert np.abs(o_drr).max() > 0
    d_max = float(step.dvf.abs().max())
    assert 0.5 < d_max < 60.0, d_max                                  # the DVFs really move voxels (mm)
    assert np.abs(drr - o_drr).max() <= 3e-5 * np.abs(o_drr).max() + 1e-6
    assert rel_l2(grads["coef"].cpu().numpy(), o_coef) <= 2e-4
    res = check_grad_groups(("rho", "pos", "scale", "quat"), [t.cpu().numpy() for t in grads["ref"]], o_ref, tol=2e-4, label="stage3 ref")
    print("stage3 reference Gaussians: %s" % fmt(res))
    for i in range(len(levels)):
        res = check_grad_groups(("feat", "pos", "scale", "quat"), [t.cpu().numpy() for t in grads["levels"][i]], o_levels[i],
                                tol=2e-4, label="stage3 level %d" % i)
        print("stage3 level %d: %s" % (i, fmt(res)))
