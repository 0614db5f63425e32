"""GPU parity of the batched cone-beam projector (gsvox_project_forward / gsvox_project_backward;
SURVEY.md 8(f) rank 4) against oracle.project_forward / project_backward
(Joseph's method, exact transpose).  Forward max|err| <= 1e-5 max|drr| + 1e-6; backward relative
L2 <= 1e-4.  `-m gpu`, B200.
"""
import numpy as np
import pytest

import gsvox_inputs
import oracle

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


def rel_l2(a, b):
    nb = np.linalg.norm(b)
    return np.linalg.norm(a.astype(np.float64) - b) / nb if nb > 0 else float(np.abs(a).max())


def parity(pkg, case, backward=True):
    drr = pkg.project_forward(dev(case.vol), case.grid, case.geom, list(case.angles)).cpu().numpy()
    ref = oracle.project_forward(case.vol, case.grid, case.geom, case.angles)
    err = np.abs(drr - ref).max()
    tol = FWD_REL * np.abs(ref).max() + FWD_ABS
    assert err <= tol, "project forward max|err| %.3e > tol %.3e" % (err, tol)
    rel = None
    if backward:
        g = case.grad_drr()
        gv = pkg.project_backward(dev(g), case.grid, case.geom, list(case.angles)).cpu().numpy()
        rv = oracle.project_backward(g, case.grid, case.geom, case.angles)
        rel = rel_l2(gv, rv)
        assert rel <= GRAD_REL, "project backward rel L2 %.3e" % rel
    return err / tol, rel


def test_project_small_ragged_all_octants(pkg):
    """Angles in every octant (both dominant axes, both signs), anisotropic spacing, half-fan offsets,
    dims that are not multiples of the transpose tile."""
    angles = [0.0, 0.5, 1.0, 1.6, 2.4, 3.1, 3.9, 4.7, 5.5, np.pi / 4, -np.pi / 4]
    parity(pkg, gsvox_inputs.project_case(batch=len(angles), dims=(37, 45, 21), spacing=(2.0, 1.5, 2.5), nu=70, nv=40,
                                          du=3.0, dv=3.0, sad=300.0, sdd=450.0, off_u=9.0, off_v=-4.0, seed=51,
                                          angles=angles))


def test_project_wide_detector_rays_miss_the_volume(pkg):
    parity(pkg, gsvox_inputs.project_case(batch=3, dims=(24, 24, 12), nu=130, nv=90, du=4.0, dv=4.0, sad=200.0,
                                          sdd=300.0, seed=52))


def test_project_steep_cone_z_dominant_rays(pkg):
    """Outer detector rows run mostly along z: the third dominant-axis branch, forward and transpose."""
    case = gsvox_inputs.project_case(batch=3, dims=(14, 12, 30), nu=9, nv=41, du=6.0, dv=12.0, sad=60.0, sdd=90.0,
                                     seed=56, angles=[0.3, 1.7, 4.0])
    assert (oracle.cone_rays(case.grid, case.geom, np.float32(0.3))["axis"] == 2).any()
    parity(pkg, case)


def test_project_shared_volume_equals_batched_copies(pkg):
    case = gsvox_inputs.project_case(batch=4, dims=(32, 28, 16), nu=64, nv=32, du=2.5, dv=2.5, sad=250.0, sdd=400.0, seed=53)
    v0 = dev(case.vol[0])
    a = pkg.project_forward(v0, case.grid, case.geom, list(case.angles)).cpu().numpy()
    b = pkg.project_forward(dev(np.stack([case.vol[0]] * 4)), case.grid, case.geom, list(case.angles)).cpu().numpy()
    assert np.array_equal(a, b)
    ref = oracle.project_forward(case.vol[0], case.grid, case.geom, case.angles)
    assert np.abs(a - ref).max() <= FWD_REL * np.abs(ref).max() + FWD_ABS


def test_project_transpose_identity_on_the_gpu(pkg):
    """<P x, y> = <x, P^T y> with both sides from the CUDA path (fp32 sums: 1e-5)."""
    case = gsvox_inputs.project_case(batch=2, dims=(40, 36, 20), nu=96, nv=48, du=2.0, dv=2.0, sad=300.0, sdd=450.0, seed=54)
    rng = np.random.default_rng(54)
    x = rng.standard_normal(case.vol.shape).astype(np.float32)
    y = case.grad_drr()
    Px = pkg.project_forward(dev(x), case.grid, case.geom, list(case.angles)).cpu().numpy().astype(np.float64)
    PTy = pkg.project_backward(dev(y), case.grid, case.geom, list(case.angles)).cpu().numpy().astype(np.float64)
    lhs, rhs = float((Px * y).sum()), float((x * PTy).sum())
    assert lhs == pytest.approx(rhs, rel=1e-5)


def test_project_argument_checks(pkg):
    case = gsvox_inputs.project_case(batch=1, dims=(8, 8, 8), nu=8, nv=8, seed=55)
    bad = dict(case.geom, sdd=0.0)
    with pytest.raises(pkg.GsvoxError):
        pkg.project_forward(dev(case.vol), case.grid, bad, list(case.angles))
    with pytest.raises(pkg.GsvoxError):
        pkg.project_forward(dev(case.vol), case.grid, case.geom, [0.1] * 65)      # more than 64 angles per call


def test_project_full_size_paper_geometry(pkg):
    """Table I geometry: 200x200x100 voxels of 2 mm, 512x384 pixels of 0.776 mm, SAD 1000 / SDD 1500; B = 2
    keeps the numpy oracle to under a minute."""
    ratio, rel = parity(pkg, gsvox_inputs.project_case(batch=2))
    print("project full size: forward err/tol %.3f, backward rel L2 %.3e" % (ratio, rel))


@pytest.mark.parametrize("dims", [(12, 8, 1100), (9, 10, 1100)])
def test_project_many_slices(pkg, dims):
    """nz x B = 70 400 (b, z) slices: the transposes index slices on a 1-D grid (a gridDim.z of slices would stop
    at 65 535).  (12, 8, .) takes the float4 transpose, (9, 10, .) the scalar one."""
    B = 64
    angles = np.linspace(0.0, 2 * np.pi, B, endpoint=False) + 0.05
    case = gsvox_inputs.project_case(batch=B, dims=dims, spacing=(3.0, 3.0, 0.25), nu=10, nv=12, du=8.0, dv=30.0,
                                     sad=150.0, sdd=220.0, seed=57, angles=angles)
    parity(pkg, case)
