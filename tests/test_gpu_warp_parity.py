"""GPU parity of the warp (gsvox_warp_forward / gsvox_warp_backward; SURVEY.md 8(f) rank 2;
PAPER.md:55 Eq. 2) against oracle.warp_forward / warp_backward.  Forward max|err| <=
1e-5 max|out| + 1e-6; gradients relative L2 <= 1e-4 per group (I_ref, d).  `-m gpu`, B200.
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


def cell_disagreements(case):
    """The oracle decides the cell as floor(d / h) in fp64 (Eq. 2 read plainly).  The kernel decides it on
    t = fp32(d * fp32(1 / h)) — two fp32 roundings, |t - d/h| <= 2^-23 |t| — so its cell differs from the oracle's
    only for samples within that distance of a cell face: an expected fraction of E|t| 2^-23 per component, ~1e-7
    for displacements of a few voxels, and exactly none when h is a power of two (then t is exact).  Returns
    (number of (sample, axis) components whose cell differs, number of components).  The interpolant is continuous
    across a face, so the forward does not see these samples; grad d does (the slope changes at a face), which is
    why the gradient tolerance below is asserted on ALL samples, these included."""
    d32 = np.asarray(case.dvf, np.float32)
    h32 = np.asarray(case.spacing, np.float32).reshape(1, 3, 1, 1, 1)
    with np.errstate(invalid="ignore", over="ignore"):
        t32 = (d32 * (np.float32(1.0) / h32).astype(np.float32)).astype(np.float32)
        t64 = d32.astype(np.float64) / h32.astype(np.float64)
    ok = np.isfinite(t64) & (np.abs(t64) < 4194304.0)
    return int((np.floor(t32)[ok] != np.floor(t64)[ok]).sum()), int(ok.sum())


def parity(pkg, case, grads=True):
    iref, dvf = dev(case.iref), dev(case.dvf)
    nbad, ncomp = cell_disagreements(case)
    assert nbad <= 2 + 4e-6 * ncomp, "cell decisions differ on %d of %d components" % (nbad, ncomp)
    print("warp cells decided differently by the fp32 reciprocal-multiply: %d of %d components" % (nbad, ncomp))
    out = pkg.warp_forward(iref, dvf, case.grid).cpu().numpy()
    ref = oracle.warp_forward(case.iref, case.dvf, case.grid)
    err = np.abs(out - ref).max()
    tol = FWD_REL * np.abs(ref).max() + FWD_ABS
    assert err <= tol, "warp forward max|err| %.3e > tol %.3e" % (err, tol)
    rels = {}
    if grads:
        g = case.grad_out()
        gi, gd = pkg.warp_backward(iref, dvf, case.grid, dev(g))
        ri, rd = oracle.warp_backward(case.iref, case.dvf, case.grid, g)
        rels = {"iref": rel_l2(gi.cpu().numpy(), ri), "dvf": rel_l2(gd.cpu().numpy(), rd)}
        for k, r in rels.items():
            assert r <= GRAD_REL, "warp grad %s rel L2 %.3e > %.1e" % (k, r, GRAD_REL)
    return err / tol, rels


def test_warp_small_ragged_anisotropic(pkg):
    parity(pkg, gsvox_inputs.warp_case(batch=3, dims=(37, 29, 21), spacing=(2.0, 1.5, 0.75), amp_vox=6.0, seed=41))


def test_warp_large_displacements_leave_the_grid(pkg):
    parity(pkg, gsvox_inputs.warp_case(batch=2, dims=(40, 24, 16), amp_vox=30.0, seed=42, rough=2.0))


def test_warp_zero_and_integer_displacements_are_exact(pkg):
    case = gsvox_inputs.warp_case(batch=2, dims=(32, 16, 8), seed=43)
    case.dvf[0] = 0.0
    case.dvf[1, 0] = 2 * case.spacing[0]; case.dvf[1, 1] = -1 * case.spacing[1]; case.dvf[1, 2] = 3 * case.spacing[2]
    out = pkg.warp_forward(dev(case.iref), dev(case.dvf), case.grid).cpu().numpy()
    assert np.array_equal(out[0], case.iref)
    want = np.zeros_like(case.iref)
    want[:8 - 3, 1:, :32 - 2] = case.iref[3:, :16 - 1, 2:]
    assert np.array_equal(out[1], want)


def test_warp_non_finite_displacement(pkg):
    case = gsvox_inputs.warp_case(batch=1, dims=(24, 16, 8), seed=44)
    case.dvf[0, 1, 3, 4, 5] = np.nan; case.dvf[0, 0, 2, 2, 2] = np.inf; case.dvf[0, 2, 1, 1, 1] = -np.inf
    ratio, rels = parity(pkg, case)
    out = pkg.warp_forward(dev(case.iref), dev(case.dvf), case.grid).cpu().numpy()
    assert out[0, 3, 4, 5] == 0.0 and out[0, 2, 2, 2] == 0.0 and out[0, 1, 1, 1] == 0.0


def test_warp_far_origin_does_not_matter(pkg):
    """origin cancels in Eq. 2 on a voxel grid (x_v + d - o) / h = i + d / h."""
    case = gsvox_inputs.warp_case(batch=1, dims=(24, 16, 8), seed=45)
    a = pkg.warp_forward(dev(case.iref), dev(case.dvf), case.grid).cpu().numpy()
    case.origin = (1.0e6, -3.0e5, 7.0e4)
    b = pkg.warp_forward(dev(case.iref), dev(case.dvf), case.grid).cpu().numpy()
    assert np.array_equal(a, b)


def test_warp_argument_checks(pkg):
    case = gsvox_inputs.warp_case(batch=1, dims=(8, 8, 8), seed=46)
    bad = (case.grid[0], np.array([1.0, 0.0, 1.0], np.float32), case.grid[2])
    with pytest.raises(pkg.GsvoxError):
        pkg.warp_forward(dev(case.iref), dev(case.dvf), bad)


def test_warp_medium_batch8(pkg):
    parity(pkg, gsvox_inputs.warp_case(batch=8, dims=(128, 96, 64), seed=47))


def test_warp_medium_spacing_not_a_power_of_two(pkg):
    """1/h is inexact in fp32 on all three axes and displacements reach +-12 voxels: the case in which the kernel's
    reciprocal-multiply can put a sample in the neighbouring cell (1.9e7 components).  Tolerances as everywhere."""
    ratio, rels = parity(pkg, gsvox_inputs.warp_case(batch=8, dims=(128, 96, 64), spacing=(1.5, 0.7, 2.3), amp_vox=12.0, seed=48))
    print("warp non-power-of-two spacing: forward err/tol %.3f, grads %s" % (ratio, rels))


def test_warp_full_size_256x256x128(pkg):
    """The size bench times (config-2 grid, 2 mm voxels); B = 2 keeps the numpy oracle to ~1 min."""
    ratio, rels = parity(pkg, gsvox_inputs.warp_case(batch=2))
    print("warp full size: forward err/tol %.3f, grads %s" % (ratio, rels))
