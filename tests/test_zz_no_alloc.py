"""gsvox_project_forward_static — the forward projector with its scratch built into the library (no device
allocation; include/gsvox.h) — against the existing path gsvox_project_forward with caller-owned scratch.  Same
kernels, same launch order: bit-identical results are required (tighter than the projector's parity tolerance
1e-5 max|drr| + 1e-6, which is checked too).  Two calls in a row with different inputs: the second must not see
anything the first left in the shared array.  Collected last on purpose (`pytest -x` stops at the first failure).
`-m gpu`, B200.
"""
import numpy as np
import pytest

import gsvox_inputs

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

FWD_REL, FWD_ABS = 1e-5, 1e-6


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


def both_paths(pkg, case, shared=False):
    vol = dev(case.vol[0] if shared else case.vol)
    angles = list(case.angles)
    ref = pkg.project_forward(vol, case.grid, case.geom, angles)
    out = torch.full_like(ref, float("nan"))                       # every pixel must be written
    torch.cuda.synchronize()
    before = torch.cuda.memory_allocated()
    pkg.project_forward_static(vol, case.grid, case.geom, angles, out)
    torch.cuda.synchronize()
    assert torch.cuda.memory_allocated() == before                 # nothing allocated through torch either
    tol = FWD_REL * float(ref.abs().max()) + FWD_ABS
    err = float((out - ref).abs().max())
    assert err <= tol, "static-scratch projector differs from the scratch path: %.3e > %.3e" % (err, tol)
    assert torch.equal(out, ref), "same kernels, same order: expected identical bits (max diff %.3e)" % err
    return out


def test_static_scratch_projector_matches_scratch_path_on_two_calls_in_a_row(pkg):
    # call 1: 11 angles in every octant, ragged dims, anisotropic spacing, half-fan offsets
    angles = [0.0, 0.5, 1.0, 1.6, 2.4, 3.1, 3.9, 4.7, 5.5, np.pi / 4, -np.pi / 4]
    a = gsvox_inputs.project_case(batch=len(angles), dims=(37, 45, 21), spacing=(2.0, 1.5, 2.5), nu=70, nv=40,
                                  du=3.0, dv=3.0, sad=300.0, sdd=450.0, off_u=9.0, off_v=-4.0, seed=51, angles=angles)
    both_paths(pkg, a)
    # call 2, right after it on the same stream: other volumes, a SMALLER footprint in the shared array (what call 1
    # left beyond it must not matter), then one volume shared by all angles (vol_stride = 0)
    b = gsvox_inputs.project_case(batch=3, dims=(24, 20, 18), nu=48, nv=32, seed=52)
    both_paths(pkg, b)
    both_paths(pkg, b, shared=True)
    # and call 1 again: the array now holds call 2's volumes
    both_paths(pkg, a)


def test_static_scratch_projector_at_its_limit_and_beyond(pkg):
    """One 200x200x100 volume (4 000 000 <= 4 194 304 voxels) is accepted; two are refused with
    GSVOX_ELIMIT by the library and with a message that names the limit by the binding; nothing is enqueued."""
    case = gsvox_inputs.project_case(batch=1, seed=53)
    assert int(np.prod(case.dims)) == 4_000_000
    both_paths(pkg, case)
    two = gsvox_inputs.project_case(batch=2, seed=54)
    out = torch.zeros((2, int(two.geom["nv"]), int(two.geom["nu"])), device="cuda")
    with pytest.raises(pkg.GsvoxError, match="built-in scratch"):
        pkg.project_forward_static(dev(two.vol), two.grid, two.geom, list(two.angles), out)
    import ctypes as C
    from paper_2503_22139_b200 import binding as B_
    g, cg = B_.make_grid(*two.grid), B_.make_cone_geometry(two.geom)
    ang = (C.c_float * 2)(*[float(x) for x in two.angles])
    vol = dev(two.vol)
    rc = pkg.lib().gsvox_project_forward_static(vol.data_ptr(), int(np.prod(two.dims)), C.byref(g), C.byref(cg), ang, 2,
                                                out.data_ptr(), 0)
    assert rc == -5                                                 # GSVOX_ELIMIT
    torch.cuda.synchronize()
    assert not out.any()
