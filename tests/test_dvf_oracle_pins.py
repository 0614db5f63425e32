"""Pins of the MBC -> DVF oracle (oracle.dvf_forward / dvf_backward, SURVEY.md 8(f) rank 1;
PAPER.md:58-61 Eq. 3, :106, :141) to things other than itself: an independent brute force through
library routines (scipy rotations, numpy.linalg.inv), reductions to the plain voxelizer, closed
forms, Euler identities of the (bi)linear map, and central finite differences.  CPU only.
"""
import math

import numpy as np
import pytest
from scipy.spatial.transform import Rotation

import gsvox_inputs
import oracle

TWO_PI_32 = (2.0 * math.pi) ** 1.5


def small_case(batch=3, counts=(4, 9, 25), dims=(22, 18, 14), seed=21, scales=((5.0, 8.0), (2.5, 4.0), (0.8, 2.0))):
    return gsvox_inputs.dvf_case(batch=batch, counts=counts, dims=dims, seed=seed, scales=scales)


def brute_dvf(case, kappa=3.0):
    """d[b,k,x] = sum_i coef[b,i,k] sum_{j in level i} feat[j,k] exp(-1/2 d^T Sigma_j^-1 d) inside the
    3-sigma box, written with library routines only (no oracle call)."""
    nx, ny, nz = case.dims
    o = np.asarray(case.origin, np.float64); h = np.asarray(case.spacing, np.float64)
    out = np.zeros((case.batch, 3, nz, ny, nx))
    coef = case.coef.astype(np.float64)
    for j in range(case.n):
        q = case.quat[j].astype(np.float64)
        R = Rotation.from_quat([q[1], q[2], q[3], q[0]]).as_matrix()       # scipy is (x,y,z,w)
        s = case.scale[j].astype(np.float64)
        Sigma = R @ np.diag(s * s) @ R.T
        Minv = np.linalg.inv(Sigma)
        p = case.pos[j].astype(np.float64)
        r = kappa * np.sqrt(np.diag(Sigma))
        lo = np.maximum(0, np.ceil((p - r - o) / h)).astype(int)
        hi = np.minimum(np.array([nx, ny, nz]) - 1, np.floor((p + r - o) / h)).astype(int)
        if np.any(hi < lo):
            continue
        i = int(case.level[j])
        f = case.feat[j].astype(np.float64)
        for z in range(lo[2], hi[2] + 1):
            for y in range(lo[1], hi[1] + 1):
                xs = np.arange(lo[0], hi[0] + 1)
                d = np.stack([o[0] + xs * h[0] - p[0], np.full(xs.size, o[1] + y * h[1] - p[1]),
                              np.full(xs.size, o[2] + z * h[2] - p[2])], axis=1)
                G = np.exp(-0.5 * np.einsum("na,ab,nb->n", d, Minv, d))
                for b in range(case.batch):
                    for k in range(3):
                        out[b, k, z, y, lo[0]:hi[0] + 1] += coef[b, i, k] * f[k] * G
    return out


def test_dvf_forward_equals_independent_brute_force():
    case = small_case()
    lv, _ = case.levels()
    d = oracle.dvf_forward(lv, case.coef, case.grid)
    ref = brute_dvf(case)
    assert d.shape == ref.shape == (3, 3, 14, 18, 22)
    assert np.abs(d - ref).max() <= 1e-12 * max(1.0, np.abs(ref).max())


def test_single_level_unit_coefficients_reduce_to_the_voxelizer():
    case = small_case(batch=1, counts=(30,), scales=((1.0, 4.0),))
    lv, _ = case.levels()
    coef = np.ones((1, 1, 3), np.float32)
    d = oracle.dvf_forward(lv, coef, case.grid)
    e = oracle.forward(case.pos, case.scale, case.quat, case.feat, case.grid)
    assert np.array_equal(d[0], e)


def test_each_output_component_sees_only_its_own_axis_and_levels():
    """d[b,k] depends on coef[b,:,k] and feat[:,k] only (Eq. 3 per Cartesian direction)."""
    case = small_case()
    lv, _ = case.levels()
    d0 = oracle.dvf_forward(lv, case.coef, case.grid)
    coef = case.coef.copy(); coef[1, :, 2] *= 4.0                     # projection 1, axis z only (exact in fp32)
    d1 = oracle.dvf_forward(lv, coef, case.grid)
    assert np.array_equal(d1[0], d0[0]) and np.array_equal(d1[2], d0[2])
    assert np.array_equal(d1[1, :2], d0[1, :2])
    assert np.allclose(d1[1, 2], 4.0 * d0[1, 2], rtol=1e-13, atol=1e-13)
    coef = case.coef.copy(); coef[:, 1, :] = 0.0                       # drop level 1 entirely
    lv2 = [lv[0], lv[2]]
    d2 = oracle.dvf_forward(lv, coef, case.grid)
    d3 = oracle.dvf_forward(lv2, case.coef[:, [0, 2], :], case.grid)
    assert np.allclose(d2, d3, rtol=0, atol=1e-13)


def test_peak_value_at_a_voxel_centre():
    """Three isotropic Gaussians (one per level) centred on the same voxel centre, nothing else
    nearby: d[b,k] at that voxel is sum_i coef[b,i,k] feat_i[k] exactly (G = 1)."""
    dims = (17, 17, 17)
    pos = np.array([[8, 8, 8]] * 3, np.float32)
    scale = np.array([[3, 3, 3], [2, 2, 2], [1, 1, 1]], np.float32)
    quat = np.array([[1, 0, 0, 0]] * 3, np.float32)
    feat = np.array([[0.5, -1.0, 2.0], [1.5, 0.25, -0.75], [-2.0, 3.0, 1.0]], np.float32)
    coef = np.array([[[1, 2, 3], [4, 5, 6], [7, 8, 9]], [[-1, 0, 1], [0.5, 0.5, 0.5], [2, -2, 2]]], np.float32)
    grid = (np.zeros(3, np.float32), np.ones(3, np.float32), np.asarray(dims, np.int32))
    lv = [(pos[i:i + 1], scale[i:i + 1], quat[i:i + 1], feat[i:i + 1]) for i in range(3)]
    d = oracle.dvf_forward(lv, coef, grid)
    want = np.einsum("bik,ik->bk", coef.astype(np.float64), feat.astype(np.float64))
    assert np.allclose(d[:, :, 8, 8, 8], want, rtol=1e-14, atol=0)


def test_grad_coef_closed_form_for_unit_upstream():
    """g = 1 on one (b,k) volume, wide Gaussians well inside the grid, cutoff 7.5 sigma:
    dL/dcoef[b,i,k] = sum_x e_{i,k}(x) = sum_{j in i} feat[j,k] (2 pi)^{3/2} s0 s1 s2."""
    rng = np.random.default_rng(3)
    dims = (64, 64, 64)
    grid = (np.zeros(3, np.float32), np.ones(3, np.float32), np.asarray(dims, np.int32))
    lv = []
    for n in (2, 3):
        pos = rng.uniform(29, 34, size=(n, 3)).astype(np.float32)
        scale = rng.uniform(2.0, 3.0, size=(n, 3)).astype(np.float32)
        quat = rng.standard_normal((n, 4)).astype(np.float32)
        feat = rng.standard_normal((n, 3)).astype(np.float32)
        lv.append((pos, scale, quat, feat))
    coef = rng.standard_normal((2, 2, 3)).astype(np.float32)
    g = np.zeros((2, 3, 64, 64, 64), np.float32); g[1, 2] = 1.0
    gc, per = oracle.dvf_backward(lv, coef, grid, g, kappa=7.5)
    for i, (pos, scale, quat, feat) in enumerate(lv):
        want = float(np.sum(feat[:, 2].astype(np.float64) * TWO_PI_32 * np.prod(scale.astype(np.float64), axis=1)))
        assert gc[1, i, 2] == pytest.approx(want, rel=1e-9)
        # only the z column of the features is reached, with factor coef[1,i,2]
        gf = per[i][0]
        assert np.allclose(gf[:, :2], 0.0, atol=1e-12)
        want_f = float(coef[1, i, 2]) * TWO_PI_32 * np.prod(scale.astype(np.float64), axis=1)
        assert np.allclose(gf[:, 2], want_f, rtol=1e-9)
    mask = np.ones_like(gc, dtype=bool); mask[1, :, 2] = False
    assert np.all(gc[mask] == 0.0)


def test_euler_identities_of_the_bilinear_map():
    """d is linear in coef and in feat: <coef, dL/dcoef> = <feat, dL/dfeat> = <g, d>."""
    case = small_case()
    lv, _ = case.levels()
    g = case.grad_dvf()
    d = oracle.dvf_forward(lv, case.coef, case.grid)
    gc, per = oracle.dvf_backward(lv, case.coef, case.grid, g)
    L = float(np.sum(g.astype(np.float64) * d))
    assert float(np.sum(case.coef.astype(np.float64) * gc)) == pytest.approx(L, rel=1e-11)
    lf = sum(float(np.sum(f.astype(np.float64) * gl[0])) for (_, _, _, f), gl in zip(lv, per))
    assert lf == pytest.approx(L, rel=1e-11)


def test_backward_against_central_differences_frozen_support():
    """L = <g, d>.  kappa = 60 puts every box on the whole grid, so the support cannot move under
    the perturbation (reading A12).  Central differences with Richardson extrapolation."""
    case = small_case(batch=2, counts=(2, 3, 4), dims=(12, 11, 10), scales=((3.0, 5.0), (2.0, 3.0), (1.2, 2.0)))
    lv, _ = case.levels()
    g = case.grad_dvf()
    kap = 60.0

    def loss(levels, coef):
        return float(np.sum(g.astype(np.float64) * oracle.dvf_forward(levels, coef, case.grid, kappa=kap)))

    gc, per = oracle.dvf_backward(lv, case.coef, case.grid, g, kappa=kap)

    def fd(fun, x, idx, eps):
        def at(e):
            y = x.astype(np.float64).copy(); y[idx] += e
            return fun(y)
        d1 = (at(eps) - at(-eps)) / (2 * eps)
        d2 = (at(2 * eps) - at(-2 * eps)) / (4 * eps)
        return (4 * d1 - d2) / 3

    # the oracle takes fp32 inputs: perturb in steps that fp32 represents exactly (powers of two)
    eps = 2.0 ** -9
    for idx in [(0, 0, 0), (1, 2, 1), (0, 1, 2)]:
        base = case.coef.copy()
        val = fd(lambda c: loss(lv, c.astype(np.float32)), base, idx, eps)
        assert val == pytest.approx(gc[idx], rel=2e-6, abs=1e-7)
    names = ["pos", "scale", "quat", "feat"]
    order = {"feat": 0, "pos": 1, "scale": 2, "quat": 3}
    for i in range(3):
        for which in range(4):
            arr = lv[i][which]
            for idx in [(0, 0), (arr.shape[0] - 1, arr.shape[1] - 1)]:
                def fun(y, i=i, which=which):
                    lev = list(lv)
                    t = list(lev[i]); t[which] = y.astype(np.float32); lev[i] = tuple(t)
                    return loss(lev, case.coef)
                # keep base + k eps exactly representable in fp32
                base = np.round(arr.astype(np.float64) * 64) / 64
                lev0 = list(lv); t = list(lev0[i]); t[which] = base.astype(np.float32); lev0[i] = tuple(t)
                gc0, per0 = oracle.dvf_backward(lev0, case.coef, case.grid, g, kappa=kap)

                def fun0(y, i=i, which=which, lev0=lev0):
                    lev = list(lev0)
                    t = list(lev[i]); t[which] = y.astype(np.float32); lev[i] = tuple(t)
                    return loss(lev, case.coef)
                val = fd(fun0, base, idx, eps)
                got = per0[i][order[names[which]]][idx]
                assert val == pytest.approx(got, rel=5e-5, abs=5e-6), (i, names[which], idx)


def test_mbc_combine_backward_pinned_by_differences_adjoint_and_library_contraction():
    """oracle.mbc_combine_backward (the reference of gsvox_mbc_combine_backward, the batch path) against
    things other than itself: (i) mbc_combine is bilinear, so central differences of L = <g, combine(e, coef)>
    are exact up to rounding; (ii) the adjoint identities <g, combine(e, c)> = <dL/de, e> = <dL/dcoef, c>;
    (iii) numpy's tensor contraction of the same index pattern d[b,k] = sum_i c[b,i,k] e[i,k] (PAPER.md:58-61,
    Eq. 3; :141 for the index meaning); (iv) zero pattern: coefficient (b,i,k) sees only e[i,k] and g[b,k]."""
    rng = np.random.default_rng(77)
    B, L, shp = 3, 4, (3, 4, 5)
    e = rng.standard_normal((L, 3) + shp)
    coef = rng.standard_normal((B, L, 3)).astype(np.float32)
    g = rng.standard_normal((B, 3) + shp)
    ge, gc = oracle.mbc_combine_backward(e, coef, g)
    assert ge.shape == e.shape and gc.shape == (B, L, 3)
    loss = lambda ee, cc: float(np.sum(g * oracle.mbc_combine(ee, cc)))
    base = loss(e, coef)
    # (ii)
    assert float(np.sum(ge * e)) == pytest.approx(base, rel=1e-12)
    assert float(np.sum(gc * coef.astype(np.float64))) == pytest.approx(base, rel=1e-12)
    # (i) bilinear => a central difference with any step is exact
    for idx in [(0, 0, 0), (2, 3, 1), (1, 2, 2)]:
        cp, cm = coef.copy(), coef.copy()
        cp[idx] += 0.5; cm[idx] -= 0.5
        assert loss(e, cp) - loss(e, cm) == pytest.approx(gc[idx], rel=1e-11, abs=1e-12)
    for idx in [(0, 0, 0, 0, 0), (3, 2, 2, 3, 4), (1, 1, 0, 2, 1)]:
        ep, em = e.copy(), e.copy()
        ep[idx] += 0.5; em[idx] -= 0.5
        assert loss(ep, coef) - loss(em, coef) == pytest.approx(ge[idx], rel=1e-11, abs=1e-12)
    # (iii)
    c64 = coef.astype(np.float64)
    assert np.allclose(oracle.mbc_combine(e, coef), np.einsum("bik,ikzyx->bkzyx", c64, e), rtol=1e-13, atol=1e-13)
    assert np.allclose(ge, np.einsum("bik,bkzyx->ikzyx", c64, g), rtol=1e-13, atol=1e-13)
    assert np.allclose(gc, np.einsum("bkzyx,ikzyx->bik", g, e), rtol=1e-13, atol=1e-13)
    # (iv)
    g1 = np.zeros_like(g); g1[1, 2] = g[1, 2]
    ge1, gc1 = oracle.mbc_combine_backward(e, coef, g1)
    mask = np.zeros((B, L, 3), bool); mask[1, :, 2] = True
    assert np.all(gc1[~mask] == 0.0) and np.all(gc1[mask] != 0.0)
    assert np.all(ge1[:, :2] == 0.0) and np.all(ge1[:, 2] != 0.0)


def test_dvf_backward_goes_through_mbc_combine_backward():
    """dvf_backward's coefficient gradient IS mbc_combine_backward's on the voxelized MBC volumes (so the pins of
    dvf_backward above — closed form, Euler identities, central differences — also hold it in place)."""
    case = small_case()
    lv, _ = case.levels()
    g = case.grad_dvf()
    gc, _ = oracle.dvf_backward(lv, case.coef, case.grid, g)
    _, gc2 = oracle.mbc_combine_backward(oracle.mbc_volumes(lv, case.grid), case.coef, g)
    assert np.array_equal(gc, gc2)
