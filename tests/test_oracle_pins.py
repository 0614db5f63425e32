"""Pins of the fp64 oracle (oracle/) to things other than itself.

Each test names what fixes the expected value: a closed form, an invariant, a library
routine (scipy rotations, numpy.linalg.inv), brute force through those library routines,
central finite differences, or a worked value from tests/golden/ (with its citation).
A plausible mistake in the oracle (a dropped term, a wrong sign or index, a transposed
operand, an off-by-one box bound, a wrong layout) must fail at least one test here.
CPU only; the CUDA path is never imported.
"""
import json
import math
import os

import numpy as np
import pytest
from scipy.spatial.transform import Rotation
from scipy.special import ndtr

import oracle

TWO_PI_32 = (2.0 * math.pi) ** 1.5


def f32(x):
    return np.asarray(x, dtype=np.float32)


def grid_of(dims, origin=(0, 0, 0), spacing=(1, 1, 1)):
    return (f32(origin), f32(spacing), np.asarray(dims, np.int32))


def rand_quat(rng, n=1):
    q = rng.standard_normal((n, 4))
    return f32(q * rng.uniform(0.3, 3.0, size=(n, 1)))      # deliberately unnormalised


# ----------------------------------------------------------------------------- golden
def test_survey_worked_values(golden_dir):
    """Worked values of SURVEY.md 8(c) 'Pins' (independent numpy script, fp64 inputs).
    The oracle takes fp32 inputs, so w = fp32(0.7) rescales the sums by fp32(0.7)/0.7
    exactly (forward is linear in w); p rounds by < 1 ulp(fp32), which the sums of a wide
    Gaussian do not see at 1e-9 but the truncation remainder dL/dp (kappa = 3) does."""
    G = json.load(open(os.path.join(golden_dir, "survey_worked_values.json")))
    grid = grid_of(G["grid"]["dims"], G["grid"]["origin"], G["grid"]["spacing"])
    p = f32([G["p"]]); w = f32([[G["w"]]])
    wfix = float(w[0, 0]) / G["w"]
    for case in G["forward"]:
        s, q, k = f32([case["s"]]), f32([case["q"]]), case["kappa"]
        geo = oracle.geometry(p, s, q, grid, kappa=k)
        assert geo["box"][0].tolist() == case["box_lo"] + case["box_hi"]
        out, pairs = oracle.forward(p, s, q, w, grid, kappa=k, return_pairs=True)
        assert out.sum() == pytest.approx(case["sum_out"] * wfix, rel=2e-9)
        ext = np.array(case["box_hi"]) - np.array(case["box_lo"]) + 1
        assert pairs == int(np.prod(ext))
        if "closed_form" in case:
            assert out.sum() == pytest.approx(case["closed_form"] * wfix, rel=2e-9)
    g1 = np.ones((1, 64, 64, 64), np.float32)
    for case in G["backward_g_equal_1"]:
        s, q, k = f32([case["s"]]), f32([case["q"]]), case["kappa"]
        gw, gp, gs, gq = oracle.backward(p, s, q, w, grid, g1, kappa=k)
        assert gw[0, 0] == pytest.approx(case["dw"], rel=2e-9)
        np.testing.assert_allclose(gs[0], np.array(case["ds"]) * wfix, rtol=3e-8)
        if "dp" in case:
            np.testing.assert_allclose(gp[0], case["dp"], rtol=2e-5, atol=2e-8)
        else:
            assert np.abs(gp).max() < 10 * case["dp_abs_below"]
            assert np.abs(gq).max() < 10 * case["dq_abs_below"]


# ----------------------------------------------------------------------- closed forms
@pytest.mark.parametrize("seed", [0, 1, 2])
def test_untruncated_integral_closed_form(seed):
    """sum_x out * voxel volume = w (2 pi)^{3/2} s0 s1 s2 for a Gaussian wide relative to
    the voxel, any rotation, any spacing/origin, kappa >= 7.5 (Gaussian integral)."""
    rng = np.random.default_rng(seed)
    spacing = rng.uniform(0.8, 1.25, 3)
    dims = (100, 104, 98)
    origin = rng.uniform(-20, 20, 3)
    centre = origin + spacing * (np.array(dims) - 1) / 2 + rng.uniform(-0.5, 0.5, 3)
    s = rng.uniform(2.2, 3.0, 3) * spacing.max()          # 7.5 sigma stays inside the grid
    q = rand_quat(rng)
    w = f32([[rng.uniform(-2, 2)]])
    grid = grid_of(dims, origin, spacing)
    out = oracle.forward(f32([centre]), f32([s]), q, w, grid, kappa=7.5)
    s32 = f32(s).astype(np.float64); h32 = f32(spacing).astype(np.float64)
    expect = float(w[0, 0]) * TWO_PI_32 * s32.prod()
    assert out.sum() * h32.prod() == pytest.approx(expect, rel=1e-9)


def test_box_truncated_closed_form_kappa3():
    """kappa = 3, axis-aligned: the box sum factorises into three 1-D sums, each close to
    s sqrt(2 pi) [Phi((hi+1/2-p)/s) - Phi((lo-1/2-p)/s)] (midpoint rule; reading A16)."""
    p = np.array([31.3, 31.7, 31.5]); s = np.array([4.0, 3.0, 5.0])
    grid = grid_of((64, 64, 64))
    geo = oracle.geometry(f32([p]), f32([s]), f32([[1, 0, 0, 0]]), grid)
    lo, hi = geo["box"][0, :3], geo["box"][0, 3:]
    out = oracle.forward(f32([p]), f32([s]), f32([[1, 0, 0, 0]]), f32([[0.7]]), grid)
    p32 = f32(p).astype(float)
    expect = float(f32(0.7))
    for k in range(3):
        expect *= s[k] * math.sqrt(2 * math.pi) * (ndtr((hi[k] + 0.5 - p32[k]) / s[k])
                                                   - ndtr((lo[k] - 0.5 - p32[k]) / s[k]))
    assert out.sum() == pytest.approx(expect, rel=5e-4)
    # and the 3-sigma mass fraction erf(3/sqrt2)^3 = 0.99192 within the +-1 voxel slack
    full = float(f32(0.7)) * TWO_PI_32 * s.prod()
    assert 0.985 < out.sum() / full < 0.997


def test_peak_value_and_sign():
    """out(p) = w when p sits exactly on a voxel centre; negative weights give negative
    output (negative-permitting voxelizer)."""
    grid = grid_of((20, 18, 16), origin=(1.0, -2.0, 0.5), spacing=(0.5, 0.25, 2.0))
    p = np.array([1.0 + 0.5 * 7, -2.0 + 0.25 * 9, 0.5 + 2.0 * 5])
    rng = np.random.default_rng(5)
    out = oracle.forward(f32([p]), f32([[0.9, 1.7, 1.2]]), rand_quat(rng), f32([[-1.25]]), grid)
    assert out[0, 5, 9, 7] == pytest.approx(-1.25, abs=1e-15)     # layout [c, k, j, i]
    assert out.min() == out[0, 5, 9, 7] and out.max() <= 0.0


def test_axis_aligned_is_outer_product_with_layout():
    """Identity rotation: out[k,j,i] = w gx[i] gy[j] gz[k] inside the box, 0 outside.
    Distinct nx, ny, nz and distinct scales catch any axis/layout transposition."""
    dims = (23, 17, 11)
    spacing = (1.0, 1.25, 0.8); origin = (-3.0, 2.0, 7.0)
    grid = grid_of(dims, origin, spacing)
    p = np.array([8.3, 12.1, 10.4]); s = np.array([1.7, 2.9, 1.1]); w = 0.6
    out = oracle.forward(f32([p]), f32([s]), f32([[2, 0, 0, 0]]), f32([[w]]), grid)[0]
    p32, s32 = f32(p).astype(float), f32(s).astype(float)
    axes = []
    for k in range(3):
        x = float(f32(origin[k])) + np.arange(dims[k]) * float(f32(spacing[k]))
        g = np.exp(-0.5 * ((x - p32[k]) / s32[k]) ** 2)
        g[np.abs(x - p32[k]) > 3.0 * s32[k]] = 0.0               # reading A3/A4: closed box
        axes.append(g)
    expect = float(f32(w)) * axes[2][:, None, None] * axes[1][None, :, None] * axes[0][None, None, :]
    np.testing.assert_allclose(out, expect, rtol=1e-12, atol=1e-300)
    assert (expect == 0).sum() > 0 and (expect != 0).sum() > 0


# ---------------------------------------------------------- library-routine geometry
def test_rotation_matches_scipy_and_inverse_matches_numpy():
    """R(q) against scipy's Rotation (scalar-LAST there), M against numpy.linalg.inv of
    Sigma = R S S^T R^T (north_star's parameterisation, reading A1)."""
    rng = np.random.default_rng(7)
    n = 64
    q = rand_quat(rng, n); s = f32(rng.uniform(0.4, 5.0, (n, 3))); p = f32(rng.uniform(0, 30, (n, 3)))
    geo = oracle.geometry(p, s, q, grid_of((32, 32, 32)))
    q64 = q.astype(np.float64)
    Rs = Rotation.from_quat(q64[:, [1, 2, 3, 0]]).as_matrix()
    np.testing.assert_allclose(geo["R"], Rs, atol=1e-14)
    for i in range(n):
        S2 = np.diag(s[i].astype(np.float64) ** 2)
        Minv = np.linalg.inv(Rs[i] @ S2 @ Rs[i].T)
        M = geo["M"][i]
        Mfull = np.array([[M[0], M[1], M[2]], [M[1], M[3], M[4]], [M[2], M[4], M[5]]])
        np.testing.assert_allclose(Mfull, Minv, rtol=1e-10, atol=1e-13)


def test_forward_brute_force_through_library_routines():
    """Tiny case, pure-Python loops over every (Gaussian, voxel) pair: R from scipy,
    Sigma^-1 from numpy.linalg.inv, support from the ellipsoid-tangent box
    kappa*sqrt(diag(Sigma)) evaluated with numpy on the voxel-centre coordinates."""
    rng = np.random.default_rng(3)
    dims = (9, 7, 6); origin = np.array([-1.0, 0.5, 2.0]); spacing = np.array([1.0, 0.5, 1.5])
    n, C = 4, 2
    p = f32(origin + rng.uniform(0, 1, (n, 3)) * spacing * np.array(dims))
    s = f32(rng.uniform(0.5, 1.6, (n, 3))); q = rand_quat(rng, n); w = f32(rng.standard_normal((n, C)))
    out = oracle.forward(p, s, q, w, grid_of(dims, origin, spacing))
    expect = np.zeros((C, dims[2], dims[1], dims[0]))
    for g in range(n):
        R = Rotation.from_quat(q[g].astype(float)[[1, 2, 3, 0]]).as_matrix()
        Sig = R @ np.diag(s[g].astype(float) ** 2) @ R.T
        Minv = np.linalg.inv(Sig)
        half = 3.0 * np.sqrt(np.diag(Sig))
        for k in range(dims[2]):
            for j in range(dims[1]):
                for i in range(dims[0]):
                    x = origin + np.array([i, j, k]) * spacing
                    d = x - p[g].astype(float)
                    if np.all(np.abs(d) <= half):
                        expect[:, k, j, i] += w[g].astype(float) * math.exp(-0.5 * d @ Minv @ d)
    np.testing.assert_allclose(out, expect, rtol=1e-11, atol=1e-14)
    assert np.count_nonzero(expect) > 50


def test_box_is_tangent_to_the_kappa_sigma_ellipsoid():
    """The box is the AABB of {d : d^T Sigma^-1 d <= kappa^2}: points p + kappa R S u
    (|u| = 1) sampled on the surface never leave it and come within a voxel of each face."""
    rng = np.random.default_rng(11)
    h = 0.05
    grid = grid_of((4000, 4000, 4000), origin=(-100, -100, -100), spacing=(h, h, h))
    for _ in range(5):
        p = rng.uniform(-5, 5, 3); s = rng.uniform(0.5, 6.0, 3); q = rand_quat(rng)
        geo = oracle.geometry(f32([p]), f32([s]), q, grid)
        lo, hi = geo["box"][0, :3], geo["box"][0, 3:]
        u = rng.standard_normal((200000, 3)); u /= np.linalg.norm(u, axis=1, keepdims=True)
        R = Rotation.from_quat(q[0].astype(float)[[1, 2, 3, 0]]).as_matrix()
        pts = f32(p).astype(float) + 3.0 * (u * f32(s).astype(float)) @ R.T
        idx = (pts + 100.0) / h
        # lo = ceil(extreme), hi = floor(extreme): the surface stays within one voxel outside
        assert np.all(idx.min(0) > lo - 1 - 1e-9) and np.all(idx.max(0) < hi + 1 + 1e-9)
        # and the sampled extremes reach the faces up to the sampling resolution of the sphere
        slack = 0.002 * (hi - lo)
        assert np.all(idx.min(0) <= lo + slack) and np.all(idx.max(0) >= hi - slack)


def test_box_bounds_inclusive_closed_interval():
    """A voxel centre exactly at distance 3*sigma is inside (closed interval, reading A4);
    one ulp further out it is not."""
    grid = grid_of((32, 8, 8))
    # s = 2 (exact in fp32): r = 6, p = 10 -> centres 4 and 16 lie exactly on the faces
    geo = oracle.geometry(f32([[10, 4, 4]]), f32([[2, 1, 1]]), f32([[1, 0, 0, 0]]), grid)
    assert geo["box"][0].tolist() == [4, 1, 1, 16, 7, 7]
    p_up = np.nextafter(np.float32(10), np.float32(11))
    geo = oracle.geometry(f32([[p_up, 4, 4]]), f32([[2, 1, 1]]), f32([[1, 0, 0, 0]]), grid)
    assert geo["box"][0].tolist() == [5, 1, 1, 16, 7, 7]
    out = oracle.forward(f32([[10, 4, 4]]), f32([[2, 1, 1]]), f32([[1, 0, 0, 0]]), f32([[1]]), grid)
    assert out[0, 4, 4, 4] == pytest.approx(math.exp(-4.5), rel=1e-14)       # included face voxel
    assert out[0, 4, 4, 3] == 0.0 and out[0, 4, 4, 17] == 0.0


# ------------------------------------------------------------------------- invariants
def _random_case(rng, n, C, dims, smin=0.6, smax=3.0):
    p = f32(rng.uniform(-2, np.array(dims) + 1, (n, 3)))
    s = f32(np.exp(rng.uniform(np.log(smin), np.log(smax), (n, 3))))
    q = rand_quat(rng, n)
    w = f32(rng.standard_normal((n, C)))
    return p, s, q, w


def test_linearity_superposition_and_channels():
    rng = np.random.default_rng(21)
    dims = (20, 22, 18); grid = grid_of(dims)
    p, s, q, w = _random_case(rng, 30, 3, dims)
    out = oracle.forward(p, s, q, w, grid)
    # channels are independent scalar problems sharing geometry (reading A10)
    for c in range(3):
        oc = oracle.forward(p, s, q, w[:, c:c + 1], grid)
        np.testing.assert_allclose(out[c], oc[0], rtol=1e-13, atol=1e-15)
    # linear in w
    w2 = f32(rng.standard_normal(w.shape))
    o2 = oracle.forward(p, s, q, w2, grid)
    wsum = f32(w.astype(np.float64) * 2 + w2.astype(np.float64))       # exact? keep fp32-representable
    os_ = oracle.forward(p, s, q, wsum, grid)
    # compare against the fp32-rounded combination actually passed in
    ref = np.zeros_like(out)
    unit = oracle.forward(p, s, q, f32(np.ones_like(w)), grid)         # not used for scaling check
    for i in range(30):
        oi = oracle.forward(p[i:i + 1], s[i:i + 1], q[i:i + 1], f32(np.ones((1, 3))), grid)
        ref += oi * wsum[i].astype(np.float64)[:, None, None, None]
    np.testing.assert_allclose(os_, ref, rtol=1e-12, atol=1e-13)
    # superposition: voxelize(A u B) = voxelize(A) + voxelize(B)
    oa = oracle.forward(p[:13], s[:13], q[:13], w[:13], grid)
    ob = oracle.forward(p[13:], s[13:], q[13:], w[13:], grid)
    np.testing.assert_allclose(out, oa + ob, rtol=1e-12, atol=1e-14)
    assert unit.shape == out.shape and o2.shape == out.shape


def test_rotation_identities():
    rng = np.random.default_rng(22)
    dims = (24, 24, 24); grid = grid_of(dims)
    p = f32([[11.3, 12.6, 10.2]]); w = f32([[0.8]])
    # isotropic: output independent of q
    s_iso = f32([[2.5, 2.5, 2.5]])
    o1 = oracle.forward(p, s_iso, rand_quat(rng), w, grid)
    o2 = oracle.forward(p, s_iso, rand_quat(rng), w, grid)
    np.testing.assert_allclose(o1, o2, rtol=1e-10, atol=1e-14)
    # q, -q and lambda*q (lambda > 0) are the same rotation (reading A2)
    s = f32([[1.5, 2.5, 3.5]]); q = rand_quat(rng)
    o = oracle.forward(p, s, q, w, grid)
    np.testing.assert_array_equal(o, oracle.forward(p, s, -q, w, grid))
    np.testing.assert_allclose(o, oracle.forward(p, s, f32(4.0 * q), w, grid), rtol=1e-12, atol=1e-15)
    # 90 degrees about z maps local x -> world y, local y -> -world x: same as swapping s0,s1
    c = math.sqrt(0.5)
    o_rot = oracle.forward(p, s, f32([[c, 0, 0, c]]), w, grid)
    o_perm = oracle.forward(p, f32([[2.5, 1.5, 3.5]]), f32([[1, 0, 0, 0]]), w, grid)
    np.testing.assert_allclose(o_rot, o_perm, rtol=1e-6, atol=1e-9)     # c is rounded to fp32
    # 90 degrees about x swaps s1,s2
    o_rot = oracle.forward(p, s, f32([[c, c, 0, 0]]), w, grid)
    o_perm = oracle.forward(p, f32([[1.5, 3.5, 2.5]]), f32([[1, 0, 0, 0]]), w, grid)
    np.testing.assert_allclose(o_rot, o_perm, rtol=1e-6, atol=1e-9)
    # an anisotropic Gaussian rotated by +30 deg about z is elongated along (cos30, sin30):
    # a sign error in R would put the ridge at -30 deg
    th = math.radians(30)
    qz = f32([[math.cos(th / 2), 0, 0, math.sin(th / 2)]])
    o = oracle.forward(f32([[12, 12, 12]]), f32([[3.0, 0.7, 0.7]]), qz, w, grid)[0]
    assert o[12, 12 + 2, 12 + 3] > 10 * o[12, 12 - 2, 12 + 3]


def test_outside_clipped_degenerate_and_empty():
    dims = (16, 12, 10); grid = grid_of(dims)
    q = f32([[1, 0, 0, 0]])
    # wholly outside -> empty box, zero output, zero pairs (reading A11)
    out, pairs = oracle.forward(f32([[-40, 5, 5]]), f32([[1, 1, 1]]), q, f32([[1]]), grid, return_pairs=True)
    assert pairs == 0 and not out.any()
    # partly outside -> box clipped to the grid
    geo = oracle.geometry(f32([[0.2, 11.0, 9.4]]), f32([[1, 1, 1]]), q, grid)
    assert geo["box"][0].tolist() == [0, 8, 7, 3, 11, 9] and geo["flags"][0] == 0
    # sub-voxel Gaussian between voxel centres -> empty box even though it is inside the grid
    geo = oracle.geometry(f32([[5.5, 5.5, 5.5]]), f32([[0.1, 0.1, 0.1]]), q, grid)
    assert geo["flags"][0] == 2 and geo["box"][0].tolist() == [0, 0, 0, -1, -1, -1]
    # degenerate inputs are skipped, counted via flag bit 0, contribute nothing
    P = f32([[5, 5, 5]] * 6); S = f32([[1, 1, 1]] * 6); Q = f32([[1, 0, 0, 0]] * 6)
    S[1, 2] = 0.0; S[2, 0] = -1.0; Q[3] = 0.0; P[4, 1] = np.nan; S[5, 1] = np.inf
    geo = oracle.geometry(P, S, Q, grid)
    assert geo["flags"].tolist() == [0, 1, 1, 1, 1, 1]
    W = f32(np.ones((6, 1)))
    out = oracle.forward(P, S, Q, W, grid)
    np.testing.assert_array_equal(out, oracle.forward(P[:1], S[:1], Q[:1], W[:1], grid))
    g = np.ones((1, 10, 12, 16), np.float32)
    gw, gp, gs, gq = oracle.backward(P, S, Q, W, grid, g)
    assert not gw[1:].any() and not gp[1:].any() and not gs[1:].any() and not gq[1:].any()
    assert np.isfinite(gw).all() and gw[0, 0] > 0
    # no Gaussians at all
    out = oracle.forward(np.zeros((0, 3)), np.zeros((0, 3)), np.zeros((0, 4)), np.zeros((0, 1)), grid)
    assert out.shape == (1, 10, 12, 16) and not out.any()


def test_pair_count_is_sum_of_box_volumes():
    rng = np.random.default_rng(23)
    dims = (30, 26, 22); grid = grid_of(dims)
    p, s, q, w = _random_case(rng, 200, 1, dims)
    geo = oracle.geometry(p, s, q, grid)
    ext = np.clip(geo["box"][:, 3:] - geo["box"][:, :3] + 1, 0, None)
    _, pairs = oracle.forward(p, s, q, w, grid, return_pairs=True)
    assert pairs == int(ext.prod(1).sum())


# ---------------------------------------------------------------------------- backward
def test_backward_closed_form_unit_gradient():
    """g = 1, kappa >= 7.5: L = sum out = w (2pi)^{3/2} s0 s1 s2 / voxel volume, hence
    dL/dw = L/w, dL/ds_k = L/s_k, dL/dp = 0, dL/dq = 0 (SURVEY 8(c) pins)."""
    rng = np.random.default_rng(31)
    dims = (70, 70, 70); spacing = np.array([1.0, 0.8, 1.25]); origin = np.array([3.0, -4.0, 5.0])
    grid = grid_of(dims, origin, spacing)
    p = f32([origin + spacing * 34.5 + rng.uniform(-0.4, 0.4, 3)])
    s = f32([rng.uniform(2.6, 3.4, 3)]); q = rand_quat(rng); w = f32([[-0.85]])
    g = np.ones((1,) + dims[::-1], np.float32)
    gw, gp, gs, gq = oracle.backward(p, s, q, w, grid, g, kappa=7.5)
    vol = float(np.prod(f32(spacing).astype(float)))
    base = TWO_PI_32 * float(np.prod(s.astype(float))) / vol
    assert gw[0, 0] == pytest.approx(base, rel=1e-9)
    np.testing.assert_allclose(gs[0], float(w[0, 0]) * base / s[0].astype(float), rtol=1e-8)
    assert np.abs(gp).max() < 1e-8 * base and np.abs(gq).max() < 1e-8 * base


def _loss(p, s, q, w, grid, g, kappa):
    return float((oracle.forward(p, s, q, w, grid, kappa=kappa) * g).sum())


def _fd(fun, x, idx, eps):
    """Richardson-extrapolated central difference; eps and eps/2 are exact in fp32
    because every parameter is a multiple of 2^-10 and eps is a power of two."""
    def cd(e):
        xp = x.copy(); xm = x.copy()
        xp[idx] += e; xm[idx] -= e
        assert float(xp[idx]) - float(x[idx]) == e and float(x[idx]) - float(xm[idx]) == e
        return (fun(xp) - fun(xm)) / (2 * e)
    return (4.0 * cd(eps / 2) - cd(eps)) / 3.0


@pytest.mark.parametrize("kappa,frozen_by", [(60.0, "grid"), (3.0, "margin")])
def test_backward_matches_finite_differences(kappa, frozen_by):
    """Central finite differences of the oracle's own forward with frozen boxes (reading
    A12).  kappa = 60: every box is the whole (tiny) grid, so the support cannot move and
    the truncation at the grid faces is live.  kappa = 3: boxes strictly inside; the test
    asserts that no box changes under the +-eps perturbations it applies."""
    rng = np.random.default_rng(41)
    dims = (13, 11, 12)
    spacing = (1.0, 0.75, 1.5); origin = (-2.0, 1.0, 0.5)
    grid = grid_of(dims, origin, spacing)
    n, C = 3, 2
    quant = lambda a: f32(np.round(np.asarray(a) * 1024) / 1024)
    ext = np.array(dims) * np.array(spacing)
    p = quant(np.array(origin) + rng.uniform(0.35, 0.65, (n, 3)) * ext)
    s = quant(rng.uniform(0.8, 1.3, (n, 3)) if kappa == 3.0 else rng.uniform(1.5, 3.0, (n, 3)))
    q = quant(rng.standard_normal((n, 4)) * 1.7)
    w = quant(rng.standard_normal((n, C)))
    g = rng.standard_normal((C, dims[2], dims[1], dims[0])).astype(np.float32)
    g64 = g.astype(np.float64)
    eps = 2.0 ** -7
    box0 = oracle.geometry(p, s, q, grid, kappa=kappa)["box"]
    if frozen_by == "grid":
        assert (box0 == np.array([0, 0, 0, dims[0] - 1, dims[1] - 1, dims[2] - 1])).all()
    gw, gp, gs, gq = oracle.backward(p, s, q, w, grid, g, kappa=kappa)
    checks = [("w", w, gw, lambda v: _loss(p, s, q, v, grid, g64, kappa)),
              ("p", p, gp, lambda v: _loss(v, s, q, w, grid, g64, kappa)),
              ("s", s, gs, lambda v: _loss(p, v, q, w, grid, g64, kappa)),
              ("q", q, gq, lambda v: _loss(p, s, v, w, grid, g64, kappa))]
    for name, x, grad, fun in checks:
        fd = np.zeros_like(grad)
        for idx in np.ndindex(*x.shape):
            if frozen_by == "margin" and name != "w":
                for e in (eps, eps / 2):
                    for sgn in (1, -1):
                        xx = x.copy(); xx[idx] += sgn * e
                        args = {"p": (xx, s, q), "s": (p, xx, q), "q": (p, s, xx)}[name]
                        assert (oracle.geometry(*args, grid, kappa=kappa)["box"] == box0).all(), \
                            "box moved under perturbation; pick another seed"
            fd[idx] = _fd(fun, x, idx, eps)
        err = np.linalg.norm(fd - grad) / np.linalg.norm(grad)
        assert err < 2e-7, (name, err)


def test_backward_invariants():
    """q . dL/dq = 0 (gradient wrt the unnormalised quaternion, reading A2); dL/dw does not
    depend on w; every gradient is linear in the upstream gradient."""
    rng = np.random.default_rng(51)
    dims = (18, 16, 14); grid = grid_of(dims, (0.5, 0.5, 0.5), (1.0, 1.2, 0.9))
    p, s, q, w = _random_case(rng, 40, 3, dims)
    g = rng.standard_normal((3, dims[2], dims[1], dims[0])).astype(np.float32)
    gw, gp, gs, gq = oracle.backward(p, s, q, w, grid, g)
    dots = np.abs((gq * q.astype(np.float64)).sum(1))
    assert dots.max() < 1e-12 * max(1.0, np.abs(gq).max())
    gw2, gp2, _, _ = oracle.backward(p, s, q, f32(4 * w), grid, g)      # x4 is exact in fp32
    np.testing.assert_allclose(gw2, gw, rtol=1e-13)
    np.testing.assert_allclose(gp2, 4 * gp, rtol=1e-12, atol=1e-13)
    r = oracle.backward(p, s, q, w, grid, f32(2 * g))
    for a, b in zip(r, (gw, gp, gs, gq)):
        np.testing.assert_allclose(a, 2 * b, rtol=1e-12, atol=1e-13)
    # a rescaled quaternion gives a rescaled-by-1/lambda gradient (same rotation)
    r = oracle.backward(p, s, f32(2 * q), w, grid, g)
    np.testing.assert_allclose(r[3], gq / 2, rtol=1e-10, atol=1e-12)
    np.testing.assert_allclose(r[2], gs, rtol=1e-10, atol=1e-12)


def test_spot_check_entry_points_agree_with_full_versions():
    rng = np.random.default_rng(61)
    dims = (21, 19, 17); grid = grid_of(dims, (1, 2, 3), (0.9, 1.1, 1.3))
    p, s, q, w = _random_case(rng, 80, 2, dims)
    g = rng.standard_normal((2, dims[2], dims[1], dims[0])).astype(np.float32)
    out = oracle.forward(p, s, q, w, grid)
    vox = rng.choice(dims[0] * dims[1] * dims[2], 500, replace=False)
    at = oracle.forward_at(p, s, q, w, grid, vox)
    np.testing.assert_allclose(at, out.reshape(2, -1)[:, vox], rtol=1e-13, atol=1e-16)
    full = oracle.backward(p, s, q, w, grid, g)
    ids = rng.choice(80, 25, replace=False)
    some = oracle.backward_for(p, s, q, w, grid, g, ids)
    for a, b in zip(some, full):
        np.testing.assert_array_equal(a, b[ids])
