"""Pins of the X-ray splat oracle (oracle/splat.py; Eq. 6-9) to things
other than itself: the closed-form line integral of a 3D Gaussian (Eq. 6-7) — exactly on the ray
through the centre, and to O(sigma / distance) elsewhere, shrinking with sigma as a local affine
approximation must; agreement with the OTHER two operators (voxelize, then cone-beam project);
linearity, isotropy, cutoff semantics, and finite differences of the autograd gradients.  CPU only.
"""
import math

import numpy as np
import pytest
from scipy.spatial.transform import Rotation

import oracle

GEOM = dict(sad=1000.0, sdd=1500.0, nu=65, nv=49, du=1.0, dv=1.0, off_u=0.0, off_v=0.0, iso=[0.0, 0.0, 0.0])


def f32(a):
    return np.asarray(a, dtype=np.float32)


def scanner(geom, angle):
    a = float(np.float32(angle))
    ca, sa = math.cos(a), math.sin(a)
    src = np.array(geom["iso"], np.float64) + geom["sad"] * np.array([ca, sa, 0.0])
    detc = src - geom["sdd"] * np.array([ca, sa, 0.0])
    return src, detc, np.array([-sa, ca, 0.0]), np.array([0.0, 0.0, 1.0])


def pixel_world(geom, angle, iu, iv):
    src, detc, uh, vh = scanner(geom, angle)
    u = (iu - (geom["nu"] - 1) / 2.0) * geom["du"] + geom["off_u"]
    v = (iv - (geom["nv"] - 1) / 2.0) * geom["dv"] + geom["off_v"]
    return src, detc + u * uh + v * vh


def exact_line_integral(pos, scale, quat, rho, geom, angle, iu, iv):
    """Eq. 6-7 in closed form: int rho exp(-1/2 (o + t d - p)^T M (o + t d - p)) dt over the whole line."""
    q = np.asarray(quat, np.float64)
    R = Rotation.from_quat([q[1], q[2], q[3], q[0]]).as_matrix()
    M = np.linalg.inv(R @ np.diag(np.asarray(scale, np.float64) ** 2) @ R.T)
    src, pix = pixel_world(geom, angle, iu, iv)
    d = (pix - src) / np.linalg.norm(pix - src)
    delta = src - np.asarray(pos, np.float64)
    dMd, dMD, DMD = d @ M @ d, d @ M @ delta, delta @ M @ delta
    return float(rho) * math.sqrt(2 * math.pi / dMd) * math.exp(-0.5 * (DMD - dMD * dMD / dMd))


def one(pos, scale, quat, rho=0.8):
    return f32([pos]), f32([scale]), f32([quat]), f32([rho])


@pytest.mark.parametrize("angle,iu,iv,depth", [(0.0, 32, 24, 0.62), (0.9, 40, 10, 0.7), (2.6, 12, 37, 0.66), (-1.2, 50, 30, 0.58)])
def test_value_on_the_ray_through_the_centre_is_the_exact_line_integral(angle, iu, iv, depth):
    """On the ray through the Gaussian's centre the local affine approximation is exact:
    rho^ = rho sqrt(2 pi |Sigma~| / |Sigma^|) = rho sqrt(2 pi / (d^T Sigma^-1 d))."""
    src, pix = pixel_world(GEOM, angle, iu, iv)
    p = src + depth * (pix - src)
    pos, scale, quat, rho = one(p, (6.0, 3.0, 9.0), (0.8, -0.3, 0.4, 0.2))
    got = oracle.splat_forward_at(pos, scale, quat, rho, GEOM, angle, [(iu, iv)])[0]
    want = exact_line_integral(pos[0], scale[0], quat[0], rho[0], GEOM, angle, iu, iv)
    assert got == pytest.approx(want, rel=2e-6)            # the fp32 position is ~1e-4 pixel off the pixel centre


def test_splat_approaches_the_exact_line_integral_as_sigma_over_distance_shrinks():
    errs = []
    for sig in (8.0, 2.0):
        pos, scale, quat, rho = one((30.0, -20.0, 10.0), (sig, 0.6 * sig, 1.4 * sig), (0.9, 0.1, -0.3, 0.2))
        geom = dict(GEOM, nu=257, nv=257, du=0.25 * sig, dv=0.25 * sig)
        img = oracle.splat_forward(pos, scale, quat, rho, geom, [0.4], kappa=3.0)[0]
        cu, cv, A, B, C, amp, box, valid = oracle.splat_terms(*[oracle.splat._t(x) for x in (pos, scale, quat)],
                                                              oracle.splat._t(rho).reshape(-1), geom, 0.4)
        u0, v0, u1, v1 = (int(x) for x in box[0])
        assert bool(valid[0]) and u1 - u0 > 10 and v1 - v0 > 10
        worst = 0.0
        for iv in range(v0, v1 + 1, 3):
            for iu in range(u0, u1 + 1, 3):
                ex = exact_line_integral(pos[0], scale[0], quat[0], rho[0], geom, 0.4, iu, iv)
                worst = max(worst, abs(img[iv, iu] - ex))
        errs.append(worst / img.max())
    assert errs[0] < 0.03 and errs[1] < 0.008
    assert errs[1] < 0.4 * errs[0]                          # first order in sigma / distance


def test_agrees_with_voxelize_then_project():
    """The two routes of PAPER.md:104 — splat the Gaussians, or voxelize them (Eq. 5) and project the
    volume (Eq. 6) — must give the same DRR up to discretisation: pins the scanner conventions of
    the three operators against each other."""
    rng = np.random.default_rng(3)
    n = 6
    pos = rng.uniform(-25, 25, (n, 3)); scale = rng.uniform(5.0, 9.0, (n, 3))
    quat = rng.standard_normal((n, 4)); rho = rng.uniform(0.2, 1.0, n)
    dims, h = (64, 64, 64), 2.0
    grid = (f32([-(d - 1) / 2 * h for d in dims]), f32([h] * 3), np.asarray(dims, np.int32))
    geom = dict(GEOM, nu=96, nv=96, du=2.0, dv=2.0, off_u=3.0, off_v=-5.0)
    vol = oracle.forward(f32(pos), f32(scale), f32(quat), f32(rho).reshape(n, 1), grid, kappa=5.0)[0]
    for angle in (0.3, 2.0):
        drr = oracle.project_forward(vol, grid, geom, [angle])[0]
        spl = oracle.splat_forward(f32(pos), f32(scale), f32(quat), f32(rho), geom, [angle], kappa=5.0)[0]
        assert np.abs(drr - spl).max() <= 0.03 * spl.max()
        assert abs(drr.sum() - spl.sum()) <= 0.01 * spl.sum()


def test_linear_in_rho_superposition_and_isotropy():
    rng = np.random.default_rng(4)
    n = 8
    pos = f32(rng.uniform(-20, 20, (n, 3))); scale = f32(rng.uniform(3, 8, (n, 3)))
    quat = f32(rng.standard_normal((n, 4))); rho = f32(rng.standard_normal(n))          # signed values are fine
    a = oracle.splat_forward(pos, scale, quat, rho, GEOM, [0.5])
    assert np.allclose(oracle.splat_forward(pos, scale, quat, 2 * rho, GEOM, [0.5]), 2 * a, rtol=1e-13, atol=0)
    b = oracle.splat_forward(pos[:3], scale[:3], quat[:3], rho[:3], GEOM, [0.5]) + \
        oracle.splat_forward(pos[3:], scale[3:], quat[3:], rho[3:], GEOM, [0.5])
    assert np.allclose(a, b, rtol=0, atol=1e-12)
    iso = f32(np.repeat(rng.uniform(3, 8, (n, 1)), 3, axis=1))
    c = oracle.splat_forward(pos, iso, quat, rho, GEOM, [0.5])
    d = oracle.splat_forward(pos, iso, f32(rng.standard_normal((n, 4))), rho, GEOM, [0.5])
    assert np.allclose(c, d, rtol=0, atol=1e-10)                                          # isotropic: q is irrelevant
    e = oracle.splat_forward(pos, scale, 4.0 * quat, rho, GEOM, [0.5])                    # unnormalised quaternion (x4 is exact in fp32)
    assert np.allclose(a, e, rtol=0, atol=1e-10)


def test_cutoff_is_the_inclusive_pixel_box_and_pairs_are_counted():
    pos, scale, quat, rho = one((5.0, -8.0, 3.0), (4.0, 2.0, 6.0), (0.7, 0.2, 0.1, -0.5))
    img, pairs = oracle.splat_forward(pos, scale, quat, rho, GEOM, [1.0], return_pairs=True)
    cu, cv, A, B, C, amp, box, valid = oracle.splat_terms(*[oracle.splat._t(x) for x in (pos, scale, quat)],
                                                          oracle.splat._t(rho).reshape(-1), GEOM, 1.0)
    u0, v0, u1, v1 = (int(x) for x in box[0])
    assert pairs == (u1 - u0 + 1) * (v1 - v0 + 1)
    nz = np.argwhere(img[0] != 0)
    assert nz[:, 1].min() == u0 and nz[:, 1].max() == u1 and nz[:, 0].min() == v0 and nz[:, 0].max() == v1
    # box half-widths are 3 sigma of the marginals of Sigma^ in pixels
    Sig = np.linalg.inv(np.array([[float(A[0]), float(B[0])], [float(B[0]), float(C[0])]]))
    assert u0 == max(0, math.ceil(float(cu[0]) - 3 * math.sqrt(Sig[0, 0])))
    assert u1 == min(GEOM["nu"] - 1, math.floor(float(cu[0]) + 3 * math.sqrt(Sig[0, 0])))
    assert v0 == max(0, math.ceil(float(cv[0]) - 3 * math.sqrt(Sig[1, 1])))
    assert v1 == min(GEOM["nv"] - 1, math.floor(float(cv[0]) + 3 * math.sqrt(Sig[1, 1])))
    assert v1 == GEOM["nv"] - 1 and u0 > 0                       # this case is clipped by the detector edge in v only


def test_gaussians_behind_the_source_or_off_the_detector_contribute_nothing():
    pos = f32([[1200.0, 0.0, 0.0], [0.0, 0.0, 400.0], [0.0, 0.0, 0.0]])                 # behind the source at angle 0; far off in v
    scale = f32([[5, 5, 5]] * 3); quat = f32([[1, 0, 0, 0]] * 3); rho = f32([1, 1, 1])
    img = oracle.splat_forward(pos, scale, quat, rho, GEOM, [0.0])[0]
    only = oracle.splat_forward(pos[2:], scale[2:], quat[2:], rho[2:], GEOM, [0.0])[0]
    assert np.array_equal(img, only) and img.max() > 0
    g = np.ones((1, GEOM["nv"], GEOM["nu"]), np.float32)
    gr, gp, gs, gq = oracle.splat_backward(pos, scale, quat, rho, GEOM, [0.0], g)
    assert np.all(gr[:2] == 0) and np.all(gp[:2] == 0) and np.all(gs[:2] == 0) and np.all(gq[:2] == 0)
    assert gr[2] > 0


def test_autograd_gradients_against_central_differences_and_invariants():
    rng = np.random.default_rng(6)
    n = 4
    pos = f32(np.round(rng.uniform(-15, 15, (n, 3)) * 64) / 64); scale = f32(np.round(rng.uniform(4, 8, (n, 3)) * 64) / 64)
    quat = f32(np.round(rng.standard_normal((n, 4)) * 64) / 64); rho = f32(np.round(rng.uniform(0.3, 1, n) * 64) / 64)
    angles = [0.3, 1.9]
    g = rng.standard_normal((2, GEOM["nv"], GEOM["nu"])).astype(np.float32)
    kap = 40.0                                              # every box is the whole detector: the support cannot move
    gr, gp, gs, gq = oracle.splat_backward(pos, scale, quat, rho, GEOM, angles, g, kappa=kap)
    assert np.abs((quat.astype(np.float64) * gq).sum(1)).max() <= 1e-9 * np.abs(gq).max()      # q . dL/dq = 0

    def loss(p, s, q, r):
        return float((oracle.splat_forward(p, s, q, r, GEOM, angles, kappa=kap) * g).sum())
    eps = 2.0 ** -7
    for arr, grad, idx in [(pos, gp, (1, 0)), (pos, gp, (2, 2)), (scale, gs, (0, 1)), (scale, gs, (3, 2)),
                           (quat, gq, (1, 3)), (quat, gq, (2, 0)), (rho, gr, (3,))]:
        def at(e):
            a2 = arr.copy(); a2[idx] += e
            args = [a2 if x is arr else x for x in (pos, scale, quat, rho)]
            return loss(*args)
        d1 = (at(eps) - at(-eps)) / (2 * eps); d2 = (at(2 * eps) - at(-2 * eps)) / (4 * eps)
        assert (4 * d1 - d2) / 3 == pytest.approx(grad[idx], rel=2e-5, abs=1e-7)


def test_sampled_backward_equals_the_full_backward_on_a_masked_upstream_gradient():
    """splat_backward(pixels=...) (what the full-size GPU parity uses) = the full backward — pinned above by
    central differences — with the upstream gradient zeroed outside the listed pixels.  kappa = 3: live boxes,
    Gaussians clipped by the detector edge and Gaussians whose box holds none of the sampled pixels included."""
    rng = np.random.default_rng(8)
    n = 12
    pos = f32(rng.uniform(-60, 60, (n, 3))); scale = f32(rng.uniform(2, 9, (n, 3)))
    quat = f32(rng.standard_normal((n, 4))); rho = f32(rng.standard_normal(n))
    angles = [0.3, 1.9, 4.4]
    g = rng.standard_normal((3, GEOM["nv"], GEOM["nu"])).astype(np.float32)
    pix = [(int(rng.integers(0, 3)), int(rng.integers(0, GEOM["nu"])), int(rng.integers(0, GEOM["nv"]))) for _ in range(400)]
    pix = sorted(set(pix))
    gm = np.zeros_like(g)
    for b, iu, iv in pix:
        gm[b, iv, iu] = g[b, iv, iu]
    full = oracle.splat_backward(pos, scale, quat, rho, GEOM, angles, gm)
    samp = oracle.splat_backward(pos, scale, quat, rho, GEOM, angles, g, pixels=pix)
    assert np.abs(full[0]).max() > 0
    for a, b in zip(full, samp):
        assert np.allclose(a, b, rtol=1e-12, atol=1e-14 * max(1.0, np.abs(a).max()))
    # and the forward sampler agrees with the image
    img = oracle.splat_forward(pos, scale, quat, rho, GEOM, angles)
    for bsel in range(3):
        sel = [(iu, iv) for (b, iu, iv) in pix if b == bsel]
        vals = oracle.splat_forward_at(pos, scale, quat, rho, GEOM, np.float32(angles[bsel]), sel)
        assert np.allclose(vals, [img[bsel, iv, iu] for iu, iv in sel], rtol=1e-13, atol=1e-15)


def test_autograd_gradients_against_central_differences_with_live_3_sigma_boxes():
    """kappa = 3 (the product's cutoff): the boxes are strictly inside the detector and live (pixels outside
    contribute nothing), the support is frozen (R6) — asserted: no box changes under any perturbation applied —
    and Richardson central differences of the oracle's own forward match its autograd backward."""
    rng = np.random.default_rng(16)
    n = 2
    q64 = lambda a: f32(np.round(np.asarray(a) * 64) / 64)
    angles = [0.3, 1.9]

    def boxes(p, s, q, r):
        out = []
        for a in angles:
            t = oracle.splat_terms(*[oracle.splat._t(x) for x in (p, s, q)], oracle.splat._t(r).reshape(-1), GEOM, a)
            assert bool(t[7].all())
            out.append(t[6].numpy().copy())
        return np.stack(out)

    eps = 2.0 ** -10
    for attempt in range(200):                                # deterministic search for a set whose boxes stay put
        pos = q64(rng.uniform(-8, 8, (n, 3))); scale = q64(rng.uniform(1.5, 3.0, (n, 3)))
        quat = q64(rng.standard_normal((n, 4))); rho = q64(rng.uniform(0.3, 1, n))
        box0 = boxes(pos, scale, quat, rho)
        ok = (box0[..., 0] > 0).all() and (box0[..., 1] > 0).all() and (box0[..., 2] < GEOM["nu"] - 1).all() \
            and (box0[..., 3] < GEOM["nv"] - 1).all()
        for arr in (pos, scale, quat):
            for idx in np.ndindex(*arr.shape):
                for e in (eps, -eps, 2 * eps, -2 * eps):
                    a2 = arr.copy(); a2[idx] += e
                    args = [a2 if x is arr else x for x in (pos, scale, quat, rho)]
                    ok = ok and np.array_equal(boxes(*args), box0)
        if ok:
            break
    assert ok, "no frozen-box configuration found"
    area = (box0[..., 2] - box0[..., 0] + 1) * (box0[..., 3] - box0[..., 1] + 1)
    assert area.max() < 0.5 * GEOM["nu"] * GEOM["nv"]        # the cutoff is live: each box is a small part of the detector
    g = rng.standard_normal((2, GEOM["nv"], GEOM["nu"])).astype(np.float32)
    gr, gp, gs, gq = oracle.splat_backward(pos, scale, quat, rho, GEOM, angles, g)

    def loss(p, s, q, r):
        return float((oracle.splat_forward(p, s, q, r, GEOM, angles) * g).sum())
    for arr, grad in [(pos, gp), (scale, gs), (quat, gq), (rho, gr)]:
        fd = np.zeros_like(grad)
        for idx in np.ndindex(*arr.shape):
            def at(e):
                a2 = arr.copy(); a2[idx] += e
                args = [a2 if x is arr else x for x in (pos, scale, quat, rho)]
                return loss(*args)
            d1 = (at(eps) - at(-eps)) / (2 * eps); d2 = (at(2 * eps) - at(-2 * eps)) / (4 * eps)
            fd[idx] = (4 * d1 - d2) / 3
        err = np.linalg.norm(fd - grad) / np.linalg.norm(grad)
        assert err < 2e-5, err


def test_per_gaussian_box_form_equals_the_per_pixel_form():
    """splat_forward_boxes (what the every-pixel GPU parity at the bench size uses) against splat_forward, which the
    pins above hold in place: clipped boxes, Gaussians behind the source and off the detector, signed amplitudes."""
    rng = np.random.default_rng(12)
    n = 40
    pos = f32(rng.uniform(-70, 70, (n, 3))); scale = f32(rng.uniform(1.0, 9.0, (n, 3)))
    quat = f32(rng.standard_normal((n, 4))); rho = f32(rng.standard_normal(n))
    pos[0] = (1200.0, 0.0, 0.0); pos[1] = (0.0, 0.0, 400.0)                 # behind the source at angle 0 / far off in v
    angles = [0.0, 0.8, 2.9, 5.1]
    a = oracle.splat_forward(pos, scale, quat, rho, GEOM, angles)
    b = oracle.splat_forward_boxes(pos, scale, quat, rho, GEOM, angles)
    assert a.shape == b.shape and np.abs(a).max() > 0
    assert np.allclose(a, b, rtol=1e-13, atol=1e-13 * np.abs(a).max())
    assert np.array_equal(a == 0.0, b == 0.0)                                # the same pixels are untouched


def test_box_restricted_backward_equals_the_full_backward():
    """splat_backward_boxes (every-pixel gradient parity at the bench size) against splat_backward, which central
    differences hold in place: groups smaller than the set, clipped boxes, dropped Gaussians, signed amplitudes."""
    rng = np.random.default_rng(14)
    n = 50
    pos = f32(rng.uniform(-70, 70, (n, 3))); scale = f32(rng.uniform(1.0, 9.0, (n, 3)))
    quat = f32(rng.standard_normal((n, 4))); rho = f32(rng.standard_normal(n))
    pos[0] = (1200.0, 0.0, 0.0); pos[1] = (0.0, 0.0, 400.0)
    angles = [0.0, 2.9, 5.1]
    g = rng.standard_normal((3, GEOM["nv"], GEOM["nu"])).astype(np.float32)
    full = oracle.splat_backward(pos, scale, quat, rho, GEOM, angles, g)
    for group in (7, 64):
        part = oracle.splat_backward_boxes(pos, scale, quat, rho, GEOM, angles, g, group=group)
        for a, b in zip(full, part):
            assert np.allclose(a, b, rtol=1e-11, atol=1e-13 * max(1.0, np.abs(a).max()))
    assert np.abs(full[1]).max() > 0 and not full[1][0].any()
