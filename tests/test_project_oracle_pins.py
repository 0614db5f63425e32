"""Pins of the cone-beam projector oracle (oracle.project_forward / project_backward; SURVEY.md 8(f)
rank 4; Eq. 6, :141, :275, Table I) to things other than itself: an independent ray
sampler through scipy map_coordinates, closed-form chord lengths, exact axis-aligned sums, the
predicted detector position of a point (magnification SDD / (SAD - depth)), a 90-degree gantry /
volume rotation identity, and the transpose identities of the backward.  CPU only.
"""
import numpy as np
import pytest
from scipy.ndimage import map_coordinates

import oracle


def setup(dims=(20, 16, 10), h=(2.0, 2.0, 2.0), nu=25, nv=13, du=3.0, dv=3.0, sad=100.0, sdd=150.0,
          off_u=0.0, off_v=0.0):
    nx, ny, nz = dims
    origin = [-(n - 1) / 2.0 * hh for n, hh in zip(dims, h)]          # isocentre at the grid centre
    grid = (np.array(origin, np.float32), np.array(h, np.float32), np.array(dims, np.int32))
    geom = dict(sad=sad, sdd=sdd, nu=nu, nv=nv, du=du, dv=dv, off_u=off_u, off_v=off_v, iso=[0.0, 0.0, 0.0])
    return grid, geom


def independent_projection(vol, grid, geom, angle):
    """Geometry rebuilt from its description, samples through scipy (order 1, zero outside)."""
    o, h, dims = (np.asarray(a, np.float64) for a in grid)
    nx, ny, nz = (int(v) for v in grid[2])
    ca, sa = np.cos(angle), np.sin(angle)
    src = np.array([geom["sad"] * ca, geom["sad"] * sa, 0.0]) + np.asarray(geom["iso"], np.float64)
    out = np.zeros((geom["nv"], geom["nu"]))
    for iv in range(geom["nv"]):
        for iu in range(geom["nu"]):
            u = (iu - (geom["nu"] - 1) / 2.0) * geom["du"] + geom["off_u"]
            v = (iv - (geom["nv"] - 1) / 2.0) * geom["dv"] + geom["off_v"]
            pix = src - geom["sdd"] * np.array([ca, sa, 0.0]) + u * np.array([-sa, ca, 0.0]) + v * np.array([0.0, 0.0, 1.0])
            D = pix - src
            a = int(np.argmax(np.abs(D) + np.array([2e-12, 1e-12, 0.0])))          # first axis wins ties
            n_a = (nx, ny, nz)[a]
            planes = o[a] + np.arange(n_a) * h[a]
            t = (planes - src[a]) / D[a]
            X = src[None, :] + t[:, None] * D[None, :]
            idx = (X - o[None, :]) / h[None, :]                                    # x, y, z index coordinates
            idx[:, a] = np.arange(n_a)
            samples = map_coordinates(vol.astype(np.float64), [idx[:, 2], idx[:, 1], idx[:, 0]], order=1,
                                      mode="grid-constant", cval=0.0)
            out[iv, iu] = samples.sum() * h[a] * np.linalg.norm(D) / abs(D[a])
    return out


@pytest.mark.parametrize("angle", [0.0, 0.4, 1.1, 2.5, -2.0, np.pi / 4 + 0.01])
def test_forward_equals_independent_ray_sampler(angle):
    rng = np.random.default_rng(1)
    grid, geom = setup(h=(2.0, 1.5, 2.5), off_u=4.0, off_v=-2.0)
    vol = rng.standard_normal((10, 16, 20)).astype(np.float32)
    got = oracle.project_forward(vol, grid, geom, [angle])[0]
    ref = independent_projection(vol, grid, geom, np.float64(np.float32(angle)))
    # the oracle rounds the per-ray constants and the sample positions to fp32 (reading P3)
    assert np.abs(got - ref).max() <= 3e-5 * np.abs(ref).max()


def test_uniform_volume_gives_chord_length_between_the_outer_planes():
    grid, geom = setup(nu=9, nv=5, du=2.0, dv=2.0)                # narrow fan: every ray stays inside laterally
    vol = np.full((10, 16, 20), 0.25, np.float32)
    for angle, n_a, h_a, ax in [(0.0, 20, 2.0, 0), (np.pi / 2, 16, 2.0, 1), (np.pi, 20, 2.0, 0)]:
        d = oracle.project_forward(vol, grid, geom, [angle])[0]
        rays = oracle.cone_rays(grid, geom, np.float32(angle))
        assert np.all(rays["axis"] == ax)
        u = (np.arange(9) - 4) * 2.0
        v = (np.arange(5) - 2) * 2.0
        norm = np.sqrt(150.0 ** 2 + u[None, :] ** 2 + v[:, None] ** 2)
        want = 0.25 * n_a * h_a * norm / 150.0
        assert np.allclose(d, want, rtol=2e-7, atol=0)


def test_central_ray_sums_a_row_of_voxels():
    """Odd detector, odd ny/nz: the central ray at angle 0 runs along x through voxel centres."""
    rng = np.random.default_rng(2)
    grid, geom = setup(dims=(12, 9, 7), nu=11, nv=5)
    vol = rng.standard_normal((7, 9, 12)).astype(np.float32)
    d = oracle.project_forward(vol, grid, geom, [0.0])[0]
    assert d[2, 5] == pytest.approx(2.0 * vol[3, 4, :].astype(np.float64).sum(), rel=1e-12)
    d = oracle.project_forward(vol, grid, geom, [np.pi / 2])[0]            # along y, through x = centre column? nx even: between
    col = 0.5 * (vol[3, :, 5].astype(np.float64) + vol[3, :, 6].astype(np.float64))
    assert d[2, 5] == pytest.approx(2.0 * col.sum(), rel=1e-6)


def test_point_projects_where_the_magnification_says():
    """A single bright voxel at world (x, y, z): detector coordinates u = SDD y' / (SAD - x'),
    v = SDD z / (SAD - x') in the gantry frame (x' towards the source).  Pins the side of the source,
    the orientation of u and v and the half-fan offsets."""
    grid, geom = setup(dims=(41, 41, 21), h=(1.0, 1.0, 1.0), nu=81, nv=41, du=1.0, dv=1.0, off_u=3.0, off_v=-2.0)
    vol = np.zeros((21, 41, 41), np.float32)
    ix, iy, iz = 28, 12, 15
    vol[iz, iy, ix] = 1.0
    X = np.array([ix - 20.0, iy - 20.0, iz - 10.0])
    for angle in (0.0, 0.7, 2.2, -1.3):
        d = oracle.project_forward(vol, grid, geom, [angle])[0]
        a = np.float64(np.float32(angle))
        xp = X[0] * np.cos(a) + X[1] * np.sin(a)                     # towards the source
        yp = -X[0] * np.sin(a) + X[1] * np.cos(a)                    # along u
        mag = 150.0 / (100.0 - xp)
        u_pred, v_pred = mag * yp, mag * X[2]
        uu = (np.arange(81) - 40) * 1.0 + 3.0
        vv = (np.arange(41) - 20) * 1.0 - 2.0
        tot = d.sum()
        assert tot > 0
        assert (d.sum(0) * uu).sum() / tot == pytest.approx(u_pred, abs=0.35)
        assert (d.sum(1) * vv).sum() / tot == pytest.approx(v_pred, abs=0.35)


def test_quarter_turn_of_the_gantry_equals_quarter_turn_of_the_volume():
    """Cubic in-plane grid, isocentre at its centre: P(vol, a + pi/2) = P(vol rotated by -pi/2 about z, a)."""
    rng = np.random.default_rng(3)
    grid, geom = setup(dims=(15, 15, 7), nu=21, nv=9)
    vol = rng.standard_normal((7, 15, 15)).astype(np.float32)
    # new[x, y] = old[-y, x] in centred coordinates: array [z, y, x] -> rot90 in the (y, x) plane
    rot = np.ascontiguousarray(np.rot90(vol, k=1, axes=(1, 2)))
    for a in (0.0, 0.3):
        lhs = oracle.project_forward(vol, grid, geom, [a + np.pi / 2])[0]
        cands = [oracle.project_forward(np.ascontiguousarray(np.rot90(vol, k=k, axes=(1, 2))), grid, geom, [a])[0]
                 for k in (1, 3)]
        errs = [np.abs(lhs - c).max() for c in cands]
        assert min(errs) <= 2e-5 * np.abs(lhs).max(), errs
        assert max(errs) > 1e-2 * np.abs(lhs).max()                  # and the other sense is really different
    assert rot.shape == vol.shape


def test_backward_is_the_transpose():
    rng = np.random.default_rng(4)
    grid, geom = setup(dims=(9, 8, 5), nu=10, nv=6, du=4.0, dv=4.0)
    angles = np.array([0.2, 1.9], np.float32)
    x = rng.standard_normal((2, 5, 8, 9)).astype(np.float32)
    y = rng.standard_normal((2, 6, 10)).astype(np.float32)
    Px = oracle.project_forward(x, grid, geom, angles)
    PTy = oracle.project_backward(y, grid, geom, angles)
    assert float((Px * y).sum()) == pytest.approx(float((x.astype(np.float64) * PTy).sum()), rel=1e-12)
    # explicit matrix of projection 0, column by column
    V = 5 * 8 * 9
    P = np.zeros((60, V))
    for j in range(V):
        e = np.zeros(V, np.float32); e[j] = 1.0
        P[:, j] = oracle.project_forward(e.reshape(1, 5, 8, 9), grid, geom, angles[:1])[0].ravel()
    assert np.allclose(P.T @ y[0].ravel().astype(np.float64), PTy[0].ravel(), rtol=1e-12, atol=1e-12)
    assert np.allclose(P @ x[0].ravel().astype(np.float64), Px[0].ravel(), rtol=1e-12, atol=1e-12)


def test_shared_volume_and_rays_missing_the_grid():
    rng = np.random.default_rng(5)
    grid, geom = setup(nu=40, nv=30, du=12.0, dv=12.0)              # wide detector: outer rays miss the volume
    vol = rng.uniform(0.0, 1.0, (10, 16, 20)).astype(np.float32)
    d = oracle.project_forward(vol, grid, geom, [0.0, 1.0])
    d2 = oracle.project_forward(np.stack([vol, vol]), grid, geom, [0.0, 1.0])
    assert np.array_equal(d, d2)
    assert d[0, 0, 0] == 0.0 and d[1, -1, -1] == 0.0 and d.max() > 0


def test_steep_cone_rays_take_z_as_the_dominant_axis():
    """A tall detector close to the source: the outer rows run mostly along z (axis 2), the branch a
    clinical geometry never reaches.  Same independent sampler."""
    rng = np.random.default_rng(6)
    grid, geom = setup(dims=(14, 12, 30), nu=9, nv=41, du=6.0, dv=12.0, sad=60.0, sdd=90.0)
    vol = rng.standard_normal((30, 12, 14)).astype(np.float32)
    rays = oracle.cone_rays(grid, geom, np.float32(0.3))
    assert (rays["axis"] == 2).any() and (rays["axis"] == 0).any()
    got = oracle.project_forward(vol, grid, geom, [0.3])[0]
    ref = independent_projection(vol, grid, geom, np.float64(np.float32(0.3)))
    assert np.abs(got - ref).max() <= 3e-5 * np.abs(ref).max()
