"""Pins of the warp oracle (oracle.warp_forward / warp_backward; PAPER.md:55
Eq. 2, I(x,p) = I_ref(x + d(x,p))) to library routines and closed forms: scipy.ndimage
map_coordinates (order 1, grid-constant), torch grid_sample on the CPU in fp64 and its autograd for
both gradients, exact integer shifts, zero padding, and central finite differences.  CPU only.
"""
import numpy as np
import pytest
import torch
from scipy.ndimage import map_coordinates

import oracle


def make(dims=(20, 14, 9), B=2, spacing=(2.0, 0.5, 0.25), amp=3.0, seed=0, exact=True):
    """exact: displacements are multiples of h/256, so d/h is exact in fp32 and the oracle's fp32
    cell decision (reading W3) coincides with the fp64 one of the library routines."""
    rng = np.random.default_rng(seed)
    nx, ny, nz = dims
    grid = (np.array([5.0, -3.0, 40.0], np.float32), np.array(spacing, np.float32), np.array(dims, np.int32))
    I = rng.standard_normal((nz, ny, nx)).astype(np.float32)
    t = rng.standard_normal((B, 3, nz, ny, nx)) * amp
    if exact:
        t = np.round(t * 256) / 256
    d = (t * np.array(spacing)[None, :, None, None, None]).astype(np.float32)
    return I, d, grid


def coords_index(d, grid):
    _, h, dims = grid
    nx, ny, nz = (int(v) for v in dims)
    zz, yy, xx = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    h = h.astype(np.float64)
    return (xx + d[:, 0].astype(np.float64) / h[0], yy + d[:, 1].astype(np.float64) / h[1],
            zz + d[:, 2].astype(np.float64) / h[2])


def test_forward_equals_scipy_map_coordinates():
    I, d, grid = make()
    out = oracle.warp_forward(I, d, grid)
    ux, uy, uz = coords_index(d, grid)
    for b in range(d.shape[0]):
        ref = map_coordinates(I.astype(np.float64), np.stack([uz[b], uy[b], ux[b]]), order=1,
                              mode="grid-constant", cval=0.0)
        assert np.abs(out[b] - ref).max() <= 1e-13


def torch_reference(I, d, grid, g=None):
    """grid_sample(bilinear, zeros, align_corners=True) in fp64; with g also both gradients."""
    _, h, dims = grid
    nx, ny, nz = (int(v) for v in dims)
    h = h.astype(np.float64)
    zz, yy, xx = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    It = torch.tensor(I.astype(np.float64), requires_grad=True)
    dt = torch.tensor(d.astype(np.float64), requires_grad=True)
    B = d.shape[0]
    ux = torch.tensor(xx, dtype=torch.float64) + dt[:, 0] / h[0]
    uy = torch.tensor(yy, dtype=torch.float64) + dt[:, 1] / h[1]
    uz = torch.tensor(zz, dtype=torch.float64) + dt[:, 2] / h[2]
    gridt = torch.stack([ux / (nx - 1) * 2 - 1, uy / (ny - 1) * 2 - 1, uz / (nz - 1) * 2 - 1], dim=-1)
    out = torch.nn.functional.grid_sample(It[None, None].expand(B, 1, nz, ny, nx), gridt, mode="bilinear",
                                          padding_mode="zeros", align_corners=True)[:, 0]
    if g is None:
        return out.detach().numpy()
    (out * torch.tensor(g.astype(np.float64))).sum().backward()
    return out.detach().numpy(), It.grad.numpy(), dt.grad.numpy()


def test_forward_and_both_gradients_equal_torch_grid_sample_autograd():
    I, d, grid = make(seed=1)
    g = np.random.default_rng(2).standard_normal((d.shape[0],) + I.shape).astype(np.float32)
    out = oracle.warp_forward(I, d, grid)
    gI, gd = oracle.warp_backward(I, d, grid, g)
    ref, rI, rd = torch_reference(I, d, grid, g)
    assert np.abs(out - ref).max() <= 1e-13
    assert np.abs(gI - rI).max() <= 1e-12
    # kinks: where a sample sits exactly on a cell face the one-sided derivative is a convention
    ux, uy, uz = coords_index(d, grid)
    interior = (ux != np.floor(ux)) & (uy != np.floor(uy)) & (uz != np.floor(uz))
    assert interior.mean() > 0.95
    assert np.abs((gd - rd) * interior[:, None]).max() <= 1e-12


def test_general_spacing_agrees_with_fp64_cells_to_fp32_rounding():
    """With d/h inexact in fp32 the oracle's cell decision is the kernel's (fp32); the value differs
    from the all-fp64 library result only by the rounding of t (continuity of the interpolant)."""
    I, d, grid = make(spacing=(2.0, 1.5, 0.75), exact=False, seed=3)
    out = oracle.warp_forward(I, d, grid)
    ref = torch_reference(I, d, grid)
    assert np.abs(out - ref).max() <= 5e-6


def test_zero_displacement_is_identity_and_integer_shifts_are_exact():
    I, _, grid = make()
    nz, ny, nx = I.shape
    h = grid[1]
    d = np.zeros((1, 3, nz, ny, nx), np.float32)
    assert np.array_equal(oracle.warp_forward(I, d, grid)[0], I.astype(np.float64))
    d[0, 0] = 2 * h[0]; d[0, 1] = -1 * h[1]; d[0, 2] = 3 * h[2]          # out[z,y,x] = I[z+3, y-1, x+2]
    out = oracle.warp_forward(I, d, grid)[0]
    want = np.zeros_like(out)
    want[:nz - 3, 1:, :nx - 2] = I[3:, :ny - 1, 2:]
    assert np.array_equal(out, want)


def test_half_voxel_shift_averages_neighbours_and_pads_with_zero():
    I, _, grid = make()
    nz, ny, nx = I.shape
    d = np.zeros((1, 3, nz, ny, nx), np.float32); d[0, 0] = 0.5 * grid[1][0]
    out = oracle.warp_forward(I, d, grid)[0]
    I64 = I.astype(np.float64)
    assert np.allclose(out[:, :, :-1], 0.5 * (I64[:, :, :-1] + I64[:, :, 1:]), rtol=0, atol=1e-15)
    assert np.allclose(out[:, :, -1], 0.5 * I64[:, :, -1], rtol=0, atol=1e-15)       # neighbour outside = 0
    d[0, 0] = 1000.0
    assert np.all(oracle.warp_forward(I, d, grid) == 0.0)


def test_non_finite_displacement_gives_zero_output_and_zero_gradients():
    I, d, grid = make(B=1)
    d[0, 1, 3, 4, 5] = np.nan; d[0, 0, 2, 2, 2] = np.inf
    out = oracle.warp_forward(I, d, grid)
    assert out[0, 3, 4, 5] == 0.0 and out[0, 2, 2, 2] == 0.0 and np.all(np.isfinite(out))
    g = np.ones((1,) + I.shape, np.float32)
    gI, gd = oracle.warp_backward(I, d, grid, g)
    assert np.all(gd[0, :, 3, 4, 5] == 0.0) and np.all(gd[0, :, 2, 2, 2] == 0.0)
    assert np.all(np.isfinite(gI)) and np.all(np.isfinite(gd))


def test_backward_against_central_differences():
    """L = <g, out>.  Linear in I_ref (differences exact); in d only inside a cell, so samples are
    placed at cell fractions 0.25..0.75 and the step keeps them there."""
    rng = np.random.default_rng(5)
    dims = (9, 8, 7)
    spacing = (2.0, 0.5, 0.25)
    grid = (np.zeros(3, np.float32), np.array(spacing, np.float32), np.array(dims, np.int32))
    nx, ny, nz = dims
    I = (np.round(rng.standard_normal((nz, ny, nx)) * 1024) / 1024).astype(np.float32)   # I +- 0.5 exact in fp32
    t = rng.integers(-2, 3, size=(2, 3, nz, ny, nx)) + rng.integers(64, 193, size=(2, 3, nz, ny, nx)) / 256.0
    d = (t * np.array(spacing)[None, :, None, None, None]).astype(np.float32)
    g = rng.standard_normal((2, nz, ny, nx)).astype(np.float32)
    gI, gd = oracle.warp_backward(I, d, grid, g)

    def loss(I_, d_):
        return float(np.sum(g.astype(np.float64) * oracle.warp_forward(I_, d_, grid)))
    for idx in [(0, 0, 0), (3, 4, 5), (6, 7, 8), (2, 1, 7)]:
        Ip, Im = I.copy(), I.copy()
        Ip[idx] += 0.5; Im[idx] -= 0.5
        assert loss(Ip, d) - loss(Im, d) == pytest.approx(gI[idx], rel=1e-9, abs=1e-12)
    for idx in [(0, 0, 1, 2, 3), (1, 1, 4, 4, 4), (0, 2, 6, 7, 8), (1, 0, 0, 0, 0), (1, 2, 3, 0, 8)]:
        eps = spacing[idx[1]] / 1024.0                    # exact in fp32, stays inside the cell
        dp, dm = d.copy(), d.copy()
        dp[idx] += eps; dm[idx] -= eps
        fd = (loss(I, dp) - loss(I, dm)) / (2 * eps)
        assert fd == pytest.approx(gd[idx], rel=1e-8, abs=1e-10)
