"""ctypes front end of the fp64 CPU oracle (oracle/gsvox_oracle.c).

TEST INFRASTRUCTURE ONLY.  Importers allowed: tests/, __graft_entry__.smoke(),
bench.py's cpu_baseline and --impl reference legs.  The product package
(paper_2503_22139_b200) never imports this module and this module never imports it.

All functions take numpy arrays (fp32 inputs, as handed to the CUDA path) and
return fp64 numpy arrays.  `grid` is (origin[3], spacing[3], dims[3]) with
dims = (nx, ny, nz); volumes are laid out [C, nz, ny, nx] (reading A7).
"""
import ctypes as C

import numpy as np

from .build import build as _build

KAPPA = 3.0          # the product's fixed cutoff (north_star: "3-sigma"); a parameter here

_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build())
        fp, dp, ip, lp, bp = (C.POINTER(C.c_float), C.POINTER(C.c_double),
                              C.POINTER(C.c_int32), C.POINTER(C.c_int64), C.POINTER(C.c_uint8))
        L.gsvox_oracle_threads.restype = C.c_int
        L.gsvox_oracle_geometry.argtypes = [fp, fp, fp, C.c_int64, fp, fp, ip, C.c_double,
                                            dp, dp, ip, bp]
        L.gsvox_oracle_forward.argtypes = [fp, fp, fp, fp, C.c_int64, C.c_int32, fp, fp, ip,
                                           C.c_double, dp, lp]
        L.gsvox_oracle_forward_at.argtypes = [fp, fp, fp, fp, C.c_int64, C.c_int32, fp, fp, ip,
                                              C.c_double, lp, C.c_int64, dp]
        L.gsvox_oracle_backward.argtypes = [fp, fp, fp, fp, C.c_int64, C.c_int32, fp, fp, ip,
                                            C.c_double, fp, dp, dp, dp, dp]
        L.gsvox_oracle_backward_for.argtypes = [fp, fp, fp, fp, C.c_int64, C.c_int32, fp, fp, ip,
                                                C.c_double, fp, lp, C.c_int64, dp, dp, dp, dp]
        _lib = L
    return _lib


def threads() -> int:
    return int(lib().gsvox_oracle_threads())


def _f32(a, shape=None):
    a = np.ascontiguousarray(a, dtype=np.float32)
    if shape is not None:
        a = a.reshape(shape)
    return a


def _p(a, ct):
    return a.ctypes.data_as(C.POINTER(ct))


def _grid(grid):
    origin, spacing, dims = grid
    o = _f32(origin, (3,))
    h = _f32(spacing, (3,))
    d = np.ascontiguousarray(dims, dtype=np.int32).reshape(3)
    return o, h, d


def _check(rc):
    if rc != 0:
        raise RuntimeError("gsvox oracle error %d" % rc)


def _params(pos, scale, quat):
    pos, scale, quat = _f32(pos), _f32(scale), _f32(quat)
    n = pos.shape[0] if pos.ndim == 2 else pos.size // 3
    return pos.reshape(n, 3), scale.reshape(n, 3), quat.reshape(n, 4), n


def geometry(pos, scale, quat, grid, kappa=KAPPA):
    """-> dict(M [n,6] xx,xy,xz,yy,yz,zz; R [n,3,3]; box [n,6] lo xyz, hi xyz; flags [n])."""
    pos, scale, quat, n = _params(pos, scale, quat)
    o, h, d = _grid(grid)
    M = np.zeros((n, 6)); R = np.zeros((n, 9))
    box = np.zeros((n, 6), dtype=np.int32); flags = np.zeros(n, dtype=np.uint8)
    _check(lib().gsvox_oracle_geometry(_p(pos, C.c_float), _p(scale, C.c_float), _p(quat, C.c_float),
                                       n, _p(o, C.c_float), _p(h, C.c_float), _p(d, C.c_int32),
                                       float(kappa), _p(M, C.c_double), _p(R, C.c_double),
                                       _p(box, C.c_int32), _p(flags, C.c_uint8)))
    return {"M": M, "R": R.reshape(n, 3, 3), "box": box, "flags": flags}


def forward(pos, scale, quat, weight, grid, kappa=KAPPA, return_pairs=False):
    """-> out [C, nz, ny, nx] fp64 (and P_def, the number of pairs inside the cutoff)."""
    pos, scale, quat, n = _params(pos, scale, quat)
    weight = _f32(weight).reshape(n, -1) if n else _f32(weight).reshape(0, max(1, np.shape(weight)[-1]))
    ch = weight.shape[1]
    o, h, d = _grid(grid)
    out = np.empty((ch, int(d[2]), int(d[1]), int(d[0])))
    pairs = C.c_int64(0)
    _check(lib().gsvox_oracle_forward(_p(pos, C.c_float), _p(scale, C.c_float), _p(quat, C.c_float),
                                      _p(weight, C.c_float), n, ch, _p(o, C.c_float),
                                      _p(h, C.c_float), _p(d, C.c_int32), float(kappa),
                                      _p(out, C.c_double), C.byref(pairs)))
    return (out, int(pairs.value)) if return_pairs else out


def forward_at(pos, scale, quat, weight, grid, voxels, kappa=KAPPA):
    """Brute force at linear voxel indices v = (k*ny + j)*nx + i  -> [C, m] fp64."""
    pos, scale, quat, n = _params(pos, scale, quat)
    weight = _f32(weight).reshape(n, -1)
    ch = weight.shape[1]
    o, h, d = _grid(grid)
    vox = np.ascontiguousarray(voxels, dtype=np.int64).reshape(-1)
    out = np.zeros((ch, vox.size))
    _check(lib().gsvox_oracle_forward_at(_p(pos, C.c_float), _p(scale, C.c_float), _p(quat, C.c_float),
                                         _p(weight, C.c_float), n, ch, _p(o, C.c_float),
                                         _p(h, C.c_float), _p(d, C.c_int32), float(kappa),
                                         _p(vox, C.c_int64), vox.size, _p(out, C.c_double)))
    return out


def backward(pos, scale, quat, weight, grid, grad_out, kappa=KAPPA):
    """-> (dL/dw [n,C], dL/dp [n,3], dL/ds [n,3], dL/dq [n,4]) fp64."""
    pos, scale, quat, n = _params(pos, scale, quat)
    weight = _f32(weight).reshape(n, -1)
    ch = weight.shape[1]
    o, h, d = _grid(grid)
    g = _f32(grad_out).reshape(ch, int(d[2]), int(d[1]), int(d[0]))
    gw = np.zeros((n, ch)); gp = np.zeros((n, 3)); gs = np.zeros((n, 3)); gq = np.zeros((n, 4))
    _check(lib().gsvox_oracle_backward(_p(pos, C.c_float), _p(scale, C.c_float), _p(quat, C.c_float),
                                       _p(weight, C.c_float), n, ch, _p(o, C.c_float),
                                       _p(h, C.c_float), _p(d, C.c_int32), float(kappa),
                                       _p(g, C.c_float), _p(gw, C.c_double), _p(gp, C.c_double),
                                       _p(gs, C.c_double), _p(gq, C.c_double)))
    return gw, gp, gs, gq


def backward_for(pos, scale, quat, weight, grid, grad_out, ids, kappa=KAPPA):
    """Gradients of the listed Gaussians only -> (gw [m,C], gp [m,3], gs [m,3], gq [m,4])."""
    pos, scale, quat, n = _params(pos, scale, quat)
    weight = _f32(weight).reshape(n, -1)
    ch = weight.shape[1]
    o, h, d = _grid(grid)
    g = _f32(grad_out).reshape(ch, int(d[2]), int(d[1]), int(d[0]))
    ids = np.ascontiguousarray(ids, dtype=np.int64).reshape(-1)
    m = ids.size
    gw = np.zeros((m, ch)); gp = np.zeros((m, 3)); gs = np.zeros((m, 3)); gq = np.zeros((m, 4))
    _check(lib().gsvox_oracle_backward_for(_p(pos, C.c_float), _p(scale, C.c_float),
                                           _p(quat, C.c_float), _p(weight, C.c_float), n, ch,
                                           _p(o, C.c_float), _p(h, C.c_float), _p(d, C.c_int32),
                                           float(kappa), _p(g, C.c_float), _p(ids, C.c_int64), m,
                                           _p(gw, C.c_double), _p(gp, C.c_double),
                                           _p(gs, C.c_double), _p(gq, C.c_double)))
    return gw, gp, gs, gq


# --------------------------------------------------------------------------------------------
# motion-basis components -> deformation vector fields.
#   PAPER.md:106   "three spatial levels (i = 1, 2, 3) are employed for e_i(x) along each Cartesian
#                   direction (x, y, z), resulting in a total of nine MBC volumes"
#   PAPER.md:58-61 Eq. 3:  d(x,p) = sum_i w_i(p) e_i(x);  PAPER.md:141: w_{i,k}(p), i = level, k = axis
# The oracle follows the paper's order literally: voxelize every level into its three MBC volumes
# e_{i,k} (Eq. 5 with the level's feature column k as the weight), THEN combine them with the
# per-projection coefficients.  (The CUDA path never forms the nine volumes; it folds the
# coefficients into per-Gaussian weights.  Nothing of that is used here.)
# --------------------------------------------------------------------------------------------
def mbc_volumes(levels, grid, kappa=KAPPA):
    """levels = [(pos, scale, quat, feat[n_i,3]), ...]  ->  e [L, 3, nz, ny, nx] fp64."""
    return np.stack([forward(p, s, q, f, grid, kappa) for (p, s, q, f) in levels])


def mbc_combine(e, coef):
    """Eq. 3 on given MBC volumes: e [L,3,...] , coef [B,L,3] -> d [B,3,...] fp64."""
    coef = np.asarray(_f32(coef), dtype=np.float64)
    e = np.asarray(e, dtype=np.float64)
    B, L = coef.shape[0], coef.shape[1]
    d = np.zeros((B, 3) + e.shape[2:])
    for b in range(B):
        for i in range(L):
            for k in range(3):
                d[b, k] += coef[b, i, k] * e[i, k]
    return d


def mbc_combine_backward(e, coef, grad_dvf):
    """-> (dL/de [L,3,...], dL/dcoef [B,L,3]) of mbc_combine, fp64."""
    coef = np.asarray(_f32(coef), dtype=np.float64)
    e = np.asarray(e, dtype=np.float64)
    g = np.asarray(grad_dvf, dtype=np.float64)
    B, L = coef.shape[0], coef.shape[1]
    ge = np.zeros_like(e)
    gc = np.zeros((B, L, 3))
    for b in range(B):
        for i in range(L):
            for k in range(3):
                ge[i, k] += coef[b, i, k] * g[b, k]
                gc[b, i, k] = float(np.sum(g[b, k] * e[i, k]))
    return ge, gc


def dvf_forward(levels, coef, grid, kappa=KAPPA):
    """coef [B, L, 3] (w_{i,k}(p) of PAPER.md:141)  ->  d [B, 3, nz, ny, nx] fp64 (Eq. 3)."""
    return mbc_combine(mbc_volumes(levels, grid, kappa), coef)


def _split_f32(a):
    """fp64 array -> (hi, lo) fp32 arrays with hi + lo == a to ~1e-15 relative."""
    hi = a.astype(np.float32)
    lo = (a - hi.astype(np.float64)).astype(np.float32)
    return hi, lo


def dvf_backward(levels, coef, grid, grad_dvf, kappa=KAPPA):
    """Chain rule of dvf_forward.  grad_dvf [B,3,nz,ny,nx] (fp32 as handed to the CUDA path) ->
    (grad_coef [B,L,3], [(grad_feat [n_i,3], grad_pos, grad_scale, grad_quat) per level]).
      dL/dcoef[b,i,k] = <grad_dvf[b,k], e_{i,k}>
      dL/de_{i,k}     = sum_b coef[b,i,k] grad_dvf[b,k]      then the voxelizer's analytic backward.
    The C oracle takes fp32 upstream gradients; dL/de is handed over as an exact hi+lo fp32 split
    (the backward is linear in the upstream gradient)."""
    g = np.asarray(_f32(grad_dvf), dtype=np.float64)
    e = mbc_volumes(levels, grid, kappa)
    grad_e, grad_coef = mbc_combine_backward(e, coef, g)
    per_level = []
    for i, (p, s, q, f) in enumerate(levels):
        hi, lo = _split_f32(grad_e[i])
        a = backward(p, s, q, f, grid, hi, kappa)
        c = backward(p, s, q, f, grid, lo, kappa)
        per_level.append(tuple(x + y for x, y in zip(a, c)))
    return grad_coef, per_level


# --------------------------------------------------------------------------------------------
# the warp  I(x,p) = I_ref(x + d(x,p))   (PAPER.md:55, Eq. 2; :136).
# The paper does not say how I_ref is evaluated between voxel centres or outside the volume.
# Readings (W1-W4): trilinear interpolation of the voxel-centre samples; a corner
# outside the grid contributes 0 (zero padding, corner by corner); d is in world units like
# origin/spacing, so the sample position in index units is u_k = i_k + d_k / h_k (the origin cancels);
# the cell is floor(d_k / h_k) and the interpolation fraction d_k / h_k - floor(d_k / h_k), both in
# fp64 on the fp32 inputs promoted exactly — the plain reading of Eq. 2, no fp32 step anywhere; a
# non-finite displacement, or one of 2^22 voxels or more, yields 0 and zero gradients.  Backward is
# the exact derivative of the piecewise-trilinear interpolant (kinks at integer u have measure zero).
# --------------------------------------------------------------------------------------------
def _warp_cells(dvf, spacing, dims):
    """-> integer base corner i0 [B,3,nz,ny,nx] (int64), fraction f [B,3,nz,ny,nx] fp64, finite mask."""
    nx, ny, nz = (int(v) for v in dims)
    d = np.asarray(_f32(dvf), dtype=np.float64).reshape(-1, 3, nz, ny, nx)
    h = np.asarray(_f32(spacing), dtype=np.float64).reshape(3)
    with np.errstate(invalid="ignore", over="ignore"):
        t = d / h[None, :, None, None, None]                   # displacement in voxels, fp64
    finite = np.all(np.isfinite(t), axis=1) & np.all(np.abs(t) < 4194304.0, axis=1)   # |t| < 2^22 voxels
    t = np.where(finite[:, None], t, 0.0)
    tf = np.floor(t)
    frac = t - tf
    idx = np.stack(np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij"))   # z,y,x
    base = np.empty(t.shape, dtype=np.int64)
    base[:, 0] = idx[2][None] + tf[:, 0].astype(np.int64)      # x
    base[:, 1] = idx[1][None] + tf[:, 1].astype(np.int64)      # y
    base[:, 2] = idx[0][None] + tf[:, 2].astype(np.int64)      # z
    return base, frac, finite


def warp_forward(iref, dvf, grid):
    """iref [nz,ny,nx], dvf [B,3,nz,ny,nx] (components x,y,z, world units) -> out [B,nz,ny,nx] fp64."""
    _, h, dims = _grid(grid)
    nx, ny, nz = (int(v) for v in dims)
    I = np.asarray(_f32(iref), dtype=np.float64).reshape(nz, ny, nx)
    base, f, finite = _warp_cells(dvf, h, dims)
    B = base.shape[0]
    out = np.zeros((B, nz, ny, nx))
    for az in (0, 1):
        for ay in (0, 1):
            for ax in (0, 1):
                cx, cy, cz = base[:, 0] + ax, base[:, 1] + ay, base[:, 2] + az
                w = (f[:, 0] if ax else 1.0 - f[:, 0]) * (f[:, 1] if ay else 1.0 - f[:, 1]) * \
                    (f[:, 2] if az else 1.0 - f[:, 2])
                ok = (cx >= 0) & (cx < nx) & (cy >= 0) & (cy < ny) & (cz >= 0) & (cz < nz) & finite
                val = I[np.clip(cz, 0, nz - 1), np.clip(cy, 0, ny - 1), np.clip(cx, 0, nx - 1)]
                out += np.where(ok, w * val, 0.0)
    return out


def warp_backward(iref, dvf, grid, grad_out):
    """-> (dL/dI_ref [nz,ny,nx], dL/ddvf [B,3,nz,ny,nx]) fp64."""
    _, h, dims = _grid(grid)
    nx, ny, nz = (int(v) for v in dims)
    I = np.asarray(_f32(iref), dtype=np.float64).reshape(nz, ny, nx)
    base, f, finite = _warp_cells(dvf, h, dims)
    B = base.shape[0]
    g = np.asarray(_f32(grad_out), dtype=np.float64).reshape(B, nz, ny, nx)
    gI = np.zeros(nz * ny * nx)
    gd = np.zeros((B, 3, nz, ny, nx))
    h64 = np.asarray(h, dtype=np.float64)
    for az in (0, 1):
        for ay in (0, 1):
            for ax in (0, 1):
                cx, cy, cz = base[:, 0] + ax, base[:, 1] + ay, base[:, 2] + az
                wx = f[:, 0] if ax else 1.0 - f[:, 0]
                wy = f[:, 1] if ay else 1.0 - f[:, 1]
                wz = f[:, 2] if az else 1.0 - f[:, 2]
                ok = (cx >= 0) & (cx < nx) & (cy >= 0) & (cy < ny) & (cz >= 0) & (cz < nz) & finite
                lin = (np.clip(cz, 0, nz - 1) * ny + np.clip(cy, 0, ny - 1)) * nx + np.clip(cx, 0, nx - 1)
                gI += np.bincount(lin[ok], weights=(g * wx * wy * wz)[ok], minlength=gI.size)   # scatter-add
                val = np.where(ok, I.reshape(-1)[lin], 0.0)
                sx, sy, sz = (1.0 if ax else -1.0), (1.0 if ay else -1.0), (1.0 if az else -1.0)
                gd[:, 0] += g * val * sx * wy * wz / h64[0]
                gd[:, 1] += g * val * wx * sy * wz / h64[1]
                gd[:, 2] += g * val * wx * wy * sz / h64[2]
    return gI.reshape(nz, ny, nx), gd


# --------------------------------------------------------------------------------------------
# batched cone-beam forward projector, one DISTINCT volume per gantry angle
# (Eq. 12 "P denotes the ODL cone-beam projector that generates DRRs from the dynamic
# CBCT I(x,p)"; "requires a distinct DRR for each dynamic CBCT at each gantry angle ...
# future work could implement GPU-based parallelization to compute DRRs from multiple dynamic CBCTs
# simultaneously"; Eq. 6 I(r) = int sigma(r(t)) dt; Table I: SAD/SDD, detector size and pitch).
# The paper does not state ODL's discretisation.  Readings (P1-P5):
#  P1 geometry: circular orbit about the axis through `iso` parallel to z; source at
#     iso + SAD (cos a, sin a, 0); flat detector perpendicular to the central ray, SDD from the source,
#     u = (-sin a, cos a, 0), v = (0, 0, 1); pixel (iu, iv) centre at
#     det_centre + ((iu - (nu-1)/2) du + off_u) u + ((iv - (nv-1)/2) dv + off_v) v.
#  P2 line integral by Joseph's method (Joseph 1982): along the axis a on which the ray direction is
#     largest (first of x,y,z on ties), one sample per voxel-centre plane m of that axis, bilinear
#     interpolation in the plane, corners outside the grid read 0, each sample weighted by the path
#     length between planes h_a |D| / |D_a|.
#  P3 everything in fp64: per-ray constants (p0, ps, q0, qs, weight), the in-plane sample position
#     p0 + m ps of plane m, its cell floor(.) and the bilinear fractions.  (The interpolant is continuous
#     in the position, so an implementation that rounds the position differs by |grad I| x its rounding.)
#  P4 backward is the exact transpose (the projector is linear in the volume); no geometry gradients.
# --------------------------------------------------------------------------------------------
def cone_rays(grid, geom, angle):
    """geom = dict(sad, sdd, nu, nv, du, dv, off_u, off_v, iso[3]).  -> per-pixel [nv, nu] arrays:
    dominant axis a, and fp64 (p0, ps, q0, qs, weight) for the two in-plane axes (b, c) = the axes
    other than a in ascending order, all in voxel index units."""
    from .splat import geom32
    geom = geom32(geom)                                       # fp32 scalars, as gsvox_cone_geometry carries them
    o, h, dims = _grid(grid)
    o = o.astype(np.float64); h = h.astype(np.float64)
    ca, sa = np.cos(np.float64(angle)), np.sin(np.float64(angle))
    iso = np.asarray(geom["iso"], dtype=np.float64)
    src = iso + float(geom["sad"]) * np.array([ca, sa, 0.0])
    det_c = src - float(geom["sdd"]) * np.array([ca, sa, 0.0])
    nu, nv = int(geom["nu"]), int(geom["nv"])
    uu = (np.arange(nu) - (nu - 1) / 2.0) * float(geom["du"]) + float(geom["off_u"])
    vv = (np.arange(nv) - (nv - 1) / 2.0) * float(geom["dv"]) + float(geom["off_v"])
    P = det_c[None, None, :] + uu[None, :, None] * np.array([-sa, ca, 0.0]) + vv[:, None, None] * np.array([0.0, 0.0, 1.0])
    D = P - src                                               # [nv, nu, 3]
    absD = np.abs(D)
    a = np.where((absD[..., 0] >= absD[..., 1]) & (absD[..., 0] >= absD[..., 2]), 0,
                 np.where(absD[..., 1] >= absD[..., 2], 1, 2))
    norm = np.sqrt((D * D).sum(-1))
    out = {"axis": a}
    others = {0: (1, 2), 1: (0, 2), 2: (0, 1)}
    p0 = np.zeros(a.shape); ps = np.zeros(a.shape); q0 = np.zeros(a.shape); qs = np.zeros(a.shape); w = np.zeros(a.shape)
    for ax in range(3):
        sel = a == ax
        b, c = others[ax]
        Da = D[..., ax]
        with np.errstate(divide="ignore", invalid="ignore"):
            rb, rc = D[..., b] / Da, D[..., c] / Da
            p0a = (src[b] - o[b] + (o[ax] - src[ax]) * rb) / h[b]
            q0a = (src[c] - o[c] + (o[ax] - src[ax]) * rc) / h[c]
            psa, qsa = (h[ax] / h[b]) * rb, (h[ax] / h[c]) * rc
            wa = h[ax] * norm / np.abs(Da)
        p0[sel], ps[sel], q0[sel], qs[sel], w[sel] = p0a[sel], psa[sel], q0a[sel], qsa[sel], wa[sel]
    for k, v in (("p0", p0), ("ps", ps), ("q0", q0), ("qs", qs), ("w", w)):
        out[k] = v
    return out


def _project_terms(grid, geom, angle):
    """Yield, per dominant axis and plane m, (pixel mask, flat voxel index [4 corners], weight [4 corners])."""
    _, _, dims = _grid(grid)
    nx, ny, nz = (int(v) for v in dims)
    n = (nx, ny, nz)
    stride = (1, nx, nx * ny)
    rays = cone_rays(grid, geom, angle)
    others = {0: (1, 2), 1: (0, 2), 2: (0, 1)}
    for ax in range(3):
        sel = rays["axis"] == ax
        if not sel.any():
            continue
        b, c = others[ax]
        p0, ps, q0, qs = (rays[k][sel] for k in ("p0", "ps", "q0", "qs"))
        w = rays["w"][sel]
        for m in range(n[ax]):
            p = p0 + m * ps                                                 # fp64 (P3)
            q = q0 + m * qs
            good = (np.abs(p) < 4194304.0) & (np.abs(q) < 4194304.0)
            pf, qf = np.floor(np.where(good, p, 0)), np.floor(np.where(good, q, 0))
            fp_, fq = np.where(good, p, 0) - pf, np.where(good, q, 0) - qf
            ib, ic = pf.astype(np.int64), qf.astype(np.int64)
            idx, wt = [], []
            for db in (0, 1):
                for dc in (0, 1):
                    jb, jc = ib + db, ic + dc
                    ok = good & (jb >= 0) & (jb < n[b]) & (jc >= 0) & (jc < n[c])
                    lin = m * stride[ax] + np.clip(jb, 0, n[b] - 1) * stride[b] + np.clip(jc, 0, n[c] - 1) * stride[c]
                    wgt = (fp_ if db else 1.0 - fp_) * (fq if dc else 1.0 - fq) * w
                    idx.append(lin); wt.append(np.where(ok, wgt, 0.0))
            yield sel, idx, wt


def project_forward(vol, grid, geom, angles):
    """vol [B,nz,ny,nx] (or [nz,ny,nx], shared by all angles); angles [B] radians -> drr [B,nv,nu] fp64."""
    _, _, dims = _grid(grid)
    nx, ny, nz = (int(v) for v in dims)
    angles = np.atleast_1d(np.asarray(angles, dtype=np.float32))
    v = np.asarray(_f32(vol), dtype=np.float64).reshape(-1, nz * ny * nx)
    nu, nv = int(geom["nu"]), int(geom["nv"])
    out = np.zeros((angles.size, nv, nu))
    for bi, ang in enumerate(angles):
        vb = v[bi if v.shape[0] > 1 else 0]
        for sel, idx, wt in _project_terms(grid, geom, ang):
            acc = np.zeros(int(sel.sum()))
            for lin, w in zip(idx, wt):
                acc += w * vb[lin]
            out[bi][sel] += acc
    return out


def project_backward(grad_drr, grid, geom, angles):
    """Transpose of project_forward: grad_drr [B,nv,nu] -> grad_vol [B,nz,ny,nx] fp64."""
    _, _, dims = _grid(grid)
    nx, ny, nz = (int(v) for v in dims)
    angles = np.atleast_1d(np.asarray(angles, dtype=np.float32))
    g = np.asarray(_f32(grad_drr), dtype=np.float64).reshape(angles.size, int(geom["nv"]), int(geom["nu"]))
    out = np.zeros((angles.size, nz * ny * nx))
    for bi, ang in enumerate(angles):
        for sel, idx, wt in _project_terms(grid, geom, ang):
            gs = g[bi][sel]
            for lin, w in zip(idx, wt):
                out[bi] += np.bincount(lin, weights=w * gs, minlength=out.shape[1])
    return out.reshape(angles.size, nz, ny, nx)


# Gaussian-splat X-ray rasterizer (Eq. 6-9) — oracle/splat.py (torch fp64)
from .splat import (splat_backward, splat_backward_boxes, splat_forward, splat_forward_at, splat_forward_boxes,   # noqa: E402,F401
                    splat_terms)
