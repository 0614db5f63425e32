"""Seeded synthetic inputs for the five BASELINE.json configs (and small test variants).

This module is the ONLY code shared by the fp64 oracle (oracle/) and the CUDA path
(paper_2503_22139_b200/).  It holds none of the voxelizer's arithmetic: it only draws
positions, scales, quaternions, weights and upstream gradients with numpy's PCG64
(`numpy.random.default_rng`), in fp64, and casts to fp32 ONCE; both sides are handed
the same fp32 arrays.  The recipe is SURVEY.md section 8(d) "Concrete synthetic inputs",
restated in DESIGN.md; these inputs stand in for the paper's XCAT / MDACC / SPARE
volumes, which are not available — only shapes are borrowed.

Conventions common to all configs: origin (0,0,0), spacing (1,1,1) (voxel units),
"uniform in the grid" = U(-0.5, n_k - 0.5) per axis, unit quaternions = normalised
N(0, I4) in (w,x,y,z) order, "log-uniform a-b" = exp(U(ln a, ln b)), upstream gradient
N(0,1) in the output layout [C, nz, ny, nx], seed = config number - 1.
"""
from dataclasses import dataclass, field

import numpy as np


@dataclass
class Case:
    name: str
    dims: tuple                 # (nx, ny, nz)
    channels: int
    pos: np.ndarray             # [n,3] fp32
    scale: np.ndarray           # [n,3] fp32
    quat: np.ndarray            # [n,4] fp32 (w,x,y,z)
    weight: np.ndarray          # [n,C] fp32
    origin: tuple = (0.0, 0.0, 0.0)
    spacing: tuple = (1.0, 1.0, 1.0)
    seed: object = 0
    _grad_seed: object = field(default=None, repr=False)

    @property
    def n(self):
        return int(self.pos.shape[0])

    @property
    def grid(self):
        return (np.asarray(self.origin, np.float32), np.asarray(self.spacing, np.float32),
                np.asarray(self.dims, np.int32))

    @property
    def voxels(self):
        return int(self.dims[0]) * int(self.dims[1]) * int(self.dims[2])

    def grad_out(self):
        """Upstream gradient N(0,1), fp32, [C, nz, ny, nx]; drawn on demand (it is large)."""
        rng = np.random.default_rng(self._grad_seed)
        nx, ny, nz = self.dims
        return rng.standard_normal((self.channels, nz, ny, nx), dtype=np.float32)


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def _uniform_in_grid(rng, n, dims):
    d = np.asarray(dims, dtype=np.float64)
    return rng.uniform(-0.5, d - 0.5, size=(n, 3))


def _log_uniform(rng, a, b, size):
    return np.exp(rng.uniform(np.log(a), np.log(b), size=size))


def _unit_quats(rng, n):
    q = rng.standard_normal((n, 4))
    return q / np.linalg.norm(q, axis=1, keepdims=True)


def _case(name, dims, ch, pos, scale, quat, weight, seed, **kw):
    gs = [int(x) for x in np.atleast_1d(seed)] + [0x67726164]   # separate stream for grad_out
    return Case(name, tuple(int(d) for d in dims), ch, _f32(pos), _f32(scale), _f32(quat),
                _f32(weight).reshape(len(pos), ch), seed=seed, _grad_seed=gs, **kw)


def config1(n=2000, dims=(64, 64, 64), seed=0):
    """Tiny voxelizer: 64^3, 2,000 Gaussians, scales logU(0.5,3) per axis, w U(0,1)."""
    rng = np.random.default_rng(seed)
    pos = _uniform_in_grid(rng, n, dims)
    scale = _log_uniform(rng, 0.5, 3.0, (n, 3))
    quat = _unit_quats(rng, n)
    w = rng.uniform(0.0, 1.0, size=(n, 1))
    return _case("config1_tiny", dims, 1, pos, scale, quat, w, seed)


def config2(n=100_000, dims=(256, 256, 128), seed=1):
    """Reference-frame CBCT: centres uniform in volume inside a torso-like ellipsoid,
    scales logU(1,4), 3-tissue attenuation mix {0.02,0.2,0.5} with p=(0.6,0.3,0.1) + N(0,0.01)."""
    rng = np.random.default_rng(seed)
    d = np.asarray(dims, dtype=np.float64)
    centre = (d - 1.0) / 2.0
    semi = np.array([0.45, 0.35, 0.48]) * d
    pts = np.empty((0, 3))
    while pts.shape[0] < n:                       # rejection sampling in the unit ball
        u = rng.uniform(-1.0, 1.0, size=(2 * n, 3))
        pts = np.concatenate([pts, u[(u * u).sum(1) <= 1.0]])
    pos = centre + semi * pts[:n]
    scale = _log_uniform(rng, 1.0, 4.0, (n, 3))
    quat = _unit_quats(rng, n)
    tissue = rng.choice(np.array([0.02, 0.2, 0.5]), size=n, p=[0.6, 0.3, 0.1])
    w = (tissue + rng.normal(0.0, 0.01, size=n)).reshape(n, 1)
    return _case("config2_cbct", dims, 1, pos, scale, quat, w, seed)


_LEVELS = {1: (1_000, 16.0, 32.0), 2: (8_000, 6.0, 12.0), 3: (64_000, 2.0, 5.0)}


def config3(level, dims=(128, 128, 64), seed=2, n=None, channels=9):
    """Motion-basis DVF field, one level (1, 2 or 3): 9-channel features N(0,1),
    N = 1k / 8k / 64k, scales logU(16,32) / (6,12) / (2,5)."""
    n0, a, b = _LEVELS[level]
    n = n0 if n is None else n
    rng = np.random.default_rng([seed, level])
    pos = _uniform_in_grid(rng, n, dims)
    scale = _log_uniform(rng, a, b, (n, 3))
    quat = _unit_quats(rng, n)
    w = rng.standard_normal((n, channels))
    return _case("config3_dvf_level%d" % level, dims, channels, pos, scale, quat, w, [seed, level])


def config4(n=500_000, dims=(256, 256, 256), seed=3):
    """Training step at scale: 70% isotropic s0~logU(0.7,5); 30% anisotropic, three
    independent logU(0.7,5) draws redrawn until max/min <= 6; w U(0,0.5)."""
    rng = np.random.default_rng(seed)
    pos = _uniform_in_grid(rng, n, dims)
    iso = rng.uniform(size=n) < 0.7
    s0 = _log_uniform(rng, 0.7, 5.0, n)
    scale = np.repeat(s0[:, None], 3, axis=1)
    aniso = np.flatnonzero(~iso)
    s = _log_uniform(rng, 0.7, 5.0, (aniso.size, 3))
    bad = np.flatnonzero(s.max(1) / s.min(1) > 6.0)
    while bad.size:
        s[bad] = _log_uniform(rng, 0.7, 5.0, (bad.size, 3))
        bad = bad[s[bad].max(1) / s[bad].min(1) > 6.0]
    scale[aniso] = s
    quat = _unit_quats(rng, n)
    w = rng.uniform(0.0, 0.5, size=(n, 1))
    return _case("config4_train", dims, 1, pos, scale, quat, w, seed)


def config5(n=2_000_000, dims=(512, 512, 256), seed=4):
    """Load-imbalance stress: 95% small Gaussians (s logU(0.5,2)) in 16 Gaussian blobs
    (centres in the central 70% of each axis, blob sigma U(8,24), positions not clipped),
    5% needles s = (U(10,20), 0.5, 0.5) uniform in the grid; w U(0,1)."""
    rng = np.random.default_rng(seed)
    d = np.asarray(dims, dtype=np.float64)
    n_needle = int(round(0.05 * n))
    n_blob = n - n_needle
    blob_c = rng.uniform(0.15 * d - 0.5, 0.85 * d - 0.5, size=(16, 3))
    blob_sigma = rng.uniform(8.0, 24.0, size=16)
    which = rng.integers(0, 16, size=n_blob)
    pos_b = blob_c[which] + blob_sigma[which, None] * rng.standard_normal((n_blob, 3))
    scale_b = _log_uniform(rng, 0.5, 2.0, (n_blob, 3))
    pos_n = _uniform_in_grid(rng, n_needle, dims)
    scale_n = np.stack([rng.uniform(10.0, 20.0, size=n_needle),
                        np.full(n_needle, 0.5), np.full(n_needle, 0.5)], axis=1)
    pos = np.concatenate([pos_b, pos_n])
    scale = np.concatenate([scale_b, scale_n])
    perm = rng.permutation(n)                      # interleave needles with blob members
    pos, scale = pos[perm], scale[perm]
    quat = _unit_quats(rng, n)
    w = rng.uniform(0.0, 1.0, size=(n, 1))
    return _case("config5_stress", dims, 1, pos, scale, quat, w, seed)


def subvolume_case(n=600, dims=(37, 29, 21), channels=3, seed=11,
                   origin=(-13.5, 4.25, 100.0), spacing=(2.0, 1.5, 0.75)):
    """A ragged, anisotropic-spacing sub-grid with a non-zero origin and unnormalised
    quaternions, most Gaussians partly or wholly outside (the 32^3 TV sub-volume query of
    PAPER.md:128-130 and the coarse Stage-2 grid of PAPER.md:136 exercise these arguments)."""
    rng = np.random.default_rng(seed)
    d = np.asarray(dims, dtype=np.float64)
    o = np.asarray(origin, dtype=np.float64)
    h = np.asarray(spacing, dtype=np.float64)
    ext = d * h
    pos = o + rng.uniform(-0.4, 1.4, size=(n, 3)) * ext
    scale = _log_uniform(rng, 0.6, 6.0, (n, 3))
    quat = rng.standard_normal((n, 4)) * rng.uniform(0.2, 5.0, size=(n, 1))
    w = rng.standard_normal((n, channels))
    return _case("subvolume", dims, channels, pos, scale, quat, w, seed,
                 origin=tuple(origin), spacing=tuple(spacing))


@dataclass
class DvfCase:
    """Inputs of the fused MBC -> DVF op: the
    three MBC levels as ONE Gaussian set with a level id per Gaussian, a 3-vector feature per
    Gaussian (the Cartesian components k of e_{i,k}) and per-projection coefficients w_{i,k}(p)."""
    name: str
    dims: tuple
    pos: np.ndarray             # [n,3]
    scale: np.ndarray           # [n,3]
    quat: np.ndarray            # [n,4]
    feat: np.ndarray            # [n,3] fp32
    level: np.ndarray           # [n] int32 in 0..L-1
    coef: np.ndarray            # [B,L,3] fp32
    origin: tuple = (0.0, 0.0, 0.0)
    spacing: tuple = (1.0, 1.0, 1.0)
    seed: object = 0

    @property
    def n(self):
        return int(self.pos.shape[0])

    @property
    def batch(self):
        return int(self.coef.shape[0])

    @property
    def nlevels(self):
        return int(self.coef.shape[1])

    @property
    def grid(self):
        return (np.asarray(self.origin, np.float32), np.asarray(self.spacing, np.float32),
                np.asarray(self.dims, np.int32))

    def levels(self):
        """The same Gaussians split per level, as the oracle's (pos, scale, quat, feat) tuples,
        plus the index arrays that map each level back into the concatenated set."""
        out, ids = [], []
        for i in range(self.nlevels):
            sel = np.flatnonzero(self.level == i)
            ids.append(sel)
            out.append((self.pos[sel], self.scale[sel], self.quat[sel], self.feat[sel]))
        return out, ids

    def grad_dvf(self):
        rng = np.random.default_rng([77, self.batch] + list(np.atleast_1d(self.seed)))
        nx, ny, nz = self.dims
        return rng.standard_normal((self.batch, 3, nz, ny, nx), dtype=np.float32)


def dvf_case(batch=8, counts=(1_000, 8_000, 64_000), dims=(128, 128, 64), seed=5, shuffle=True,
             scales=((16.0, 32.0), (6.0, 12.0), (2.0, 5.0))):
    """Config 3's three MBC levels (same counts and scale ranges) as one set for the fused op:
    features N(0,1) per Cartesian component, coefficients w_{i,k}(p) ~ N(0,1) for `batch`
    projections (N_batch = 8 in Stage 3, 32 in Stage 2).  Level membership is
    interleaved (shuffle) so that the level id really is per Gaussian."""
    rng = np.random.default_rng(seed)
    pos, scale, quat, feat, level = [], [], [], [], []
    for i, (n, (a, b)) in enumerate(zip(counts, scales)):
        pos.append(_uniform_in_grid(rng, n, dims))
        scale.append(_log_uniform(rng, a, b, (n, 3)))
        quat.append(_unit_quats(rng, n))
        feat.append(rng.standard_normal((n, 3)))
        level.append(np.full(n, i, dtype=np.int32))
    pos, scale, quat, feat, level = (np.concatenate(x) for x in (pos, scale, quat, feat, level))
    if shuffle:
        perm = rng.permutation(pos.shape[0])
        pos, scale, quat, feat, level = pos[perm], scale[perm], quat[perm], feat[perm], level[perm]
    coef = rng.standard_normal((batch, len(counts), 3))
    return DvfCase("dvf_fused_b%d" % batch, tuple(dims), _f32(pos), _f32(scale), _f32(quat), _f32(feat),
                   np.ascontiguousarray(level, dtype=np.int32), _f32(coef), seed=seed)


@dataclass
class WarpCase:
    """Inputs of the warp I(x,p) = I_ref(x + d(x,p)) (Eq. 2)."""
    name: str
    dims: tuple
    iref: np.ndarray            # [nz,ny,nx] fp32
    dvf: np.ndarray             # [B,3,nz,ny,nx] fp32, world units, components x,y,z
    origin: tuple = (0.0, 0.0, 0.0)
    spacing: tuple = (2.0, 2.0, 2.0)
    seed: object = 0

    @property
    def batch(self):
        return int(self.dvf.shape[0])

    @property
    def grid(self):
        return (np.asarray(self.origin, np.float32), np.asarray(self.spacing, np.float32),
                np.asarray(self.dims, np.int32))

    def grad_out(self):
        rng = np.random.default_rng([78, self.batch] + list(np.atleast_1d(self.seed)))
        nx, ny, nz = self.dims
        return rng.standard_normal((self.batch, nz, ny, nx), dtype=np.float32)


def warp_case(batch=8, dims=(256, 256, 128), spacing=(2.0, 2.0, 2.0), amp_vox=4.0, seed=6, rough=0.15):
    """Stand-in for a reference CBCT and a batch of breathing DVFs (2 mm voxels):
    I_ref = an ellipsoidal body (0.45/0.35/0.48 of the grid, as config 2) of attenuation 0.2 with a
    few low-frequency cosine modulations plus N(0, 0.01) noise, 0 outside; d = per-projection
    amplitude U(-amp, amp) voxels per axis times a smooth cosine field, plus `rough` voxels of
    white noise (so neighbouring samples do not share cells exactly); world units = voxels x spacing.
    A thin shell of samples leaves the grid (zero padding is exercised)."""
    rng = np.random.default_rng(seed)
    nx, ny, nz = dims
    z, y, x = np.meshgrid(np.arange(nz, dtype=np.float32), np.arange(ny, dtype=np.float32),
                          np.arange(nx, dtype=np.float32), indexing="ij")
    c = (np.array([nx, ny, nz], np.float32) - 1) / 2
    semi = np.array([0.45 * nx, 0.35 * ny, 0.48 * nz], np.float32)
    r2 = ((x - c[0]) / semi[0]) ** 2 + ((y - c[1]) / semi[1]) ** 2 + ((z - c[2]) / semi[2]) ** 2
    body = (r2 <= 1.0).astype(np.float32)
    tex = np.zeros_like(body)
    for _ in range(4):
        k = rng.uniform(0.5, 4.0, size=3) * 2 * np.pi / np.array([nx, ny, nz])
        ph = rng.uniform(0, 2 * np.pi)
        tex += np.cos(k[0] * x + k[1] * y + k[2] * z + ph).astype(np.float32)
    iref = body * (0.2 + 0.05 * tex) + rng.normal(0.0, 0.01, size=body.shape).astype(np.float32) * body
    dvf = np.empty((batch, 3, nz, ny, nx), np.float32)
    for b in range(batch):
        for a in range(3):
            k = rng.uniform(0.3, 1.5, size=3) * 2 * np.pi / np.array([nx, ny, nz])
            ph = rng.uniform(0, 2 * np.pi)
            field = np.cos(k[0] * x + k[1] * y + k[2] * z + ph)
            field = rng.uniform(-amp_vox, amp_vox) * field + rough * rng.standard_normal(field.shape, dtype=np.float32)
            dvf[b, a] = (field * spacing[a]).astype(np.float32)
    return WarpCase("warp_b%d" % batch, tuple(dims), _f32(iref), dvf, spacing=tuple(spacing), seed=seed)


@dataclass
class ProjectCase:
    """Inputs of the batched cone-beam projector (Table I)."""
    name: str
    dims: tuple
    vol: np.ndarray             # [B,nz,ny,nx] fp32: one dynamic CBCT per gantry angle
    angles: np.ndarray          # [B] fp32 radians
    geom: dict                  # sad, sdd, nu, nv, du, dv, off_u, off_v, iso[3]
    origin: tuple = (0.0, 0.0, 0.0)
    spacing: tuple = (2.0, 2.0, 2.0)
    seed: object = 0

    @property
    def batch(self):
        return int(self.vol.shape[0])

    @property
    def grid(self):
        return (np.asarray(self.origin, np.float32), np.asarray(self.spacing, np.float32),
                np.asarray(self.dims, np.int32))

    def grad_drr(self):
        rng = np.random.default_rng([79, self.batch] + list(np.atleast_1d(self.seed)))
        return rng.standard_normal((self.batch, self.geom["nv"], self.geom["nu"]), dtype=np.float32)


def project_case(batch=8, dims=(200, 200, 100), spacing=(2.0, 2.0, 2.0), nu=512, nv=384, du=0.776, dv=0.776,
                 sad=1000.0, sdd=1500.0, off_u=0.0, off_v=0.0, seed=7, angles=None):
    """The paper's acquisition geometry (Table I: 512x384 pixels of 0.776 mm, SAD 1000 / SDD 1500 mm;
    200x200x100 voxels of 2 mm) with the isocentre at the grid centre.  Volumes: the
    ellipsoidal body of warp_case with a different low-frequency modulation per projection (stand-ins
    for the dynamic CBCTs); gantry angles uniform over a full turn unless given."""
    rng = np.random.default_rng(seed)
    nx, ny, nz = dims
    origin = tuple(-(n - 1) / 2.0 * h for n, h in zip(dims, spacing))
    z, y, x = np.meshgrid(np.arange(nz, dtype=np.float32), np.arange(ny, dtype=np.float32),
                          np.arange(nx, dtype=np.float32), indexing="ij")
    c = (np.array([nx, ny, nz], np.float32) - 1) / 2
    semi = np.array([0.45 * nx, 0.35 * ny, 0.48 * nz], np.float32)
    body = ((((x - c[0]) / semi[0]) ** 2 + ((y - c[1]) / semi[1]) ** 2 + ((z - c[2]) / semi[2]) ** 2) <= 1.0)
    body = body.astype(np.float32)
    vol = np.empty((batch, nz, ny, nx), np.float32)
    for b in range(batch):
        k = rng.uniform(0.5, 4.0, size=3) * 2 * np.pi / np.array([nx, ny, nz])
        tex = np.cos(k[0] * x + k[1] * y + k[2] * z + rng.uniform(0, 2 * np.pi)).astype(np.float32)
        vol[b] = body * (0.02 + 0.005 * tex) + body * rng.normal(0.0, 0.001, size=body.shape).astype(np.float32)
    if angles is None:
        angles = rng.uniform(0.0, 2 * np.pi, size=batch)
    geom = dict(sad=float(sad), sdd=float(sdd), nu=int(nu), nv=int(nv), du=float(du), dv=float(dv),
                off_u=float(off_u), off_v=float(off_v), iso=[0.0, 0.0, 0.0])
    return ProjectCase("project_b%d" % batch, tuple(dims), vol, np.asarray(angles, np.float32), geom,
                       origin=origin, spacing=tuple(spacing), seed=seed)


@dataclass
class SplatCase:
    """Inputs of the Gaussian-splat X-ray rasterizer (Eq. 6-9, Table I)."""
    name: str
    pos: np.ndarray             # [n,3] fp32, world units (mm), isocentre at the origin
    scale: np.ndarray           # [n,3]
    quat: np.ndarray            # [n,4]
    rho: np.ndarray             # [n]
    angles: np.ndarray          # [B] fp32 radians
    geom: dict
    seed: object = 0

    @property
    def n(self):
        return int(self.pos.shape[0])

    @property
    def batch(self):
        return int(self.angles.shape[0])

    def grad_drr(self):
        rng = np.random.default_rng([80, self.batch] + list(np.atleast_1d(self.seed)))
        return rng.standard_normal((self.batch, self.geom["nv"], self.geom["nu"]), dtype=np.float32)


def splat_case(n=50_000, batch=8, extent=(400.0, 400.0, 200.0), voxel=2.0, nu=512, nv=384, du=0.776, dv=0.776,
               sad=1000.0, sdd=1500.0, off_u=0.0, off_v=0.0, seed=8, angles=None, scales=(1.0, 4.0)):
    """Stage-1 stand-in: the reference-frame CBCT Gaussians of config 2 in world
    units — M = 50 000 (XCAT), centres uniform in an ellipsoid with semi-axes
    0.45/0.35/0.48 of a 400 x 400 x 200 mm field of view (200 x 200 x 100 voxels of 2 mm), scales
    log-uniform 1-4 voxels, random quaternions, 3-tissue attenuation mix — splatted onto the Table I
    detector (512 x 384 pixels of 0.776 mm, SAD 1000 / SDD 1500) at `batch` gantry angles."""
    rng = np.random.default_rng(seed)
    semi = np.array([0.45, 0.35, 0.48]) * np.asarray(extent)
    pts = np.empty((0, 3))
    while pts.shape[0] < n:
        c = rng.uniform(-1.0, 1.0, size=(2 * n + 16, 3))
        pts = np.concatenate([pts, c[(c * c).sum(1) <= 1.0]])
    pos = semi * pts[:n]
    scale = _log_uniform(rng, scales[0] * voxel, scales[1] * voxel, (n, 3))
    quat = _unit_quats(rng, n)
    tissue = rng.choice(np.array([0.02, 0.2, 0.5]), size=n, p=[0.6, 0.3, 0.1])
    rho = tissue + rng.normal(0.0, 0.01, size=n)
    if angles is None:
        angles = rng.uniform(0.0, 2 * np.pi, size=batch)
    geom = dict(sad=float(sad), sdd=float(sdd), nu=int(nu), nv=int(nv), du=float(du), dv=float(dv),
                off_u=float(off_u), off_v=float(off_v), iso=[0.0, 0.0, 0.0])
    return SplatCase("splat_n%d_b%d" % (n, len(angles)), _f32(pos), _f32(scale), _f32(quat), _f32(rho),
                     np.asarray(angles, np.float32), geom, seed=seed)


@dataclass
class Stage3Case:
    """Inputs of one Stage-2/3 step: reference Gaussians, three MBC levels, per-projection
    coefficients, gantry angles, all in world units (mm) on one voxel grid centred at the isocentre."""
    name: str
    dims: tuple
    spacing: tuple
    origin: tuple
    ref: tuple                  # (pos, scale, quat, rho[n,1])
    levels: list                # [(pos, scale, quat, feat[n,3]), ...]
    coef: np.ndarray            # [B, L, 3]
    angles: np.ndarray          # [B]
    geom: dict
    seed: object = 0

    @property
    def grid(self):
        return (np.asarray(self.origin, np.float32), np.asarray(self.spacing, np.float32),
                np.asarray(self.dims, np.int32))

    @property
    def batch(self):
        return int(self.angles.shape[0])

    def grad_drr(self):
        rng = np.random.default_rng([81, self.batch] + list(np.atleast_1d(self.seed)))
        return rng.standard_normal((self.batch, self.geom["nv"], self.geom["nu"]), dtype=np.float32)


def stage3_case(batch=8, dims=(200, 200, 100), voxel=2.0, n_ref=100_000, n_levels=(8_000, 10_648, 13_824),
                nu=512, nv=384, du=0.776, dv=0.776, sad=1000.0, sdd=1500.0, seed=9, dvf_mm=4.0):
    """The paper's patient-study sizes (M = 100 000 reference Gaussians, MBC levels 20^3 / 22^3 /
    24^3 Gaussians; 200 x 200 x 100 voxels of 2 mm; Table I detector).  Reference Gaussians as config 2 (scales
    logU(1,4) voxels, 3-tissue rho).  MBC Gaussians: the paper gives the counts but not the sizes; with 20-24
    Gaussians per axis the lattice pitch is ~10 x 10 x 5 voxels, so the three coarse-to-fine levels take scales
    logU(6,12) / (4,8) / (2,5) voxels (a reading; config 3's 16-32 voxels belong to its 1 000-Gaussian level),
    features N(0,1) mm; coefficients N(0, dvf_mm / sqrt(levels * mean overlap)), sized so that displacements are a
    few mm."""
    rng = np.random.default_rng(seed)
    ext = np.asarray(dims, np.float64) * voxel
    origin = tuple(-(n - 1) / 2.0 * voxel for n in dims)

    def in_ellipsoid(n):
        pts = np.empty((0, 3))
        while pts.shape[0] < n:
            c = rng.uniform(-1.0, 1.0, size=(2 * n + 16, 3))
            pts = np.concatenate([pts, c[(c * c).sum(1) <= 1.0]])
        return np.array([0.45, 0.35, 0.48]) * ext * pts[:n]
    pos = in_ellipsoid(n_ref)
    scale = _log_uniform(rng, 1.0 * voxel, 4.0 * voxel, (n_ref, 3))
    tissue = rng.choice(np.array([0.02, 0.2, 0.5]), size=n_ref, p=[0.6, 0.3, 0.1])
    rho = (tissue + rng.normal(0.0, 0.01, size=n_ref)).reshape(n_ref, 1)
    ref = (_f32(pos), _f32(scale), _f32(_unit_quats(rng, n_ref)), _f32(rho))
    k = voxel
    level_scales = ((6.0, 12.0), (4.0, 8.0), (2.0, 5.0))
    levels = []
    for n, (a, b) in zip(n_levels, level_scales):
        p = rng.uniform(-0.5, 0.5, size=(n, 3)) * ext
        levels.append((_f32(p), _f32(_log_uniform(rng, a * k, b * k, (n, 3))), _f32(_unit_quats(rng, n)),
                       _f32(rng.standard_normal((n, 3)))))
    # typical |e_{i,k}(x)| ~ sqrt(number of Gaussians overlapping a voxel): keep |d| at a few mm
    overlap = [n * (2.5 * k * (a + b) / 2) ** 3 / float(np.prod(ext)) for n, (a, b) in zip(n_levels, level_scales)]
    coef = rng.standard_normal((batch, len(n_levels), 3)) * dvf_mm / np.sqrt(3.0 * np.maximum(1.0, np.asarray(overlap)))[None, :, None]
    angles = rng.uniform(0.0, 2 * np.pi, size=batch)
    geom = dict(sad=float(sad), sdd=float(sdd), nu=int(nu), nv=int(nv), du=float(du), dv=float(dv),
                off_u=0.0, off_v=0.0, iso=[0.0, 0.0, 0.0])
    return Stage3Case("stage3_b%d" % batch, tuple(dims), (voxel,) * 3, origin, ref, levels, _f32(coef),
                      np.asarray(angles, np.float32), geom, seed=seed)


FULL = {
    "config1": lambda: [config1()],
    "config2": lambda: [config2()],
    "config3": lambda: [config3(1), config3(2), config3(3)],
    "config4": lambda: [config4()],
    "config5": lambda: [config5()],
}
