"""Thin Python binding of the gsvox C ABI (include/gsvox.h): argument marshalling only.

PyTorch is used for device memory and streams; every step of the path runs in the CUDA
kernels of libgsvox.so.  There is no CPU fallback: if the library is missing or cannot be
loaded the import of this module's functions fails loudly.
"""
import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libgsvox.so")

K_NAMES = ["preprocess", "count", "scan", "scatter", "forward", "backward", "epilogue", "memset", "dvf"]

EXPORTS = [
    "gsvox_workspace_bytes", "gsvox_plan_create", "gsvox_plan_destroy", "gsvox_preprocess",
    "gsvox_forward", "gsvox_backward", "gsvox_plan_status", "gsvox_plan_geometry_host",
    "gsvox_plan_bins_host", "gsvox_plan_set_timing", "gsvox_plan_timings",
    "gsvox_host_staging_bytes", "gsvox_step_host", "gsvox_error_string",
    "gsvox_last_cuda_error", "gsvox_version", "gsvox_dvf_forward", "gsvox_dvf_backward",
    "gsvox_mbc_combine_forward", "gsvox_mbc_combine_backward", "gsvox_warp_forward", "gsvox_warp_backward",
    "gsvox_plan_set_slab", "gsvox_backward_accumulate", "gsvox_backward_finish", "gsvox_plan_accumulators",
    "gsvox_project_scratch_bytes", "gsvox_project_forward", "gsvox_project_backward", "gsvox_project_forward_static",
    "gsvox_splat_workspace_bytes", "gsvox_splat_forward", "gsvox_splat_backward", "gsvox_splat_status",
    "gsvox_splat_drops", "gsvox_plan_set_deterministic", "gsvox_plan_unsorted_bins",
]
PROBE_EXPORTS = ["gsvox_probe_peaks"]            # include/gsvox_probe.h, libgsvox_probe.so (bench only)


class GsvoxGrid(C.Structure):
    _fields_ = [("origin", C.c_float * 3), ("spacing", C.c_float * 3), ("dims", C.c_int32 * 3)]


class GsvoxStatus(C.Structure):
    _fields_ = [("keys_needed", C.c_int64), ("pairs", C.c_int64),
                ("skipped_gaussians", C.c_int32), ("overflow", C.c_int32),
                ("culled_keys", C.c_int64), ("pairs_exec", C.c_int64)]


class GsvoxConeGeometry(C.Structure):
    _fields_ = [("sad", C.c_float), ("sdd", C.c_float), ("nu", C.c_int32), ("nv", C.c_int32),
                ("du", C.c_float), ("dv", C.c_float), ("off_u", C.c_float), ("off_v", C.c_float),
                ("iso", C.c_float * 3)]


class GsvoxError(RuntimeError):
    pass


_lib = None


def lib():
    """Load libgsvox.so (built in-tree by paper_2503_22139_b200/build.py).  Never falls back."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise GsvoxError("libgsvox.so is not built: run `python -c 'import __graft_entry__ as g; g.build()'` "
                         "(or python paper_2503_22139_b200/build.py); there is no CPU fallback")
    L = C.CDLL(LIB_PATH)
    vp, i64, i32, szp = C.c_void_p, C.c_int64, C.c_int32, C.POINTER(C.c_size_t)
    gp = C.POINTER(GsvoxGrid)
    L.gsvox_workspace_bytes.argtypes = [i64, i32, gp, i64, szp]
    L.gsvox_plan_create.argtypes = [i64, i32, gp, i64, vp, C.c_size_t, C.POINTER(vp)]
    L.gsvox_plan_destroy.argtypes = [vp]
    L.gsvox_plan_destroy.restype = None
    L.gsvox_preprocess.argtypes = [vp, vp, vp, vp, i64, vp]
    L.gsvox_forward.argtypes = [vp, vp, i32, vp, vp]
    L.gsvox_backward.argtypes = [vp, vp, i32, vp, vp, vp, vp, vp, vp]
    L.gsvox_plan_status.argtypes = [vp, C.POINTER(GsvoxStatus), vp]
    L.gsvox_plan_geometry_host.argtypes = [vp, vp, vp, vp]
    L.gsvox_plan_bins_host.argtypes = [vp, vp, vp, i64, vp]
    L.gsvox_plan_set_timing.argtypes = [vp, i32]
    L.gsvox_plan_timings.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(C.c_int64), i32, vp]
    L.gsvox_host_staging_bytes.argtypes = [i64, i32, gp, szp]
    L.gsvox_step_host.argtypes = [vp, vp, C.c_size_t, vp, vp, vp, vp, i64, i32, vp, vp, vp, vp, vp, vp, vp]
    L.gsvox_dvf_forward.argtypes = [vp, vp, vp, vp, i32, i32, vp, vp, vp]
    L.gsvox_dvf_backward.argtypes = [vp, vp, vp, vp, i32, i32, vp, vp, vp, vp, vp, vp, vp, vp, vp]
    L.gsvox_mbc_combine_forward.argtypes = [vp, vp, i32, i32, i64, vp, vp]
    L.gsvox_mbc_combine_backward.argtypes = [vp, vp, vp, i32, i32, i64, vp, vp, vp]
    L.gsvox_warp_forward.argtypes = [vp, vp, gp, i32, vp, vp]
    L.gsvox_warp_backward.argtypes = [vp, vp, gp, i32, vp, vp, vp, vp]
    L.gsvox_plan_set_slab.argtypes = [vp, i32, i32]
    L.gsvox_plan_set_deterministic.argtypes = [vp, i32]
    L.gsvox_plan_unsorted_bins.argtypes = [vp, C.POINTER(i64), vp]
    L.gsvox_backward_accumulate.argtypes = [vp, vp, i32, vp, vp]
    L.gsvox_backward_finish.argtypes = [vp, i32, vp, vp, vp, vp, vp]
    L.gsvox_plan_accumulators.argtypes = [vp, i32, C.POINTER(vp), C.POINTER(i64)]
    cgp = C.POINTER(GsvoxConeGeometry)
    L.gsvox_project_scratch_bytes.argtypes = [gp, i32, szp]
    L.gsvox_project_forward.argtypes = [vp, i64, gp, cgp, vp, i32, vp, vp, vp]
    L.gsvox_project_forward_static.argtypes = [vp, i64, gp, cgp, vp, i32, vp, vp]
    L.gsvox_project_backward.argtypes = [vp, gp, cgp, vp, i32, vp, vp, vp]
    L.gsvox_splat_workspace_bytes.argtypes = [i64, cgp, i32, i64, szp]
    L.gsvox_splat_forward.argtypes = [vp, vp, vp, vp, i64, cgp, vp, i32, vp, C.c_size_t, i64, vp, vp]
    L.gsvox_splat_backward.argtypes = [vp, vp, vp, vp, i64, cgp, vp, i32, vp, C.c_size_t, i64, vp, vp, vp, vp, vp, vp]
    L.gsvox_splat_status.argtypes = [vp, C.POINTER(i64), C.POINTER(i64), C.POINTER(i32), C.POINTER(i32), vp]
    L.gsvox_splat_drops.argtypes = [vp, C.POINTER(i64), C.POINTER(i64), C.POINTER(i64), vp]
    L.gsvox_error_string.argtypes = [C.c_int]
    L.gsvox_error_string.restype = C.c_char_p
    L.gsvox_last_cuda_error.restype = C.c_char_p
    L.gsvox_version.restype = C.c_int
    _lib = L
    return L


def _check(rc):
    if rc != 0:
        L = lib()
        msg = L.gsvox_error_string(rc).decode()
        extra = L.gsvox_last_cuda_error().decode()
        raise GsvoxError("gsvox error %d: %s%s" % (rc, msg, (" [" + extra + "]") if extra and rc == -3 else ""))


def make_grid(origin, spacing, dims):
    g = GsvoxGrid()
    for k in range(3):
        g.origin[k] = float(origin[k]); g.spacing[k] = float(spacing[k]); g.dims[k] = int(dims[k])
    return g


def _stream():
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _dev(t, name, shape=None):
    """Device pointer of a contiguous float32 CUDA tensor.  The C ABI takes raw pointers, so this binding is the only
    place a size can be checked: `shape` (a tuple; None entries are free) is what the call will read or write."""
    if t is None:
        return None
    if not (t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()):
        raise GsvoxError("%s must be a contiguous float32 CUDA tensor" % name)
    if shape is not None:
        got = tuple(int(v) for v in t.shape)
        if len(got) == len(shape) - 1 and shape[-1] == 1:      # [n] is accepted for [n, 1]
            got = got + (1,)
        if len(got) != len(shape) or any(w is not None and g != w for g, w in zip(got, shape)):
            raise GsvoxError("%s has shape %s, expected %s" % (name, tuple(t.shape), tuple(shape)))
    return C.c_void_p(t.data_ptr())


def _host(t, name, shape=None):
    if t is None:
        return None
    if t.is_cuda or t.dtype != torch.float32 or not t.is_contiguous():
        raise GsvoxError("%s must be a contiguous float32 CPU tensor" % name)
    if shape is not None and tuple(int(v) for v in t.shape) != tuple(shape):
        raise GsvoxError("%s has shape %s, expected %s" % (name, tuple(t.shape), tuple(shape)))
    return C.c_void_p(t.data_ptr())


_probe_lib = None


def probe_lib():
    """The bench-only microbenchmark library (include/gsvox_probe.h); separate from the product library."""
    global _probe_lib
    if _probe_lib is None:
        lib()                                        # raises if the build has not run (build.py makes both shared objects)
        path = os.path.join(os.path.dirname(LIB_PATH), "libgsvox_probe.so")
        L = C.CDLL(path)
        dp = C.POINTER(C.c_double)
        L.gsvox_probe_peaks.argtypes = [C.c_void_p, dp, dp, dp, C.POINTER(C.c_int32), C.c_void_p]
        _probe_lib = L
    return _probe_lib


def probe_peaks():
    """Measured FP32 (scalar FFMA, packed FFMA2) and MUFU ex2 rates of the current device."""
    scratch = torch.zeros(64, dtype=torch.float32, device="cuda")
    a, b, c, sms = C.c_double(0), C.c_double(0), C.c_double(0), C.c_int32(0)
    _check(probe_lib().gsvox_probe_peaks(C.c_void_p(scratch.data_ptr()), C.byref(a), C.byref(b), C.byref(c),
                                   C.byref(sms), _stream()))
    return {"fp32_tflops": a.value, "fp32x2_tflops": b.value, "ex2_tera_per_s": c.value, "sm_count": sms.value}


def mbc_combine_forward(e, coef, out=None):
    """e [L,3,nz,ny,nx], coef [B,L,3] -> dvf [B,3,nz,ny,nx] (Eq. 3), HBM-bound combine."""
    L_, B = int(e.shape[0]), int(coef.shape[0])
    V = int(e[0, 0].numel())
    vol = tuple(int(v) for v in e.shape[2:])
    if out is None:
        out = torch.empty((B, 3) + vol, dtype=torch.float32, device=e.device)
    _check(lib().gsvox_mbc_combine_forward(_dev(e, "e", (L_, 3) + vol), _dev(coef, "coef", (B, L_, 3)), B, L_, V,
                                           _dev(out, "dvf", (B, 3) + vol), _stream()))
    return out


def mbc_combine_backward(e, coef, grad_dvf, grads=None):
    """-> (grad_e [L,3,nz,ny,nx], grad_coef [B,L,3])."""
    L_, B = int(e.shape[0]), int(coef.shape[0])
    V = int(e[0, 0].numel())
    if grads is None:
        grads = (torch.empty_like(e), torch.empty((B, L_, 3), dtype=torch.float32, device=e.device))
    ge, gc = grads
    vol = tuple(int(v) for v in e.shape[2:])
    _check(lib().gsvox_mbc_combine_backward(_dev(e, "e", (L_, 3) + vol), _dev(coef, "coef", (B, L_, 3)),
                                            _dev(grad_dvf, "grad_dvf", (B, 3) + vol), B, L_, V,
                                            _dev(ge, "grad_e", (L_, 3) + vol), _dev(gc, "grad_coef", (B, L_, 3)), _stream()))
    return grads


def warp_forward(iref, dvf, grid, out=None):
    """iref [nz,ny,nx], dvf [B,3,nz,ny,nx] (world units), grid = (origin, spacing, dims) -> [B,nz,ny,nx]."""
    g = make_grid(*grid)
    B = int(dvf.shape[0])
    if out is None:
        out = torch.empty((B,) + tuple(iref.shape), dtype=torch.float32, device=iref.device)
    vol = (g.dims[2], g.dims[1], g.dims[0])
    _check(lib().gsvox_warp_forward(_dev(iref, "iref", vol), _dev(dvf, "dvf", (B, 3) + vol), C.byref(g), B,
                                    _dev(out, "out", (B,) + vol), _stream()))
    return out


def warp_backward(iref, dvf, grid, grad_out, grads=None):
    """-> (grad_iref [nz,ny,nx], grad_dvf [B,3,nz,ny,nx])."""
    g = make_grid(*grid)
    B = int(dvf.shape[0])
    if grads is None:
        grads = (torch.empty_like(iref), torch.empty_like(dvf))
    gi, gd = grads
    vol = (g.dims[2], g.dims[1], g.dims[0])
    _check(lib().gsvox_warp_backward(_dev(iref, "iref", vol), _dev(dvf, "dvf", (B, 3) + vol), C.byref(g), B,
                                     _dev(grad_out, "grad_out", (B,) + vol), _dev(gi, "grad_iref", vol),
                                     _dev(gd, "grad_dvf", (B, 3) + vol), _stream()))
    return grads


def make_cone_geometry(geom):
    g = GsvoxConeGeometry()
    g.sad, g.sdd, g.nu, g.nv = float(geom["sad"]), float(geom["sdd"]), int(geom["nu"]), int(geom["nv"])
    g.du, g.dv, g.off_u, g.off_v = float(geom["du"]), float(geom["dv"]), float(geom["off_u"]), float(geom["off_v"])
    for k in range(3):
        g.iso[k] = float(geom["iso"][k])
    return g


def _project_scratch(grid, B, device):
    nb = C.c_size_t(0)
    _check(lib().gsvox_project_scratch_bytes(C.byref(grid), B, C.byref(nb)))
    return torch.empty(int(nb.value) // 4, dtype=torch.float32, device=device)


def project_forward(vol, grid, geom, angles, out=None, scratch=None):
    """vol [B,nz,ny,nx] (or [nz,ny,nx] shared by all angles), angles: sequence of B radians (host)
    -> drr [B,nv,nu] (cone-beam line integrals, Joseph's method)."""
    g, cg = make_grid(*grid), make_cone_geometry(geom)
    ang = (C.c_float * len(angles))(*[float(a) for a in angles])
    B = len(angles)
    shared = vol.dim() == 3
    if out is None:
        out = torch.empty((B, cg.nv, cg.nu), dtype=torch.float32, device=vol.device)
    if scratch is None:
        scratch = _project_scratch(g, B, vol.device)
    V = int(vol[0].numel()) if not shared else int(vol.numel())
    vshape = (g.dims[2], g.dims[1], g.dims[0])
    nb = C.c_size_t(0)
    _check(lib().gsvox_project_scratch_bytes(C.byref(g), B, C.byref(nb)))
    if scratch.numel() * 4 < int(nb.value):
        raise GsvoxError("project scratch holds %d bytes, %d needed" % (scratch.numel() * 4, int(nb.value)))
    _check(lib().gsvox_project_forward(_dev(vol, "vol", vshape if shared else (B,) + vshape), 0 if shared else V,
                                       C.byref(g), C.byref(cg), ang, B, _dev(scratch, "scratch"),
                                       _dev(out, "drr", (B, cg.nv, cg.nu)), _stream()))
    return out


PROJECT_STATIC_MAX_VOXELS = 4194304          # GSVOX_PROJECT_STATIC_MAX_VOXELS (include/gsvox.h)


def project_forward_static(vol, grid, geom, angles, out):
    """project_forward for callers that cannot allocate device memory: `out` [B,nv,nu] is required, the scratch is a
    16 MB array built into libgsvox.so (B * voxels <= PROJECT_STATIC_MAX_VOXELS; shared by all calls on a device, so
    calls that overlap on the GPU race).  Allocates nothing on the device."""
    g, cg = make_grid(*grid), make_cone_geometry(geom)
    ang = (C.c_float * len(angles))(*[float(a) for a in angles])
    B = len(angles)
    shared = vol.dim() == 3
    vshape = (g.dims[2], g.dims[1], g.dims[0])
    V = vshape[0] * vshape[1] * vshape[2]
    if V * B > PROJECT_STATIC_MAX_VOXELS:
        raise GsvoxError("project_forward_static: %d volumes of %d voxels exceed the built-in scratch of %d voxels; "
                         "use project_forward with caller-owned scratch" % (B, V, PROJECT_STATIC_MAX_VOXELS))
    _check(lib().gsvox_project_forward_static(_dev(vol, "vol", vshape if shared else (B,) + vshape), 0 if shared else V,
                                              C.byref(g), C.byref(cg), ang, B,
                                              _dev(out, "drr", (B, cg.nv, cg.nu)), _stream()))
    return out


def project_backward(grad_drr, grid, geom, angles, out=None, scratch=None):
    """grad_drr [B,nv,nu] -> grad_vol [B,nz,ny,nx] (exact transpose of project_forward)."""
    g, cg = make_grid(*grid), make_cone_geometry(geom)
    ang = (C.c_float * len(angles))(*[float(a) for a in angles])
    B = len(angles)
    if out is None:
        out = torch.empty((B, g.dims[2], g.dims[1], g.dims[0]), dtype=torch.float32, device=grad_drr.device)
    if scratch is None:
        scratch = _project_scratch(g, B, grad_drr.device)
    nb = C.c_size_t(0)
    _check(lib().gsvox_project_scratch_bytes(C.byref(g), B, C.byref(nb)))
    if scratch.numel() * 4 < int(nb.value):
        raise GsvoxError("project scratch holds %d bytes, %d needed" % (scratch.numel() * 4, int(nb.value)))
    _check(lib().gsvox_project_backward(_dev(grad_drr, "grad_drr", (B, cg.nv, cg.nu)), C.byref(g), C.byref(cg), ang, B,
                                        _dev(scratch, "scratch"),
                                        _dev(out, "grad_vol", (B, g.dims[2], g.dims[1], g.dims[0])), _stream()))
    return out


class Splatter:
    """Gaussian-splat X-ray rasterizer (gsvox_splat_*): owns the torch workspace for n Gaussians, B angles."""

    def __init__(self, n_max, geom, batch, key_capacity=None, device="cuda"):
        self.geom, self.cg = dict(geom), make_cone_geometry(geom)
        self.n_max, self.batch = int(n_max), int(batch)
        if key_capacity is None:
            key_capacity = max(1 << 20, 48 * self.n_max * self.batch)
        self.key_capacity = int(key_capacity)
        self.device = torch.device(device)
        nb = C.c_size_t(0)
        _check(lib().gsvox_splat_workspace_bytes(self.n_max, C.byref(self.cg), self.batch, self.key_capacity, C.byref(nb)))
        self.workspace_bytes = int(nb.value)
        self._ws = torch.zeros(self.workspace_bytes + 256, dtype=torch.uint8, device=self.device)   # zeroed: no stale stamp
        self._base = (self._ws.data_ptr() + 255) & ~255
        self._n_fwd = None                                    # Gaussians of the latest forward

    def _angles(self, angles):
        if len(angles) != self.batch:
            raise GsvoxError("expected %d angles" % self.batch)
        return (C.c_float * len(angles))(*[float(a) for a in angles])

    def forward(self, pos, scale, quat, rho, angles, out=None):
        n = int(pos.shape[0])
        if n > self.n_max:
            raise GsvoxError("%d Gaussians, the Splatter was sized for %d" % (n, self.n_max))
        if out is None:
            out = torch.empty((self.batch, self.cg.nv, self.cg.nu), dtype=torch.float32, device=self.device)
        _check(lib().gsvox_splat_forward(_dev(pos, "pos", (n, 3)), _dev(scale, "scale", (n, 3)), _dev(quat, "quat", (n, 4)),
                                         _dev(rho, "rho", (n, 1)), n,
                                         C.byref(self.cg), self._angles(angles), self.batch, C.c_void_p(self._base),
                                         self.workspace_bytes, self.key_capacity,
                                         _dev(out, "drr", (self.batch, self.cg.nv, self.cg.nu)), _stream()))
        self._n_fwd = n
        return out

    def backward(self, pos, scale, quat, rho, angles, grad_drr, grads=None):
        n = int(pos.shape[0])
        if self._n_fwd is None or n != self._n_fwd:
            raise GsvoxError("Splatter.backward must follow Splatter.forward with the same Gaussians "
                             "(forward saw %s, backward %d)" % (self._n_fwd, n))
        if grads is None:
            mk = lambda *sh: torch.empty(sh, dtype=torch.float32, device=self.device)
            grads = (mk(n), mk(n, 3), mk(n, 3), mk(n, 4))
        gr, gp, gs, gq = grads
        _check(lib().gsvox_splat_backward(_dev(pos, "pos", (n, 3)), _dev(scale, "scale", (n, 3)), _dev(quat, "quat", (n, 4)),
                                          _dev(rho, "rho", (n, 1)), n,
                                          C.byref(self.cg), self._angles(angles), self.batch, C.c_void_p(self._base),
                                          self.workspace_bytes, self.key_capacity,
                                          _dev(grad_drr, "grad_drr", (self.batch, self.cg.nv, self.cg.nu)),
                                          _dev(gr, "grad_rho", (n, 1)), _dev(gp, "grad_pos", (n, 3)),
                                          _dev(gs, "grad_scale", (n, 3)), _dev(gq, "grad_quat", (n, 4)), _stream()))
        return grads

    def status(self):
        k, p, o, sk = C.c_int64(0), C.c_int64(0), C.c_int32(0), C.c_int32(0)
        _check(lib().gsvox_splat_status(C.c_void_p(self._base), C.byref(k), C.byref(p), C.byref(o), C.byref(sk), _stream()))
        a, b, c = C.c_int64(0), C.c_int64(0), C.c_int64(0)
        _check(lib().gsvox_splat_drops(C.c_void_p(self._base), C.byref(a), C.byref(b), C.byref(c), _stream()))
        return {"keys_needed": int(k.value), "pairs": int(p.value), "overflow": bool(o.value), "skipped": int(sk.value),
                "dropped_behind_source": int(a.value), "dropped_out_of_range": int(b.value), "dropped_empty_box": int(c.value)}


class Plan:
    """gsvox_plan + the torch-owned workspace it lives in."""

    def __init__(self, n_max, grid, max_channels=1, key_capacity=None, device="cuda", workspace=None):
        """workspace: optional caller-owned uint8 CUDA tensor (>= workspace_bytes + 255) to place the plan in."""
        origin, spacing, dims = grid
        self.grid = make_grid(origin, spacing, dims)
        self.dims = tuple(int(d) for d in dims)
        self.n_max = int(n_max)
        self.max_channels = int(max_channels)
        if key_capacity is None:
            # a key is one Gaussian touching one 8^3 brick; never more than n * nbricks
            nbricks = 1
            for d in self.dims:
                nbricks *= (d + 7) // 8
            key_capacity = min(self.n_max * nbricks, max(1 << 22, 64 * self.n_max))
        self.key_capacity = int(key_capacity)
        self.device = torch.device(device)
        nbytes = C.c_size_t(0)
        _check(lib().gsvox_workspace_bytes(self.n_max, self.max_channels, C.byref(self.grid),
                                           self.key_capacity, C.byref(nbytes)))
        self.workspace_bytes = int(nbytes.value)
        if workspace is None:
            workspace = torch.empty(self.workspace_bytes + 256, dtype=torch.uint8, device=self.device)
        if not (workspace.is_cuda and workspace.dtype == torch.uint8 and workspace.is_contiguous()):
            raise GsvoxError("workspace must be a contiguous uint8 CUDA tensor")
        self.workspace = workspace
        base = (self.workspace.data_ptr() + 255) & ~255
        if base + self.workspace_bytes > self.workspace.data_ptr() + self.workspace.numel():
            raise GsvoxError("workspace holds %d bytes, %d (+ alignment) needed" % (self.workspace.numel(), self.workspace_bytes))
        self.workspace_offset = base - self.workspace.data_ptr()
        self._h = C.c_void_p(None)
        _check(lib().gsvox_plan_create(self.n_max, self.max_channels, C.byref(self.grid), self.key_capacity,
                                       C.c_void_p(base), self.workspace_bytes, C.byref(self._h)))
        self.n = None
        self._staging = None

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            lib().gsvox_plan_destroy(self._h)
            self._h = C.c_void_p(None)

    def __del__(self):
        try:                 # at interpreter shutdown the module globals close() uses may already be gone
            self.close()
        except Exception:
            pass

    # --- the three hot-path calls -----------------------------------------------------
    def preprocess(self, pos, scale, quat):
        n = int(pos.shape[0])
        if n > self.n_max:
            raise GsvoxError("%d Gaussians, the plan was sized for %d" % (n, self.n_max))
        _check(lib().gsvox_preprocess(self._h, _dev(pos, "pos", (n, 3)), _dev(scale, "scale", (n, 3)),
                                      _dev(quat, "quat", (n, 4)), n, _stream()))
        self.n = n

    def _need_n(self):
        if self.n is None:
            raise GsvoxError("no preprocess on this plan yet")
        return self.n

    def forward(self, weight, out=None):
        ch = int(weight.shape[1])
        nx, ny, nz = self.dims
        if out is None:
            out = torch.empty((ch, nz, ny, nx), dtype=torch.float32, device=self.device)
        _check(lib().gsvox_forward(self._h, _dev(weight, "weight", (self._need_n(), ch)), ch,
                                   _dev(out, "out", (ch, nz, ny, nx)), _stream()))
        return out

    def backward(self, weight, grad_out, grads=None):
        n, ch = int(weight.shape[0]), int(weight.shape[1])
        if grads is None:
            mk = lambda k: torch.empty((n, k), dtype=torch.float32, device=self.device)
            grads = (mk(ch), mk(3), mk(3), mk(4))
        gw, gp, gs, gq = grads
        nx, ny, nz = self.dims
        n = self._need_n()
        _check(lib().gsvox_backward(self._h, _dev(weight, "weight", (n, ch)), ch, _dev(grad_out, "grad_out", (ch, nz, ny, nx)),
                                    _dev(gw, "grad_weight", (n, ch)), _dev(gp, "grad_pos", (n, 3)),
                                    _dev(gs, "grad_scale", (n, 3)), _dev(gq, "grad_quat", (n, 4)), _stream()))
        return grads

    # --- CUDA graph of one training step ----------------------------------------------
    def capture_step(self, pos, scale, quat, weight, grad_out, out=None, grads=None):
        """Capture gsvox_preprocess + gsvox_forward + gsvox_backward on the given (static) tensors into a
        CUDA graph and return (graph, out, grads): graph.replay() re-runs the step on whatever the tensors
        hold then.  The three calls never synchronise or allocate, so they are capturable as they are; for
        launch-bound sizes (config 1: 11 launches for 20 us of work) the replay removes the launch gaps."""
        ch = int(weight.shape[1])
        nx, ny, nz = self.dims
        n = int(pos.shape[0])
        if out is None:
            out = torch.empty((ch, nz, ny, nx), dtype=torch.float32, device=self.device)
        if grads is None:
            mk = lambda k: torch.empty((n, k), dtype=torch.float32, device=self.device)
            grads = (mk(ch), mk(3), mk(3), mk(4))
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(side):                      # warm-up outside the capture (first-launch module loads)
            self.preprocess(pos, scale, quat); self.forward(weight, out=out); self.backward(weight, grad_out, grads=grads)
        torch.cuda.current_stream().wait_stream(side)
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph):
            self.preprocess(pos, scale, quat)
            self.forward(weight, out=out)
            self.backward(weight, grad_out, grads=grads)
        return graph, out, grads

    # --- multi-GPU z-slabs --------------------------------------
    def set_slab(self, bz_begin, bz_end):
        _check(lib().gsvox_plan_set_slab(self._h, int(bz_begin), int(bz_end)))
        self.n = None

    def set_deterministic(self, on=True):
        """Sort every (brick, class) bin by Gaussian id and run a3 without atomics: bitwise repeatable forward."""
        _check(lib().gsvox_plan_set_deterministic(self._h, 1 if on else 0))
        self.n = None

    def unsorted_bins(self):
        v = C.c_int64(0)
        _check(lib().gsvox_plan_unsorted_bins(self._h, C.byref(v), _stream()))
        return int(v.value)

    def backward_accumulate(self, weight, grad_out):
        ch = int(weight.shape[1])
        nx, ny, nz = self.dims
        _check(lib().gsvox_backward_accumulate(self._h, _dev(weight, "weight", (self._need_n(), ch)), ch,
                                               _dev(grad_out, "grad_out", (ch, nz, ny, nx)), _stream()))

    def accumulators(self, channels):
        """torch view (no copy) of the [n, round4(9 + C)] accumulators: the all-reduce payload."""
        ptr, cnt = C.c_void_p(None), C.c_int64(0)
        _check(lib().gsvox_plan_accumulators(self._h, int(channels), C.byref(ptr), C.byref(cnt)))
        off = int(ptr.value) - self.workspace.data_ptr()
        return self.workspace[off:off + 4 * int(cnt.value)].view(torch.float32)

    def backward_finish(self, channels, grads=None):
        n = self.n
        if grads is None:
            mk = lambda k: torch.empty((n, k), dtype=torch.float32, device=self.device)
            grads = (mk(channels), mk(3), mk(3), mk(4))
        gw, gp, gs, gq = grads
        n = self._need_n()
        _check(lib().gsvox_backward_finish(self._h, int(channels), _dev(gw, "grad_weight", (n, int(channels))),
                                           _dev(gp, "grad_pos", (n, 3)), _dev(gs, "grad_scale", (n, 3)),
                                           _dev(gq, "grad_quat", (n, 4)), _stream()))
        return grads

    # --- 8(f) rank 1: fused MBC -> DVF ------------------------------------------------
    def _dvf_scratch(self, n, ch):
        key = (n, ch)
        if getattr(self, "_dvf_key", None) != key:
            self._dvf_mixed = torch.empty((n, ch), dtype=torch.float32, device=self.device)
            self._dvf_gmixed = torch.empty((n, ch), dtype=torch.float32, device=self.device)
            self._dvf_key = key
        return self._dvf_mixed, self._dvf_gmixed

    @staticmethod
    def _dev_i32(t, name):
        if not (t.is_cuda and t.dtype == torch.int32 and t.is_contiguous()):
            raise GsvoxError("%s must be a contiguous int32 CUDA tensor" % name)
        return C.c_void_p(t.data_ptr())

    def dvf_forward(self, feat, level, coef, out=None):
        n, B, L = int(feat.shape[0]), int(coef.shape[0]), int(coef.shape[1])
        nx, ny, nz = self.dims
        if out is None:
            out = torch.empty((B, 3, nz, ny, nx), dtype=torch.float32, device=self.device)
        mixed, _ = self._dvf_scratch(n, 3 * B)
        if n != self._need_n() or int(level.numel()) != n:
            raise GsvoxError("feat / level must have one row per preprocessed Gaussian (%d)" % self.n)
        _check(lib().gsvox_dvf_forward(self._h, _dev(feat, "feat", (n, 3)), self._dev_i32(level, "level"),
                                       _dev(coef, "coef", (B, L, 3)), B, L, _dev(mixed, "mixed"),
                                       _dev(out, "dvf", (B, 3, nz, ny, nx)), _stream()))
        return out

    def dvf_backward(self, feat, level, coef, grad_dvf, grads=None):
        n, B, L = int(feat.shape[0]), int(coef.shape[0]), int(coef.shape[1])
        if grads is None:
            mk = lambda *shape: torch.empty(shape, dtype=torch.float32, device=self.device)
            grads = (mk(n, 3), mk(B, L, 3), mk(n, 3), mk(n, 3), mk(n, 4))
        gf, gc, gp, gs, gq = grads
        mixed, gmixed = self._dvf_scratch(n, 3 * B)
        nx, ny, nz = self.dims
        if n != self._need_n() or int(level.numel()) != n:
            raise GsvoxError("feat / level must have one row per preprocessed Gaussian (%d)" % self.n)
        _check(lib().gsvox_dvf_backward(self._h, _dev(feat, "feat", (n, 3)), self._dev_i32(level, "level"),
                                        _dev(coef, "coef", (B, L, 3)), B, L, _dev(mixed, "mixed"),
                                        _dev(grad_dvf, "grad_dvf", (B, 3, nz, ny, nx)), _dev(gmixed, "grad_mixed"),
                                        _dev(gf, "grad_feat", (n, 3)), _dev(gc, "grad_coef", (B, L, 3)),
                                        _dev(gp, "grad_pos", (n, 3)), _dev(gs, "grad_scale", (n, 3)),
                                        _dev(gq, "grad_quat", (n, 4)), _stream()))
        return grads

    # --- synchronising helpers --------------------------------------------------------
    def status(self):
        s = GsvoxStatus()
        _check(lib().gsvox_plan_status(self._h, C.byref(s), _stream()))
        return {"keys_needed": int(s.keys_needed), "pairs": int(s.pairs),
                "skipped_gaussians": int(s.skipped_gaussians), "overflow": bool(s.overflow),
                "culled_keys": int(s.culled_keys), "pairs_exec": int(s.pairs_exec)}

    def geometry(self):
        box = torch.empty((self.n, 6), dtype=torch.int32)
        minv = torch.empty((self.n, 6), dtype=torch.float32)
        _check(lib().gsvox_plan_geometry_host(self._h, C.c_void_p(box.data_ptr()), C.c_void_p(minv.data_ptr()),
                                              _stream()))
        return box.numpy(), minv.numpy()

    def bins(self):
        nb = [(d + 7) // 8 for d in self.dims]
        nbricks = nb[0] * nb[1] * nb[2]
        start = torch.empty(nbricks + 1, dtype=torch.int64)
        _check(lib().gsvox_plan_bins_host(self._h, C.c_void_p(start.data_ptr()), None, 0, _stream()))
        total = int(start[-1])
        keys = torch.empty(max(total, 1), dtype=torch.int32)
        _check(lib().gsvox_plan_bins_host(self._h, C.c_void_p(start.data_ptr()), C.c_void_p(keys.data_ptr()),
                                          total, _stream()))
        return start.numpy(), keys.numpy()[:total]

    def layer_keys(self):
        """Keys per brick layer along z of the latest binning (SYNCHRONISES): what dist.slab_bounds_by_keys cuts on."""
        start, _ = self.bins()
        nb = [(d + 7) // 8 for d in self.dims]
        per_brick = start[1:] - start[:-1]
        return per_brick.reshape(nb[2], nb[1] * nb[0]).sum(axis=1).tolist()

    def set_timing(self, on):
        _check(lib().gsvox_plan_set_timing(self._h, 1 if on else 0))

    def timings(self, reset=True):
        ms = (C.c_double * len(K_NAMES))()
        cnt = (C.c_int64 * len(K_NAMES))()
        _check(lib().gsvox_plan_timings(self._h, ms, cnt, 1 if reset else 0, _stream()))
        return ({k: float(ms[i]) for i, k in enumerate(K_NAMES)},
                {k: int(cnt[i]) for i, k in enumerate(K_NAMES)})

    # --- end-to-end on host buffers ---------------------------------------------------
    def step_host(self, pos, scale, quat, weight, grad_out=None, out=None, grads=None):
        """Host (pinned) tensors in, host tensors out; H2D/D2H copies happen inside the call."""
        n, ch = int(pos.shape[0]), int(weight.shape[1])
        if self._staging is None:
            nbytes = C.c_size_t(0)
            _check(lib().gsvox_host_staging_bytes(self.n_max, self.max_channels, C.byref(self.grid), C.byref(nbytes)))
            self._staging_bytes = int(nbytes.value)
            self._staging = torch.empty(self._staging_bytes + 256, dtype=torch.uint8, device=self.device)
        base = (self._staging.data_ptr() + 255) & ~255
        gw = gp = gs = gq = None
        if grad_out is not None:
            gw, gp, gs, gq = grads
        nx, ny, nz = self.dims
        vol = (ch, nz, ny, nx)
        _check(lib().gsvox_step_host(self._h, C.c_void_p(base), self._staging_bytes,
                                     _host(pos, "pos", (n, 3)), _host(scale, "scale", (n, 3)), _host(quat, "quat", (n, 4)),
                                     _host(weight, "weight", (n, ch)), n, ch, _host(grad_out, "grad_out", vol),
                                     _host(out, "out", vol), _host(gw, "grad_weight", (n, ch)), _host(gp, "grad_pos", (n, 3)),
                                     _host(gs, "grad_scale", (n, 3)), _host(gq, "grad_quat", (n, 4)), _stream()))
        self.n = n
        return out, grads
