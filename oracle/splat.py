"""fp64 CPU oracle of the Gaussian-splat X-ray rasterizer (PAPER.md:76-94,
Eq. 6-9).  TEST INFRASTRUCTURE ONLY (same rules as oracle/__init__.py).  Plain PyTorch CPU ops in
fp64; the backward is torch autograd of this forward.

PAPER.md Eq. 8: each 3D Gaussian is mapped to ray space by the local affine approximation of the
projective mapping phi, Sigma~ = J W Sigma W^T J^T; Eq. 9: integrating over the ray coordinate x2
leaves a 2D Gaussian with Sigma^ = Sigma~[0:2, 0:2], centre p^ = (p~0, p~1) and amplitude
rho^ = rho sqrt(2 pi |Sigma~| / |Sigma^|).  "phi, J and W are determined by scanner parameters"
 — the paper defers them to R2-Gaussian; the readings taken:
  R1 scanner = the projector's (P1): source at iso + SAD (cos a, sin a, 0), flat detector at SDD,
     u = (-sin a, cos a, 0), v = (0, 0, 1).  Camera frame: origin at the source, rows of W =
     (u, v, c) with c = -(cos a, sin a, 0) the central-ray direction; t = W (p - source).
  R2 ray space (EWA splatting): phi(t) = (t0/t2, t1/t2, |t|); the third coordinate is the path
     length along the ray, so Eq. 6's integral over t is the integral over x2.  J = d phi / d t at t.
  R3 pixel (iu, iv) has ray-space coordinates x^ = (u/SDD, v/SDD), u = (iu - (nu-1)/2) du + off_u.
  R4 cutoff: the axis-aligned box of the 3-sigma ellipse on the detector, in pixels, inclusive,
     clipped to the detector, decided in fp64; nothing else is tested inside the box (as A3/A4).
  R5 a Gaussian with t2 <= 0 (at or behind the source plane), with degenerate parameters, or whose
     centre projects more than 30000 pixels off the detector origin is skipped.  R6 backward: supports frozen.
"""
import math

import numpy as np
import torch

KAPPA = 3.0


def _t(a):
    return torch.as_tensor(np.ascontiguousarray(np.asarray(a, dtype=np.float32)), dtype=torch.float32).to(torch.float64)


def geom32(geom):
    """The scanner geometry as the boundary carries it: gsvox_cone_geometry holds fp32 scalars (sad, sdd, du, dv,
    off_u, off_v, iso), so — like every other input ("inputs are fp32; the oracle promotes them
    exactly") — they are rounded to fp32 once and promoted to fp64.  0.776 mm is not an fp32 number: taking it as the
    Python double moved cu + 3 sigma by 1e-6 pixel and one box edge of 400 000 across an integer (found by the
    every-pixel parity at the bench size)."""
    g = dict(geom)
    for k in ("sad", "sdd", "du", "dv", "off_u", "off_v"):
        g[k] = float(np.float32(geom[k]))
    g["iso"] = [float(np.float32(v)) for v in geom["iso"]]
    return g


def splat_terms(pos, scale, quat, rho, geom, angle, kappa=KAPPA):
    """Per-Gaussian 2D quantities for one gantry angle (torch fp64, differentiable):
    centre in pixel coordinates (cu, cv), conic (A, B, C) in pixel units, amplitude, inclusive
    integer box (u0, v0, u1, v1) and validity."""
    geom = geom32(geom)
    qn = quat / quat.norm(dim=1, keepdim=True)
    r, x, y, z = qn[:, 0], qn[:, 1], qn[:, 2], qn[:, 3]
    R = torch.stack([1 - 2 * (y * y + z * z), 2 * (x * y - r * z), 2 * (x * z + r * y),
                     2 * (x * y + r * z), 1 - 2 * (x * x + z * z), 2 * (y * z - r * x),
                     2 * (x * z - r * y), 2 * (y * z + r * x), 1 - 2 * (x * x + y * y)], dim=1).reshape(-1, 3, 3)
    Sigma = R @ torch.diag_embed(scale * scale) @ R.transpose(1, 2)
    a = float(np.float64(np.float32(angle)))
    ca, sa = math.cos(a), math.sin(a)
    iso = torch.tensor([float(v) for v in geom["iso"]], dtype=torch.float64)
    src = iso + float(geom["sad"]) * torch.tensor([ca, sa, 0.0], dtype=torch.float64)
    W = torch.tensor([[-sa, ca, 0.0], [0.0, 0.0, 1.0], [-ca, -sa, 0.0]], dtype=torch.float64)
    t = (pos - src) @ W.T
    t0, t1, t2 = t[:, 0], t[:, 1], t[:, 2]
    valid = t2 > 0
    t2s = torch.where(valid, t2, torch.ones_like(t2))
    ell = torch.sqrt(t0 * t0 + t1 * t1 + t2s * t2s)
    zero = torch.zeros_like(t0)
    J = torch.stack([1 / t2s, zero, -t0 / (t2s * t2s),
                     zero, 1 / t2s, -t1 / (t2s * t2s),
                     t0 / ell, t1 / ell, t2s / ell], dim=1).reshape(-1, 3, 3)
    T = J @ W
    St = T @ Sigma @ T.transpose(1, 2)
    det_t = torch.linalg.det(St)
    # detector pixels: u = SDD x0, pixel index = (u - off_u) / du + (nu - 1) / 2
    ku, kv = float(geom["sdd"]) / float(geom["du"]), float(geom["sdd"]) / float(geom["dv"])
    s00, s01, s11 = St[:, 0, 0], St[:, 0, 1], St[:, 1, 1]
    det_h = s00 * s11 - s01 * s01
    amp = rho * torch.sqrt(2 * math.pi * det_t / det_h)
    p00, p01, p11 = s00 * ku * ku, s01 * ku * kv, s11 * kv * kv          # Sigma^ in pixel units
    dp = p00 * p11 - p01 * p01
    A, B, C = p11 / dp, -p01 / dp, p00 / dp
    cu = (float(geom["sdd"]) * t0 / t2s - float(geom["off_u"])) / float(geom["du"]) + (int(geom["nu"]) - 1) / 2.0
    cv = (float(geom["sdd"]) * t1 / t2s - float(geom["off_v"])) / float(geom["dv"]) + (int(geom["nv"]) - 1) / 2.0
    with torch.no_grad():
        ru, rv = kappa * torch.sqrt(p00), kappa * torch.sqrt(p11)
        u0 = torch.clamp(torch.ceil(cu - ru), min=0)
        u1 = torch.clamp(torch.floor(cu + ru), max=int(geom["nu"]) - 1)
        v0 = torch.clamp(torch.ceil(cv - rv), min=0)
        v1 = torch.clamp(torch.floor(cv + rv), max=int(geom["nv"]) - 1)
        finite = torch.isfinite(cu) & torch.isfinite(cv) & torch.isfinite(ru) & torch.isfinite(rv) & (det_h > 0) & (det_t > 0)
        near = (cu.abs() <= 30000.0) & (cv.abs() <= 30000.0)          # R5: centres beyond +-30000 pixels are skipped
        valid = valid & finite & near & (u1 >= u0) & (v1 >= v0)
        box = torch.stack([u0, v0, u1, v1], dim=1)
    return cu, cv, A, B, C, amp, box, valid


def _chunk_size(npix):
    return max(1, min(512, int(2.0e7 // max(1, npix))))


def _render_subset(ids, cu, cv, A, B, C, amp, box, pix_u, pix_v):
    """Contribution of the Gaussians `ids` at the listed pixels, and the number of pairs in their boxes."""
    sh = (-1,) + (1,) * pix_u.dim()
    du, dv = pix_u[None] - cu[ids].reshape(sh), pix_v[None] - cv[ids].reshape(sh)
    inside = ((pix_u[None] >= box[ids, 0].reshape(sh)) & (pix_u[None] <= box[ids, 2].reshape(sh)) &
              (pix_v[None] >= box[ids, 1].reshape(sh)) & (pix_v[None] <= box[ids, 3].reshape(sh)))
    q = A[ids].reshape(sh) * du * du + 2 * B[ids].reshape(sh) * du * dv + C[ids].reshape(sh) * dv * dv
    val = amp[ids].reshape(sh) * torch.exp(-0.5 * q)
    return torch.where(inside, val, torch.zeros_like(val)).sum(0), int(inside.sum())


def _render(pos, scale, quat, rho, geom, angle, pix_u, pix_v, kappa):
    """Sum of the 2D Gaussians at the listed pixels (pix_u, pix_v: fp64 tensors of equal shape)."""
    cu, cv, A, B, C, amp, box, valid = splat_terms(pos, scale, quat, rho, geom, angle, kappa)
    out = torch.zeros_like(pix_u)
    pairs = 0
    idx = torch.nonzero(valid).reshape(-1)
    chunk = _chunk_size(pix_u.numel())
    for s in range(0, idx.numel(), chunk):
        part, k = _render_subset(idx[s:s + chunk], cu, cv, A, B, C, amp, box, pix_u, pix_v)
        out = out + part
        pairs += k
    return out, pairs


def splat_forward(pos, scale, quat, rho, geom, angles, kappa=KAPPA, return_pairs=False):
    """pos [n,3], scale [n,3], quat [n,4] (w,x,y,z), rho [n] (fp32 arrays); angles [B] radians
    -> drr [B, nv, nu] fp64 (and the number of (Gaussian, pixel) pairs inside the cutoff)."""
    p, s, q, r = _t(pos), _t(scale), _t(quat), _t(rho).reshape(-1)
    nu, nv = int(geom["nu"]), int(geom["nv"])
    vv, uu = torch.meshgrid(torch.arange(nv, dtype=torch.float64), torch.arange(nu, dtype=torch.float64), indexing="ij")
    out, pairs = [], 0
    with torch.no_grad():
        for a in np.atleast_1d(np.asarray(angles, dtype=np.float32)):
            img, k = _render(p, s, q, r, geom, a, uu, vv, kappa)
            out.append(img.numpy()); pairs += k
    out = np.stack(out)
    return (out, pairs) if return_pairs else out


def splat_forward_boxes(pos, scale, quat, rho, geom, angles, kappa=KAPPA):
    """The same sum as splat_forward, organised per Gaussian instead of per pixel chunk: for every valid
    (angle, Gaussian) the 2D Gaussian of Eq. 9 is added on the pixels of its inclusive box, nothing else — a plain
    double loop with numpy rows.  Cost is proportional to the pairs inside the cutoff, so the bench size (50 000
    Gaussians, 8 angles, 512 x 384 pixels, 1e9 pairs) takes about a minute where the masked form above would take
    hours; tests/test_splat_oracle_pins.py pins it to splat_forward.  -> drr [B, nv, nu] fp64."""
    p, s, q, r = _t(pos), _t(scale), _t(quat), _t(rho).reshape(-1)
    nu, nv = int(geom["nu"]), int(geom["nv"])
    out = np.zeros((len(np.atleast_1d(angles)), nv, nu))
    with torch.no_grad():
        for b, a in enumerate(np.atleast_1d(np.asarray(angles, dtype=np.float32))):
            cu, cv, A, B, C, amp, box, valid = (x.numpy() for x in splat_terms(p, s, q, r, geom, a, kappa))
            img = out[b]
            for i in np.flatnonzero(valid):
                u0, v0, u1, v1 = (int(x) for x in box[i])
                du = np.arange(u0, u1 + 1, dtype=np.float64) - cu[i]
                dv = np.arange(v0, v1 + 1, dtype=np.float64) - cv[i]
                qf = A[i] * du[None, :] ** 2 + 2.0 * B[i] * du[None, :] * dv[:, None] + C[i] * dv[:, None] ** 2
                img[v0:v1 + 1, u0:u1 + 1] += amp[i] * np.exp(-0.5 * qf)
    return out


def splat_forward_at(pos, scale, quat, rho, geom, angle, pixels, kappa=KAPPA):
    """Values at listed pixels [(iu, iv), ...] of one projection -> [m] fp64."""
    p, s, q, r = _t(pos), _t(scale), _t(quat), _t(rho).reshape(-1)
    pix = np.asarray(pixels, dtype=np.float64).reshape(-1, 2)
    with torch.no_grad():
        img, _ = _render(p, s, q, r, geom, angle, torch.tensor(pix[:, 0]), torch.tensor(pix[:, 1]), kappa)
    return img.numpy()


def splat_backward(pos, scale, quat, rho, geom, angles, grad_drr, kappa=KAPPA, pixels=None):
    """Gradients of L = <grad_drr, drr> (grad_drr [B,nv,nu] fp32) -> (d rho [n], d pos [n,3],
    d scale [n,3], d quat [n,4]) fp64, by autograd of the forward above.  L is a sum over
    Gaussians, so it is differentiated in chunks of Gaussians (bounded memory).  With `pixels`
    ([(b, iu, iv), ...]) only those pixels enter L (sampled parity at full size)."""
    P, S, Q, Rh = _t(pos), _t(scale), _t(quat), _t(rho).reshape(-1)
    n = P.shape[0]
    angles = np.atleast_1d(np.asarray(angles, dtype=np.float32))
    nu, nv = int(geom["nu"]), int(geom["nv"])
    g = torch.as_tensor(np.asarray(grad_drr, dtype=np.float32)).to(torch.float64).reshape(angles.size, nv, nu)
    gr, gp, gs, gq = torch.zeros(n, dtype=torch.float64), torch.zeros(n, 3, dtype=torch.float64), \
        torch.zeros(n, 3, dtype=torch.float64), torch.zeros(n, 4, dtype=torch.float64)
    for b, a in enumerate(angles):
        if pixels is None:
            vv, uu = torch.meshgrid(torch.arange(nv, dtype=torch.float64), torch.arange(nu, dtype=torch.float64), indexing="ij")
            gb = g[b]
        else:
            sel = np.asarray([(iu, iv) for (bb, iu, iv) in pixels if bb == b], dtype=np.int64).reshape(-1, 2)
            if sel.shape[0] == 0:
                continue
            uu, vv = torch.tensor(sel[:, 0], dtype=torch.float64), torch.tensor(sel[:, 1], dtype=torch.float64)
            gb = g[b][sel[:, 1], sel[:, 0]]
        chunk = _chunk_size(uu.numel())
        for s0 in range(0, n, chunk):
            sl = slice(s0, min(n, s0 + chunk))
            p, s, q, r = (P[sl].clone().requires_grad_(True), S[sl].clone().requires_grad_(True),
                          Q[sl].clone().requires_grad_(True), Rh[sl].clone().requires_grad_(True))
            cu, cv, A, B_, C, amp, box, valid = splat_terms(p, s, q, r, geom, a, kappa)
            ids = torch.nonzero(valid).reshape(-1)
            if ids.numel() == 0:
                continue
            img, _ = _render_subset(ids, cu, cv, A, B_, C, amp, box, uu, vv)
            (img * gb).sum().backward()
            gr[sl] += r.grad; gp[sl] += p.grad; gs[sl] += s.grad; gq[sl] += q.grad
    return gr.numpy(), gp.numpy(), gs.numpy(), gq.numpy()


def splat_backward_boxes(pos, scale, quat, rho, geom, angles, grad_drr, kappa=KAPPA, group=64):
    """splat_backward over ALL pixels at a cost proportional to the pairs inside the cutoff: the same autograd of the
    same _render_subset, but each group of Gaussians (taken in the order of their projected centre, so that a group is
    compact on the detector) is rendered only on the union of its boxes — outside every box `inside` is false and
    the pixel contributes nothing to the loss, so the result is that of splat_backward.  Pinned to it on the CPU
    (tests/test_splat_oracle_pins.py).  -> (d rho [n], d pos [n,3], d scale [n,3], d quat [n,4]) fp64."""
    P, S, Q, Rh = _t(pos), _t(scale), _t(quat), _t(rho).reshape(-1)
    n = P.shape[0]
    angles = np.atleast_1d(np.asarray(angles, dtype=np.float32))
    nu, nv = int(geom["nu"]), int(geom["nv"])
    g = torch.as_tensor(np.asarray(grad_drr, dtype=np.float32)).to(torch.float64).reshape(angles.size, nv, nu)
    gr, gp, gs, gq = torch.zeros(n, dtype=torch.float64), torch.zeros(n, 3, dtype=torch.float64), \
        torch.zeros(n, 3, dtype=torch.float64), torch.zeros(n, 4, dtype=torch.float64)
    for b, a in enumerate(angles):
        with torch.no_grad():
            cu0, cv0, _, _, _, _, box0, valid0 = splat_terms(P, S, Q, Rh, geom, a, kappa)
        ids_all = torch.nonzero(valid0).reshape(-1)
        if ids_all.numel() == 0:
            continue
        # order by 32-pixel detector cell of the centre: neighbours on the detector end up in the same group
        cell = (torch.floor(cv0[ids_all] / 32.0) * 4096 + torch.floor(cu0[ids_all] / 32.0))
        ids_all = ids_all[torch.argsort(cell, stable=True)]
        for s0 in range(0, ids_all.numel(), group):
            ids = ids_all[s0:s0 + group]
            bx = box0[ids]
            u0, v0 = int(bx[:, 0].min()), int(bx[:, 1].min())
            u1, v1 = int(bx[:, 2].max()), int(bx[:, 3].max())
            vv, uu = torch.meshgrid(torch.arange(v0, v1 + 1, dtype=torch.float64),
                                    torch.arange(u0, u1 + 1, dtype=torch.float64), indexing="ij")
            p, s, q, r = (P[ids].clone().requires_grad_(True), S[ids].clone().requires_grad_(True),
                          Q[ids].clone().requires_grad_(True), Rh[ids].clone().requires_grad_(True))
            cu, cv, A, B_, C, amp, box, valid = splat_terms(p, s, q, r, geom, a, kappa)
            img, _ = _render_subset(torch.arange(ids.numel()), cu, cv, A, B_, C, amp, box, uu, vv)
            (img * g[b, v0:v1 + 1, u0:u1 + 1]).sum().backward()
            gr[ids] += r.grad; gp[ids] += p.grad; gs[ids] += s.grad; gq[ids] += q.grad
    return gr.numpy(), gp.numpy(), gs.numpy(), gq.numpy()
