"""Shared checks of the `-m gpu` parity tests (no test in here; imported by tests/test_gpu_*.py).

Two gradient criteria:
  * the pass criterion of record, north_star's: relative L2 error <= 1e-4 per parameter group over ALL Gaussians;
  * a per-Gaussian bound on top, because a group norm over 5e5 Gaussians cannot see a few hundred completely
    wrong rows (one broken key class, one brick-edge case):
        |g_gpu,i - g_ref,i|_2  <=  PER_REL |g_ref,i|_2 + PER_ABS rms_j |g_ref,j|_2      for every Gaussian i,
    PER_REL = 1e-3, PER_ABS = 1e-4 (the absolute term carries Gaussians whose gradient is a near-cancelling sum:
    fp32 accumulation error scales with the terms, not with their sum; the scale is the root mean square of the
    row norms, not their median: 70 % of config 4's Gaussians are isotropic, their dL/dq is exactly 0 in the
    oracle and so is the median).  The worst offender is reported.
"""
import numpy as np

GRAD_REL = 1e-4
PER_REL, PER_ABS = 1e-3, 1e-4


def rel_l2(a, b):
    a = np.asarray(a, dtype=np.float64).reshape(np.shape(b))
    nb = np.linalg.norm(b)
    return float(np.linalg.norm(a - b) / nb) if nb > 0 else float(np.abs(a).max(initial=0.0))


def per_row_worst(a, b):
    """-> (worst ratio err_i / (PER_REL |b_i| + PER_ABS rms|b|), its row index, err_i, |b_i|)."""
    b = np.asarray(b, dtype=np.float64)
    a = np.asarray(a, dtype=np.float64).reshape(b.shape)
    if b.size == 0:
        return 0.0, -1, 0.0, 0.0
    b2 = b.reshape(b.shape[0], -1)
    a2 = a.reshape(b.shape[0], -1)
    nb = np.linalg.norm(b2, axis=1)
    err = np.linalg.norm(a2 - b2, axis=1)
    rms = float(np.sqrt(np.mean(nb * nb)))
    allow = PER_REL * nb + PER_ABS * rms
    ratio = np.where(allow > 0, err / np.where(allow > 0, allow, 1.0), np.where(err > 0, np.inf, 0.0))
    i = int(np.argmax(ratio))
    return float(ratio[i]), i, float(err[i]), float(nb[i])


def check_grad_groups(names, grads, refs, tol=GRAD_REL, per_row=True, describe=None, label=""):
    """Assert both criteria for every group; returns {name: (rel L2, worst per-row ratio, row)}.
    describe(i) -> str adds context (box, scales, class) to the message about row i."""
    out = {}
    for name, a, b in zip(names, grads, refs):
        rel = rel_l2(a, b)
        assert rel <= tol, "%s grad %s rel L2 %.3e > %.1e" % (label, name, rel, tol)
        if per_row and np.ndim(b) >= 1 and np.shape(b)[0] > 0:
            worst, i, err, nb = per_row_worst(a, b)
            extra = (" [" + describe(i) + "]") if (describe is not None and i >= 0) else ""
            assert worst <= 1.0, "%s grad %s: Gaussian %d is off by %.3e (|ref| %.3e): %.2f x the per-Gaussian bound%s" % (
                label, name, i, err, nb, worst, extra)
            out[name] = (rel, worst, i)
        else:
            out[name] = (rel, 0.0, -1)
    return out


def fmt(res):
    return ", ".join("%s: L2 %.1e worst/bound %.2f (#%d)" % (k, v[0], v[1], v[2]) for k, v in res.items())
