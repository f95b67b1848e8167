"""Tolerance rules of the GPU-vs-oracle parity tests (BASELINE.json north_star; readings in DESIGN.md "Tolerances").

Integer outputs (keys, sort order, counts, positions that decide them) are compared bit for bit elsewhere.  Here:
  * moments:   |d| <= 1e-6 * max(|ref|, <|c|^k>) for a k-th order central moment (k = 2 P, 3 t/h, 4 F, 5 g), with
               <|c|^k> the cell's own absolute moment (``abs_moments``); without particle data the smaller
               (3 theta)^(k/2) <= <|c|^k> is used instead (stricter);
               |dU_i| <= 1e-6 * max(|U_i|, sqrt(theta));  N exact.
  * coefficients (exact closure and fp32 MLP): per cell, ||d||_inf <= tol * max(||ref||_inf, floor) separately on
               the C block (6, floor 1/tau) and the Gamma block (3, floor 1e-3/(tau sqrt(theta))).
  * velocities: |dv_i| <= tol * max(|v_i|, sqrt(theta_cell)).
Every function returns the worst ratio err/allowed (<= 1 passes) so that tests can print the margin.
"""
import numpy as np

ORDER_FULL = np.array([0, 0, 0, 0] + [2] * 6 + [3] * 10 + [4] * 6 + [5] * 3)
ORDER_LITE = np.array([0, 0, 0, 0] + [2] * 6 + [3] * 3)


def abs_moments(vx, vy, vz, cell_start, ref):
    """<|c|^k> per cell for k = 0..5 (columns), from the particles and the reference mean velocity."""
    n = np.diff(cell_start)
    ncell = n.shape[0]
    seg = np.repeat(np.arange(ncell), n)
    c2 = np.zeros(seg.shape[0])
    for i, v in enumerate((vx, vy, vz)):
        c2 += (np.asarray(v, dtype=np.float64) - ref[seg, 1 + i]) ** 2
    cabs = np.sqrt(c2)
    out = np.zeros((ncell, 6))
    for k in range(2, 6):
        out[:, k] = np.bincount(seg, weights=cabs ** k, minlength=ncell) / np.maximum(n, 1)
    return out


def moment_ratio(got, ref, tol=1e-6, absmom=None, mask=None):
    got, ref = np.asarray(got, dtype=np.float64), np.asarray(ref, dtype=np.float64)
    assert got.shape == ref.shape
    assert np.array_equal(got[:, 0], ref[:, 0]), "per-cell counts differ"
    assert np.isfinite(got).all()
    if mask is not None:
        got, ref = got[mask], ref[mask]
        absmom = absmom[mask] if absmom is not None else None
        if got.shape[0] == 0:
            return 0.0
    theta = (ref[:, 4] + ref[:, 7] + ref[:, 9]) / 3.0
    order = ORDER_FULL if ref.shape[1] == 29 else ORDER_LITE
    s = np.sqrt(np.maximum(3.0 * theta, 0.0))
    worst = 0.0
    # U
    allowed = tol * np.maximum(np.abs(ref[:, 1:4]), np.sqrt(np.maximum(theta, 0.0))[:, None])
    err = np.abs(got[:, 1:4] - ref[:, 1:4])
    nz = ref[:, 0] > 0
    if nz.any():
        with np.errstate(divide="ignore", invalid="ignore"):
            r = np.where(allowed[nz] > 0, err[nz] / allowed[nz], np.where(err[nz] > 0, np.inf, 0.0))
        worst = max(worst, float(r.max()))
    for k in range(4, ref.shape[1]):
        scale = s ** order[k] if absmom is None else absmom[:, order[k]]
        allowed = tol * np.maximum(np.abs(ref[:, k]), scale)
        err = np.abs(got[:, k] - ref[:, k])
        with np.errstate(divide="ignore", invalid="ignore"):
            r = np.where(allowed > 0, err / allowed, np.where(err > 0, np.inf, 0.0))
        worst = max(worst, float(r.max()))
    return worst


def coef_ratio(got, ref, tau, theta, tol=1e-5, mask=None):
    """got, ref [ncell, 9]; tau scalar or [ncell]; theta [ncell].  mask: cells to check."""
    got, ref = np.asarray(got, dtype=np.float64), np.asarray(ref, dtype=np.float64)
    tau = np.broadcast_to(np.asarray(tau, dtype=np.float64), theta.shape)
    if mask is None:
        mask = np.ones(ref.shape[0], dtype=bool)
    if not mask.any():
        return 0.0
    d = np.abs(got - ref)
    fc = 1.0 / tau
    with np.errstate(divide="ignore", invalid="ignore"):
        fg = np.where(theta > 0, 1e-3 / (tau * np.sqrt(np.maximum(theta, 1e-300))), 1.0)
    rc = d[:, :6].max(axis=1) / (tol * np.maximum(np.abs(ref[:, :6]).max(axis=1), fc))
    rg = d[:, 6:].max(axis=1) / (tol * np.maximum(np.abs(ref[:, 6:]).max(axis=1), fg))
    return float(max(rc[mask].max(), rg[mask].max()))


def velocity_ratio(got, ref, cell_start, theta, tol=1e-6):
    """got, ref: tuples (vx, vy, vz) of the cell-sorted arrays; theta [ncell] of the pre-update cell."""
    n = np.diff(cell_start)
    th = np.repeat(np.sqrt(np.maximum(theta, 0.0)), n)
    worst = 0.0
    for g, r in zip(got, ref):
        g, r = np.asarray(g, dtype=np.float64), np.asarray(r, dtype=np.float64)
        assert np.isfinite(g).all()
        allowed = tol * np.maximum(np.abs(r), th)
        err = np.abs(g - r)
        with np.errstate(divide="ignore", invalid="ignore"):
            ratio = np.where(allowed > 0, err / allowed, np.where(err > 0, np.inf, 0.0))
        if ratio.size:
            worst = max(worst, float(ratio.max()))
    return worst
