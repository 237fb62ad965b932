"""Double-precision, numpy-only restatements used to PIN the oracle (they are not the oracle and share
nothing with it or with the CUDA path).  Everything here is the textbook form: atan2 for angles, the
circle equation x^2+y^2-2Ax-2By=0 solved for B in float64."""
from __future__ import annotations

import numpy as np


def a_centres(bn) -> np.ndarray:
    """Bin centres of A in float64 (reading R5)."""
    d = (float(bn.a_max) - float(bn.a_min)) / bn.n_a
    return float(bn.a_min) + (np.arange(bn.n_a, dtype=np.float64) + 0.5) * d


def b_edges(bn) -> np.ndarray:
    d = (float(bn.b_max) - float(bn.b_min)) / bn.n_b
    return float(bn.b_min) + np.arange(bn.n_b + 1, dtype=np.float64) * d


def b_star(x, y, a):
    """B of the circle through the origin and (x,y) with centre abscissa a; float64."""
    x = np.asarray(x, np.float64); y = np.asarray(y, np.float64)
    with np.errstate(divide="ignore", invalid="ignore"):
        return (x * x + y * y - 2.0 * a * x) / (2.0 * y)


def b_eps(x, y, a, bn):
    """Bound on |B_fp32 - B*| and on the binning of t: a few binary32 roundings, amplified by 1/(2y)."""
    x = np.asarray(x, np.float64); y = np.asarray(y, np.float64)
    bs = b_star(x, y, a)
    with np.errstate(divide="ignore", invalid="ignore"):
        return 2.0 ** -21 * ((x * x + y * y + np.abs(2.0 * a * x)) / np.abs(2.0 * y) + np.abs(bs) + abs(float(bn.b_min)))


def angles(x, y, z):
    """(theta, phi) of the hit position: polar angle from +z in [0,pi], azimuth in [0,2pi)."""
    x = np.asarray(x, np.float64); y = np.asarray(y, np.float64); z = np.asarray(z, np.float64)
    theta = np.arctan2(np.hypot(x, y), z)
    phi = np.mod(np.arctan2(y, x), 2.0 * np.pi)
    return theta, phi


def plane_atan2(bn, x, y, z):
    """Plane index by uniform angular bins (R2, R4) in float64, and the distance (rad) to the nearest edge."""
    theta, phi = angles(x, y, z)
    tlo, thi = float(bn.theta_min), float(bn.theta_max)
    plo, phi_hi = float(bn.phi_min), float(bn.phi_max)
    ft = (theta - tlo) / ((thi - tlo) / bn.n_theta)
    fp = (phi - plo) / ((phi_hi - plo) / bn.n_phi)
    it = np.floor(ft).astype(np.int64)
    ip = np.floor(fp).astype(np.int64)
    ok = (it >= 0) & (it < bn.n_theta) & (ip >= 0) & (ip < bn.n_phi)
    margin_t = np.abs(ft - np.round(ft)) * ((thi - tlo) / bn.n_theta)
    margin_p = np.abs(fp - np.round(fp)) * ((phi_hi - plo) / bn.n_phi)
    plane = np.where(ok, it * bn.n_phi + ip, -1)
    return plane, np.minimum(margin_t, margin_p)


def brute_fill(bn, x, y, z):
    """Cell-centric enumeration (pin P4): for each plane, row, column and hit -- is the hit in the plane and
    does B*(A_c[a]) fall in [B_b, B_{b+1})?  Returns M (float64 logic, int counts) and the smallest margin
    (in units of the rounding bound) of any decision, so the caller can assert the case is unambiguous."""
    ac = a_centres(bn)
    be = b_edges(bn)
    plane, _ = plane_atan2(bn, x, y, z)
    m = np.zeros((bn.n_theta * bn.n_phi, bn.n_a, bn.n_b), np.int64)
    worst = np.inf
    for p in range(bn.n_theta * bn.n_phi):
        for a in range(bn.n_a):
            for b in range(bn.n_b):
                for h in range(len(x)):
                    if plane[h] != p:
                        continue
                    bs = b_star(x[h], y[h], ac[a])
                    eps = b_eps(x[h], y[h], ac[a], bn)
                    worst = min(worst, abs(bs - be[b]) / eps, abs(bs - be[b + 1]) / eps)
                    if be[b] <= bs < be[b + 1]:
                        m[p, a, b] += 1
    return m.reshape(bn.n_theta, bn.n_phi, bn.n_a, bn.n_b), worst


def brute_peaks(m4, threshold):
    """Peak set by the rule of SPEC.md section 3 written as whole-array comparisons on a padded copy
    (a different formulation from the oracle's per-cell loop).  Returns sorted linear cell indices."""
    m4 = np.asarray(m4).astype(np.int64)
    nt, npi, na, nb = m4.shape
    pad = np.pad(m4, ((0, 0), (0, 0), (1, 1), (1, 1)), constant_values=-1)
    c = pad[:, :, 1:-1, 1:-1]
    ok = c >= threshold
    for da in (-1, 0, 1):
        for db in (-1, 0, 1):
            if da == 0 and db == 0:
                continue
            nbr = pad[:, :, 1 + da:1 + da + na, 1 + db:1 + db + nb]
            earlier = da < 0 or (da == 0 and db < 0)
            ok &= (c > nbr) if earlier else (c >= nbr)
    return np.flatnonzero(ok.reshape(-1))
