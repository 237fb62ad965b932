"""Pins of the oracle's FILL against what the paper and the mathematics fix (no GPU, no CUDA code).

P1 circle equation, P2 noiseless 12-layer track, P3 vote conservation
("incremented by one"), P4 cell-centric brute force in float64 with atan2 binning,
P5 single-hit geometry, P6 mirror symmetry, P7 permutation/batching invariance, P10 table binning vs
atan2, and the closed-form in-range fraction.  Each would fail on a dropped term, a wrong sign, a
transposed index or an off-by-one bin.
"""
import math

import numpy as np
import pytest

import dref
from oracle import oracle_fill, oracle_fill_batch, oracle_tables, oracle_votes
from paper_1507_03074_b200.events import (Binning, WORKLOADS, batch_from_arrays, generate_batch, layer_radii)


def _hits(cfg, **kw):
    b = generate_batch(cfg, **kw)
    return b, WORKLOADS[cfg].binning


# ---------------------------------------------------------------- tables (SPEC.md section 1)
def test_tables_are_exact_for_the_paper_binnings():
    # range 8000 mm over 128 / 1024 / 2048 bins: dA, A_c and 2A_c are exactly representable in binary32
    for n in (128, 1024, 2048):
        bn = Binning(4, 16, n, n)
        two_a, t_theta, p_phi, dA, dB = oracle_tables(bn)
        assert float(dA) == 8000.0 / n and float(dB) == 8000.0 / n
        np.testing.assert_array_equal(two_a.astype(np.float64), 2.0 * dref.a_centres(bn))


def test_angle_tables_closed_form():
    two_a, t_theta, p_phi, _, _ = oracle_tables(Binning(4, 16, 8, 8))
    # cot(0)=+inf, cot(pi/4)=1, cot(pi/2)~0, cot(3pi/4)=-1, cot(pi)=-inf
    assert t_theta[0] == np.inf and t_theta[4] == -np.inf
    assert t_theta[1] == np.float32(1.0) and t_theta[3] == np.float32(-1.0) and abs(t_theta[2]) < 1e-15
    # diamond pseudo-angle at k*22.5 deg: k*pi/8 -> quarter q, 1 - c/(|c|+|s|) within the quarter
    k = np.arange(17)
    ang = k * (2 * np.pi / 16)
    c, s = np.cos(ang), np.sin(ang)
    expect = np.where(s >= 0, 1 - c / (np.abs(c) + np.abs(s)), 3 + c / (np.abs(c) + np.abs(s)))
    expect[0], expect[16] = 0.0, 4.0
    np.testing.assert_allclose(p_phi, expect, rtol=0, atol=3e-7)
    assert p_phi[4] == 1.0 and p_phi[8] == 2.0 and p_phi[12] == 3.0
    assert np.all(np.diff(p_phi) > 0) and np.all(np.diff(t_theta) < 0)


def test_partial_angle_ranges():
    bn = Binning(2, 3, 4, 4, theta_min=0.5, theta_max=2.5, phi_min=1.0, phi_max=4.0)
    _, t_theta, p_phi, _, _ = oracle_tables(bn)
    f = np.float32
    np.testing.assert_allclose(t_theta, [1 / math.tan(float(f(0.5))), 1 / math.tan(1.5), 1 / math.tan(float(f(2.5)))], rtol=2e-7)
    assert np.all(np.diff(p_phi) > 0) and p_phi[0] > 0 and p_phi[-1] < 4


# ---------------------------------------------------------------- P1: circle equation for every vote
@pytest.mark.parametrize("cfg", [1, 2])
def test_P1_every_vote_satisfies_the_circle_equation(cfg):
    batch, bn = _hits(cfg)
    x, y, z = batch.event(0)
    if cfg == 2:                                   # keep the (hit, row) table small: 600 hits x 1024 rows
        x, y, z = x[:600], y[:600], z[:600]
    plane, bins = oracle_votes(bn, x, y, z)
    ac = dref.a_centres(bn)
    be = dref.b_edges(bn)
    X, Y = x.astype(np.float64)[:, None], y.astype(np.float64)[:, None]
    A = ac[None, :]
    bs = dref.b_star(X, Y, A)
    eps = dref.b_eps(X, Y, A, bn)
    r2 = X * X + Y * Y
    # the circle equation itself, with the B the vote stands for
    resid = np.abs(r2 - 2 * A * X - 2 * bs * Y)
    assert np.all(resid <= 1e-6 * np.maximum(r2, 1.0))
    voted = bins >= 0
    assert voted.sum() > 0.6 * voted.size
    # a voted cell must contain B* up to the binary32 rounding bound ...
    lo = be[np.where(voted, bins, 0)]
    hi = be[np.where(voted, bins, 0) + 1]
    assert np.all((bs >= lo - eps)[voted]) and np.all((bs < hi + eps)[voted])
    # ... and a row without a vote must have B* outside the range (up to the same bound)
    inside = (bs >= be[0] + eps) & (bs < be[-1] - eps)
    assert not np.any(inside & ~voted & (plane[:, None] >= 0))
    # exact agreement away from edges: b == floor((B*-Bmin)/dB)
    dB = be[1] - be[0]
    far = voted & (np.abs((bs - be[0]) / dB - np.round((bs - be[0]) / dB)) * dB > eps)
    assert far.sum() > 0.99 * voted.sum()
    np.testing.assert_array_equal(bins[far], np.floor((bs[far] - be[0]) / dB).astype(np.int64))


# ---------------------------------------------------------------- P2: noiseless track => 12
def _ideal_track(bn, ia, ib, eta=0.3, sign=-1.0):
    """12 hits, one per layer, exactly on the circle through the origin whose centre is the centre of
    cell (ia, ib); float64 geometry rounded once to float32.  Built from the circle itself (chord of length
    r subtends the angle acos(r/2R) at the origin with the centre direction), not from events.py."""
    ac = dref.a_centres(bn)
    be = dref.b_edges(bn)
    a0, b0 = ac[ia], 0.5 * (be[ib] + be[ib + 1])
    R = math.hypot(a0, b0)
    phic = math.atan2(b0, a0)
    r = layer_radii()
    alpha = np.arccos(r / (2 * R))
    ph = phic + sign * alpha
    x, y = r * np.cos(ph), r * np.sin(ph)
    psi = 2 * np.arcsin(r / (2 * R))
    z = R * psi * math.sinh(eta)
    assert np.allclose(x * x + y * y - 2 * a0 * x - 2 * b0 * y, 0, atol=1e-6)
    return x.astype(np.float32), y.astype(np.float32), z.astype(np.float32)


@pytest.mark.parametrize("n", [128, 1024, 2048])
def test_P2_noiseless_track_puts_12_in_its_cell(n):
    bn = Binning(4, 16, n, n)
    ia, ib = int(0.70 * n), int(0.80 * n)
    x, y, z = _ideal_track(bn, ia, ib)
    plane, _ = dref.plane_atan2(bn, x, y, z)
    assert len(set(plane.tolist())) == 1 and plane[0] >= 0          # all 12 hits in one (theta,phi) plane
    m, votes = oracle_fill(bn, x, y, z)
    it, ip = divmod(int(plane[0]), bn.n_phi)
    assert m[it, ip, ia, ib] == 12                                   # 12 layers
    assert m.max() == 12
    assert int(m.sum(dtype=np.uint64)) == votes == int(m[it, ip].sum(dtype=np.uint64))
    others = m.copy(); others[it, ip] = 0
    assert others.max() == 0


def test_P2_negative_soft_track_splits_across_phi_sectors():
    # R ~ 930 mm: the 12 hits sweep ~33 deg of azimuth > one 22.5 deg sector => no single cell gets 12 (reading R2)
    bn = Binning(4, 16, 128, 128)
    ac = dref.a_centres(bn)
    ia = int(np.argmin(np.abs(ac - 700.0)))
    ib = int((600.0 + 4000.0) / 62.5)
    x, y, z = _ideal_track(bn, ia, ib)
    plane, _ = dref.plane_atan2(bn, x, y, z)
    assert len(set(plane.tolist())) >= 2
    m, _ = oracle_fill(bn, x, y, z)
    assert m.max() < 12
    assert m.sum(axis=(0, 1))[ia, ib] == 12                          # summed over planes the track is whole again


# ---------------------------------------------------------------- P3: conservation
@pytest.mark.parametrize("cfg", [1, 2])
def test_P3_conservation(cfg):
    batch, bn = _hits(cfg)
    x, y, z = batch.event(0)
    m, votes = oracle_fill(bn, x, y, z)
    total = int(m.sum(dtype=np.uint64))
    assert total == votes <= len(x) * bn.n_a
    # independent count in float64: rows whose B* is in range, for hits that have a plane
    plane, margin = dref.plane_atan2(bn, x, y, z)
    ac = dref.a_centres(bn)
    bs = dref.b_star(x.astype(np.float64)[:, None], y.astype(np.float64)[:, None], ac[None, :])
    eps = dref.b_eps(x.astype(np.float64)[:, None], y.astype(np.float64)[:, None], ac[None, :], bn)
    sure = (bs >= bn.b_min + eps) & (bs < bn.b_max - eps)
    maybe = (bs >= bn.b_min - eps) & (bs < bn.b_max + eps)
    assert sure.sum() <= total <= maybe.sum()
    assert maybe.sum() - sure.sum() < 1e-3 * total + 20
    # per plane: sum of the plane == votes of its hits; every row sum and every cell <= hits in the plane
    hp = np.bincount(plane[plane >= 0], minlength=bn.planes)
    m3 = m.reshape(bn.planes, bn.n_a, bn.n_b)
    row_sums = m3.sum(axis=2)
    assert np.all(row_sums.max(axis=1) <= hp)
    assert np.all(m3.reshape(bn.planes, -1).max(axis=1) <= hp)
    per_plane_sure = np.array([sure[plane == p].sum() for p in range(bn.planes)])
    per_plane_maybe = np.array([maybe[plane == p].sum() for p in range(bn.planes)])
    tot_p = m3.reshape(bn.planes, -1).sum(axis=1)
    assert np.all(per_plane_sure <= tot_p) and np.all(tot_p <= per_plane_maybe)
    # closed form: mean over uniform azimuth of min(1,|tan phi|) = (2/pi)(pi/4 + ln sqrt2) = 0.7206
    assert abs(total / (len(x) * bn.n_a) - 0.7206) < 0.02


def test_in_range_fraction_closed_form():
    # hits close to the origin, uniform in azimuth: B = r/(2 sin phi) - A cot phi ~ -A cot phi, so the fraction of
    # rows in a square (A,B) range is min(1,|tan phi|); its mean is (2/pi)(pi/4 + ln sqrt 2).
    rng = np.random.default_rng(7)
    n = 4000
    ph = rng.uniform(0, 2 * np.pi, n)
    r = 1.0
    x, y, z = (r * np.cos(ph)).astype(np.float32), (r * np.sin(ph)).astype(np.float32), np.full(n, 0.3, np.float32)
    bn = Binning(1, 1, 256, 256)
    m, votes = oracle_fill(bn, x, y, z)
    expect = (2 / np.pi) * (np.pi / 4 + 0.5 * np.log(2.0))
    assert abs(votes / (n * bn.n_a) - expect) < 0.01


# ---------------------------------------------------------------- P4: brute force on tiny binnings
@pytest.mark.parametrize("dims,seed", [((1, 1, 2, 2), 0), ((2, 3, 4, 5), 1), ((3, 2, 8, 6), 2), ((2, 2, 7, 8), 3),
                                       ((3, 3, 5, 3), 4)])
def test_P4_cell_centric_brute_force(dims, seed):
    bn = Binning(*dims, a_min=-900.0, a_max=1100.0, b_min=-1000.0, b_max=800.0)
    rng = np.random.default_rng(100 + seed)
    n = 10
    while True:
        ph = rng.uniform(0, 2 * np.pi, n)
        r = rng.uniform(60.0, 1000.0, n)
        x, y = r * np.cos(ph), r * np.sin(ph)
        z = rng.uniform(-1500, 1500, n)
        x, y, z = x.astype(np.float32), y.astype(np.float32), z.astype(np.float32)
        _, margin = dref.plane_atan2(bn, x, y, z)
        if np.all(np.abs(y) > 50.0) and np.all(margin > 1e-5):
            break
    want, worst = dref.brute_fill(bn, x, y, z)
    assert worst > 1.0, "case not unambiguous: pick another seed"     # every decision farther than the rounding bound
    got, votes = oracle_fill(bn, x, y, z)
    np.testing.assert_array_equal(got.astype(np.int64), want)
    assert votes == want.sum() > 0


# ---------------------------------------------------------------- P5: one hit
def test_P5_single_hit_geometry():
    bn = Binning(4, 16, 128, 128)
    ac = dref.a_centres(bn)
    for (i0, yv, zv) in [(80, 300.0, 100.0), (40, -520.0, -900.0), (100, 77.0, 5.0)]:
        xv = 2.0 * ac[i0]                                   # x/2 is exactly the centre of row i0
        x, y, z = (np.array([v], np.float32) for v in (xv, yv, zv))
        m, votes = oracle_fill(bn, x, y, z)
        plane, bins = oracle_votes(bn, x, y, z)
        p_ref, _ = dref.plane_atan2(bn, x, y, z)
        assert plane[0] == p_ref[0] >= 0
        m3 = m.reshape(bn.planes, bn.n_a, bn.n_b)
        nz_planes = np.flatnonzero(m3.reshape(bn.planes, -1).sum(axis=1))
        assert nz_planes.tolist() == [int(plane[0])]        # exactly one plane is touched
        rows = m3[plane[0]].sum(axis=1)
        assert rows.max() <= 1 and rows.sum() == votes      # at most one vote per A row (R7)
        b = bins[0]
        v = b[b >= 0]
        d = np.diff(v)
        slope_sign = -np.sign(xv / yv)                      # dB/dA = -x/y
        assert np.all(d * slope_sign >= 0)                  # monotone in the direction of the slope
        # perpendicular bisector of origin-hit: at A = x/2 the circle centre has B = y/2
        assert b[i0] == int(math.floor((yv / 2 - bn.b_min) / ((bn.b_max - bn.b_min) / bn.n_b)))


# ---------------------------------------------------------------- P6: mirror
@pytest.mark.parametrize("n", [128, 1024])
def test_P6_mirror_through_the_origin(n):
    bn = Binning(4, 16, n, n)
    batch = generate_batch(1)
    x, y, z = batch.event(0)
    m, v = oracle_fill(bn, x, y, z)
    mm, vm = oracle_fill(bn, -x, -y, z)
    # (x,y)->(-x,-y): phi -> phi+pi (sector + Nphi/2), B(A) -> -B(-A): rows and columns reverse
    want = np.roll(m, bn.n_phi // 2, axis=1)[:, :, ::-1, ::-1]
    diff = int((want != mm).sum())
    # only a B within one binary32 ulp of a bin edge may land differently: (B+4000) and (4000-B) round separately.
    # Expected ~ votes * 2*ulp(4000)/dB ~ 1e-4 * votes differing cells; a sign or index mistake gives ~votes.
    assert diff <= 2e-4 * v + 8 and abs(v - vm) <= 4


# ---------------------------------------------------------------- P7: order and batching
def test_P7_permutation_and_batching_invariance():
    wl = WORKLOADS[1]
    batch = generate_batch(wl, n_events=3)
    ms, votes = oracle_fill_batch(wl.binning, batch)
    assert len(ms) == 3
    rng = np.random.default_rng(5)
    for e in range(3):
        x, y, z = batch.event(e)
        alone, v = oracle_fill(wl.binning, x, y, z)
        np.testing.assert_array_equal(alone, ms[e])
        perm = rng.permutation(len(x))
        shuffled, v2 = oracle_fill(wl.binning, x[perm], y[perm], z[perm])
        np.testing.assert_array_equal(shuffled, alone)
        assert v == v2
    assert not np.array_equal(ms[0], ms[1])


# ---------------------------------------------------------------- P10: table binning == atan2 binning
@pytest.mark.parametrize("dims", [(4, 16), (8, 32), (3, 5), (1, 1)])
def test_P10_table_binning_matches_atan2(dims):
    bn = Binning(dims[0], dims[1], 4, 4)
    batch = generate_batch(4)                               # 20000 generated hits
    x, y, z = batch.x, batch.y, batch.z
    plane, _ = oracle_votes(bn, x, y, z)
    ref, margin = dref.plane_atan2(bn, x, y, z)
    far = margin > 1e-5
    assert far.mean() > 0.99
    np.testing.assert_array_equal(plane[far], ref[far])
    assert np.all(plane >= 0)                               # full angular range: every finite hit has a plane


def test_P10_partial_ranges_drop_hits_outside():
    bn = Binning(2, 4, 4, 4, theta_min=0.6, theta_max=2.2, phi_min=0.5, phi_max=3.5)
    batch = generate_batch(2)
    x, y, z = batch.x, batch.y, batch.z
    plane, _ = oracle_votes(bn, x, y, z)
    ref, margin = dref.plane_atan2(bn, x, y, z)
    theta, phi = dref.angles(x, y, z)
    edge = np.minimum.reduce([np.abs(theta - 0.6), np.abs(theta - 2.2), np.abs(phi - 0.5), np.abs(phi - 3.5)])
    far = (margin > 1e-5) & (edge > 1e-5)
    np.testing.assert_array_equal(plane[far], ref[far])
    assert (plane < 0).sum() > 100 and (plane >= 0).sum() > 100


# ---------------------------------------------------------------- R8: degenerate hits
def test_R8_degenerate_hits_cast_no_votes():
    bn = Binning(4, 16, 16, 16)
    bad = np.array([[100.0, 0.0, 5.0], [0.0, 0.0, 1.0], [np.nan, 3.0, 1.0], [3.0, np.nan, 1.0], [3.0, 4.0, np.nan],
                    [np.inf, 4.0, 1.0], [3.0, -np.inf, 1.0], [-50.0, -0.0, 1.0]], np.float32)
    m, votes = oracle_fill(bn, bad[:, 0], bad[:, 1], bad[:, 2])
    assert votes == 0 and m.max() == 0
    good = np.array([[300.0, 400.0, 10.0]], np.float32)
    both = np.concatenate([bad, good])
    m1, v1 = oracle_fill(bn, good[:, 0], good[:, 1], good[:, 2])
    m2, v2 = oracle_fill(bn, both[:, 0], both[:, 1], both[:, 2])
    np.testing.assert_array_equal(m1, m2)
    assert v1 == v2 > 0
    # an empty event is a zero matrix
    m0, v0 = oracle_fill(bn, np.zeros(0, np.float32), np.zeros(0, np.float32), np.zeros(0, np.float32))
    assert v0 == 0 and m0.max() == 0


def test_hand_built_batch_helper():
    b = batch_from_arrays([np.zeros((2, 3)), np.zeros((0, 3)), np.ones((1, 3))])
    assert b.event_offsets.tolist() == [0, 2, 2, 3] and b.n_events == 3
