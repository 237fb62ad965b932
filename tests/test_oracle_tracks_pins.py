"""Pins of oracle_tracks (SPEC.md section 4; "rho = sqrt(A^2+B^2) and phi = tan^-1(B/A)").

P11: geometry the paper fixes -- a noiseless track is a circle through the origin; the peak it makes must
     read out the circle's radius and the azimuth of its centre, within the size of a cell.
P12: what the mathematics fixes -- polar identities, hand-computed special cells, the half-turn symmetry.
None of them re-types the oracle's formula: P11 goes through the generator's truth and the fill, P12 through the inverse
map and exact values.
"""
import math

import numpy as np

from oracle import PEAK_DTYPE, oracle_fill, oracle_peaks, oracle_tracks
from paper_1507_03074_b200.events import Binning, layer_radii


def _circle_hits(radius, q, phi0, z_slope=0.3):
    """12 exact hits of the circle of radius R through the origin that starts along phi0 (G3 without smearing)."""
    r = layer_radii()
    psi = 2.0 * np.arcsin(r / (2.0 * radius))
    ph = phi0 - q * psi / 2.0
    return (r * np.cos(ph)).astype(np.float32), (r * np.sin(ph)).astype(np.float32), (z_slope * r).astype(np.float32)


def test_p11_peak_of_a_noiseless_track_reads_out_its_circle():
    bn = Binning(1, 1, 512, 512)                                   # one (theta, phi) plane: the read-out is about (A, B)
    d = 8000.0 / 512
    for ia, ib, q in [(300, 100, 1.0), (120, 400, -1.0), (256, 350, 1.0), (60, 200, -1.0)]:
        cx, cy = -4000.0 + (ia + 0.5) * d, -4000.0 + (ib + 0.5) * d              # a circle centred on a cell centre
        radius = math.hypot(cx, cy)
        phi0 = math.atan2(q * cx, -q * cy)                         # centre = R (q sin phi0, -q cos phi0)  (G3)
        x, y, z = _circle_hits(radius, q, phi0)
        m, votes = oracle_fill(bn, x, y, z)
        assert m.max() == 12 and m[0, 0, ia, ib] == 12             # P2: all 12 lines cross in that cell
        # the cell all 12 lines cross in (a stiff track can tie with a neighbour, R12 then keeps one of the two:
        # the read-out is tested on the cell itself, and on whatever peak the rule kept next to it)
        pk = np.zeros(1, PEAK_DTYPE)
        pk["cell"], pk["count"] = ia * 512 + ib, 12
        k = 0
        rho, phi = oracle_tracks(bn, pk)
        kept = oracle_peaks(bn, m, 12)
        r_kept, _ = oracle_tracks(bn, kept)
        assert np.min(np.abs(r_kept - radius)) <= 4 * math.hypot(d, d)     # the 12-vote ridge is a few cells long
        assert abs(rho[k] - radius) < 1e-9 * radius                # radius of the circle the hits were generated on
        # azimuth of the centre: perpendicular to the initial direction phi0, on the side the charge bends to
        want = (phi0 - q * math.pi / 2 + math.pi) % (2 * math.pi) - math.pi
        dphi = (phi[k] - want + math.pi) % (2 * math.pi) - math.pi
        assert abs(dphi) < 1e-9


def test_p12_hand_computed_cells():
    bn = Binning(1, 1, 5, 5, a_min=-5.0, a_max=5.0, b_min=-5.0, b_max=5.0)     # centres -4, -2, 0, 2, 4
    cells = {(2, 3): (2.0, math.pi / 2), (0, 2): (4.0, math.pi), (3, 1): (2.0 * math.sqrt(2.0), -math.pi / 4),
             (2, 2): (0.0, 0.0), (4, 4): (4.0 * math.sqrt(2.0), math.pi / 4), (1, 0): (math.sqrt(20.0), math.atan2(-4.0, -2.0))}
    pk = np.zeros(len(cells), PEAK_DTYPE)
    pk["cell"] = [ia * 5 + ib for ia, ib in cells]
    rho, phi = oracle_tracks(bn, pk)
    for k, (want_rho, want_phi) in enumerate(cells.values()):
        assert rho[k] == want_rho or abs(rho[k] - want_rho) < 1e-15 * want_rho
        assert abs(phi[k] - want_phi) < 1e-15


def test_p12_polar_identities_planes_and_half_turn():
    bn = Binning(4, 16, 128, 64, a_min=-4000.0, a_max=4000.0, b_min=-1000.0, b_max=3000.0)
    rng = np.random.default_rng(7)
    ia, ib = rng.integers(0, 128, 500), rng.integers(0, 64, 500)
    plane = rng.integers(0, 64, 500)
    pk = np.zeros(500, PEAK_DTYPE)
    pk["cell"] = (plane * 128 + ia) * 64 + ib
    rho, phi = oracle_tracks(bn, pk)
    a_c = -4000.0 + (ia + 0.5) * (8000.0 / 128)                    # exact in binary32 and binary64 for these ranges
    b_c = -1000.0 + (ib + 0.5) * (4000.0 / 64)
    np.testing.assert_allclose(rho * np.cos(phi), a_c, rtol=0, atol=1e-9)
    np.testing.assert_allclose(rho * np.sin(phi), b_c, rtol=0, atol=1e-9)
    assert np.all((phi > -math.pi) & (phi <= math.pi))
    # the (theta, phi) plane of the cell does not enter
    pk2 = pk.copy()
    pk2["cell"] = (0 * 128 + ia) * 64 + ib
    rho2, phi2 = oracle_tracks(bn, pk2)
    assert np.array_equal(rho, rho2) and np.array_equal(phi, phi2)
    # half turn: (A, B) -> (-A, -B) keeps rho and turns phi by pi (symmetric binning)
    bs = Binning(1, 1, 64, 64)
    p = np.zeros(64 * 64, PEAK_DTYPE)
    p["cell"] = np.arange(64 * 64)
    r1, f1 = oracle_tracks(bs, p)
    r2, f2 = r1.reshape(64, 64)[::-1, ::-1].reshape(-1), f1.reshape(64, 64)[::-1, ::-1].reshape(-1)
    np.testing.assert_allclose(r1, r2, rtol=1e-15)
    d = (f1 - f2 + math.pi) % (2 * math.pi) - math.pi
    np.testing.assert_allclose(np.abs(d), math.pi, atol=1e-12)
