"""The seeded generator: shapes of BASELINE.json:configs / PAPER.md:27, determinism, geometry."""
import numpy as np

from golden_io import read_paper_shapes
from paper_1507_03074_b200.events import (WORKLOADS, event_seed, generate_batch, generate_event, layer_radii)


def test_workloads_match_the_shapes_the_paper_prints():
    s = read_paper_shapes()
    bn = WORKLOADS[2].binning
    assert [bn.n_theta, bn.n_phi, bn.n_a, bn.n_b] == s["bins"]          # PAPER.md:27 (reading R1)
    assert WORKLOADS[2].n_hits == s["max_hits_per_event"][0] == WORKLOADS[3].n_hits_range[1]
    assert WORKLOADS[3].n_events == s["events"][0]
    assert len(layer_radii()) == s["layers"][0]
    assert bn.cells == 67_108_864 and WORKLOADS[5].binning.cells == 1_073_741_824


def test_layer_radii_and_hit_radii():
    r = layer_radii()
    assert r[0] == 50.0 and abs(r[-1] - 1000.0) < 1e-9 and np.allclose(np.diff(r), 950.0 / 11)
    xyz, tr = generate_event(3, n_tracks=50, noise_frac=0.0, shuffle=False)
    rr = np.hypot(xyz[:, 0].astype(np.float64), xyz[:, 1].astype(np.float64)).reshape(50, 12)
    assert np.all(np.abs(rr - r[None, :]) < 0.2)                          # on the layers up to the 0.02 mm smearing
    assert np.all(tr["pt"] > 0.5) and np.all(tr["radius"] >= 833.0)       # pT > 500 MeV


def test_track_hits_lie_on_a_circle_through_the_origin():
    xyz, tr = generate_event(5, n_tracks=30, noise_frac=0.0, shuffle=False)
    x = xyz[:, 0].astype(np.float64).reshape(30, 12)
    y = xyz[:, 1].astype(np.float64).reshape(30, 12)
    a = tr["radius"] * tr["q"] * np.sin(tr["phi0"])
    b = -tr["radius"] * tr["q"] * np.cos(tr["phi0"])
    resid = x * x + y * y - 2 * a[:, None] * x - 2 * b[:, None] * y
    assert np.all(np.abs(resid) < 0.3 * tr["radius"][:, None])            # smearing 0.02 mm times 2R plus float32 rounding


def test_hit_totals():
    assert generate_batch(1).n_hits == 264                               # 20 tracks x 12 + round(0.1 x 240)
    b2 = generate_batch(2)
    assert b2.n_hits == 5000 and b2.truth[0]["n_noise"] == 455
    b4 = generate_batch(4)
    assert b4.n_hits == 20000 and b4.truth[0]["n_noise"] == 3333
    b3 = generate_batch(3, n_events=12)
    n = np.diff(b3.event_offsets)
    assert b3.event_offsets[0] == 0 and np.all((n >= 3000) & (n <= 5000)) and len(set(n.tolist())) > 6
    assert b3.x.dtype == np.float32 and b3.event_offsets.dtype == np.int32


def test_determinism_and_seed_scheme():
    a, b = generate_batch(3, n_events=2), generate_batch(3, n_events=2)
    np.testing.assert_array_equal(a.x, b.x); np.testing.assert_array_equal(a.z, b.z)
    c = generate_batch(3, n_events=1, first_event=1)
    lo = int(a.event_offsets[1])
    np.testing.assert_array_equal(a.y[lo:], c.y)
    assert event_seed(2, 0) == 2000 and event_seed(3, 7) == 3007
    d = generate_batch(2, seed_offset=1)
    assert not np.array_equal(d.x, generate_batch(2).x)


def test_noise_hits_within_z_and_events_are_shuffled():
    xyz, tr = generate_event(9, n_hits=2000, noise_frac=1.0, shuffle=False)
    noise = xyz[tr["n_track_hits"]:]
    assert len(noise) == 1000 and np.all(np.abs(noise[:, 2]) <= 1500.0)
    xyz_s, _ = generate_event(9, n_hits=2000, noise_frac=1.0, shuffle=True)
    assert not np.array_equal(xyz, xyz_s)
    np.testing.assert_array_equal(np.sort(xyz[:, 0]), np.sort(xyz_s[:, 0]))
