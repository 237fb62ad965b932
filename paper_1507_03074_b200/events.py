"""Seeded synthetic event generator (helix hits on a 12-layer cylindrical detector + noise).

This module serves BOTH the CPU oracle (``oracle/``) and the CUDA path; it holds none of
the Hough method's arithmetic (no circle equation, no binning, no peak rule) -- only the
recipe that produces hit coordinates.  The paper's dataset (100 simulated minimum-bias
events, pT > 500 MeV, <= 5000 hits on a cylindrical 12-layer silicon detector,
PAPER.md:27, section 2) is not available; these events stand in for it with the shapes
``BASELINE.json:configs`` names.  Recipe = DESIGN.md "Input recipe" (G1-G8).

All geometry is evaluated in float64 and rounded once to float32; hits of an event are
randomly permuted so that nothing profits from track-sorted input.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

N_LAYERS = 12                      # PAPER.md:27 "cylindrical 12-layer silicon detector"
R_INNER_MM, R_OUTER_MM = 50.0, 1000.0
B_FIELD_T = 2.0                    # BASELINE.json:configs[0]
Z_HALF_MM = 1500.0                 # |z| bound of noise hits (G4)
SMEAR_MM = 0.02                    # Gaussian smearing of track hits (G5)
ETA_MAX = 2.5
INV_PT_MAX = 2.0                   # 1/pT ~ U(0,2) GeV^-1  => pT > 0.5 GeV


def layer_radii() -> np.ndarray:
    """G1: 12 radii equally spaced from 50 mm to 1000 mm."""
    return R_INNER_MM + np.arange(N_LAYERS, dtype=np.float64) * ((R_OUTER_MM - R_INNER_MM) / (N_LAYERS - 1))


@dataclass(frozen=True)
class Binning:
    """Hough-space binning as handed to ``ht_create`` and to the oracle (ranges in mm / rad)."""
    n_theta: int
    n_phi: int
    n_a: int
    n_b: int
    a_min: float = -4000.0
    a_max: float = 4000.0
    b_min: float = -4000.0
    b_max: float = 4000.0
    theta_min: float = 0.0
    theta_max: float = math.pi
    phi_min: float = 0.0
    phi_max: float = 2.0 * math.pi

    @property
    def planes(self) -> int:
        return self.n_theta * self.n_phi

    @property
    def cells(self) -> int:
        return self.planes * self.n_a * self.n_b


@dataclass(frozen=True)
class Workload:
    """One entry of ``BASELINE.json:configs`` (index = config id - 1)."""
    config: int
    name: str
    binning: Binning
    n_events: int
    threshold: int
    n_tracks: int | None = None          # fixed number of tracks (config 1) ...
    n_hits: int | None = None            # ... or fixed hit total (configs 2, 4, 5)
    n_hits_range: tuple[int, int] | None = None   # ... or hit total ~ U{lo..hi} per event (config 3)
    noise_frac: float = 0.10


_PAPER_BINS = Binning(4, 16, 1024, 1024)       # PAPER.md:27 "4 x 16 x 1024 x 1024" (reading R1)

WORKLOADS: dict[int, Workload] = {
    1: Workload(1, "tiny", Binning(4, 16, 128, 128), n_events=1, threshold=8, n_tracks=20),
    2: Workload(2, "paper_single", _PAPER_BINS, n_events=1, threshold=8, n_hits=5000),
    3: Workload(3, "paper_batch100", _PAPER_BINS, n_events=100, threshold=8, n_hits_range=(3000, 5000)),
    4: Workload(4, "high_occupancy", _PAPER_BINS, n_events=1, threshold=10, n_hits=20000, noise_frac=0.20),
    5: Workload(5, "fine_binning_x10", Binning(8, 32, 2048, 2048), n_events=10, threshold=8, n_hits=5000),
}


@dataclass
class EventBatch:
    """SoA hit arrays of a batch of events (float32, mm) + per-event offsets (int32, n_events+1)."""
    x: np.ndarray
    y: np.ndarray
    z: np.ndarray
    event_offsets: np.ndarray
    truth: list = field(default_factory=list)     # per event: dict(q, pt, phi0, eta, radius, n_track_hits)

    @property
    def n_events(self) -> int:
        return int(self.event_offsets.shape[0] - 1)

    @property
    def n_hits(self) -> int:
        return int(self.x.shape[0])

    def event(self, e: int) -> tuple[np.ndarray, np.ndarray, np.ndarray]:
        lo, hi = int(self.event_offsets[e]), int(self.event_offsets[e + 1])
        return self.x[lo:hi], self.y[lo:hi], self.z[lo:hi]


def event_seed(config: int, event: int, seed_offset: int = 0) -> int:
    """G8: one documented scheme."""
    return 1000 * config + event + 1_000_000 * seed_offset


def _track_hits(rng: np.random.Generator, n_tracks: int):
    """G2, G3: helix from the origin (d0 = z0 = 0) crossing every layer once."""
    q = np.where(rng.random(n_tracks) < 0.5, 1.0, -1.0)
    inv_pt = rng.uniform(1e-6, INV_PT_MAX, n_tracks)          # GeV^-1; (0,2) with the < 1e-6 tail redrawn
    pt = 1.0 / inv_pt
    phi0 = rng.uniform(0.0, 2.0 * math.pi, n_tracks)
    eta = rng.uniform(-ETA_MAX, ETA_MAX, n_tracks)
    radius = 1000.0 * pt / (0.3 * B_FIELD_T)                  # mm; >= 833 mm so r <= 2R on all layers
    r = layer_radii()[None, :]
    psi = 2.0 * np.arcsin(r / (2.0 * radius[:, None]))
    phi_hit = phi0[:, None] - q[:, None] * psi / 2.0
    hx = r * np.cos(phi_hit)
    hy = r * np.sin(phi_hit)
    hz = radius[:, None] * psi * np.sinh(eta)[:, None]
    hits = np.stack([hx, hy, hz], axis=-1).reshape(-1, 3)     # track-major, layer-minor
    truth = dict(q=q, pt=pt, phi0=phi0, eta=eta, radius=radius)
    return hits, truth


def _noise_hits(rng: np.random.Generator, n_noise: int) -> np.ndarray:
    """G6: uniform on the layers, |z| < 1500 mm."""
    lay = rng.integers(0, N_LAYERS, n_noise)
    ph = rng.uniform(0.0, 2.0 * math.pi, n_noise)
    zz = rng.uniform(-Z_HALF_MM, Z_HALF_MM, n_noise)
    rr = layer_radii()[lay]
    return np.stack([rr * np.cos(ph), rr * np.sin(ph), zz], axis=-1)


def generate_event(seed: int, *, n_tracks: int | None = None, n_hits: int | None = None,
                   noise_frac: float = 0.10, shuffle: bool = True):
    """One event.  Either ``n_tracks`` (noise = round(noise_frac * track hits)) or a hit total
    ``n_hits`` (noise = round(n*f/(1+f)); tracks generated until the rest is filled, last track
    truncated) must be given.  Returns (xyz float32 [n,3], truth dict)."""
    if (n_tracks is None) == (n_hits is None):
        raise ValueError("give exactly one of n_tracks / n_hits")
    rng = np.random.default_rng(seed)
    if n_tracks is not None:
        n_sig = n_tracks * N_LAYERS
        n_noise = int(round(noise_frac * n_sig))
    else:
        n_noise = int(round(n_hits * noise_frac / (1.0 + noise_frac)))
        n_sig = n_hits - n_noise
        n_tracks = -(-n_sig // N_LAYERS)
    sig, truth = _track_hits(rng, n_tracks)
    sig = sig[:n_sig]
    sig = sig + rng.normal(0.0, SMEAR_MM, sig.shape)           # G5
    noise = _noise_hits(rng, n_noise)
    xyz = np.concatenate([sig, noise], axis=0)
    if shuffle:
        xyz = xyz[rng.permutation(xyz.shape[0])]               # G7
    truth["n_track_hits"] = n_sig
    truth["n_noise"] = n_noise
    return xyz.astype(np.float32), truth


def generate_batch(workload: Workload | int, *, n_events: int | None = None, seed_offset: int = 0,
                   first_event: int = 0) -> EventBatch:
    """All events of a workload (or its first ``n_events``), concatenated SoA + offsets."""
    wl = WORKLOADS[workload] if isinstance(workload, int) else workload
    ne = wl.n_events if n_events is None else n_events
    xs, truths, offs = [], [], [0]
    for e in range(first_event, first_event + ne):
        seed = event_seed(wl.config, e, seed_offset)
        if wl.n_tracks is not None:
            xyz, tr = generate_event(seed, n_tracks=wl.n_tracks, noise_frac=wl.noise_frac)
        else:
            if wl.n_hits_range is not None:
                lo, hi = wl.n_hits_range
                # the hit total comes from a stream of its own so that it does not shift the event's draws
                n = int(np.random.default_rng(seed + 500_000_000).integers(lo, hi + 1))
            else:
                n = wl.n_hits
            xyz, tr = generate_event(seed, n_hits=n, noise_frac=wl.noise_frac)
        xs.append(xyz)
        truths.append(tr)
        offs.append(offs[-1] + xyz.shape[0])
    allx = np.concatenate(xs, axis=0) if xs else np.zeros((0, 3), np.float32)
    return EventBatch(x=np.ascontiguousarray(allx[:, 0]), y=np.ascontiguousarray(allx[:, 1]),
                      z=np.ascontiguousarray(allx[:, 2]),
                      event_offsets=np.asarray(offs, dtype=np.int32), truth=truths)


def truth_table(batch: EventBatch, n_theta: int | None = None, n_phi: int | None = None) -> dict:
    """Generator truth of a batch as flat arrays, one entry per generated track (geometry of the generator only, G2/G3):
    ``event``; centre ``a, b`` of the track's circle through the origin, ``R * (q sin phi0, -q cos phi0)`` (mm, float64);
    its radius ``rho`` and the azimuth ``phi`` of the centre in (-pi, pi]; ``n_hits`` of the track that are in the event
    (12, fewer for the truncated last track of a fixed-total event); and, if a segmentation is given, ``max_sector_hits``:
    the largest number of the track's (unsmeared) hits inside ONE of the n_theta x n_phi equal sectors in polar angle
    and azimuth -- a soft track curls across azimuthal sectors, so not all of its 12 hits share one."""
    ev, a, b, rho, nh, msh = [], [], [], [], [], []
    r = layer_radii()[None, :]
    for e, tr in enumerate(batch.truth):
        q, radius, phi0, eta = tr["q"], tr["radius"], tr["phi0"], tr["eta"]
        n_tr = q.shape[0]
        kept = np.clip(tr["n_track_hits"] - N_LAYERS * np.arange(n_tr), 0, N_LAYERS)     # hits are track-major, layer-minor
        ev.append(np.full(n_tr, e, np.uint32))
        a.append(radius * q * np.sin(phi0))
        b.append(-radius * q * np.cos(phi0))
        rho.append(radius)
        nh.append(kept)
        if n_theta and n_phi:
            psi = 2.0 * np.arcsin(r / (2.0 * radius[:, None]))
            phi_hit = np.mod(phi0[:, None] - q[:, None] * psi / 2.0, 2.0 * math.pi)
            theta_hit = np.arctan2(r, radius[:, None] * psi * np.sinh(eta)[:, None])        # polar angle from the +z axis, (0, pi)
            sec = (np.minimum((theta_hit / (math.pi / n_theta)).astype(np.int64), n_theta - 1) * n_phi
                   + np.minimum((phi_hit / (2.0 * math.pi / n_phi)).astype(np.int64), n_phi - 1))
            have = np.arange(N_LAYERS)[None, :] < kept[:, None]
            m = np.zeros(n_tr, np.int64)
            for k in range(n_tr):
                if kept[k]:
                    m[k] = np.bincount(sec[k][have[k]]).max()
            msh.append(m)
    cat = lambda parts, dt: np.concatenate(parts).astype(dt) if parts else np.zeros(0, dt)
    out = dict(event=cat(ev, np.uint32), a=cat(a, np.float64), b=cat(b, np.float64), rho=cat(rho, np.float64),
               n_hits=cat(nh, np.int64))
    out["phi"] = np.arctan2(out["b"], out["a"])
    if n_theta and n_phi:
        out["max_sector_hits"] = cat(msh, np.int64)
    return out


def batch_from_arrays(events: list[np.ndarray]) -> EventBatch:
    """Pack hand-built events ([n_i,3] arrays) into an EventBatch (used by tests for edge cases)."""
    offs = [0]
    for ev in events:
        offs.append(offs[-1] + int(np.asarray(ev).reshape(-1, 3).shape[0]))
    allx = (np.concatenate([np.asarray(ev, dtype=np.float32).reshape(-1, 3) for ev in events], axis=0)
            if events else np.zeros((0, 3), np.float32))
    return EventBatch(x=np.ascontiguousarray(allx[:, 0]), y=np.ascontiguousarray(allx[:, 1]),
                      z=np.ascontiguousarray(allx[:, 2]), event_offsets=np.asarray(offs, dtype=np.int32))
