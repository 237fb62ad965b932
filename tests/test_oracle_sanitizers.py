"""The CPU oracle under AddressSanitizer + UndefinedBehaviorSanitizer: the tiny workload of
BASELINE.json:configs[0] plus degenerate hits goes through every oracle function inside a program built with
-fsanitize=address,undefined; any finding aborts the program (non-zero exit), and its digest must equal the digest of
the ordinary build's results."""
import os
import struct
import subprocess

import numpy as np

from oracle import TRUTH_DTYPE, oracle_fill, oracle_match_truth, oracle_merge_ridges, oracle_peaks, oracle_tracks, oracle_votes
from paper_1507_03074_b200.events import WORKLOADS, generate_batch

HERE = os.path.dirname(os.path.abspath(__file__))


def _fnv(data: bytes, h: int) -> int:
    for c in data:
        h = ((h ^ c) * 1099511628211) & 0xFFFFFFFFFFFFFFFF
    return h


def test_oracle_is_clean_under_asan_and_ubsan(tmp_path):
    exe = tmp_path / "oracle_asan"
    subprocess.run(["gcc", "-O1", "-g", "-std=c11", "-ffp-contract=off", "-fno-fast-math", "-fsanitize=address,undefined",
                    "-fno-sanitize-recover=all", "-fno-omit-frame-pointer", "-o", str(exe),
                    os.path.join(HERE, "asan_driver.c"), "-lm"], check=True)
    wl = WORKLOADS[1]
    bn = wl.binning
    x, y, z = generate_batch(wl, n_events=1).event(0)
    bad = np.array([[100.0, 0.0, 5.0], [0.0, 0.0, 1.0], [np.nan, 3.0, 1.0], [3.0, np.inf, 1.0], [1e-30, 1e-30, 1.0],
                    [1e30, 1e30, 1e30], [-50.0, -0.0, 1.0]], np.float32)
    x, y, z = (np.concatenate([v, bad[:, k]]).astype(np.float32) for k, v in enumerate((x, y, z)))
    window = 3
    inp = tmp_path / "event.bin"
    with open(inp, "wb") as f:
        f.write(struct.pack("<4i8f", bn.n_theta, bn.n_phi, bn.n_a, bn.n_b, bn.a_min, bn.a_max, bn.b_min, bn.b_max,
                            bn.theta_min, bn.theta_max, bn.phi_min, bn.phi_max))
        f.write(struct.pack("<IIq", wl.threshold, window, len(x)))
        f.write(x.tobytes() + y.tobytes() + z.tobytes())
    env = dict(os.environ, ASAN_OPTIONS="detect_leaks=1:abort_on_error=0", UBSAN_OPTIONS="halt_on_error=1")
    r = subprocess.run([str(exe), str(inp)], capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode == 0, r.stderr[-3000:]
    assert "runtime error" not in r.stderr and "AddressSanitizer" not in r.stderr, r.stderr[-3000:]
    tok = r.stdout.split()
    got = {tok[i]: int(tok[i + 1]) for i in range(0, len(tok), 2)}
    # the same through the ordinary build
    m, votes = oracle_fill(bn, x, y, z)
    pk = oracle_peaks(bn, m, wl.threshold)
    rho, phi = oracle_tracks(bn, pk)
    mg = oracle_merge_ridges(bn, pk, window)
    plane, bins = oracle_votes(bn, x, y, z)
    assert got["votes"] == votes and got["peaks"] == len(pk) > 0 and got["merged"] == len(mg) > 0
    assert got["matrix_hash"] == _fnv(m.tobytes(), 1469598103934665603)
    assert got["peaks_hash"] == _fnv(pk.tobytes(), 7)
    assert got["tracks_hash"] == _fnv(rho.tobytes(), _fnv(phi.tobytes(), 7))
    assert got["merged_hash"] == _fnv(mg.tobytes(), 7)
    assert got["planes_hash"] == _fnv(plane.tobytes(), _fnv(bins.tobytes(), 7))
    nt = min(len(x), 64)
    tr = np.zeros(nt, TRUTH_DTYPE)
    tr["event"] = np.arange(nt) & 1
    tr["a"], tr["b"] = 3.0 * x[:nt].astype(np.float64), -2.5 * y[:nt].astype(np.float64)
    cm, tm, s = oracle_match_truth(bn, mg, tr, 200.0, 0.95)
    assert got["match_rc"] == 0 and got["found"] == s["n_found"] and got["fake"] == s["n_fake"]
    assert got["match_hash"] == _fnv(cm.tobytes(), _fnv(tm.tobytes(), 7))
