"""Reader of tests/golden/peak_cases.txt (format described in the file's header)."""
from __future__ import annotations

import os

import numpy as np

HERE = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def read_peak_cases(path: str | None = None):
    path = path or os.path.join(HERE, "peak_cases.txt")
    cases, cur, plane_rows, plane_idx = [], None, None, None

    def flush_plane():
        nonlocal plane_rows, plane_idx
        if plane_idx is not None:
            arr = np.array(plane_rows, dtype=np.uint32)
            assert arr.shape == (cur["dims"][2], cur["dims"][3]), (cur["name"], arr.shape)
            cur["m"][plane_idx] = arr
        plane_rows, plane_idx = None, None

    with open(path) as f:
        for raw in f:
            line = raw.strip()
            if not line or line.startswith("#"):
                continue
            tok = line.split()
            if tok[0] == "case":
                cur = {"name": tok[1]}
            elif tok[0] == "dims":
                cur["dims"] = tuple(int(t) for t in tok[1:5])
                nt, nphi, na, nb = cur["dims"]
                cur["m"] = np.zeros((nt * nphi, na, nb), np.uint32)
            elif tok[0] == "T":
                cur["T"] = int(tok[1])
            elif tok[0] == "plane":
                flush_plane()
                plane_idx, plane_rows = int(tok[1]), []
            elif tok[0] == "peaks":
                flush_plane()
                nt, nphi, na, nb = cur["dims"]
                cells = []
                for t in tok[1:]:
                    p, a, b = (int(v) for v in t.split(":"))
                    cells.append((p * na + a) * nb + b)
                cur["peaks"] = sorted(cells)
            elif tok[0] == "end":
                nt, nphi, na, nb = cur["dims"]
                cur["m"] = cur["m"].reshape(nt, nphi, na, nb)
                cases.append(cur)
                cur = None
            else:
                plane_rows.append([int(t) for t in tok])
    return cases


def read_paper_shapes(path: str | None = None) -> dict:
    path = path or os.path.join(HERE, "paper_shapes.txt")
    out = {}
    with open(path) as f:
        for raw in f:
            line = raw.strip()
            if not line or line.startswith("#"):
                continue
            k, *v = line.split()
            out[k] = [float(t) if "." in t else int(t) for t in v]
    return out


def read_merge_cases(path=None):
    """tests/golden/merge_cases.txt -> list of dict(name, dims, window, peaks PEAK-like tuples, want tuples)."""
    path = path or os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "merge_cases.txt")
    cases, cur = [], None
    for line in open(path):
        line = line.split("#")[0].strip()
        if not line:
            continue
        tok = line.split()
        if tok[0] == "case":
            cur = dict(name=tok[1], dims=None, window=None, peaks=[], want=[])
            cases.append(cur)
        elif tok[0] == "dims":
            cur["dims"] = tuple(int(t) for t in tok[1:5])
        elif tok[0] == "window":
            cur["window"] = int(tok[1])
        elif tok[0] in ("peak", "want"):
            ev, plane, a, b, count = (int(t) for t in tok[1:6])
            _, _, n_a, n_b = cur["dims"]
            cell = (plane * n_a + a) * n_b + b
            if tok[0] == "peak":
                cur["peaks"].append((ev, cell, count))
            else:
                cur["want"].append((ev, cell, count, int(tok[6])))
        else:
            raise ValueError(f"bad line in {path}: {line}")
    return cases
