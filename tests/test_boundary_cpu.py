"""No-GPU checks of the boundary: the C-ABI library loads, exports every symbol include/ht.h declares, builds the
same tables as the oracle bit for bit, and validates arguments (no compute call is made)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from oracle import oracle_tables
from paper_1507_03074_b200 import binding as B
from paper_1507_03074_b200.build import build
from paper_1507_03074_b200.events import Binning, WORKLOADS

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module", autouse=True)
def _built():
    build()


def _declared(header):
    text = open(os.path.join(ROOT, "include", header)).read()
    return sorted(set(re.findall(r"HT_API\s+[^;(]*?\b(ht_\w+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    """include/ht.h = the method's calls, include/ht_diag.h = diagnostics; the binding names exactly those."""
    names, diag = _declared("ht.h"), _declared("ht_diag.h")
    assert len(names) >= 9 and set(names) == set(B.EXPORTS)
    assert set(diag) == set(B.DIAG_EXPORTS) and not set(diag) & set(names)
    lib = C.CDLL(B.LIB_PATH)
    for n in names + diag:
        assert getattr(lib, n) is not None


def test_no_environment_variable_is_read_by_the_library():
    """Every switch is a field of ht_tuning (read once by ht_create_ex): no getenv anywhere in the sources."""
    csrc = os.path.join(ROOT, "paper_1507_03074_b200", "csrc")
    for f in os.listdir(csrc):
        assert "getenv" not in open(os.path.join(csrc, f)).read(), f
    assert C.sizeof(B.ht_tuning) == 64


def test_record_layouts_of_the_binding_match_the_header():
    """The numpy / ctypes records the binding marshals have the sizes and field orders include/ht.h declares."""
    text = open(os.path.join(ROOT, "include", "ht.h")).read()

    def fields(struct):
        body = re.search(r"typedef struct %s \{(.*?)\} %s;" % (struct, struct), text, re.S).group(1)
        body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
        names = []
        for decl in body.split(";"):
            decl = decl.strip()
            if decl:
                names += [n.strip().split("[")[0] for n in decl.split(None, 1)[1].split(",")]
        return names

    assert fields("ht_peak") == list(B.PEAK_DTYPE.names) and B.PEAK_DTYPE.itemsize == 12
    assert fields("ht_track") == list(B.TRACK_DTYPE.names) and B.TRACK_DTYPE.itemsize == 20
    assert fields("ht_candidate") == list(B.CAND_DTYPE.names) and B.CAND_DTYPE.itemsize == 24
    assert fields("ht_truth") == list(B.TRUTH_DTYPE.names) and B.TRUTH_DTYPE.itemsize == 24
    assert fields("ht_match_summary") == list(B.SUMMARY_DTYPE.names) and B.SUMMARY_DTYPE.itemsize == 80
    assert fields("ht_tuning") == [n for n, _ in B.ht_tuning._fields_]
    assert fields("ht_config") == [n for n, _ in B.ht_config._fields_]


def test_both_bench_arms_print_the_same_config():
    import importlib.util
    spec = importlib.util.spec_from_file_location("bench_mod", os.path.join(ROOT, "bench.py"))
    bench = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(bench)
    wl = WORKLOADS[2]
    c = bench.workload_config(wl, 5000, 1)
    assert c["workload"] == "config2:paper_single" and c["bins"] == [4, 16, 1024, 1024] and c["hits_per_step"] == 5000
    src = open(os.path.join(ROOT, "bench.py")).read()
    assert src.count("= workload_config(wl,") + src.count(": workload_config(wl,") == 2      # one call per arm, nothing else builds a `config`


def test_no_torch_types_in_the_header():
    text = open(os.path.join(ROOT, "include", "ht.h")).read()
    assert "torch" not in text.replace("torch.cuda.Stream().cuda_stream", "") and "at::" not in text
    assert 'extern "C"' in text


@pytest.mark.parametrize("bn", [WORKLOADS[1].binning, WORKLOADS[2].binning, WORKLOADS[5].binning,
                                Binning(2, 3, 4, 4, theta_min=0.5, theta_max=2.5, phi_min=1.0, phi_max=4.0),
                                Binning(7, 13, 33, 17, a_min=-1234.5, a_max=3210.7, b_min=-99.9, b_max=4567.8),
                                Binning(1, 1, 1, 1)])
def test_tables_bit_identical_to_the_oracle(bn):
    cfg = B.ht_config.from_binning(bn, max_events=1, max_hits=1)
    lib_t = B.ht_tables_host(cfg)
    ora_t = oracle_tables(bn)
    for a, b in zip(lib_t, ora_t):
        np.testing.assert_array_equal(np.atleast_1d(a).view(np.uint32), np.atleast_1d(b).view(np.uint32))


def test_query_sizes_and_argument_validation():
    cfg = B.ht_config.from_binning(WORKLOADS[2].binning, max_events=2, max_hits=5000)
    mh, ws = B.ht_query_sizes(cfg)
    assert mh == 4 * 67_108_864 and 0 < ws < (1 << 24) and ws % 256 == 0     # incl. 64 plane buckets x 5000 records
    cfg_h = B.ht_config.from_binning(WORKLOADS[1].binning, max_events=2, max_hits=100, host_slots=2, host_peak_capacity=100)
    mh1, ws1 = B.ht_query_sizes(cfg_h)
    assert ws1 > 2 * mh1
    bad = [dict(n_a=0), dict(a_min=5.0, a_max=5.0), dict(b_max=float("inf")), dict(theta_max=4.0), dict(phi_min=-0.1),
           dict(n_theta=8, n_phi=32, n_a=4096, n_b=4096)]              # the last one: cells >= 2^32
    for kw in bad:
        c = B.ht_config.from_binning(WORKLOADS[1].binning, max_events=1, max_hits=1)
        for k, v in kw.items():
            setattr(c, k, v)
        with pytest.raises(B.HtError) as ei:
            B.ht_query_sizes(c)
        assert ei.value.status == B.HT_ERR_INVALID_ARG
    c = B.ht_config.from_binning(WORKLOADS[1].binning, max_events=0, max_hits=1)
    with pytest.raises(B.HtError):
        B.ht_query_sizes(c)
    assert B.ht_strerror(B.HT_OK) == "ok" and "invalid" in B.ht_strerror(B.HT_ERR_INVALID_ARG)


def test_product_path_never_touches_the_oracle():
    """The CUDA package must not import, read or run anything under oracle/ (and vice versa)."""
    pkg = os.path.join(ROOT, "paper_1507_03074_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in src.lower() or f == "events.py", f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_1507_03074_b200" not in src.replace("paper_1507_03074_b200/csrc", "") or f == "__init__.py", f
            assert "libht.so" not in src
