"""Host-side pieces of bench.py that need no GPU: the committed ncu traffic table is readable, the measured-peak loader
falls back as documented, and the reference arm (the oracle on host cores) prints the contract's JSON line."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _bench():
    sys.path.insert(0, ROOT)
    import importlib
    return importlib.import_module("bench")


def test_traffic_table_and_peaks():
    b = _bench()
    for wl, kern in (("cfg2", "k_demod_stream"), ("cfg3", "k_slide_bulk"), ("cfg4", "k_demod_tc")):
        v = b.load_traffic(wl, kern)
        assert isinstance(v, float) and v > 1e6, (wl, kern, v)
    assert b.load_traffic("cfg2", "no_such_kernel") is None
    peak, src = b.load_peaks()
    assert 3000.0 < peak < 9000.0 and ("measured" in src or "fallback" in src)


def test_reference_arm_prints_the_contract_line():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1", "--warmup", "0",
                          "--ref-rows", "2", "--workload", "cfg1"], capture_output=True, text=True, timeout=600)
    assert out.returncode == 0, out.stderr[-500:]
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["metric"] == "qld_pixel_samples_per_s" and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0 and line["config"]["workload"] == "cfg1"


def test_entry_points_parse_and_build():
    """__graft_entry__ imports cleanly on a CPU box and build() produces both libraries (smoke() itself needs the GPU)."""
    import importlib
    sys.path.insert(0, ROOT)
    g = importlib.import_module("__graft_entry__")
    g.build()
    assert os.path.exists(os.path.join(ROOT, "paper_1511_03390_b200", "libqld.so"))
    import ast
    ast.parse(open(os.path.join(ROOT, "__graft_entry__.py")).read())
    assert callable(g.smoke)
