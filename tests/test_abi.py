"""CPU: the C-ABI library loads and exports every symbol include/driftsched.h declares (no compute calls)."""
import ctypes
import os
import re

from paper_2606_02982_b200 import _lib, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_header_symbols_exported():
    build.build()
    hdr = open(os.path.join(ROOT, "include", "driftsched.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = sorted(set(re.findall(r"\b(ds_[a-z_]+)\s*\(", hdr)))
    assert declared == sorted(_lib.EXPORTS)
    L = ctypes.CDLL(_lib.LIB_PATH)
    for name in declared:
        assert hasattr(L, name), name


def test_host_only_entry_points():
    L = _lib.lib()
    assert L.ds_strerror(0) == b"ok" and L.ds_strerror(-3) == b"workspace too small"
    assert L.ds_workspace_bytes(_lib.WS_TAIL_STATS, 4, 2) >= 4 * 2 * 256 * 4
    assert L.ds_workspace_bytes(_lib.WS_SIMULATE, 1000, 10) >= 8000
    assert 16 * 1000 <= L.ds_workspace_bytes(_lib.WS_SIMULATE_TRACES, 1000, 0) <= 16 * 1000 + 256     # one 16-byte record per trace request
    # staging area of ds_latency_stats: 5 bytes per simulated request (+ alignment room); 0 requests -> the 256-byte floor
    assert 5 * 10**6 <= L.ds_workspace_bytes(_lib.WS_LATENCY_STAGE, 10**6, 0) <= 5 * 10**6 + 2048
    assert L.ds_workspace_bytes(_lib.WS_LATENCY_STAGE, 0, 0) == 256
    assert L.ds_workspace_bytes(99, 1, 1) >= 256
    assert L.ds_launch_count() == 0


def test_struct_layouts_match_header():
    assert ctypes.sizeof(_lib.DsTraces) == 64 and ctypes.sizeof(_lib.DsServer) == 80
    from paper_2606_02982_b200 import workload as wl
    assert wl.INSTANCE_DTYPE.itemsize == 24
    hdr = open(os.path.join(ROOT, "include", "driftsched.h")).read()
    assert "#define DS_AGING_UNCLAMPED 5" in hdr and wl.AGING_UNCLAMPED == 5 and wl.POLICY_NAMES[5] == "AGING_UNCLAMPED"
    assert "#define DS_WS_LATENCY_STAGE 3" in hdr and _lib.WS_LATENCY_STAGE == 3
    assert "#define DS_WS_SIMULATE_TRACES 4" in hdr and _lib.WS_SIMULATE_TRACES == 4


def test_no_oracle_in_product_path():
    pkg = os.path.join(ROOT, "paper_2606_02982_b200")
    for dp, _, fs in os.walk(pkg):
        for f in fs:
            if f.endswith((".py", ".cu", ".cuh", ".cpp", ".h")):
                src = open(os.path.join(dp, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "oracle/" not in src.replace("the oracle", ""), f


def test_k2_instruction_capture_belongs_to_the_committed_kernel():
    # bench.py prints roofline.frac only when profiles/r02_k2_counts.json.txt was captured from the simulate.cu in the tree
    # (it compares sha256); a kernel edit without a new ncu capture must show up here, not as a silently withheld number
    import hashlib
    import json
    cap = json.load(open(os.path.join(ROOT, "profiles", "r02_k2_counts.json.txt")))
    src = open(os.path.join(ROOT, "paper_2606_02982_b200", "csrc", "simulate.cu"), "rb").read()
    assert hashlib.sha256(src).hexdigest() == cap["simulate_cu_sha256"], "re-capture profiles/r02_k2_counts.json.txt (see its 'how')"
    for k in ("slots1", "slots4", "slots8"):
        assert cap[k]["inst_per_simreq"] > cap[k]["floor_inst_per_simreq"] > 0
