"""The C-ABI library loads and exports every symbol include/trafficsim.h declares (no GPU)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "trafficsim.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(ts_[a-z_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    from paper_1807_01148_b200 import binding, build
    build.build()
    lib = ctypes.CDLL(binding.LIB_PATH)
    names = _declared()
    assert len(names) >= 11
    for n in names:
        assert hasattr(lib, n), n
    assert set(names) == set(binding.EXPORTS)
    assert b"sm_100a" in binding.load().ts_version()


def test_query_workspace_and_validation_without_gpu(cfg1):
    """Host-side arithmetic only: sizes and argument checks work with no device present."""
    from paper_1807_01148_b200 import binding
    n = binding.query_workspace(cfg1)
    atlas = int((cfg1["edge_lanes"].astype(int) * ((cfg1["edge_len_m"] + 15) // 16 * 16)).sum())
    assert n > atlas + 4 * len(cfg1["route_edges"]) and n < 4 << 20
    bad = dict(cfg1); bad["edge_len_m"] = cfg1["edge_len_m"].copy(); bad["edge_len_m"][0] = 70000
    with pytest.raises(binding.TsError) as ei:
        binding.query_workspace(bad)
    assert ei.value.code == binding.TS_EINVAL and "length" in str(ei.value)


def test_emission_totals_are_paid_for_only_when_asked(cfg1):
    """ts_params.emissions adds 8 bytes per vehicle and 16 per slot to the
    workspace; without it the layout is the one it was."""
    from paper_1807_01148_b200 import binding
    plain = binding.query_workspace(cfg1)
    with_totals = binding.query_workspace(dict(cfg1, params=dict(cfg1["params"], emissions=1)))
    V, E = cfg1["n_vehicles"], cfg1["n_edges"]
    slots = V + E + 1024                       # upper bound of the slot capacity (vehicles + queues + slack)
    assert plain + 8 * V + 16 * V <= with_totals <= plain + 8 * V + 16 * slots + 512


def test_code_plane_granule_follows_the_vehicle_lengths(cfg1, monkeypatch):
    """the atlas keeps one speed-code byte per 4 cells where every vehicle is at least 4 m long
    and insert_clear_cells >= 4, one per cell otherwise (and when TS_CODE_GRANULE=0 asks for it).  Seen from outside
    as the size of the workspace: config 1 has 96 lane rows of 2 chunks of 128 cells."""
    from paper_1807_01148_b200 import binding
    chunks = int((cfg1["edge_lanes"] * ((cfg1["edge_len_m"] + 127) // 128)).sum())
    gran = binding.query_workspace(cfg1)
    short = binding.query_workspace(dict(cfg1, params=dict(cfg1["params"], veh_len=3.5)))
    tight = binding.query_workspace(dict(cfg1, params=dict(cfg1["params"], insert_clear_cells=3)))
    monkeypatch.setenv("TS_CODE_GRANULE", "0")
    forced = binding.query_workspace(cfg1)
    assert short == tight == forced
    saved = chunks * 128 - chunks * 32
    assert 0 <= (short - gran) - saved < 512          # each plane is rounded up to 256 bytes


def test_no_cpu_fallback(cfg1):
    """Without a CUDA device ts_create must fail loudly, not fall back."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_1807_01148_b200 import binding
    net, routes, dep, prm, keep = binding.marshal(cfg1)
    dev = binding.TsDevice(256, 1 << 30, None, 0)
    h = ctypes.c_void_p()
    rc = binding.load().ts_create(ctypes.byref(net), ctypes.byref(routes), ctypes.byref(dep),
                                  ctypes.byref(prm), ctypes.byref(dev), ctypes.byref(h))
    assert rc == binding.TS_ECUDA and not h.value


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_1807_01148_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle|#include.*oracle|ts_oracle|\borc_", text, re.M), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert "trafficsim.h\"" not in text and "import paper_1807" not in text and "from paper_1807" not in text, f
