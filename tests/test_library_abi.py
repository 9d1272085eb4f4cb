"""-m "not gpu": the C-ABI library builds, loads and exports every symbol include/pa_b200.h declares; the binding
agrees with the header; the product path fails loudly without a GPU (no CPU fallback)."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "pa_b200.h")


def declared_functions():
    text = open(HEADER).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(pa_[a-z_A-Z0-9]+)\s*\(", text)))


def test_header_declares_the_north_star_entry_points():
    names = declared_functions()
    for must in ["pa_init", "pa_step", "pa_energies", "pa_log_Z", "pa_observables"]:
        assert must in names


def test_library_builds_loads_and_exports_every_declared_symbol():
    from paper_2006_00561_b200 import build, binding
    path = build.build()
    assert os.path.exists(path)
    lib = C.CDLL(path)
    for name in declared_functions():
        assert hasattr(lib, name), name
    assert sorted(binding.EXPORTS) == declared_functions()
    binding.load_library()


def test_struct_layouts_match_the_header():
    from paper_2006_00561_b200 import binding
    assert C.sizeof(binding.PaConfig) == 4 + 4 + 8 + 8 + 8 + 8 + 8 + 8 + 8 + 4 + 4 + 4 + 4
    assert C.sizeof(binding.PaObs) == 8 + 8 + 4 * 16 + 5 * 8
    assert binding.PaConfig.workspace.offset == 40 and binding.PaConfig.flags.offset == 64 and binding.PaConfig.maxexc.offset == 76


def test_workspace_query_and_invalid_configs_without_gpu():
    from paper_2006_00561_b200 import binding
    lib = binding.load_library()
    cfg = binding.PaConfig(L=64, P=148, R0=1 << 21, capacity=0, seed=3, beta0=0.0, workspace=None, workspace_bytes=0,
                           stream=None, flags=0, policy=0, block=0, maxexc=0)
    nbytes = lib.pa_workspace_bytes(C.byref(cfg))
    cap = (1 << 21) + 16 * 1449  # 16*ceil(sqrt(2^21))
    cap = (cap + 1023) // 1024 * 1024
    assert 2 * cap * 512 < nbytes < 2 * cap * 512 * 1.2  # two population buffers dominate
    for bad in [dict(L=12), dict(L=64, P=0), dict(L=64, R0=0), dict(L=64, R0=1 << 31)]:
        kw = dict(L=64, P=1, R0=1024)
        kw.update(bad)
        c2 = binding.PaConfig(capacity=0, seed=0, beta0=0.0, workspace=None, workspace_bytes=0, stream=None, flags=0,
                              policy=0, block=0, maxexc=0, **kw)
        assert lib.pa_workspace_bytes(C.byref(c2)) == 0


def test_product_path_fails_loudly_without_cuda():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_2006_00561_b200 import binding
    with pytest.raises(RuntimeError):
        binding.PopulationAnnealer(8, 64)
    # the C entry point itself refuses as well (no device -> PA_ECUDA, never a CPU computation)
    lib = binding.load_library()
    cfg = binding.PaConfig(L=8, P=1, R0=64, capacity=0, seed=0, beta0=0.0, workspace=256, workspace_bytes=1 << 30,
                           stream=None, flags=0, policy=0, block=0, maxexc=0)
    ctx = C.c_void_p()
    assert lib.pa_init(C.byref(cfg), C.byref(ctx)) == binding.PA_ECUDA


def test_product_does_not_reference_the_oracle():
    pkg = os.path.join(ROOT, "paper_2006_00561_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle|pa_oracle|libpa_oracle", text, flags=re.M), (dirpath, f)


def test_bench_reference_arm_prints_the_contract_line():
    """bench.py --impl reference (the oracle as it stands, on the host cores) needs no GPU: one JSON line with the
    driver contract's keys, the same metric / unit as our arm, and the e2e / cpu_baseline objects of the tier framing"""
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    out = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--impl", "reference", "--config", "1",
                          "--steps", "2", "--warmup", "1"], capture_output=True, text=True, timeout=300, check=True).stdout
    line = json.loads(out.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["metric"] == "spin_flip_attempts_per_s" and line["unit"] == "attempts/s"
    assert line["higher_is_better"] is True and line["steps"] == 2 and line["value"] > 0 and line["vs_baseline"] is None
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"] == {"value": line["value"], "unit": "attempts/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert line["gpu_launches"] == 0 and line["config"]["workload"].startswith("config1")
