"""Host-side checks that need no GPU: the C-ABI library loads and exports every symbol include/krp.h
declares, argument errors come back as codes, the sharding plan covers the id range, the single collective of
the path (sum of the per-rank image maps) works across two processes (gloo), and the seeded input recipe
produces tables the library's own validity rules accept."""
import os
import re
import socket
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_functions():
    text = open(os.path.join(ROOT, "include", "krp.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(krp_[a-z_0-9]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    from paper_2512_01283_b200 import krp
    names = _declared_functions()
    assert len(names) >= 18 and "krp_transport" in names and "krp_image" in names
    L = krp.lib()
    for n in names:
        assert hasattr(L, n), n
    assert sorted(krp.SYMBOLS) == names           # the binding lists exactly what the header declares
    assert b"sm_100a" in L.krp_version()
    # the exported symbols are plain C (no mangling)
    out = subprocess.check_output(["nm", "-D", "--defined-only", krp.library_path()], text=True)
    exported = set(re.findall(r"\bT (krp_[a-z_0-9]+)\b", out))
    assert set(names) <= exported


def test_null_arguments_return_error_codes_without_a_gpu():
    """Calls that must fail before touching the device: they return KRP_ERR_ARG and set the message."""
    import ctypes as C
    from paper_2512_01283_b200 import krp
    L = krp.lib()
    h = C.c_void_p()
    b = (C.c_double * 6)(0, 1, 0, 1, 0, 1)
    assert L.krp_grid_create(C.byref(h), 0, 4, 4, b, None, None, 0, None, None) == krp.ERR_ARG
    assert b"dims" in L.krp_last_error()
    assert L.krp_grid_create(C.byref(h), 4, 4, 4, None, None, None, 0, None, None) == krp.ERR_ARG
    assert L.krp_transport(None, 10, 1, None) == krp.ERR_ARG
    assert L.krp_image(None, None, 0, 4, 4, 0, None) == krp.ERR_ARG
    assert L.krp_tune(None, 0, 0, 0, 0) == krp.ERR_ARG
    assert L.krp_tune_fused(None, 1000) == krp.ERR_ARG
    assert L.krp_tune_schedule(None, -1, -1, -1) == krp.ERR_ARG
    assert L.krp_timing_get(None, None, None) == krp.ERR_ARG
    assert L.krp_launch_count(None) == 0
    assert L.krp_grid_destroy(None) == krp.OK


def test_package_does_not_import_the_oracle():
    """The product path never routes through the oracle (or any CPU fallback)."""
    pkg = os.path.join(ROOT, "paper_2512_01283_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text and "krp_oracle" not in text, f


def test_shard_plans_cover_the_range():
    from paper_2512_01283_b200 import shard
    for world in (1, 2, 3, 8):
        seen = []
        for step in range(4):
            for r in range(world):
                a, c = shard.step_id_range(step, r, world, 1000, id0=7)
                seen.append((a, c))
        ids = np.concatenate([np.arange(a, a + c) for a, c in seen])
        assert np.array_equal(np.sort(ids), np.arange(7, 7 + 4 * world * 1000))
        parts = [shard.split_range(5, 1003, r, world) for r in range(world)]
        assert parts[0][0] == 5 and sum(c for _, c in parts) == 1003
        assert all(parts[i][0] + parts[i][1] == parts[i + 1][0] for i in range(world - 1))
        assert max(c for _, c in parts) - min(c for _, c in parts) <= 1
    with pytest.raises(ValueError):
        shard.step_id_range(0, 2, 2, 10)


_WORKER = r"""
import os, sys
sys.path.insert(0, %r)
import torch, torch.distributed as dist
from paper_2512_01283_b200 import shard
dist.init_process_group("gloo")
r, w = dist.get_rank(), dist.get_world_size()
first, cnt = shard.step_id_range(3, r, w, 50)
img = torch.zeros((2, 4, 3, 3), dtype=torch.float64)
img[:, 0] = float(first)            # stands for this rank's maps
img[:, 1] = float(cnt)
shard.reduce_images(img)
exp0 = sum((3 * w + k) * 50 for k in range(w))
assert torch.all(img[:, 0] == exp0), img[:, 0]
assert torch.all(img[:, 1] == 50 * w)
dist.destroy_process_group()
print("ok", r)
"""


def test_image_reduction_across_two_processes_gloo(tmp_path):
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    script = tmp_path / "worker.py"
    script.write_text(_WORKER % ROOT)
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), WORLD_SIZE="2", LOCAL_RANK=str(r), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True))
    for p in procs:
        out, _ = p.communicate(timeout=180)
        assert p.returncode == 0, out
        assert "ok" in out


def test_input_recipe_is_seeded_and_valid():
    from paper_2512_01283_b200 import inputs
    a = inputs.make("c3", n=8, n_packets=10, npix=8)
    b = inputs.make("c3", n=8, n_packets=10, npix=8)
    assert np.array_equal(a["density"], b["density"]) and np.array_equal(a["mueller"], b["mueller"])
    tau = a["density"] * (1.0 / a["nz"])
    assert tau.min() >= 1e-3 * 0.999 and tau.max() <= 1e3 * 1.001        # reading R16
    for name, kw in (("c1", dict(n=8)), ("c2", dict(n=16)), ("c4", dict(n=8)), ("c5", dict(n=8))):
        cfg = inputs.make(name, n_packets=10, npix=8, **kw)
        F = cfg["mueller"].astype(np.float64)
        assert np.all(F[:, 0] > 0) and np.all(F[:, 0] ** 2 * (1 + 1e-6) >= (F[:, 1:] ** 2).sum(1))
        th = np.linspace(0, np.pi, len(F))
        g = F[:, 0] * np.sin(th)
        assert abs(0.5 * np.sum(0.5 * (g[1:] + g[:-1])) * (th[1] - th[0]) - 1.0) < 1e-4   # (1/2) int S11 sin = 1 (exact Rayleigh: to the trapezoid error)
        op = cfg["opacity"]
        assert np.all(op[:, 0] > np.abs(op[:, 1])) and np.all((op[:, 3] >= 0) & (op[:, 3] <= 1))
        assert np.all(cfg["density"] >= 0) and cfg["density"].shape == (cfg["nz"], cfg["ny"], cfg["nx"])
    c2 = inputs.make("c2", n=32, n_packets=10, npix=8)
    row = c2["density"][16, 16, 16:]
    assert abs(row.sum() * (1.0 / 32) - 20.0) < 1e-3                       # midplane tau = 20 centre -> edge


def test_bench_reference_arm_runs_without_a_gpu():
    """`bench.py --impl reference` times the oracle on host cores and prints one JSON line with the contract's keys;
    under torchrun only rank 0 prints."""
    import json
    cmd = [sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "c1", "--n", "8",
           "--steps", "1", "--warmup", "1"]
    out = subprocess.check_output(cmd, text=True, timeout=600, env=dict(os.environ, RANK="0", WORLD_SIZE="1"))
    line = json.loads(out.strip().splitlines()[-1])
    for key in ("impl", "metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
                "vs_baseline", "dtype", "data", "config", "cpu_baseline", "e2e"):
        assert key in line, key
    assert line["impl"] == "reference" and line["value"] > 0 and line["unit"] == "packets/s"
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] == 1
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["e2e"]["d2h_bytes_per_step"] == 0
    out = subprocess.check_output(cmd, text=True, timeout=600, env=dict(os.environ, RANK="1", WORLD_SIZE="2"))
    assert out.strip() == ""


def test_bench_refuses_to_run_the_product_arm_without_a_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--workload", "c1", "--n", "8", "--steps", "1"],
                       capture_output=True, text=True, timeout=600)
    assert p.returncode != 0 and "no CPU fallback" in (p.stderr + p.stdout)
