"""bench.py --gpus N started as one plain process (the way the driver starts it) must become N ranks or fail loudly;
it may never print an N = 1 number under an N > 1 flag ("What's missing" 1).  CPU only: the launcher is
driven with a stub worker in place of bench.py."""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

STUB = """import os, sys
out = sys.argv[1]
with open(os.path.join(out, "rank%s" % os.environ["RANK"]), "w") as f:
    f.write(" ".join([os.environ["WORLD_SIZE"], os.environ["LOCAL_RANK"], os.environ["MASTER_ADDR"],
                      os.environ.get("NCCL_DEBUG", "")] + sys.argv[2:]))
"""


def test_launcher_refuses_more_ranks_than_devices():
    import bench
    with pytest.raises(SystemExit) as e:
        bench.launch_ranks(2, [], device_count=1, run=lambda *a, **k: pytest.fail("nothing may be launched"))
    assert "1 CUDA device" in str(e.value) and "--gpus 2" in str(e.value)


def test_launcher_starts_one_rank_per_device(tmp_path):
    import bench
    stub = tmp_path / "stub.py"
    stub.write_text(STUB)
    env_before = os.environ.pop("NCCL_DEBUG", None)
    try:
        rc = bench.launch_ranks(2, [str(tmp_path), "--gpus", "2", "--steps", "3"], device_count=2, script=str(stub))
    finally:
        if env_before is not None:
            os.environ["NCCL_DEBUG"] = env_before
    assert rc == 0
    for r in (0, 1):
        world, local, addr, nccl_debug, *argv = (tmp_path / ("rank%d" % r)).read_text().split(" ")
        assert (world, local, addr, nccl_debug) == ("2", str(r), "127.0.0.1", "INFO")
        assert argv == ["--gpus", "2", "--steps", "3"]          # the ranks see the caller's own flags


def test_bench_gpus_2_on_a_node_without_two_gpus_exits_nonzero():
    import torch
    if torch.cuda.device_count() >= 2:
        pytest.skip("this node has two GPUs: the launcher would really launch")
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--parallelism", "vocab"],
                       capture_output=True, text=True, timeout=300, env=env)
    assert r.returncode != 0
    assert "CUDA device" in r.stderr and "refusing" in r.stderr
    assert '"n_gpus"' not in r.stdout
