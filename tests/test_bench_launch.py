"""bench.py's own N-rank launch: `python bench.py --gpus N` outside torchrun starts N ranks by
itself, and refuses -- instead of quietly measuring one GPU -- when the node shows fewer than N devices.  No GPU needed:
device_count and the process start are replaced."""
import importlib
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture()
def bench(monkeypatch):
    monkeypatch.delenv("WORLD_SIZE", raising=False)
    monkeypatch.delenv("RANK", raising=False)
    mod = importlib.import_module("bench")
    return mod


def test_gpus_n_spawns_n_ranks_through_torchrun(bench, monkeypatch):
    calls = []
    monkeypatch.setattr(bench.torch.cuda, "device_count", lambda: 4)
    monkeypatch.setattr(subprocess, "call", lambda cmd: calls.append(cmd) or 0)
    monkeypatch.setattr(sys, "argv", ["bench.py", "--gpus", "4", "--steps", "3", "--warmup", "3"])
    with pytest.raises(SystemExit) as e:
        bench.main()
    assert e.value.code == 0 and len(calls) == 1
    cmd = calls[0]
    assert cmd[:3] == [sys.executable, "-m", "torch.distributed.run"]
    assert cmd[cmd.index("--nproc-per-node") + 1] == "4" and "--nnodes=1" in cmd
    assert cmd[cmd.index("--master-addr") + 1] == "127.0.0.1" and int(cmd[cmd.index("--master-port") + 1]) > 0
    script = cmd.index(os.path.join(ROOT, "bench.py"))
    assert cmd[script + 1:] == ["--gpus", "4", "--steps", "3", "--warmup", "3"]       # the ranks get the same arguments


def test_gpus_n_refuses_when_the_node_has_fewer_devices(bench, monkeypatch):
    monkeypatch.setattr(bench.torch.cuda, "device_count", lambda: 1)
    monkeypatch.setattr(subprocess, "call", lambda cmd: pytest.fail("nothing may be started"))
    monkeypatch.setattr(sys, "argv", ["bench.py", "--gpus", "2", "--steps", "3"])
    with pytest.raises(SystemExit) as e:
        bench.main()
    assert "needs 2 CUDA devices, 1 visible" in str(e.value.code)


def test_launcher_world_size_must_match_gpus(bench, monkeypatch):
    monkeypatch.setenv("WORLD_SIZE", "2")
    monkeypatch.setattr(sys, "argv", ["bench.py", "--gpus", "4"])
    with pytest.raises(SystemExit) as e:
        bench.main()
    assert "started 2 ranks" in str(e.value.code)


def test_under_torchrun_no_second_launch(bench, monkeypatch):
    """WORLD_SIZE present = started by torchrun (the driver's N > 1 form): the rank runs the bench itself."""
    ran = []
    monkeypatch.setenv("WORLD_SIZE", "2")
    monkeypatch.setattr(bench, "run_ours", lambda args: ran.append(args.gpus))
    monkeypatch.setattr(bench, "self_launch", lambda *a: pytest.fail("must not re-launch under torchrun"))
    monkeypatch.setattr(sys, "argv", ["bench.py", "--gpus", "2"])
    bench.main()
    assert ran == [2]
