"""Host-side multi-rank logic of bench.py on CPU (gloo, world_size 2): the path does not shard
("replicas only"), so all there is to cover is the max-over-ranks of the device
times, the replica throughput formula and the rank gating of the reference arm."""
import os
import socket
import subprocess
import sys
import textwrap

from conftest import ROOT


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_max_over_ranks_gloo_world2(tmp_path):
    script = tmp_path / "w.py"
    script.write_text(textwrap.dedent(f"""
        import os, sys
        sys.path.insert(0, {str(ROOT)!r})
        import torch.distributed as dist
        import bench
        dist.init_process_group("gloo")
        r = dist.get_rank()
        ms = bench.max_over_ranks([10.0 + r, 5.0 - r], "cpu")     # rank 0: [10, 5]; rank 1: [11, 4]
        assert ms == [11.0, 5.0], ms
        v = bench.replica_throughput(dist.get_world_size(), ms[0] / 2)   # two steps in 11 ms on each of 2 replicas
        assert abs(v - 2 * 1e3 / 5.5) < 1e-9
        dist.barrier(); dist.destroy_process_group()
        print("rank", r, "ok")
    """))
    port = _free_port()
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE, stderr=subprocess.STDOUT))
    for p in procs:
        out, _ = p.communicate(timeout=120)
        assert p.returncode == 0, out.decode()
        assert b"ok" in out


def test_single_process_is_identity():
    sys.path.insert(0, str(ROOT))
    import bench
    assert bench.max_over_ranks([3.0, 4.5], "cpu") == [3.0, 4.5]
    assert bench.replica_throughput(1, 4.0) == 250.0


def test_reference_arm_runs_on_rank0_only():
    """Under torchrun the other ranks of `--impl reference` exit 0 without work or output."""
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    r = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0"],
                       env=env, capture_output=True, timeout=60)
    assert r.returncode == 0 and r.stdout.strip() == b""


def test_algorithmic_bytes_match_the_design_table():
    sys.path.insert(0, str(ROOT))
    import bench
    k, path = bench.algorithmic_bytes(4088, 4088, 2, 6)
    r = 4088 * 4088 * 8.0
    assert path == 34 * r                                   # 13 + 4 + 7 + 10
    assert k["col_fwd_R"] == 9 * r and k["lagcol_omega"] == 6 * r and k["col_inv"] == 7 * r and k["row_inv"] == 3 * r
