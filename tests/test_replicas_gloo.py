"""world_size-2 test of the N > 1 host logic on CPU (gloo): replicas only, no data-path collective
(DESIGN.md section 9).  The replicas module must not need the CUDA library."""
import importlib.util
import os
import socket
import sys

import pytest
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _load_replicas():
    # by path: importing the package itself would build/load libfpm.so, which this test does not need
    spec = importlib.util.spec_from_file_location(
        "fpm_replicas", os.path.join(ROOT, "paper_2010_11847_b200", "replicas.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    return mod


def _worker(rank, world, port, out_dir):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    sys.path.insert(0, ROOT)
    rep = _load_replicas()
    import fpm_inputs as fi
    r, lr, w = rep.init("gloo")
    assert (r, lr, w) == (rank, rank, world)
    seed = rep.replica_seed(fi.CONFIGS["C1"].seed, r)
    field = fi.linear_field(8, 25.0, seed)
    rep.barrier()
    ms_local = 5.0 + 2.0 * rank                      # rank 1 is the slow replica
    ms_max = rep.max_over_ranks(ms_local)
    rate = rep.whole_job_rate(10, ms_max, w)         # 10 steps per rank
    rep.barrier()
    with open(os.path.join(out_dir, f"rank{rank}.txt"), "w") as f:
        f.write(f"{seed} {ms_max} {rate} {float(field.sum()):.10e}\n")
    rep.finalize()


def test_two_replicas_over_gloo(tmp_path):
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    rows = [open(tmp_path / f"rank{r}.txt").read().split() for r in range(2)]
    assert [int(rows[0][0]), int(rows[1][0])] == [1, 2]                  # distinct seeds per replica
    assert rows[0][3] != rows[1][3]                                     # hence distinct fields
    for r in rows:
        assert float(r[1]) == 7.0                                       # max over ranks, on every rank
        assert float(r[2]) == pytest.approx(2 * 10 * 1e3 / 7.0)        # whole-job rate


def test_single_process_needs_no_process_group():
    rep = _load_replicas()
    for k in ("RANK", "LOCAL_RANK", "WORLD_SIZE"):
        os.environ.pop(k, None)
    assert rep.env_world() == (0, 0, 1)
    assert rep.max_over_ranks(3.5) == 3.5
    assert rep.whole_job_rate(4, 2.0, 1) == 2000.0


def test_bench_style_self_launch_of_two_replicas(tmp_path):
    """`bench.py --gpus N` without torchrun must start N ranks itself: needs_spawn + launch_command
    run a two-rank gloo job that reports WORLD_SIZE, the per-rank seeds and the max-over-ranks."""
    import subprocess
    rep = _load_replicas()
    for k in ("RANK", "LOCAL_RANK", "WORLD_SIZE"):
        os.environ.pop(k, None)
    assert rep.needs_spawn(2) and not rep.needs_spawn(1)
    script = tmp_path / "ranks.py"
    script.write_text(
        "import importlib.util, os, sys\n"
        f"spec = importlib.util.spec_from_file_location('r', {os.path.join(ROOT, 'paper_2010_11847_b200', 'replicas.py')!r})\n"
        "rep = importlib.util.module_from_spec(spec); spec.loader.exec_module(rep)\n"
        "assert not rep.needs_spawn(int(sys.argv[1]))\n"
        "rank, local, world = rep.init('gloo')\n"
        "ms = rep.max_over_ranks(1.0 + rank)\n"
        "sys.stdout.write(f'RANK {rank} {world} {rep.replica_seed(1, rank)} {ms}\\n')\n"     # one write: the ranks share a pipe
        "sys.stdout.flush()\n"
        "rep.finalize()\n")
    cmd = rep.launch_command(2, str(script), ["2"])
    assert "--nproc-per-node=2" in cmd and "127.0.0.1" in cmd
    out = subprocess.run(cmd, capture_output=True, text=True, timeout=120)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = sorted(l for l in out.stdout.splitlines() if l.startswith("RANK"))
    assert lines == ["RANK 0 2 1 2.0", "RANK 1 2 2 2.0"]
