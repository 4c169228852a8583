"""Multi-GPU = independent replicas: one process per GPU, each running its own
simulation (seed + rank, the paper's batch dimension).  No collective touches the data
path; torch.distributed only provides the barrier around the timed region and the max-over-ranks of
the timings.  Works on any backend (nccl on GPUs; gloo in the CPU tests)."""
import os


def env_world():
    """(rank, local_rank, world_size) from the torchrun environment (1 process: 0, 0, 1)."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def needs_spawn(n_gpus):
    """True when N > 1 replicas were asked for but this process was not started by torchrun: the caller must
    start the N ranks itself (launch_command) instead of quietly running one."""
    return int(n_gpus) > 1 and "WORLD_SIZE" not in os.environ


def free_port():
    import socket
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def launch_command(n_gpus, script, argv, port=None, python=None):
    """The torchrun command line that runs `script argv` as n_gpus replica ranks on this node (one process
    per GPU, rendezvous on 127.0.0.1) -- the same launch the bench contract describes for N > 1."""
    import sys
    return [python or sys.executable, "-m", "torch.distributed.run", "--nnodes=1",
            f"--nproc-per-node={int(n_gpus)}", "--master-addr", "127.0.0.1",
            "--master-port", str(port if port is not None else free_port()), script] + list(argv)


def replica_seed(base_seed, rank):
    """Seed of the white-noise field of the replica on `rank`: distinct simulations, same cosmology."""
    return int(base_seed) + int(rank)


def init(backend, device=None):
    """Joins the process group when launched under torchrun with WORLD_SIZE > 1; returns the world."""
    import torch.distributed as dist
    rank, local_rank, world = env_world()
    if world > 1 and not dist.is_initialized():
        kwargs = {"device_id": device} if (device is not None and backend == "nccl") else {}
        dist.init_process_group(backend, **kwargs)
    return rank, local_rank, world


def barrier():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.barrier()


def max_over_ranks(value, device="cpu"):
    """MAX of a host float over all ranks (the timed region of a replica job is its slowest rank)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_rate(units_per_rank, ms_max, world):
    """Units processed by all ranks / the slowest rank's time: replicas scale weakly."""
    return world * units_per_rank * 1e3 / ms_max


def finalize():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.destroy_process_group()
