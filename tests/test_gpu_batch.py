"""batched small simulations ("splitting along the batch dimension is almost
always the most efficient").  A context with batch = B advances B independent simulations in
the same kernel launches, and fpm_nbody replays the whole run as one CUDA graph; member b must match the
oracle's run of member b (the oracle's batch is the loop over single runs, pinned in
tests/test_oracle_lpt_nbody.py) within the north_star tolerances, and equal the batch-1 GPU run."""
import numpy as np
import pytest

import fpm_inputs as fi
from gpu_util import dev, host, rel_l2

pytestmark = pytest.mark.gpu
OM = fi.COSMO["omega_m"]


@pytest.fixture(scope="module")
def fpm():
    import paper_2010_11847_b200 as m
    return m


def _fields(cfg, batch):
    return np.stack([fi.linear_field(cfg.np_side, cfg.box, cfg.seed + b) for b in range(batch)])


@pytest.mark.parametrize("name,batch", [("C1", 8), ("C2", 8)])
def test_batched_run_matches_the_oracle_member_by_member(fpm, oracle, name, batch):
    import torch
    cfg = fi.CONFIGS[name]
    ng, nps, n = cfg.ng, cfg.np_side, cfg.n_particles
    delta = _fields(cfg, batch)
    ctx = fpm.FPM(ng, nps, omega_m=OM, box=cfg.box, force_path=fpm.FORCE_FUSED, batch=batch)
    pos, mom = ctx.lpt_init(dev(delta), cfg.a0, cfg.lpt_order)
    assert tuple(pos.shape) == (batch, 3, n)
    p0, m0 = host(pos).astype(np.float64), host(mom).astype(np.float64)
    # batched paint of the initial state against the oracle, member by member
    rho = host(ctx.paint(pos))
    for b in (0, batch - 1):
        assert rel_l2(rho[b], oracle.paint(p0[b], ng, mass_const=1.0)) < 1e-5
    ctx.nbody(pos, mom, cfg.stages())                      # graph replay (FPM_GRAPH_AUTO at these sizes)
    torch.cuda.synchronize()
    members = range(batch) if name == "C1" else (0, 3, batch - 1)      # the oracle needs ~10 s per C2 run
    sel = list(members)
    rp, rm = oracle.nbody_batch(p0[sel], m0[sel], ng, nps, OM, cfg.stages())
    hp, hm = host(pos), host(mom)
    for j, b in enumerate(sel):
        d = np.abs(hp[b] - rp[j])
        d = np.minimum(d, ng - d)
        assert d.max() < 1e-3, (b, d.max())
        assert rel_l2(hm[b], rm[j]) < 1e-4
    # members are different simulations (seed + b) ...
    assert float(np.abs(hp[0] - hp[1]).max()) > 0.1
    # ... and each equals the batch-1 run of the same inputs, kernel by kernel (no graph), to round-off
    single = fpm.FPM(ng, nps, omega_m=OM, box=cfg.box, force_path=fpm.FORCE_FUSED)
    single.set_graph_mode(fpm.GRAPH_OFF)
    for b in (0, batch - 1):
        sp, sm = dev(p0[b].astype(np.float32)), dev(m0[b].astype(np.float32))
        single.nbody(sp, sm, cfg.stages())
        d = np.abs(host(sp) - hp[b])
        assert np.minimum(d, ng - d).max() < 1e-4


def test_graph_replay_equals_kernel_by_kernel_and_is_cached(fpm):
    import torch
    cfg = fi.CONFIGS["C1"]
    batch = 4
    delta = dev(_fields(cfg, batch))
    ctx = fpm.FPM(cfg.ng, cfg.np_side, omega_m=OM, box=cfg.box, force_path=fpm.FORCE_FUSED, batch=batch)
    pos0, mom0 = ctx.lpt_init(delta, cfg.a0, cfg.lpt_order)
    stages = cfg.stages()
    traj_a = torch.zeros(cfg.n_steps + 1, batch, 3, cfg.n_particles, device="cuda")
    traj_b = torch.zeros_like(traj_a)
    pa, ma = pos0.clone(), mom0.clone()
    ctx.set_graph_mode(fpm.GRAPH_OFF)
    ctx.nbody(pa, ma, stages, traj=traj_a)
    ctx.set_graph_mode(fpm.GRAPH_ALWAYS)
    pb, mb = pos0.clone(), mom0.clone()
    n0 = ctx.launch_count()
    ctx.nbody(pb, mb, stages, traj=traj_b)                 # capture + first replay
    # atomics order differs run to run: equal to fp32 round-off, not bit for bit
    assert float((pa - pb).abs().max()) < 1e-4 and rel_l2(host(ma), host(mb)) < 1e-5
    assert float((traj_a - traj_b).abs().max()) < 1e-4
    assert torch.equal(traj_b[0], pos0)
    n1 = ctx.launch_count()
    pb.copy_(pos0)
    mb.copy_(mom0)
    ctx.nbody(pb, mb, stages, traj=traj_b)                 # same arguments: cached graph, same launch count
    n2 = ctx.launch_count()
    assert n2 - n1 == n1 - n0 > 0                          # the replay reports the kernels the graph holds
    assert float((pa - pb).abs().max()) < 1e-4
    ctx.set_paint_mode(fpm.PAINT_DIRECT)                   # changes the kernel selection: the cache is dropped
    pb.copy_(pos0)
    mb.copy_(mom0)
    ctx.nbody(pb, mb, stages)
    assert float((pa - pb).abs().max()) < 1e-4


def test_calls_without_a_batched_form_say_so(fpm):
    import torch
    ctx = fpm.FPM(32, 32, force_path=fpm.FORCE_FUSED, batch=2)
    pos = torch.zeros(2, 3, 32 ** 3, device="cuda")
    with pytest.raises(fpm.FpmError, match="not available on a batched context"):
        ctx._check(fpm._lib.fpm_force(ctx._h, pos.data_ptr(), 32 ** 3, pos.data_ptr()))
    with pytest.raises(fpm.FpmError):
        fpm.FPM(32, 32, force_path=fpm.FORCE_UNFUSED, batch=2)          # a batch needs the fused path


def test_one_off_argument_sets_run_kernel_by_kernel_and_a_repeat_is_captured(fpm):
    """FPM_GRAPH_AUTO builds a graph only when an argument set repeats the previous call's (capture and
    instantiation cost more than one replay saves): fresh tensors on every call give the results of the
    kernel-by-kernel path, and so do the capture and the replays once a set does repeat."""
    import torch
    cfg = fi.CONFIGS["C1"]
    ctx = fpm.FPM(cfg.ng, cfg.np_side, omega_m=OM, box=cfg.box, force_path=fpm.FORCE_FUSED)
    pos0, mom0 = ctx.lpt_init(dev(fi.linear_field(cfg.np_side, cfg.box, cfg.seed)), cfg.a0, cfg.lpt_order)
    stages = cfg.stages()
    ctx.set_graph_mode(fpm.GRAPH_OFF)
    pr, mr = pos0.clone(), mom0.clone()
    n0 = ctx.launch_count()
    ctx.nbody(pr, mr, stages)
    per_run = ctx.launch_count() - n0
    ctx.set_graph_mode(fpm.GRAPH_AUTO)
    keep = []                                              # keep the tensors alive so that no address is reused
    for _ in range(4):                                     # a new argument set on every call
        p, m = pos0.clone(), mom0.clone()
        keep.append((p, m))
        n0 = ctx.launch_count()
        ctx.nbody(p, m, stages)
        assert ctx.launch_count() - n0 == per_run
        assert float((p - pr).abs().max()) < 1e-4 and rel_l2(host(m), host(mr)) < 1e-5
    p, m = pos0.clone(), mom0.clone()
    for _ in range(4):                                     # the same set: eager, capture + replay, replay, replay
        p.copy_(pos0)
        m.copy_(mom0)
        n0 = ctx.launch_count()
        ctx.nbody(p, m, stages)
        assert ctx.launch_count() - n0 == per_run
        assert float((p - pr).abs().max()) < 1e-4 and rel_l2(host(m), host(mr)) < 1e-5


def test_nbody_inside_the_callers_own_stream_capture(fpm):
    """Called while the context's stream is being captured (torch.cuda.graph), fpm_nbody must not start a
    capture of its own: it enqueues plain launches, the caller's graph records them, and replaying that graph
    gives the run -- in every graph mode."""
    import torch
    cfg = fi.CONFIGS["C1"]
    side = torch.cuda.Stream()
    ref = None
    for mode in (fpm.GRAPH_OFF, fpm.GRAPH_AUTO, fpm.GRAPH_ALWAYS):
        with torch.cuda.stream(side):
            ctx = fpm.FPM(cfg.ng, cfg.np_side, omega_m=OM, box=cfg.box, force_path=fpm.FORCE_FUSED, stream=side)
            ctx.set_graph_mode(mode)
            pos0, mom0 = ctx.lpt_init(dev(fi.linear_field(cfg.np_side, cfg.box, cfg.seed)), cfg.a0, cfg.lpt_order)
            pos, mom = pos0.clone(), mom0.clone()
            stages = cfg.stages()
            if ref is None:                                # the run itself, outside any capture
                pr, mr = pos0.clone(), mom0.clone()
                ctx.nbody(pr, mr, stages)
                ref = (pr, mr)
            side.synchronize()
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=side):
                ctx.nbody(pos, mom, stages)
            side.synchronize()
            for _ in range(2):
                pos.copy_(pos0)
                mom.copy_(mom0)
                g.replay()
                side.synchronize()
                assert float((pos - ref[0]).abs().max()) < 1e-4 and rel_l2(host(mom), host(ref[1])) < 1e-5
            ctx.nbody(pos, mom, stages)                    # the context still works after the capture
            side.synchronize()


def test_kick_and_drift_refuse_a_batched_context(fpm):
    """fpm.h 'Batches': the single-operator calls are not batched; on a [B][3][n] array they would update member 0
    only, so they return FPM_ENOTIMPL instead."""
    import ctypes
    import torch
    cfg = fi.CONFIGS["C1"]
    ctx = fpm.FPM(cfg.ng, cfg.np_side, omega_m=OM, force_path=fpm.FORCE_FUSED, batch=2)
    x = torch.zeros(2, 3, cfg.n_particles, device="cuda")
    y = torch.ones_like(x)
    lib = ctypes.CDLL(fpm.library_path())
    vp, dbl = ctypes.c_void_p, ctypes.c_double
    for fn in (lib.fpm_kick, lib.fpm_drift):
        fn.argtypes = [vp, vp, vp, ctypes.c_int64, dbl, dbl, dbl]
        assert fn(ctx._h, vp(x.data_ptr()), vp(y.data_ptr()), cfg.n_particles, 0.1, 0.2, 0.3) == fpm.ENOTIMPL
    torch.cuda.synchronize()
    assert float(x.abs().max()) == 0.0


def test_batch_whose_meshes_pass_two_to_the_31(fpm):
    """no batch so far put a mesh index past 2^31.  272 members of 64^3 particles on a 128^3 mesh:
    the batched real meshes are 2.28e9 bytes and the interleaved (F_x, F_y, F_z, -) force mesh of the step is
    2.28e9 floats, so both byte offsets and the float4 mesh's element offsets leave 32 bits for the late
    members.  First, middle and last member must equal batch-1 runs of the same fields."""
    import torch
    ng, nps, batch, box = 128, 64, 272, 200.0
    assert batch * ng ** 3 * 4 > 2 ** 31 and batch * ng <= 65535
    special = {0: 11, 1: 12, batch // 2: 13, batch - 2: 14, batch - 1: 15}
    filler = fi.linear_field(nps, box, 10)
    fields = np.stack([fi.linear_field(nps, box, special[b]) if b in special else filler for b in range(batch)])
    stages = [0.1, 0.3, 0.6, 1.0]
    ctx = fpm.FPM(ng, nps, omega_m=OM, box=box, force_path=fpm.FORCE_FUSED, batch=batch)
    pos, mom = ctx.lpt_init(dev(fields), 0.1, 2)
    rho = ctx.paint(pos)
    ctx.set_graph_mode(fpm.GRAPH_OFF)
    ctx.nbody(pos, mom, stages)
    torch.cuda.synchronize()
    single = fpm.FPM(ng, nps, omega_m=OM, box=box, force_path=fpm.FORCE_FUSED)
    single.set_graph_mode(fpm.GRAPH_OFF)
    for b in special:
        sp, sm = single.lpt_init(dev(fields[b]), 0.1, 2)
        assert float((single.paint(sp) - rho[b]).abs().max()) < 1e-4, b
        single.nbody(sp, sm, stages)
        d = (sp - pos[b]).abs()
        d = torch.minimum(d, ng - d)
        assert float(d.max()) < 1e-3, (b, float(d.max()))
        assert float(torch.linalg.vector_norm(sm - mom[b]) / torch.linalg.vector_norm(sm)) < 1e-4, b
    assert float((pos[0] - pos[batch - 1]).abs().max()) > 0.1          # different simulations
