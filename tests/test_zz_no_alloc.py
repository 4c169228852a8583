"""fpm_reduce_static -- REDUCE (Alg. 2) for callers that cannot allocate device memory.

Some users of libfpm run where every byte of device memory already has an owner (a framework's caching pool, a
fixed MIG/MPS budget) or inside a loop that cannot take the device-wide synchronisation of cudaMalloc; they can
create neither a context (fpm_create allocates plan tables) nor a workspace.  fpm_reduce_static serves them from
an 8 MiB array built into the library image (meshes up to 128^3), shared by all calls on a device and never
cleared.  This file checks that it gives what the context + workspace path (fpm_reduce, itself checked against
the float64 oracle in test_gpu_pyramid.py) gives -- on two calls in a row, the second on a smaller mesh so that
the array still holds the first call's intermediates -- that free device memory does not move across a call,
and that an oversized mesh is refused with a message instead of overrunning the array.

The file name sorts last on purpose: pytest -x stops at the first failure, so a failure here hides nothing.
It must pass alone in a fresh process (the first call does the one-time address lookup) and after the others.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def fpm():
    import paper_2010_11847_b200 as m
    return m


def test_reduce_static_matches_the_workspace_path_on_two_calls_in_a_row(fpm):
    import torch
    rng = np.random.default_rng(20101184)
    cases = [(128, 2), (64, 3)]            # the largest mesh the array holds, then a smaller one over its leftovers
    meshes = [torch.from_numpy(rng.standard_normal((ng, ng, ng)).astype(np.float32)).cuda() for ng, _ in cases]
    # expected values first, through the existing path (context + caller-allocated workspace)
    expected = [fpm.FPM(ng).reduce(mesh, levels) for (ng, levels), mesh in zip(cases, meshes)]
    outs = [torch.full((ng >> levels,) * 3, float("nan"), device="cuda") for ng, levels in cases]
    torch.cuda.synchronize()
    free_before = []
    for (ng, levels), mesh, out in zip(cases, meshes, outs):      # two calls back to back, nothing in between
        free_before.append(torch.cuda.mem_get_info()[0])
        fpm.reduce_static(mesh, levels, out)
    torch.cuda.synchronize()
    free_after = torch.cuda.mem_get_info()[0]
    for (ng, levels), out, ref in zip(cases, outs, expected):
        assert out.shape == ref.shape
        # the tolerance of test_gpu_pyramid.py; the two paths run the same passes, so in practice they agree bit for bit
        assert float((out - ref).abs().max()) <= 2e-6 * float(ref.abs().max()), (ng, levels)
    # no device memory was taken by the second call (the first may load the module that holds the array)
    assert free_after == free_before[1]
    # a repeat of the first case over the second call's leftovers
    again = torch.empty_like(outs[0])
    fpm.reduce_static(meshes[0], cases[0][1], again)
    assert torch.equal(again, outs[0])
    # zero levels is a copy, as in fpm_reduce
    same = torch.empty_like(meshes[1])
    fpm.reduce_static(meshes[1], 0, same)
    assert torch.equal(same, meshes[1])


def test_reduce_static_refuses_what_its_array_cannot_hold(fpm):
    import torch
    big = torch.zeros((256, 256, 256), device="cuda")
    with pytest.raises(fpm.FpmError, match="exceeds the built-in scratch"):
        fpm.reduce_static(big, 1, torch.empty((128, 128, 128), device="cuda"))
    small = torch.zeros((32, 32, 32), device="cuda")
    with pytest.raises(fpm.FpmError, match="levels out of range"):
        fpm.reduce_static(small, 3, torch.empty((4, 4, 4), device="cuda"))
    with pytest.raises(fpm.FpmError, match="distinct"):
        fpm.reduce_static(small, 0, small)
    with pytest.raises(fpm.FpmError):                               # out of the wrong size never reaches the C call
        fpm.reduce_static(small, 1, torch.empty((8, 8, 8), device="cuda"))
