"""ep_weighted_mean_noalloc (include/ep.h): the entry point that allocates nothing, for callers that cannot call cudaMalloc.
Its output is checked against the existing path, ep_mean_vm (v_bar of PAPER.md:216 / :230), on calls in a row that share
the file-scope device scratch.  The file is named so that pytest collects it last (the suite runs with pytest -x)."""
import numpy as np
import pytest

from ep_inputs import make

pytestmark = pytest.mark.gpu

TOL_MV = 1e-10   # the tolerance of test_mean_vm_parity for two summation orders of the same volumes (~1e-13 relative)


@pytest.fixture(scope="module")
def ep():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2112_12854_b200 as ep
    return ep


class _DevArray:
    """Minimal __cuda_array_interface__ holder so that torch can view a raw device pointer (no copy)."""
    def __init__(self, ptr, n, typestr):
        self.__cuda_array_interface__ = {"shape": (n,), "typestr": typestr, "data": (ptr, False), "version": 2}


def _tet_volumes(xyz, tets):
    a, b, c, d = (xyz[tets[:, k]] for k in range(4))
    return np.abs(np.einsum("ij,ij->i", np.cross(b - a, c - a), d - a)) / 6.0


def test_no_alloc_mean_matches_mean_vm_on_calls_in_a_row(ep, capsys):
    import torch
    prob = make(1)
    n = prob.mesh.n_tets
    g = ep.Sim.from_problem(prob)
    g.step(150, prob.dt)                                       # the wave is under way: v_bar is far from rest
    vm_ptr, perm_ptr = g.device_vm()
    g.synchronize()
    perm = torch.as_tensor(_DevArray(perm_ptr, n, "<i4"), device="cuda").long()
    vol = torch.as_tensor(_tet_volumes(prob.mesh.xyz, prob.mesh.tets), device="cuda")[perm].contiguous()   # device order
    out = torch.full((2,), float("nan"), dtype=torch.float64, device="cuda")
    stream = torch.cuda.current_stream().cuda_stream

    # call 1: the whole mesh
    ep.weighted_mean_noalloc(vm_ptr, vol.data_ptr(), n, out.data_ptr(), stream)
    torch.cuda.synchronize()
    got1 = out.cpu().numpy().copy()
    ref1 = g.mean_vm()
    assert abs(got1[0] - ref1) <= TOL_MV, (got1[0], ref1)
    assert abs(got1[1] - float(vol.sum())) <= 1e-12 * got1[1]
    assert ref1 > -80.0

    # call 2, straight after, on a shorter prefix (fewer blocks): the slots the first call left behind must not leak in
    m = n // 3 + 5
    vm = torch.as_tensor(_DevArray(vm_ptr, n, "<f8"), device="cuda")
    ep.weighted_mean_noalloc(vm_ptr, vol.data_ptr(), m, out.data_ptr(), stream)
    torch.cuda.synchronize()
    got2 = out.cpu().numpy().copy()
    want2 = float((vol[:m] * vm[:m]).sum() / vol[:m].sum())
    assert abs(got2[0] - want2) <= TOL_MV, (got2[0], want2)

    # calls 3 and 4 after more time steps, back to back on the whole mesh: same answer twice, equal to ep_mean_vm's
    g.step(100, prob.dt)
    vm_ptr, _ = g.device_vm()
    g.synchronize()
    out2 = torch.full((2,), float("nan"), dtype=torch.float64, device="cuda")
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]                 # kernels are loaded by now: a cudaMalloc would show here
    ep.weighted_mean_noalloc(vm_ptr, vol.data_ptr(), n, out.data_ptr(), stream)
    ep.weighted_mean_noalloc(vm_ptr, vol.data_ptr(), n, out2.data_ptr(), stream)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free_before          # no device memory was taken
    got3, got4 = out.cpu().numpy().copy(), out2.cpu().numpy().copy()
    ref3 = g.mean_vm()
    assert abs(got3[0] - ref3) <= TOL_MV, (got3[0], ref3)
    assert np.array_equal(got3, got4)                          # deterministic, and the scratch carries nothing over
    assert abs(ref3 - ref1) > 1.0                              # the field did change between the calls
    with capsys.disabled():
        print(f"\nno-alloc v_bar vs ep_mean_vm: {got1[0]:.12f} / {ref1:.12f} mV, then {got3[0]:.12f} / {ref3:.12f} mV "
              f"(|d| = {abs(got1[0] - ref1):.2e}, {abs(got3[0] - ref3):.2e}); prefix of {m}: |d| = {abs(got2[0] - want2):.2e}")
    g.close()


def test_no_alloc_spans_many_blocks_and_a_ragged_tail(ep):
    """More elements than one pass of the final kernel (1,024 partial sums) and a ragged last block, against torch in fp64."""
    import torch
    gen = torch.Generator(device="cpu").manual_seed(20211212)
    n = 4096 * 1500 + 77
    v = (torch.rand(n, generator=gen, dtype=torch.float64) * 120.0 - 90.0).cuda()
    w = (torch.rand(n, generator=gen, dtype=torch.float64) + 0.5).cuda()
    out = torch.empty(2, dtype=torch.float64, device="cuda")
    for _ in range(2):                                         # two calls in a row
        ep.weighted_mean_noalloc(v.data_ptr(), w.data_ptr(), n, out.data_ptr(), torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        want = float((w * v).sum() / w.sum())
        assert abs(float(out[0]) - want) <= 1e-11 * abs(want)
        assert abs(float(out[1]) - float(w.sum())) <= 1e-12 * float(w.sum())
        v = v.flip(0).contiguous()                             # other inputs for the second call


def test_no_alloc_refuses_sizes_beyond_the_scratch(ep):
    import torch
    buf = torch.zeros(8, dtype=torch.float64, device="cuda")
    with pytest.raises(ep.EpError) as e:
        ep.weighted_mean_noalloc(buf.data_ptr(), buf.data_ptr(), ep.NOALLOC_MAX_N + 1, buf.data_ptr())
    assert e.value.code == -1 and "EP_NOALLOC_MAX_N" in str(e.value) and str(ep.NOALLOC_MAX_N) in str(e.value)
    with pytest.raises(ep.EpError) as e:
        ep.weighted_mean_noalloc(buf.data_ptr(), buf.data_ptr(), 0, buf.data_ptr())
    assert e.value.code == -1
    with pytest.raises(ep.EpError) as e:
        ep.weighted_mean_noalloc(0, buf.data_ptr(), 8, buf.data_ptr())
    assert e.value.code == -1
    buf[:] = torch.arange(8, dtype=torch.float64)              # the refused calls touched nothing; a valid one still works
    w = torch.ones(8, dtype=torch.float64, device="cuda")
    out = torch.empty(2, dtype=torch.float64, device="cuda")
    ep.weighted_mean_noalloc(buf.data_ptr(), w.data_ptr(), 8, out.data_ptr())
    torch.cuda.synchronize()
    assert out.cpu().tolist() == [3.5, 8.0]
