"""ssm_group_stress_noalloc: the group stresses for callers that cannot allocate device memory.

Who they are: a flow solver's plug-in inside an application whose own memory pool owns the whole GPU (it is handed
the buffers of its inputs and outputs and nothing else; a raw cudaMalloc there fails or steals from the pool), and a
coupling loop that cannot afford the device-wide stall of cudaMalloc / cudaFree.  ssm_group_stress_device borrows its
intermediate integer sums from the workspace's staging area; this entry point keeps them in a fixed array inside
libssm.so instead (4096 groups at most), which all calls on a GPU share and which still holds the last call's sums
when the next call starts.

So the test makes TWO calls in a row on different states and a different group size: if the second call did not clear
what the first left behind, or if the kernels were given something other than the array's device address, the results
could not equal those of the existing path.  Both paths round each chain's stress to the same fixed point and add
integers, so the comparison is exact (the bound the other group-stress tests use, tests/test_gpu_flow.py).

This file is named so that pytest collects it last: `pytest -x` stops at the first failure, and a failure here must not
hide the parity tests.  It passes alone in a fresh process (where its first call does the per-device set-up) and after
the other tests."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ssm():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_1106_2899_b200 as m
    m.lib()
    return m


def test_no_alloc_group_stress_equals_the_workspace_path_on_two_calls_in_a_row(ssm):
    import torch
    N, M = 32, 5000                                     # 625 warp tiles; the last group of every split is ragged
    g = ssm.Ensemble(N, M, seed=11)
    g.step(40, 0.05)                                    # slip-springs have hopped, been destroyed and created; sigma_xy != 0
    # first call: 40 groups of 128 chains (last one 8); the caller owns the output buffer, nothing else is needed
    out1 = torch.full((40, 13), float("nan"), dtype=torch.float64, device="cuda")
    g.group_stress_noalloc(128, out1)
    ref1 = g.group_stress_device(128)
    # second call straight after it, on a moved state and with FEWER, larger groups: the leading part of the array still
    # holds the first call's sums unless the call clears it
    g.step(20, 0.05)
    out2 = torch.full((5, 13), float("nan"), dtype=torch.float64, device="cuda")
    g.group_stress_noalloc(1024, out2)
    ref2 = g.group_stress_device(1024)
    torch.cuda.synchronize()
    a1, b1, a2, b2 = out1.cpu().numpy(), ref1.cpu().numpy(), out2.cpu().numpy(), ref2.cpu().numpy()
    assert np.all(np.isfinite(a1)) and np.all(np.isfinite(a2))
    assert np.array_equal(a1, b1), np.abs(a1 - b1).max()
    assert np.array_equal(a2, b2), np.abs(a2 - b2).max()
    assert np.array_equal(a2, g.group_stress(1024))     # and the host-pointer call agrees
    assert not np.array_equal(a1[:5], a2)               # the two calls really saw different inputs
    assert abs(a2[:, 12].mean() - N / 4.0) < 1.0        # <Z> near N / N0 (eq 10): the sums are the chains', not leftovers
    # a third call with one chain per group up to the limit's edge is served; one group more is refused, loudly
    small = ssm.Ensemble(8, ssm.NOALLOC_MAX_GROUPS + 1, seed=3)
    out3 = torch.empty((ssm.NOALLOC_MAX_GROUPS + 1, 13), dtype=torch.float64, device="cuda")
    with pytest.raises(ssm.SsmError) as err:
        small.group_stress_noalloc(1, out3)
    assert err.value.code == ssm.SSM_ERANGE and "4096" in str(err.value)
    ng = -(-small.M // 2)
    small.group_stress_noalloc(2, out3[:ng])
    assert np.array_equal(out3[:ng].cpu().numpy(), small.group_stress(2))
    with pytest.raises(ssm.SsmError):
        small.group_stress_noalloc(2, None)             # the binding does not allocate the output either
    g.close(); small.close()
