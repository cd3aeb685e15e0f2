"""sm_trace_dk_static (include/submatrix.h): tr(D K), Eq.(10), through the entry point that allocates
nothing (scratch in a file-scope __device__ array) against the existing sm_trace_dk, on calls in a row.

Collected last on purpose (file name): the suite runs with pytest -x."""
import ctypes as C

import numpy as np
import pytest

from paper_2004_10811_b200 import workloads as W

TOL_E = 1e-10  # relative, as tests/test_gpu_parity.py


def test_static_entry_rejects_oversize_without_gpu():
    """Argument validation is host logic and comes before any CUDA call: sizes beyond the fixed scratch are rejected
    with a text that names the limit."""
    from paper_2004_10811_b200 import binding as B
    L = B.lib()
    dummy = C.c_void_p(256)  # never dereferenced: the call must fail before touching the device
    st = L.sm_trace_dk_static(B.SM_STATIC_MAX_NNZ + 1, dummy, dummy, dummy, None)
    assert st == B.SM_ERR_INVALID_ARG
    msg = L.sm_last_cuda_error().decode()
    assert "SM_STATIC_MAX_NNZ" in msg and str(B.SM_STATIC_MAX_NNZ) in msg, msg
    assert L.sm_trace_dk_static(-1, dummy, dummy, dummy, None) == B.SM_ERR_INVALID_ARG
    assert L.sm_trace_dk_static(8, None, dummy, dummy, None) == B.SM_ERR_INVALID_ARG
    assert L.sm_trace_dk_static(8, dummy, dummy, None, None) == B.SM_ERR_INVALID_ARG


@pytest.mark.gpu
def test_static_entry_matches_trace_dk_on_calls_in_a_row():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2004_10811_b200 import binding as B
    B.lib()
    # three workloads of very different size, the big one first: a later, smaller call sees the stale partials of
    # an earlier one in the shared scratch and must not pick them up (257.7 chunks, 7.3 chunks, less than one)
    mats = [W.make_config(2), W.make_config(0), W.random_block_pattern(nb=30, density=0.2, max_bs=5, seed=11)]
    cases = []
    for m in mats:
        K = torch.from_numpy(m.values).cuda()
        plan = B.plan_from_matrix(m, B.default_options())
        ws = B.alloc_workspace(plan)
        D = torch.empty_like(K)
        st = B.sm_sign_execute(plan, K, 0.0, 1e-12, D, ws, B.sm_stats_t())
        assert st >= 0
        _, ref = B.sm_trace_dk(plan, D, K)          # the existing path (plan scratch from cudaMalloc)
        cases.append((K, D, ref))
        B.sm_plan_destroy(plan)
        del ws
    out = torch.full((len(cases) * 2 + 1,), float("nan"), dtype=torch.float64, device="cuda")
    torch.cuda.synchronize()
    # first call on this device (resolves the scratch address), then every case twice more, back to back, no sync
    B.sm_trace_dk_static(cases[0][0].numel(), cases[0][1], cases[0][0], out[-1:])
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    k = 0
    for rep in range(2):
        for K, D, ref in cases:
            B.sm_trace_dk_static(K.numel(), D, K, out[k:k + 1])
            k += 1
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 >= free0, "device memory was allocated by sm_trace_dk_static"
    got = out.cpu().numpy()
    k = 0
    for rep in range(2):
        for K, D, ref in cases:
            assert abs(got[k] - ref) <= TOL_E * max(abs(ref), 1.0), (rep, k, got[k], ref)
            k += 1
    assert abs(got[-1] - cases[0][2]) <= TOL_E * max(abs(cases[0][2]), 1.0)
    # deterministic: the two rounds are bitwise equal
    n = len(cases)
    assert np.array_equal(got[:n], got[n:2 * n])
    # empty input: the sum of nothing, written (not left over)
    z = torch.full((1,), float("nan"), dtype=torch.float64, device="cuda")
    B.sm_trace_dk_static(0, None, None, z)
    torch.cuda.synchronize()
    assert float(z.item()) == 0.0
