"""cs_cone_violation_static -- the library's one allocation-free entry point (scratch in a file-scope device array)
-- against the existing path (cs_residuals' cone_viol_rel for the same iterate), on two calls in a row.  Collected
last on purpose (pytest -x: a failure here must not hide the other tests)."""
import numpy as np
import pytest

from paper_2103_00736_b200 import workloads as W

pytestmark = pytest.mark.gpu

TOL_RES = 1e-6      # the residual tolerance of tests/test_gpu_parity.py


def _device_iterate(S, n):
    import torch
    x = torch.empty(n, dtype=torch.float64, device="cuda:0")
    z = torch.empty(n, dtype=torch.float64, device="cuda:0")
    S.solution_into(x=x, z=z)
    torch.cuda.synchronize()
    return x, z


def test_static_scratch_entry_point_matches_cs_residuals_twice():
    import oracle
    import torch
    from paper_2103_00736_b200 import binding
    # call 1: mixed cones, a mid-run iterate (x, z are NOT in K yet: the distances are non-zero)
    p1 = W.sparse_socp(31, 900, 2600, 120, 6, n_lin=700, lo=1, hi=60)
    S1 = binding.Solver.from_problem(p1, device="cuda:0")
    S1.run(12, L=[6])
    want1 = S1.residuals()["cone_viol_rel"]
    x1, z1 = _device_iterate(S1, p1.n)
    got1 = binding.cone_violation_static(x1, z1, p1.n_lin, p1.soc_size)
    assert want1 > 1e-4
    assert abs(got1[4] - want1) <= TOL_RES * want1, (got1, want1)
    # the four norms against the oracle's O(n) cone operator on the same vectors
    xh, zh = x1.cpu().numpy(), z1.cpu().numpy()
    ref = [np.linalg.norm(xh - oracle.proj_cone(xh, p1.n_lin, p1.soc_size)), np.linalg.norm(zh - oracle.proj_cone(zh, p1.n_lin, p1.soc_size)),
           np.linalg.norm(xh), np.linalg.norm(zh)]
    assert np.allclose(got1[:4], ref, rtol=1e-12, atol=0)
    # call 2, straight after: another problem with FEWER cones and other sizes (the array still holds call 1's offsets
    # and partial sums), result into a device buffer
    p2 = W.sparse_socp(32, 300, 800, 25, 5, n_lin=50, lo=2, hi=90)
    S2 = binding.Solver.from_problem(p2, device="cuda:0")
    S2.run(7)
    want2 = S2.residuals()["cone_viol_rel"]
    x2, z2 = _device_iterate(S2, p2.n)
    out = torch.zeros(5, dtype=torch.float64, device="cuda:0")
    binding.cone_violation_static(x2, z2, p2.n_lin, p2.soc_size, out=out, stream=torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    got2 = out.cpu().numpy()
    assert want2 > 1e-4 and abs(got2[4] - want2) <= TOL_RES * want2, (got2, want2)
    # and the first input again: same bits as the first call (deterministic, nothing left over from call 2)
    assert np.array_equal(binding.cone_violation_static(x1, z1, p1.n_lin, p1.soc_size), got1)
    # all-orthant input (n_soc = 0)
    p3 = W.config(1, 0.05)
    S3 = binding.Solver.from_problem(p3, device="cuda:0")
    S3.run(5)
    x3, z3 = _device_iterate(S3, p3.n)
    got3 = binding.cone_violation_static(x3, z3, p3.n_lin, p3.soc_size)
    want3 = S3.residuals()["cone_viol_rel"]
    assert abs(got3[4] - want3) <= TOL_RES * want3 + 1e-15


def test_static_scratch_entry_point_rejects_what_does_not_fit():
    import torch
    from paper_2103_00736_b200 import binding
    n_soc = 32768 + 1
    x = torch.ones(2 * n_soc, dtype=torch.float64, device="cuda:0")
    with pytest.raises(binding.CsError) as ei:
        binding.cone_violation_static(x, x, 0, np.full(n_soc, 2, np.int32))
    assert ei.value.status == binding.CS_EINVAL and "32768" in str(ei.value)
    ok = binding.cone_violation_static(x[:2 * 32768], x[:2 * 32768], 0, np.full(32768, 2, np.int32))   # the maximum itself fits
    assert ok[0] == 0.0 and ok[1] == 0.0 and abs(ok[2] - np.sqrt(2 * 32768)) < 1e-9
    with pytest.raises(binding.CsError):
        binding.cone_violation_static(x[:10], x[:10], 3, np.array([4, 4], np.int32))       # sizes do not sum to n
