"""mhs_resnorm_static -- the entry point that allocates nothing (include/mhs.h; README "No-allocation entry point"):
its partial sums live in a file-scope device array instead of a buffer from mhs_create.  Checked against the existing
path (mhs_set_potential + mhs_op_resnorm on a context) on two calls in a row that share the array, and against the oracle.
This file is collected last on purpose: the run is `pytest -x`."""
import numpy as np
import pytest
import torch

from paper_1307_6720_b200 import binding, inputs

OPTOL = {torch.float64: 1e-13, torch.float32: 2e-6}     # as tests/test_gpu_parity.py


def _case(w, dtype, seed):
    """A potential with data on the bottom plane and zero side/top walls, c = 1 + f, and the existing path's norm."""
    nz, ny, nx = w.shape
    P = inputs.random_field(w.shape, seed)
    P[0] = inputs.random_field((ny, nx), seed + 1)
    Pd = torch.as_tensor(P, dtype=dtype, device="cuda").contiguous()
    with binding.Solver.from_workload(w, dtype=dtype) as S:
        S.set_potential(Pd.reshape(-1))
        want = S.op_resnorm(3, 0)
    c = torch.as_tensor(1.0 + np.asarray(w.f, dtype=np.float64), device="cuda")
    return P, Pd, c, want


@pytest.mark.gpu
@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
def test_resnorm_static_matches_the_context_path_twice_in_a_row(orc, dtype):
    big, small = inputs.config(1, shrink=2), inputs.small()          # 65^3, then a ragged 17 x 33 x 9 (fewer partial sums:
    out = torch.full((2,), -1.0, dtype=torch.float64, device="cuda")  # the array still holds the first call's beyond them)
    cases = [_case(big, dtype, 11), _case(small, dtype, 23)]
    before = torch.cuda.memory_allocated()
    for q, (w, (P, Pd, c, want)) in enumerate(zip((big, small), cases)):
        nz, ny, nx = w.shape
        hx, hy, hz = w.Lx / (nx - 1), w.Ly / (ny - 1), w.Lz / (nz - 1)
        binding.mhs_resnorm_static(Pd.reshape(-1), c, out[q:q + 1], nx, ny, nz, hx, hy, hz, w.alpha)
    assert torch.cuda.memory_allocated() == before
    got = out.cpu().numpy()
    for q, (w, (P, Pd, c, want)) in enumerate(zip((big, small), cases)):
        assert want > 0 and abs(got[q] - want) <= 50 * OPTOL[dtype] * want, (q, got[q], want)
        ref = orc.resnorm3(Pd.cpu().double().numpy(), None, 1.0 + np.asarray(w.f), w.alpha, w.L)
        assert abs(got[q] - ref) <= 50 * OPTOL[dtype] * ref, (q, got[q], ref)
    # the same call again: same bits (fixed summation order, nothing left over from the calls in between matters)
    w, (P, Pd, c, want) = big, cases[0]
    nz, ny, nx = w.shape
    again = torch.zeros(1, dtype=torch.float64, device="cuda")
    binding.mhs_resnorm_static(Pd.reshape(-1), c, again, nx, ny, nz, w.Lx / (nx - 1), w.Ly / (ny - 1), w.Lz / (nz - 1), w.alpha)
    assert again.item() == got[0]


@pytest.mark.gpu
def test_resnorm_static_rejects_what_the_scratch_cannot_hold():
    one = torch.zeros(1, dtype=torch.float64, device="cuda")
    ny, nz = 8 * 1024 + 2, 66                                          # 1024 * 64 = 65536 partial sums: the maximum
    assert (ny - 2) // 8 * (nz - 2) == binding.MHS_STATIC_SCRATCH_DOUBLES
    P = torch.zeros(3 * ny * (nz + 1), dtype=torch.float32, device="cuda")
    c = torch.ones(nz + 1, dtype=torch.float64, device="cuda")
    binding.mhs_resnorm_static(P[:3 * ny * nz], c[:nz], one, 3, ny, nz, 1.0, 1.0, 1.0, 0.0)
    assert one.item() == 0.0
    with pytest.raises(binding.MHSError) as e:                         # one more plane: 1024 * 65 partial sums
        binding.mhs_resnorm_static(P, c, one, 3, ny, nz + 1, 1.0, 1.0, 1.0, 0.0)
    assert e.value.status == binding.MHS_ERR_INVALID_ARG and "MHS_STATIC_SCRATCH_DOUBLES" in str(e.value)
