"""mbs_apply_B_static: the scattering operator B with the slab kernels' scratch in the library's static device array
(no cudaMalloc on the call path; include/mbs.h).  Checked against the existing path, mbs_apply_operator(MBS_OP_B), on two
calls in a row with different inputs (the static array keeps the first call's contents), and against the oracle.
Collected last on purpose (file name): the suite runs with `pytest -x`."""
import numpy as np
import pytest

from paper_2410_02395_b200 import workloads

pytestmark = pytest.mark.gpu

OP_TOL = 1e-5          # per-operator bar of the parity tests (BASELINE.json north_star)


def rel(a, b):
    a = np.asarray(a).astype(np.complex128).ravel()
    b = np.asarray(b).astype(np.complex128).ravel()
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2410_02395_b200 import binding
    return binding


CASES = [
    ((64, 40, 48), (2, 1, 3), (4, 4, 4), 8, None),
    ((128, 80), (2, 1), (8, 8), 8, None),
    ((80, 128), (2, 2), (4, 0), 8, (0, 1)),
    ((256,), (2,), (8,), 8, None),
]


@pytest.mark.parametrize("shape,S,W,t,periodic", CASES)
def test_static_scratch_B_matches_existing_path(B, shape, S, W, t, periodic):
    import torch
    from oracle import mbs_oracle
    n = workloads.random_medium(shape, 123, 1.0, 1.5, 0.02)
    s = B.Solver(shape, 0.25, 1.0, W, S, periodic=periodic, n_correction=t)
    s.set_potential(n)
    o = mbs_oracle.MBSOracle(n, 0.25, 1.0, W, S, periodic=periodic, n_correction=t)
    for call, seed in enumerate((7, 8)):                      # two calls in a row, different inputs
        u = workloads.random_field(shape, seed)
        ud = torch.from_numpy(u).cuda()
        ref = s.apply_operator(B.MBS_OP_B, ud)                # existing path: scratch in the context's workspace
        out = torch.empty_like(ud)
        torch.cuda.synchronize()
        before, free_before = torch.cuda.memory_allocated(), torch.cuda.mem_get_info()[0]
        B.mbs_apply_B_static(s.ctx, ud.data_ptr(), out.data_ptr())
        torch.cuda.synchronize()
        assert torch.cuda.memory_allocated() == before
        if call == 1:                                         # (the first call may load kernels lazily)
            assert torch.cuda.mem_get_info()[0] == free_before    # no device allocation by anyone during the call
        assert rel(out.cpu().numpy(), ref.cpu().numpy()) <= OP_TOL, (call, rel(out.cpu().numpy(), ref.cpu().numpy()))
        assert torch.equal(out, ref)                          # same kernels, same launch geometry: bit for bit
        assert rel(out.cpu().numpy(), o.apply_B(u.astype(np.complex128))) <= OP_TOL
        # in == out is allowed
        B.mbs_apply_B_static(s.ctx, ud.data_ptr(), ud.data_ptr())
        assert torch.equal(ud, ref)
    s.close()


def test_static_scratch_limit_is_reported(B):
    """A grid whose edge corrections do not fit the static array is refused with a clear error, not truncated."""
    import torch
    # (256, 256, 128), 2x2x1, t = 8: 8 + 8 + 8 MiB of compact correction buffers > 16 MiB
    s = B.Solver((256, 256, 128), 0.25, 1.0, (4, 4, 4), (2, 2, 1), n_correction=8)
    s.set_potential(workloads.random_medium((256, 256, 128), 5))
    u = torch.zeros((256, 256, 128), dtype=torch.complex64, device="cuda")
    with pytest.raises(B.MBSError) as e:
        B.mbs_apply_B_static(s.ctx, u.data_ptr(), u.data_ptr())
    assert e.value.status == B.MBS_ERR_INVALID_ARG
    assert "MBS_STATIC_SCRATCH_BYTES" in str(e.value) and str(B.MBS_STATIC_SCRATCH_BYTES) in str(e.value)
    s.close()
    s2 = B.Solver((64,), 0.25, 1.0, (4,), (2,), n_correction=8)
    with pytest.raises(B.MBSError) as e:                      # before set_potential
        B.mbs_apply_B_static(s2.ctx, u.data_ptr(), u.data_ptr())
    assert e.value.status == B.MBS_ERR_STATE
    s2.close()
