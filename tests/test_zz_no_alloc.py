"""The allocation-free entry point rgf_inverse_batched_static (include/rgf.h) against the existing rgf_inverse_batched.

Collected last on purpose (pytest -x: a failure here hides nothing after it).  Passes alone in a fresh
process (the scratch address is resolved on first use) and after the other tests (the shared static array then holds
whatever an earlier call left)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def test_static_inverse_matches_existing_path_twice_in_a_row():
    import torch
    from paper_1107_5300_b200 import binding as rgf
    stream = torch.cuda.current_stream()
    with rgf.Plan(0) as plan:
        # second call smaller than the first: it must not see the first call's leftovers (maps, flags, work copies)
        for n, batch, seed in ((100, 5, 1), (33, 3, 2)):
            rng = np.random.default_rng(seed)
            A = rng.standard_normal((batch, n, n)) + 1j * rng.standard_normal((batch, n, n))
            A[-1, 0, 0] = 0.0                      # forces a row exchange
            ref = np.empty_like(A)
            rgf.rgf_inverse_batched(plan.handle, n, batch, A, ref)          # existing path
            A_dev = torch.from_numpy(A).cuda()
            out_dev = torch.full_like(A_dev, float("nan"))
            st_dev = torch.full((batch,), 7, dtype=torch.int32, device="cuda")
            rgf.rgf_inverse_batched_static(0, stream.cuda_stream, n, batch, A_dev, out_dev, st_dev)
            torch.cuda.synchronize()
            out = out_dev.cpu().numpy()
            assert torch.equal(A_dev.cpu(), torch.from_numpy(A))            # input untouched
            assert np.all(st_dev.cpu().numpy() == 0)
            for b in range(batch):
                scale = np.max(np.abs(ref[b]))
                assert np.max(np.abs(out[b] - ref[b])) < 1e-9 * scale, (n, b, np.max(np.abs(out[b] - ref[b])) / scale)
                assert np.max(np.abs(out[b] - np.linalg.inv(A[b]))) < 1e-9 * scale


def test_static_inverse_reports_singular_and_rejects_what_it_cannot_hold():
    import torch
    from paper_1107_5300_b200 import binding as rgf
    A = torch.zeros((2, 8, 8), dtype=torch.complex128, device="cuda")
    A[0] = torch.eye(8, dtype=torch.complex128)
    out = torch.empty_like(A)
    st = torch.zeros(2, dtype=torch.int32, device="cuda")
    rgf.rgf_inverse_batched_static(0, None, 8, 2, A, out, st)
    torch.cuda.synchronize()
    assert st.cpu().tolist() == [0, 1]
    for n, batch in ((300, 1), (256, 5), (8, 65)):
        with pytest.raises(rgf.RgfError) as e:
            rgf.rgf_inverse_batched_static(0, None, n, batch, A, out, None)
        assert e.value.code == rgf.RGF_EUNSUPPORTED and "exceeds the static scratch" in str(e.value)
    with pytest.raises(rgf.RgfError) as e:
        rgf.rgf_inverse_batched_static(0, None, 8, 2, np.zeros((2, 8, 8), dtype=complex), out, None)      # host pointer
    assert e.value.code == rgf.RGF_EINVAL
