"""qsgw_chi0_to_coulomb_basis_static (include/qsgw.h): the basis rotation U^H chi0 U on the library's file-scope device
scratch, for callers that cannot call cudaMalloc.  Checked against the existing entry point qsgw_chi0_to_coulomb_basis
(stream-ordered workspace) and against the oracle, tolerance of tests/test_gpu_wc.py (1e-12 relative Frobenius per
frequency), on two calls in a row of DIFFERENT size (the second, smaller problem finds the first call's data in the
scratch).  Collected last on purpose (file name): the suite runs with pytest -x."""
import numpy as np
import pytest

import oracle

pytestmark = pytest.mark.gpu

TOL = 1e-12


def hermitian_stack(rng, n_freq, n_m):
    a = rng.standard_normal((n_freq, n_m, n_m)) + 1j * rng.standard_normal((n_freq, n_m, n_m))
    return np.ascontiguousarray(-(a @ np.conj(np.transpose(a, (0, 2, 1)))) / n_m)      # negative semidefinite, as chi0(i omega)


def rel_fro_per_freq(a, b):
    return np.array([np.linalg.norm(a[j] - b[j]) / np.linalg.norm(b[j]) for j in range(a.shape[0])])


def test_static_scratch_rotation_two_calls_in_a_row():
    import torch
    import paper_2506_03477_b200 as q
    from qsgw_synth import haar_unitary
    rng = np.random.default_rng(250603477)
    free_after = []
    for n_freq, n_m in ((16, 240), (5, 99)):          # cfg-1 shape (fills 33 * 256^2 exactly), then a ragged smaller one
        chi = hermitian_stack(rng, n_freq, n_m)
        U = haar_unitary(rng, n_m)
        d_chi, d_U = torch.from_numpy(chi).cuda(), torch.from_numpy(U).cuda()
        ref_gpu = q.chi0_to_coulomb_basis(d_chi, d_U)                 # existing path (allocating workspace)
        out = torch.full_like(d_chi, complex(float("nan"), float("nan")))
        torch.cuda.synchronize()
        free0 = torch.cuda.mem_get_info()[0]
        q.chi0_to_coulomb_basis_static(d_chi, d_U, out)
        torch.cuda.synchronize()
        free_after.append(torch.cuda.mem_get_info()[0] - free0)
        got, ref_g = out.cpu().numpy(), ref_gpu.cpu().numpy()
        assert np.isfinite(got.view(np.float64)).all()
        assert rel_fro_per_freq(got, ref_g).max() <= TOL
        assert rel_fro_per_freq(got, oracle.rotate_to_coulomb_basis_ref(chi, U)).max() <= TOL
        assert np.array_equal(got, np.conj(np.transpose(got, (0, 2, 1))))
    assert free_after[1] == 0, free_after            # the second call (kernel images loaded) changed no device memory


def test_static_scratch_rejects_sizes_beyond_the_limit():
    import torch
    import paper_2506_03477_b200 as q
    chi = torch.zeros((16, 320, 320), dtype=torch.complex128, device="cuda")      # 33 * 320^2 > 33 * 256^2
    U = torch.eye(320, dtype=torch.complex128, device="cuda")
    out = torch.empty_like(chi)
    with pytest.raises(q.QsgwError) as e:
        q.chi0_to_coulomb_basis_static(chi, U, out)
    assert e.value.code == 4 and "static scratch" in str(e.value)
    chi3 = torch.zeros((3, 512, 512), dtype=torch.complex128, device="cuda")      # 7 * 512^2 <= 33 * 256^2: accepted
    q.chi0_to_coulomb_basis_static(chi3, torch.eye(512, dtype=torch.complex128, device="cuda"), torch.empty_like(chi3))
    torch.cuda.synchronize()
