"""GPU parity of qsgw_wc_from_chi0 (Eqs. 10, 19) against the NumPy oracle.

Tolerance: relative Frobenius error per frequency <= 1e-10.  Derivation: a backward-stable Cholesky inverse of
eps (condition number kappa = 1 + ||sqrt(v) chi0 sqrt(v)|| <~ 1e3 for these inputs) carries ~ kappa * n * 2^-53
~ 1e-11 relative error; the 3M complex product adds a few ulp normwise."""
import numpy as np
import pytest

import oracle
from qsgw_synth import coulomb_eigenvalues, generate, get_config
from gpu_helpers import rel_fro_per_freq, run_cuda
from test_gpu_parity import RAGGED, oracle_chi

pytestmark = pytest.mark.gpu

TOL_WC = 1e-10


def _gpu_wc(chi, v):
    import torch
    import paper_2506_03477_b200 as q
    w, info = q.wc_from_chi0(torch.from_numpy(chi).cuda(), torch.from_numpy(v).cuda())
    torch.cuda.synchronize()
    return w.cpu().numpy(), int(info.item())


@pytest.mark.parametrize("idx", [0, 1])
def test_wc_from_oracle_chi0(idx):
    """chi0 from the oracle (cfg 0: N_M = 80 -> two 64-blocks with a ragged tail; cfg 1: 240 -> 4 blocks)."""
    cfg = get_config(idx)
    prob = generate(cfg, n_k=4 if idx else None)
    chi = oracle_chi(prob)
    v = coulomb_eigenvalues(cfg)
    got, info = _gpu_wc(chi, v)
    assert info == 0
    assert rel_fro_per_freq(got, oracle.wc_ref(chi, v)).max() <= TOL_WC
    assert np.array_equal(got, np.conj(np.transpose(got, (0, 2, 1))))          # exact Hermitian mirror


def test_wc_ragged_and_single_block():
    prob = generate(RAGGED)                                                     # N_M = 99
    chi = oracle_chi(prob)
    v = coulomb_eigenvalues(prob.cfg)
    got, info = _gpu_wc(chi, v)
    assert info == 0 and rel_fro_per_freq(got, oracle.wc_ref(chi, v)).max() <= TOL_WC
    chi1 = np.array([[[-0.37 + 0j]], [[-0.02 + 0j]]])                          # scalar closed form
    got1, info1 = _gpu_wc(chi1, np.array([2.5]))
    assert info1 == 0
    for j, c in enumerate((-0.37, -0.02)):
        assert got1[j, 0, 0].real == pytest.approx(2.5 ** 2 * c / (1 - 2.5 * c), rel=1e-13)


def test_wc_chained_after_gpu_chi0_cfg2_shape():
    """The metal (cfg 2 shapes, 6 k-points, both signs of D): chi0 built on the GPU feeds W^c on the GPU."""
    import torch
    import paper_2506_03477_b200 as q
    cfg = get_config(2)
    prob = generate(cfg, n_k=6)
    chi_gpu = run_cuda(prob, spin=0)
    v = coulomb_eigenvalues(cfg)
    got, info = _gpu_wc(chi_gpu, v)
    assert info == 0
    assert rel_fro_per_freq(got, oracle.wc_ref(oracle_chi(prob), v)).max() <= TOL_WC


def test_wc_not_positive_definite_is_reported():
    """eps with a negative eigenvalue (chi0 > 0 and large): info names a pivot, nothing hangs or throws."""
    n = 70
    chi = np.zeros((1, n, n), dtype=np.complex128)
    chi[0, 5, 5] = 3.0                                                          # eps_55 = 1 - 3 v_5 < 0
    got, info = _gpu_wc(chi, np.full(n, 1.0))
    assert info == 1 + 5


def test_wc_argument_errors():
    import torch
    import paper_2506_03477_b200 as q
    chi = torch.zeros((1, 4, 4), dtype=torch.complex128, device="cuda")
    v = torch.ones(4, dtype=torch.float64, device="cuda")
    with pytest.raises(q.QsgwError) as ei:
        q.wc_from_chi0(chi, v, out=chi)
    assert ei.value.code == 1


@pytest.mark.parametrize("idx", [0, 1])
def test_rotation_to_coulomb_basis(idx):
    """U^H chi0 U on the GPU (two batched DMMA GEMMs) against the oracle; then the chain rotate -> W^c."""
    import torch
    import paper_2506_03477_b200 as q
    from qsgw_synth import haar_unitary
    cfg = get_config(idx)
    prob = generate(cfg, n_k=3)
    chi = oracle_chi(prob)
    U = haar_unitary(np.random.default_rng(21 + idx), cfg.n_m)
    got = q.chi0_to_coulomb_basis(torch.from_numpy(chi).cuda(), torch.from_numpy(U).cuda())
    torch.cuda.synchronize()
    got = got.cpu().numpy()
    ref = oracle.rotate_to_coulomb_basis_ref(chi, U)
    assert rel_fro_per_freq(got, ref).max() <= 1e-12
    assert np.array_equal(got, np.conj(np.transpose(got, (0, 2, 1))))
    v = coulomb_eigenvalues(cfg)
    w, info = _gpu_wc(got, v)
    assert info == 0 and rel_fro_per_freq(w, oracle.wc_ref(ref, v)).max() <= TOL_WC


@pytest.mark.parametrize("n", [1, 7, 63, 64, 65, 127, 128, 130, 200])
def test_wc_and_rotation_block_edges(n):
    """Orders around the 64-block edges (one block, exactly full blocks, one element over, odd block counts:
    the two-blocks-per-step Cholesky ends on a single block) with a seeded negative-semidefinite chi0."""
    import torch
    import paper_2506_03477_b200 as q
    from qsgw_synth import haar_unitary
    rng = np.random.default_rng(300 + n)
    a = rng.standard_normal((2, n, max(1, n // 2))) + 1j * rng.standard_normal((2, n, max(1, n // 2)))
    chi = -(a @ np.conj(np.transpose(a, (0, 2, 1)))) / n                      # rank-deficient, <= 0
    chi[1] *= 0.01
    v = rng.uniform(0.3, 30.0, n)
    got, info = _gpu_wc(chi, v)
    assert info == 0 and rel_fro_per_freq(got, oracle.wc_ref(chi, v)).max() <= TOL_WC
    U = haar_unitary(rng, n)
    rot = q.chi0_to_coulomb_basis(torch.from_numpy(chi).cuda(), torch.from_numpy(U).cuda())
    torch.cuda.synchronize()
    assert rel_fro_per_freq(rot.cpu().numpy(), oracle.rotate_to_coulomb_basis_ref(chi, U)).max() <= 1e-12


@pytest.mark.parametrize("mode", [2, 0])
def test_wc_graph_and_plain_launch_paths(mode):
    """Option "wc_graph" = 2 makes the CUDA-graph path mandatory (an error if the capture fails), = 0 forces plain
    launches on the caller's stream: both give the oracle's result, also on a non-default stream."""
    import torch
    import paper_2506_03477_b200 as q
    q.set_global_option("wc_graph", mode)
    cfg = get_config(1)
    prob = generate(cfg, n_k=2)
    chi = oracle_chi(prob)
    v = coulomb_eigenvalues(cfg)
    ref = oracle.wc_ref(chi, v)
    d_chi, d_v = torch.from_numpy(chi).cuda(), torch.from_numpy(v).cuda()
    for stream in (None, torch.cuda.Stream()):
        with torch.cuda.stream(stream) if stream is not None else torch.cuda.stream(torch.cuda.current_stream()):
            w, info = q.wc_from_chi0(d_chi, d_v)
            w2, info2 = q.wc_from_chi0(d_chi, d_v)          # back to back: the first graph is still in flight
        torch.cuda.synchronize()
        for x, i in ((w, info), (w2, info2)):
            assert int(i.item()) == 0
            assert rel_fro_per_freq(x.cpu().numpy(), ref).max() <= TOL_WC
    q.set_global_option("wc_graph", 1)
