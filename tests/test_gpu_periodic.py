"""Row f3 (periodic boundary conditions, Eq. 6-12) on the GPU: the real-space calls run unchanged on a periodic
bundle (cell atoms + images, points mapped into the cell), and aims_gpu_bloch_fold forms h_ij(k), s_ij(k).  Parity with the
oracle on the same seeded inputs: H^uc, S^uc <= 1e-11 relative Frobenius norm, n / grad n <= 1e-11 max-norm relative,
folded matrices <= 1e-11 relative Frobenius norm; plus properties of the GPU outputs alone."""
import numpy as np
import pytest

import aims_synth
from oracle.oracle import Oracle

pytestmark = pytest.mark.gpu

KPTS = [np.zeros(3), np.array([0.31, -0.17, 0.23]), np.array([0.7, 0.2, -0.4])]


@pytest.fixture(scope="module")
def per():
    import paper_1912_06636_b200 as aims
    bun = aims_synth.make_periodic(n_rad=20, n_ang=38, max_batch=100)
    ctx = aims.aims_gpu_create(bun, device=0)
    yield bun, Oracle(bun), ctx
    ctx.close()


def _rel_fro(a, b):
    return np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300)


def test_real_space_calls_run_unchanged_on_the_periodic_bundle(per):
    bun, orc, ctx = per
    fn_ptr, fn_index, _, _, _ = (t.cpu().numpy() if t is not None else None for t in ctx.eval_basis(0, None))
    for b in range(bun.n_batches):
        assert np.array_equal(fn_index[fn_ptr[b]:fn_ptr[b + 1]], orc.batch_nnz(b)[0])
    H = ctx.integrate_hamiltonian(bun.v, bun.g, kinetic=True).cpu().numpy()
    assert _rel_fro(H, orc.integrate_hamiltonian_ks(bun.v, bun.g, kinetic=True)) <= 1e-11
    n, gn = ctx.update_density(bun.D_values, want_grad=True)
    ctx.synchronize()
    n_ref, gn_ref = orc.update_density(bun.D_values, want_grad=True)
    assert np.abs(n.cpu().numpy() - n_ref).max() <= 1e-11 * np.abs(n_ref).max()
    assert np.abs(gn.cpu().numpy() - gn_ref).max() <= 1e-11 * np.abs(gn_ref).max()


def test_bloch_fold_matches_oracle_and_is_hermitian(per):
    bun, orc, ctx = per
    nhb = int(bun.atom_fn_ptr[bun.n_home])
    S_uc = ctx.integrate_hamiltonian(np.ones(bun.n_points))
    H_uc = ctx.integrate_hamiltonian(bun.v, bun.g)
    ctx.synchronize()
    S_ref_uc, H_ref_uc = orc.integrate_hamiltonian(np.ones(bun.n_points)), orc.integrate_hamiltonian(bun.v, bun.g)
    for k in KPTS:
        S = ctx.bloch_fold(S_uc, bun.atom_home, bun.atom_T, bun.n_home, k, nhb).cpu().numpy()
        H = ctx.bloch_fold(H_uc, bun.atom_home, bun.atom_T, bun.n_home, k, nhb).cpu().numpy()
        assert _rel_fro(S, orc.bloch_fold(S_ref_uc, bun.atom_home, bun.atom_T, bun.n_home, k)) <= 1e-11
        assert _rel_fro(H, orc.bloch_fold(H_ref_uc, bun.atom_home, bun.atom_T, bun.n_home, k)) <= 1e-11
        assert np.abs(S - S.conj().T).max() <= 1e-13 * np.abs(S).max()
        assert np.linalg.eigvalsh(0.5 * (S + S.conj().T)).min() > 0.0
        if not k.any():
            assert np.abs(S.imag).max() == 0.0


def test_bloch_fold_bad_arguments(per):
    bun, orc, ctx = per
    import paper_1912_06636_b200 as aims
    nhb = int(bun.atom_fn_ptr[bun.n_home])
    H = ctx.integrate_hamiltonian(bun.v)
    bad_home = bun.atom_home.copy()
    bad_home[3] = bun.n_home                                  # not a cell atom
    with pytest.raises(aims.AimsError):
        ctx.bloch_fold(H, bad_home, bun.atom_T, bun.n_home, KPTS[1], nhb)
    with pytest.raises(aims.AimsError):
        ctx.bloch_fold(H, bun.atom_home, bun.atom_T, 0, KPTS[1], nhb)
