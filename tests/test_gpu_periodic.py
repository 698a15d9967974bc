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


# ---- geometry of reading P23 behind the boundary: image enumeration and the point map
@pytest.mark.parametrize("case", ["toy", "si54"])
def test_periodic_images_and_point_wrap_are_bit_exact(case):
    import paper_1912_06636_b200 as aims
    from oracle.periodic import periodic_images, wrap_points
    bun = aims_synth.make_periodic(n_rad=12, n_ang=26) if case == "toy" else aims_synth.make_periodic_si(n_rad=16, n_ang=38, max_batch=16)
    for reach in (bun.rcut, 0.0, 2.5 * bun.rcut):
        home, n = aims.aims_gpu_periodic_images(bun.lattice, bun.frac, reach)
        home_ref, n_ref = periodic_images(bun.lattice, bun.frac, reach)
        assert np.array_equal(home, home_ref) and np.array_equal(n, n_ref)
    w = aims.aims_gpu_wrap_points(bun.lattice, bun.xyz_unwrapped).cpu().numpy()
    assert np.array_equal(w, wrap_points(bun.lattice, bun.xyz_unwrapped))            # separately rounded operations: one result
    # points a hair below a cell face, on faces and on lattice translates of the origin: f - floor(f) rounds to 1.0 for the first
    # kind, and both sides put those on f = 0 (reading P23: [0, 1)); cubic cell, so the expected coordinates are exact
    cube = 4.0 * np.eye(3)
    edge_pts = np.array([[-1e-20, 1.0, 2.0], [1.0, -1e-20, -1e-20], [4.0, 8.0, -4.0], [-1.0, 5.0, 3.5], [-4.0 * 2.0 ** -60, 0.5, 0.5]])
    we = aims.aims_gpu_wrap_points(cube, edge_pts).cpu().numpy()
    assert np.array_equal(we, wrap_points(cube, edge_pts))
    assert np.array_equal(we, np.array([[0.0, 1.0, 2.0], [1.0, 0.0, 0.0], [0.0, 0.0, 0.0], [3.0, 1.0, 3.5], [0.0, 0.5, 0.5]]))
    hair = bun.xyz_unwrapped[:64] * 0.0 - 1e-18 * bun.lattice.sum(axis=0)              # a hair outside the corner of the real cell
    wh = aims.aims_gpu_wrap_points(bun.lattice, hair).cpu().numpy()
    assert np.array_equal(wh, wrap_points(bun.lattice, hair))
    # degenerate inputs
    assert aims.aims_gpu_wrap_points(bun.lattice, np.zeros((0, 3))).shape[0] == 0
    with pytest.raises(aims.AimsError):
        aims.aims_gpu_wrap_points(np.array([[1.0, 0, 0], [2.0, 0, 0], [0, 0, 1.0]]), bun.xyz_unwrapped[:4])   # singular lattice
    # the library consumes what it produced: a context over (images, wrapped points) has the oracle's lists
    import copy
    b2 = copy.copy(bun)
    home, n = aims.aims_gpu_periodic_images(bun.lattice, bun.frac, bun.rcut)
    b2.atom_xyz = np.ascontiguousarray((bun.frac[home] + n) @ bun.lattice)
    b2.xyz = np.ascontiguousarray(w)
    assert np.abs(b2.atom_xyz - bun.atom_xyz).max() < 1e-12
    ctx = aims.aims_gpu_create(b2, device=0)
    orc = Oracle(b2)
    nnz = ctx.batch_nnz()
    for b in range(0, b2.n_batches, max(1, b2.n_batches // 12)):
        assert nnz[b] == len(orc.batch_nnz(b)[0])
    ctx.close()


def test_si54_supercell_at_full_size_on_sampled_batches():
    """The periodic workload shaped like the paper's main benchmark (54-atom diamond-Si supercell, config-2 basis,
    60 x 302 points per atom, batches of <= 200): whole-grid calls as bench.py --config 6 launches them; lists, n / grad n and
    H^uc restricted to a seeded sample of batches against the oracle; Bloch sums at Gamma and one general k."""
    import torch
    import paper_1912_06636_b200 as aims
    bun = aims_synth.make_periodic_si()
    assert bun.n_home == 54 and bun.n_points == 54 * 60 * 302
    ctx = aims.aims_gpu_create(bun, device=0)
    orc = Oracle(bun)
    nnz = ctx.batch_nnz()
    rng = np.random.default_rng(54)
    sel = np.unique(np.concatenate([[0, bun.n_batches - 1, int(np.argmax(nnz)), int(np.argmin(nnz))],
                                    rng.integers(0, bun.n_batches, 12)])).astype(np.int32)
    for b in sel:
        _, fn_index, _, _, _ = ctx.eval_basis(int(b), int(b) + 1, want_grad=False)
        assert np.array_equal(fn_index.cpu().numpy(), orc.batch_nnz(int(b))[0])
    n, gn = ctx.update_density(bun.D_values, want_grad=True)                       # whole grid
    vd, gd = torch.as_tensor(bun.v).cuda(), torch.as_tensor(bun.g).cuda()
    H = torch.zeros(bun.n_values, dtype=torch.float64, device="cuda")
    for b in sel:
        ctx.integrate_hamiltonian(vd, gd, H=H, b0=int(b), b1=int(b) + 1, accumulate=True)
    ctx.synchronize()
    n_ref, gn_ref = orc.update_density(bun.D_values, want_grad=True, batches=sel)
    idx = np.concatenate([np.arange(bun.batch_ptr[b], bun.batch_ptr[b + 1]) for b in sel])
    assert np.abs(n.cpu().numpy()[idx] - n_ref[idx]).max() <= 1e-11 * np.abs(n_ref[idx]).max()
    assert np.abs(gn.cpu().numpy()[:, idx] - gn_ref[:, idx]).max() <= 1e-11 * np.abs(gn_ref[:, idx]).max()
    H_ref = orc.integrate_hamiltonian(bun.v, bun.g, batches=sel)
    assert _rel_fro(H.cpu().numpy(), H_ref) <= 1e-11
    nhb = int(bun.atom_fn_ptr[bun.n_home])
    for k in (np.zeros(3), np.array([0.11, -0.07, 0.05])):
        Hk = ctx.bloch_fold(H, bun.atom_home, bun.atom_T, bun.n_home, k, nhb).cpu().numpy()
        assert _rel_fro(Hk, orc.bloch_fold(H_ref, bun.atom_home, bun.atom_T, bun.n_home, k)) <= 1e-11
        assert np.abs(Hk - Hk.conj().T).max() <= 1e-12 * np.abs(Hk).max()
    # whole-grid overlap folded at Gamma: Hermitian and positive definite (a property of the GPU outputs alone)
    S = ctx.integrate_hamiltonian(np.ones(bun.n_points))
    Sk = ctx.bloch_fold(S, bun.atom_home, bun.atom_T, bun.n_home, np.zeros(3), nhb).cpu().numpy()
    assert np.linalg.eigvalsh(0.5 * (Sk + Sk.conj().T)).min() > 0.0
    ctx.close()


def test_forces_stress_and_density_hessian_on_the_periodic_bundle(per):
    """The widened rows run unchanged on a periodic bundle too ("the exact same real-space integration code"):
    Pulay forces on all periodic atoms, the Pulay stress with the cell volume (Eq. 20: sigma = (1/V) dE/d eps), hess n."""
    from aims_synth import make_q_values
    bun, orc, ctx = per
    Q = make_q_values(bun)
    vol = abs(float(np.linalg.det(bun.lattice)))
    F, sig = ctx.pulay_forces_stress(bun.v, bun.D_values, g=bun.g, Q=Q, volume=vol, kinetic=True)
    Hn = ctx.density_hessian(bun.D_values)
    ctx.synchronize()
    F_ref = orc.pulay_forces(bun.v, bun.D_values, g=bun.g, Q_values=Q, kinetic=True)
    sig_ref = orc.pulay_stress(bun.v, bun.D_values, g=bun.g, Q_values=Q, kinetic=True, volume=vol)
    Hn_ref = orc.density_hessian(bun.D_values)
    assert np.abs(F.cpu().numpy() - F_ref).max() <= 1e-11 * np.abs(F_ref).max()
    assert np.abs(sig.cpu().numpy() - sig_ref).max() <= 1e-11 * np.abs(sig_ref).max()
    assert np.abs(Hn.cpu().numpy() - Hn_ref).max() <= 1e-11 * np.abs(Hn_ref).max()
    # forces of the images fold onto their cell atoms: sum over images of one cell atom is what a periodic code reports
    F_home = np.zeros((bun.n_home, 3))
    np.add.at(F_home, bun.atom_home, F.cpu().numpy())
    F_home_ref = np.zeros((bun.n_home, 3))
    np.add.at(F_home_ref, bun.atom_home, F_ref)
    assert np.abs(F_home - F_home_ref).max() <= 1e-11 * np.abs(F_ref).max()
