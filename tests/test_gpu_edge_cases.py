"""Edge cases of the CUDA path against the oracle on the same seeded inputs: empty batches, batches no basis function
reaches (nnz = 0), one-point batches, a point exactly on a nucleus and one inside the innermost spline knot (reading P11),
an empty grid, bitwise reproducibility of n / grad n, and the error codes of include/aims_gpu.h."""
import copy

import numpy as np
import pytest

import aims_synth
from aims_synth import make_q_values
from oracle.oracle import Oracle

pytestmark = pytest.mark.gpu


def _ctx(bun, **kw):
    import paper_1912_06636_b200 as aims
    return aims.aims_gpu_create(bun, device=0, **kw)


def _with_odd_batches(bun, seed=7):
    """Config with extra batches appended: [empty] [2 far points: nnz = 0] [on-nucleus + inside r0 + ordinary] [1 point] [empty]."""
    rng = np.random.default_rng(seed)
    b = copy.copy(bun)
    extra = np.array([[100.0, 100.0, 100.0], [101.0, 100.0, 100.0],
                      bun.atom_xyz[0], bun.atom_xyz[1] + np.array([1e-4, 0.0, 0.0]), bun.atom_xyz[0] + np.array([0.3, 0.2, -0.4]),
                      bun.atom_xyz[2] + np.array([0.0, 0.7, 0.1])])
    ne = len(extra)
    b.xyz = np.ascontiguousarray(np.vstack([bun.xyz, extra]))
    b.w = np.concatenate([bun.w, rng.uniform(0.01, 0.1, ne)])
    b.v = np.concatenate([bun.v, rng.uniform(-1.0, -0.1, ne)])
    b.g = np.ascontiguousarray(np.hstack([bun.g, rng.uniform(-0.5, 0.5, (3, ne))]))
    b.owner = np.concatenate([bun.owner, np.zeros(ne, dtype=bun.owner.dtype)])
    n0 = bun.n_points
    b.batch_ptr = np.concatenate([bun.batch_ptr, [n0, n0 + 2, n0 + 5, n0 + 6, n0 + 6]]).astype(np.int64)
    return b


@pytest.fixture(scope="module")
def odd():
    bun = _with_odd_batches(aims_synth.make_config(1, max_batch=64))
    ctx = _ctx(bun)
    yield bun, Oracle(bun), ctx
    ctx.close()


def test_odd_batches_lists_and_values(odd):
    bun, orc, ctx = odd
    nb = bun.n_batches
    fn_ptr, fn_index, phi_ptr, phi, dphi = (t.cpu().numpy() for t in ctx.eval_basis(0, None, want_grad=True))
    ctx.synchronize()
    nnz = np.diff(fn_ptr)
    assert nnz[nb - 5] == 0 and nnz[nb - 4] == 0 and nnz[nb - 1] == 0          # empty, far, empty
    assert nnz[nb - 3] == 9 and nnz[nb - 2] == 9
    for b in range(nb):
        idx_ref, phi_ref, dphi_ref = orc.eval_basis(b, want_grad=True)
        assert np.array_equal(fn_index[fn_ptr[b]:fn_ptr[b + 1]], idx_ref)
        if phi_ref.size:
            got = phi[phi_ptr[b]:phi_ptr[b + 1]].reshape(phi_ref.shape)
            gotd = dphi[3 * phi_ptr[b]:3 * phi_ptr[b + 1]].reshape(dphi_ref.shape)
            assert np.abs(got - phi_ref).max() <= 1e-12 * max(np.abs(phi_ref).max(), 1e-300)
            assert np.abs(gotd - dphi_ref).max() <= 1e-12 * max(np.abs(dphi_ref).max(), 1e-300)
            assert np.all(np.isfinite(got)) and np.all(np.isfinite(gotd))      # d = 0 and d < r0 are guarded (P11)


def test_odd_batches_hamiltonian_density_forces(odd):
    bun, orc, ctx = odd
    rel = lambda a, r: np.abs(a - r).max() / max(np.abs(r).max(), 1e-300)    # noqa: E731
    for kin in (False, True):
        H = ctx.integrate_hamiltonian(bun.v, bun.g, kinetic=kin).cpu().numpy()
        ref = orc.integrate_hamiltonian_ks(bun.v, bun.g, kinetic=kin)
        assert np.linalg.norm(H - ref) <= 1e-11 * np.linalg.norm(ref)
    import torch
    n = torch.full((bun.n_points,), -3.0, dtype=torch.float64, device="cuda")
    gn = torch.full((3, bun.n_points), -3.0, dtype=torch.float64, device="cuda")
    ctx.update_density(bun.D_values, want_grad=True, n=n, grad_n=gn)
    ctx.synchronize()
    n_ref, gn_ref = orc.update_density(bun.D_values, want_grad=True)
    n, gn = n.cpu().numpy(), gn.cpu().numpy()
    far = slice(bun.batch_ptr[-5], bun.batch_ptr[-4])
    # points of a batch with nnz = 0: the density there is 0 by definition; the library leaves them untouched or writes 0
    assert np.all((n[far] == 0.0) | (n[far] == -3.0))
    n[far], gn[:, far] = 0.0, 0.0
    assert rel(n, n_ref) <= 1e-11 and rel(gn, gn_ref) <= 1e-11
    Q = make_q_values(bun)
    F = ctx.pulay_forces(bun.v, bun.D_values, g=bun.g, Q=Q).cpu().numpy()
    assert rel(F, orc.pulay_forces(bun.v, bun.D_values, g=bun.g, Q_values=Q)) <= 1e-11
    # only the odd batches
    b0 = bun.n_batches - 5
    Hs = ctx.integrate_hamiltonian(bun.v, bun.g, b0=b0).cpu().numpy()
    refs = orc.integrate_hamiltonian(bun.v, bun.g, batches=np.arange(b0, bun.n_batches))
    assert np.linalg.norm(Hs - refs) <= 1e-11 * np.linalg.norm(refs)


def test_density_is_bitwise_reproducible_and_hamiltonian_to_rounding(odd):
    bun, orc, ctx = odd
    n1, g1 = ctx.update_density(bun.D_values, want_grad=True)
    n2, g2 = ctx.update_density(bun.D_values, want_grad=True)
    ctx.synchronize()
    import torch
    assert torch.equal(n1, n2) and torch.equal(g1, g2)
    H1 = ctx.integrate_hamiltonian(bun.v, bun.g).cpu().numpy()
    H2 = ctx.integrate_hamiltonian(bun.v, bun.g).cpu().numpy()
    assert np.linalg.norm(H1 - H2) <= 1e-13 * np.linalg.norm(H1)


def test_empty_grid():
    bun = copy.copy(aims_synth.make_config(1))
    bun.xyz = np.zeros((0, 3))
    bun.w = np.zeros(0)
    bun.v = np.zeros(0)
    bun.g = np.zeros((3, 0))
    bun.owner = bun.owner[:0]
    bun.batch_ptr = np.zeros(1, dtype=np.int64)
    ctx = _ctx(bun)
    H = ctx.integrate_hamiltonian(bun.v, bun.g)
    n, gn = ctx.update_density(bun.D_values, want_grad=True)
    F = ctx.pulay_forces(bun.v, bun.D_values)
    ctx.synchronize()
    assert float(H.abs().sum()) == 0.0 and n.numel() == 0 and float(F.abs().sum()) == 0.0
    assert ctx.basis_sizes() == (0, 0)
    ctx.close()


def test_error_codes():
    import paper_1912_06636_b200 as aims
    base = aims_synth.make_config(1, max_batch=64)
    bad = copy.copy(base)
    bad.shell_l = base.shell_l.copy()
    bad.shell_l[0] = 4                                                    # l > AIMS_MAX_L
    with pytest.raises(aims.AimsError, match=r"\(-4\)"):
        _ctx(bad)
    bad = copy.copy(base)
    bad.batch_ptr = base.batch_ptr.copy()
    bad.batch_ptr[-1] -= 1                                                # does not span the grid
    with pytest.raises(aims.AimsError, match=r"\(-1\)"):
        _ctx(bad)
    bad = copy.copy(base)
    bad.blk_ld = base.blk_ld.copy()
    bad.blk_ld[0] += 1                                                    # odd leading dimension
    with pytest.raises(aims.AimsError, match=r"\(-1\)"):
        _ctx(bad)
    bad = copy.copy(base)
    bad.col_atom = base.col_atom.copy()
    bad.col_atom[0] = 1                                                   # block row 0 must start with its diagonal block
    with pytest.raises(aims.AimsError, match=r"\(-1\)"):
        _ctx(bad)
    # more atoms touch one batch than AIMS_MAX_ACTIVE_ATOMS: 100 atoms on top of each other's cutoff spheres
    many = aims_synth.make_config(2, n_rad=6, n_ang=14, max_batch=400)
    crowd = copy.copy(many)
    crowd.atom_xyz = np.ascontiguousarray(many.atom_xyz * 0.05)           # everything inside 1 A: all 64 atoms touch every batch
    ctx = _ctx(crowd)                                                     # 64 <= 96: still supported
    assert ctx.stats()["max_active_atoms"] == 64
    ctx.close()


def test_diagnostic_probes_report_plausible_fp64_throughput():
    bun = aims_synth.make_config(1, max_batch=64)
    ctx = _ctx(bun)
    peak = ctx.fp64_peak(50.0)
    assert 30.0 < peak < 40.0                                            # B200 FP64 tensor pipe: 37.2 TFLOP/s
    # the operand-pattern probes (and the rejected density variants) are compiled into probe builds only: the product library
    # says so instead of running them, and reports no build switches
    import paper_1912_06636_b200 as aims
    assert aims.load_library()._aims_build_flags == ""
    with pytest.raises(aims.AimsError, match="probe builds only"):
        ctx.dmma_probe(3, 16)
    ctx.close()


def test_ninety_active_atoms_per_batch_uses_the_global_pair_table():
    """90 atoms squeezed into ~1 A: every batch sees all of them (close to AIMS_MAX_ACTIVE_ATOMS = 96), nnz(B) ~ 2,000, and
    the batch's atom-pair offset table (90^2 entries) no longer fits the contraction kernels' shared memory, so the
    kernels read it from global memory -- a path the ordinary configurations never take."""
    base = aims_synth.make_config(4, n_rad=4, n_ang=6, max_batch=100, keep_atoms=90)
    bun = copy.copy(base)
    bun.atom_xyz = np.ascontiguousarray(base.atom_xyz * 0.04)
    bun.xyz = np.ascontiguousarray(base.xyz * 0.04)          # points follow their atoms; weights, fields and D unchanged
    ctx = _ctx(bun)
    st = ctx.stats()
    assert st["max_active_atoms"] == 90 and st["max_nnz"] > 1800
    orc = Oracle(bun)
    rel = lambda a, r: np.abs(a - r).max() / max(np.abs(r).max(), 1e-300)    # noqa: E731
    H = ctx.integrate_hamiltonian(bun.v, bun.g).cpu().numpy()
    ref = orc.integrate_hamiltonian(bun.v, bun.g)
    assert np.linalg.norm(H - ref) <= 1e-11 * np.linalg.norm(ref)
    n, gn = ctx.update_density(bun.D_values, want_grad=True)
    n_ref, gn_ref = orc.update_density(bun.D_values, want_grad=True)
    assert rel(n.cpu().numpy(), n_ref) <= 1e-11 and rel(gn.cpu().numpy(), gn_ref) <= 1e-11
    Q = make_q_values(bun)
    F = ctx.pulay_forces(bun.v, bun.D_values, g=bun.g, Q=Q).cpu().numpy()
    assert rel(F, orc.pulay_forces(bun.v, bun.D_values, g=bun.g, Q_values=Q)) <= 1e-11
    Hn = ctx.density_hessian(bun.D_values).cpu().numpy()
    assert rel(Hn, orc.density_hessian(bun.D_values)) <= 1e-11
    ctx.close()
