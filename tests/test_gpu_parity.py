"""Parity of the CUDA path (through the C ABI, via the ctypes binding) with the CPU oracle, element by element on
the same seeded inputs.  Bars (BASELINE.json north_star):
  nnz(B) index lists            bit-exact
  Phi, grad Phi                 <= 1e-12 max-norm relative
  H, S                          <= 1e-11 relative Frobenius norm over the stored values
  n, grad n                     <= 1e-11 max-norm relative
"""
import numpy as np
import pytest

import aims_synth
from aims_synth import bsr_pad_mask
from oracle.oracle import Oracle

pytestmark = pytest.mark.gpu

TOL_PHI = 1e-12
TOL_H = 1e-11
TOL_N = 1e-11


def _ctx(bun, **kw):
    import paper_1912_06636_b200 as aims
    return aims.aims_gpu_create(bun, device=0, **kw)


def _rel_fro(a, b):
    return np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300)


def _rel_max(a, b):
    return np.abs(a - b).max() / max(np.abs(b).max(), 1e-300)


CASES = {
    # name: (config, overrides) -- sizes the oracle finishes in seconds, several tiles and ragged tails
    "cfg1_full": (1, {}),
    "cfg1_ragged37": (1, dict(max_batch=37)),
    "cfg2_coarse": (2, dict(n_rad=10, n_ang=26)),                 # nnz up to ~700 -> 6x6 tiles of 120
    "cfg3_coarse": (3, dict(n_rad=8, n_ang=26, max_batch=200)),
    "cfg4_toy_b500": (4, dict(n_rad=8, n_ang=38, max_batch=500, keep_atoms=40)),   # batches > 208 points: 3 point tiles
    "cfg5_toy": (5, dict(n_rad=8, n_ang=26, keep_atoms=30)),      # l = 3 shells, two species
}


@pytest.fixture(scope="module", params=list(CASES))
def case(request):
    cfg, kw = CASES[request.param]
    bun = aims_synth.make_config(cfg, **kw)
    ctx = _ctx(bun)
    yield request.param, bun, Oracle(bun), ctx
    ctx.close()


def _sample_batches(bun, k, seed=0):
    rng = np.random.default_rng(seed)
    nb = bun.n_batches
    if nb <= k:
        return np.arange(nb)
    return np.unique(np.concatenate([[0, nb - 1], rng.integers(0, nb, k)]))


def test_eval_basis_lists_bit_exact_and_values(case):
    name, bun, orc, ctx = case
    fn_ptr, fn_index, phi_ptr, phi, dphi = (t.cpu().numpy() for t in ctx.eval_basis(0, None, want_grad=True))
    ctx.synchronize()
    assert fn_ptr[0] == 0 and phi_ptr[0] == 0 and len(fn_ptr) == bun.n_batches + 1
    worst_phi = worst_d = 0.0
    scale_phi = scale_d = 0.0
    sel = _sample_batches(bun, 40)
    for b in range(bun.n_batches):
        idx_ref = orc.batch_nnz(b)[0]
        got = fn_index[fn_ptr[b]:fn_ptr[b + 1]]
        assert np.array_equal(got, idx_ref), "nnz(B) list of batch %d differs" % b       # bit-exact, every batch
    for b in sel:
        idx_ref, phi_ref, dphi_ref = orc.eval_basis(int(b), want_grad=True)
        nnz, npts = phi_ref.shape
        assert phi_ptr[b + 1] - phi_ptr[b] == nnz * npts
        got = phi[phi_ptr[b]:phi_ptr[b + 1]].reshape(nnz, npts)
        gotd = dphi[3 * phi_ptr[b]:3 * phi_ptr[b + 1]].reshape(3, nnz, npts)
        if nnz:
            worst_phi = max(worst_phi, np.abs(got - phi_ref).max())
            worst_d = max(worst_d, np.abs(gotd - dphi_ref).max())
            scale_phi = max(scale_phi, np.abs(phi_ref).max())
            scale_d = max(scale_d, np.abs(dphi_ref).max())
            assert np.array_equal(got == 0.0, phi_ref == 0.0)        # exact zeros beyond the cutoff at the same places
    assert worst_phi <= TOL_PHI * scale_phi
    assert worst_d <= TOL_PHI * scale_d


def test_eval_basis_subrange_and_no_grad(case):
    name, bun, orc, ctx = case
    b0, b1 = bun.n_batches // 3, min(bun.n_batches, bun.n_batches // 3 + 5)
    fn_ptr, fn_index, phi_ptr, phi, dphi = ctx.eval_basis(b0, b1, want_grad=False)
    ctx.synchronize()
    assert dphi is None
    fn_ptr, fn_index, phi_ptr, phi = (t.cpu().numpy() for t in (fn_ptr, fn_index, phi_ptr, phi))
    for k, b in enumerate(range(b0, b1)):
        idx_ref, phi_ref, _ = orc.eval_basis(b)
        assert np.array_equal(fn_index[fn_ptr[k]:fn_ptr[k + 1]], idx_ref)
        got = phi[phi_ptr[k]:phi_ptr[k + 1]].reshape(phi_ref.shape)
        assert np.abs(got - phi_ref).max() <= TOL_PHI * max(np.abs(phi_ref).max(), 1e-300)


@pytest.mark.parametrize("mode", ["lda", "gga", "overlap"])
def test_hamiltonian_matches_oracle(case, mode):
    name, bun, orc, ctx = case
    v = np.ones(bun.n_points) if mode == "overlap" else bun.v
    g = bun.g if mode == "gga" else None
    H = ctx.integrate_hamiltonian(v, g).cpu().numpy()
    ctx.synchronize()
    ref = orc.integrate_hamiltonian(v, g)
    assert _rel_fro(H, ref) <= TOL_H
    assert np.all(H[bsr_pad_mask(bun)] == 0.0)                      # padding columns are never written


@pytest.mark.parametrize("mode", ["kin_lda", "kin_gga", "kin_only", "off"])
def test_hamiltonian_with_kinetic_term_matches_oracle(case, mode):
    """Row f2: (h phi) = -1/2 lap phi + v phi, symmetrised as Fig. 6a's DSYR2K (aims_gpu_integrate_hamiltonian_ks)."""
    name, bun, orc, ctx = case
    v = np.zeros(bun.n_points) if mode == "kin_only" else bun.v
    g = bun.g if mode == "kin_gga" else None
    kin = mode != "off"
    H = ctx.integrate_hamiltonian(v, g, kinetic=kin).cpu().numpy()
    ctx.synchronize()
    ref = orc.integrate_hamiltonian_ks(v, g, kinetic=kin)
    assert _rel_fro(H, ref) <= TOL_H
    assert np.all(H[bsr_pad_mask(bun)] == 0.0)
    if mode == "off":
        assert np.array_equal(H, ctx.integrate_hamiltonian(v, g).cpu().numpy()) or _rel_fro(H, ctx.integrate_hamiltonian(v, g).cpu().numpy()) <= 1e-13


def test_tau_matrix_matches_oracle_and_is_added_to_H(case):
    """Row f2, meta-GGA tau matrix (reading P1c): aims_gpu_add_tau_matrix."""
    name, bun, orc, ctx = case
    xi = aims_synth.make_xi(bun)
    M = ctx.add_tau_matrix(xi).cpu().numpy()
    ctx.synchronize()
    ref = orc.tau_matrix(xi)
    assert _rel_fro(M, ref) <= TOL_H
    assert np.all(M[bsr_pad_mask(bun)] == 0.0)
    H = ctx.integrate_hamiltonian(bun.v, bun.g, kinetic=True)
    mid = bun.n_batches // 2
    ctx.add_tau_matrix(xi, H=H, b0=0, b1=mid)
    ctx.add_tau_matrix(xi, H=H, b0=mid)
    ctx.synchronize()
    full = orc.tau_matrix(xi, H_values=orc.integrate_hamiltonian_ks(bun.v, bun.g, kinetic=True))
    assert _rel_fro(H.cpu().numpy(), full) <= TOL_H


def test_hamiltonian_accumulate_and_subranges(case):
    name, bun, orc, ctx = case
    import torch
    mid = bun.n_batches // 2
    H = torch.zeros(bun.n_values, dtype=torch.float64, device="cuda")
    ctx.integrate_hamiltonian(bun.v, bun.g, H=H, b0=0, b1=mid, accumulate=True)
    ctx.integrate_hamiltonian(bun.v, bun.g, H=H, b0=mid, b1=None, accumulate=True)
    ctx.synchronize()
    ref = orc.integrate_hamiltonian(bun.v, bun.g)
    assert _rel_fro(H.cpu().numpy(), ref) <= TOL_H
    # a sub-range alone equals the oracle on the same batch list (Eq. 28: per-task partial sums)
    part = ctx.integrate_hamiltonian(bun.v, None, b0=mid, b1=min(mid + 3, bun.n_batches)).cpu().numpy()
    ctx.synchronize()
    refp = orc.integrate_hamiltonian(bun.v, None, batches=np.arange(mid, min(mid + 3, bun.n_batches)))
    assert _rel_fro(part, refp) <= TOL_H


@pytest.mark.parametrize("want_grad", [False, True])
def test_density_matches_oracle(case, want_grad):
    name, bun, orc, ctx = case
    n, gn = ctx.update_density(bun.D_values, want_grad=want_grad)
    ctx.synchronize()
    n_ref, gn_ref = orc.update_density(bun.D_values, want_grad=want_grad)
    assert _rel_max(n.cpu().numpy(), n_ref) <= TOL_N
    if want_grad:
        assert _rel_max(gn.cpu().numpy(), gn_ref) <= TOL_N


def test_density_subrange_touches_only_its_points(case):
    name, bun, orc, ctx = case
    import torch
    b0, b1 = 1, min(4, bun.n_batches)
    n = torch.full((bun.n_points,), -7.0, dtype=torch.float64, device="cuda")
    ctx.update_density(bun.D_values, n=n, b0=b0, b1=b1)
    ctx.synchronize()
    n = n.cpu().numpy()
    lo, hi = bun.batch_ptr[b0], bun.batch_ptr[b1]
    assert np.all(n[:lo] == -7.0) and np.all(n[hi:] == -7.0)
    ref, _ = orc.update_density(bun.D_values, batches=np.arange(b0, b1))
    assert _rel_max(n[lo:hi], ref[lo:hi]) <= TOL_N


def test_gpu_outputs_satisfy_trace_identities(case):
    """I1-I3 of SURVEY 8(c) evaluated on the GPU outputs alone (properties that hold at any size)."""
    name, bun, orc, ctx = case
    one = np.ones(bun.n_points)
    S = ctx.integrate_hamiltonian(one).cpu().numpy()
    Hl = ctx.integrate_hamiltonian(bun.v).cpu().numpy()
    Hg = ctx.integrate_hamiltonian(bun.v, bun.g).cpu().numpy()
    n, gn = ctx.update_density(bun.D_values, want_grad=True)
    ctx.synchronize()
    n, gn = n.cpu().numpy(), gn.cpu().numpy()
    # Tr(D M) over the stored upper blocks: off-diagonal blocks count twice
    wgt = np.full(bun.n_values, 2.0)
    for a in range(bun.n_atoms):
        q = bun.row_ptr[a]
        nfa = bun.atom_fn_ptr[a + 1] - bun.atom_fn_ptr[a]
        wgt[bun.blk_off[q]: bun.blk_off[q] + nfa * bun.blk_ld[q]] = 1.0
    tr = lambda M: float((wgt * bun.D_values * M).sum())  # noqa: E731
    scale = max(abs(tr(S)), abs(tr(Hl)), 1.0)
    assert abs((bun.w * n).sum() - tr(S)) <= 1e-10 * scale
    assert abs((bun.w * bun.v * n).sum() - tr(Hl)) <= 1e-10 * scale
    assert abs((bun.w * (bun.g * gn).sum(0)).sum() - tr(Hg - Hl)) <= 1e-10 * scale


def test_empty_range_and_bad_arguments(case):
    name, bun, orc, ctx = case
    import paper_1912_06636_b200 as aims
    H = ctx.integrate_hamiltonian(bun.v, b0=2, b1=2)
    ctx.synchronize()
    assert float(H.abs().max()) == 0.0
    with pytest.raises(aims.AimsError):
        ctx.integrate_hamiltonian(bun.v, b0=0, b1=bun.n_batches + 1)
    with pytest.raises(aims.AimsError):
        ctx.update_density(bun.D_values, b0=3, b1=2)
    assert ctx.launch_count() > 0
