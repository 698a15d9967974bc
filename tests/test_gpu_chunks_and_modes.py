"""Launch configurations the other parity files do not reach:
  * a SMALL workspace_bytes, so that every call streams its Phi planes through several chunks (aims_gpu.cu: chunk_end) on
    configs the oracle checks element by element -- H (LDA, GGA, kinetic, tau), n / grad n, Pulay forces, stress, hess n;
  * the ordered scatter of aims_gpu_set_deterministic: bit-identical reruns of H, same numbers as the default path;
  * two contexts alive at once (the dynamic shared-memory opt-in is per function and device, not per context);
  * a single tiny batch with the tau matrix (the 6-plane layout sizes the workspace);
  * more than AIMS_MAX_ACTIVE_ATOMS atoms touching one batch -> AIMS_ERR_UNSUPPORTED from aims_gpu_create.
Bars as in test_gpu_parity.py: 1e-11 relative Frobenius (H), 1e-11 max-norm relative (n, grad n, F, sigma, hess n).
"""
import copy

import numpy as np
import pytest

import aims_synth
from aims_synth import make_q_values, make_xi
from oracle.oracle import Oracle

pytestmark = pytest.mark.gpu

TOL = 1e-11


def _ctx(bun, **kw):
    import paper_1912_06636_b200 as aims
    return aims.aims_gpu_create(bun, device=0, **kw)


def _rel_fro(a, b):
    return np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300)


def _rel_max(a, b):
    return np.abs(a - b).max() / max(np.abs(b).max(), 1e-300)


CHUNKED = {
    "cfg3_coarse": (3, dict(n_rad=8, n_ang=26, max_batch=200)),
    "cfg5_toy": (5, dict(n_rad=8, n_ang=26, keep_atoms=30)),
    "cfg4_toy_b500": (4, dict(n_rad=8, n_ang=38, max_batch=500, keep_atoms=40)),
}


@pytest.fixture(scope="module", params=list(CHUNKED))
def chunked(request):
    cfg, kw = CHUNKED[request.param]
    bun = aims_synth.make_config(cfg, **kw)
    ctx = _ctx(bun, workspace_bytes=1)            # clamped up to "one batch in every plane layout": the smallest legal workspace
    yield request.param, bun, Oracle(bun), ctx
    ctx.close()


def _launches(ctx, fn):
    n0 = ctx.launch_count()
    out = fn()
    ctx.synchronize()
    return out, ctx.launch_count() - n0


def test_hamiltonian_variants_in_many_chunks(chunked):
    name, bun, orc, ctx = chunked
    assert bun.n_batches >= 8
    for g, kin in ((None, False), (bun.g, False), (bun.g, True), (None, True)):
        H, nl = _launches(ctx, lambda: ctx.integrate_hamiltonian(bun.v, g, kinetic=kin))
        assert nl >= 1 + 2 * 3, "expected >= 3 chunks (k_cull + 3 x (k_eval, k_hamiltonian)), saw %d launches" % nl
        ref = orc.integrate_hamiltonian_ks(bun.v, g, kinetic=kin)
        assert _rel_fro(H.cpu().numpy(), ref) <= TOL
    xi = make_xi(bun)
    Ht, nl = _launches(ctx, lambda: ctx.add_tau_matrix(xi))
    assert nl >= 1 + 2 * 3
    assert _rel_fro(Ht.cpu().numpy(), orc.tau_matrix(xi)) <= TOL


def test_density_forces_hessian_in_many_chunks(chunked):
    name, bun, orc, ctx = chunked
    (n, gn), nl = _launches(ctx, lambda: ctx.update_density(bun.D_values, want_grad=True))
    assert nl >= 1 + 2 * 3
    n_ref, gn_ref = orc.update_density(bun.D_values, want_grad=True)
    assert _rel_max(n.cpu().numpy(), n_ref) <= TOL and _rel_max(gn.cpu().numpy(), gn_ref) <= TOL
    (n1, _), nl = _launches(ctx, lambda: ctx.update_density(bun.D_values, want_grad=False))
    assert _rel_max(n1.cpu().numpy(), n_ref) <= TOL
    Q = make_q_values(bun)
    F, nl = _launches(ctx, lambda: ctx.pulay_forces(bun.v, bun.D_values, g=bun.g, Q=Q))
    assert nl >= 1 + 2 * 3
    assert _rel_max(F.cpu().numpy(), orc.pulay_forces(bun.v, bun.D_values, g=bun.g, Q_values=Q)) <= TOL
    Hn, nl = _launches(ctx, lambda: ctx.density_hessian(bun.D_values))
    assert nl >= 1 + 2 * 3
    assert _rel_max(Hn.cpu().numpy(), orc.density_hessian(bun.D_values)) <= TOL


def test_chunked_equals_unchunked_density_bitwise(chunked):
    """n, grad n are reduced without atomics: chunk boundaries must not change a single bit."""
    import torch
    name, bun, orc, ctx = chunked
    big = _ctx(bun)
    n0, g0 = big.update_density(bun.D_values, want_grad=True)
    n1, g1 = ctx.update_density(bun.D_values, want_grad=True)
    big.synchronize(); ctx.synchronize()
    assert torch.equal(n0, n1) and torch.equal(g0, g1)
    big.close()


@pytest.mark.parametrize("case", ["cfg3_coarse", "cfg5_toy"])
def test_deterministic_mode_is_bitwise_reproducible(case):
    import torch
    cfg, kw = CHUNKED[case]
    bun = aims_synth.make_config(cfg, **kw)
    orc = Oracle(bun)
    for ws in (0, 1):                                    # one chunk, and many chunks
        ctx = _ctx(bun, workspace_bytes=ws)
        ctx.set_deterministic(True)
        xi = make_xi(bun)
        runs = []
        for _ in range(3):
            H = ctx.integrate_hamiltonian(bun.v, bun.g, kinetic=True)
            ctx.add_tau_matrix(xi, H=H)
            Hl = ctx.integrate_hamiltonian(bun.v)
            ctx.synchronize()
            runs.append((H.clone(), Hl.clone()))
        for H, Hl in runs[1:]:
            assert torch.equal(H, runs[0][0]) and torch.equal(Hl, runs[0][1])
        ref = orc.tau_matrix(xi, H_values=orc.integrate_hamiltonian_ks(bun.v, bun.g, kinetic=True))
        assert _rel_fro(runs[0][0].cpu().numpy(), ref) <= TOL
        assert _rel_fro(runs[0][1].cpu().numpy(), orc.integrate_hamiltonian(bun.v, None)) <= TOL
        # sub-ranges accumulate in the same fixed order
        H2 = torch.zeros(bun.n_values, dtype=torch.float64, device="cuda")
        mid = bun.n_batches // 3
        ctx.integrate_hamiltonian(bun.v, bun.g, H=H2, b0=0, b1=mid, accumulate=True, kinetic=True)
        ctx.integrate_hamiltonian(bun.v, bun.g, H=H2, b0=mid, b1=bun.n_batches, accumulate=True, kinetic=True)
        ctx.synchronize()
        assert _rel_fro(H2.cpu().numpy(), orc.integrate_hamiltonian_ks(bun.v, bun.g, kinetic=True)) <= TOL
        ctx.set_deterministic(False)
        Hd = ctx.integrate_hamiltonian(bun.v, bun.g, kinetic=True)
        ctx.synchronize()
        assert _rel_fro(Hd.cpu().numpy(), orc.integrate_hamiltonian_ks(bun.v, bun.g, kinetic=True)) <= TOL
        ctx.close()


def test_two_contexts_alive_large_then_small_then_large_again():
    """the dynamic shared-memory attribute is per function and device; a second, smaller context must not
    shrink it under the first one."""
    big_bun = aims_synth.make_config(5, n_rad=8, n_ang=26, keep_atoms=30)         # nnz up to ~700
    small_bun = aims_synth.make_config(1, max_batch=64)                           # nnz = 9
    big = _ctx(big_bun)
    ref_n, ref_g = Oracle(big_bun).update_density(big_bun.D_values, want_grad=True)
    n0, _ = big.update_density(big_bun.D_values, want_grad=True)
    small = _ctx(small_bun)
    ns, _ = small.update_density(small_bun.D_values, want_grad=True)
    H = big.integrate_hamiltonian(big_bun.v, big_bun.g)                           # the large context again
    n1, g1 = big.update_density(big_bun.D_values, want_grad=True)
    F = big.pulay_forces(big_bun.v, big_bun.D_values, g=big_bun.g)
    Hn = big.density_hessian(big_bun.D_values)
    big.synchronize(); small.synchronize()
    assert _rel_max(n1.cpu().numpy(), ref_n) <= TOL and _rel_max(g1.cpu().numpy(), ref_g) <= TOL
    assert _rel_max(ns.cpu().numpy(), Oracle(small_bun).update_density(small_bun.D_values)[0]) <= TOL
    assert _rel_fro(H.cpu().numpy(), Oracle(big_bun).integrate_hamiltonian(big_bun.v, big_bun.g)) <= TOL
    assert np.isfinite(F.cpu().numpy()).all() and np.isfinite(Hn.cpu().numpy()).all()
    small.close(); big.close()


def test_single_tiny_batch_with_tau_matrix():
    """One 5-point batch: the tau matrix's 6 planes of pad8(nnz) x 16 padded points exceed 10 planes of the density layout
    (round_up(nnz,16) x 8 points); the workspace must be sized for the largest layout."""
    base = aims_synth.make_config(5, n_rad=8, n_ang=26, keep_atoms=6)
    bun = copy.copy(base)
    keep = slice(int(base.batch_ptr[3]), int(base.batch_ptr[3]) + 5)
    bun.xyz = np.ascontiguousarray(base.xyz[keep]); bun.w = base.w[keep].copy(); bun.v = base.v[keep].copy()
    bun.g = np.ascontiguousarray(base.g[:, keep]); bun.owner = base.owner[keep].copy()
    bun.batch_ptr = np.array([0, 5], dtype=np.int64)
    ctx = _ctx(bun, workspace_bytes=1)
    orc = Oracle(bun)
    xi = make_xi(bun)
    H = ctx.integrate_hamiltonian(bun.v, bun.g, kinetic=True)
    ctx.add_tau_matrix(xi, H=H)
    n, gn = ctx.update_density(bun.D_values, want_grad=True)
    Hn = ctx.density_hessian(bun.D_values)
    ctx.synchronize()
    ref = orc.tau_matrix(xi, H_values=orc.integrate_hamiltonian_ks(bun.v, bun.g, kinetic=True))
    assert _rel_fro(H.cpu().numpy(), ref) <= TOL
    n_ref, gn_ref = orc.update_density(bun.D_values, want_grad=True)
    assert _rel_max(n.cpu().numpy(), n_ref) <= TOL and _rel_max(gn.cpu().numpy(), gn_ref) <= TOL
    assert _rel_max(Hn.cpu().numpy(), orc.density_hessian(bun.D_values)) <= TOL
    ctx.close()


def test_more_than_max_active_atoms_is_refused():
    """100 atoms squeezed into ~1 A: every batch is touched by all of them, 100 > AIMS_MAX_ACTIVE_ATOMS = 96."""
    import paper_1912_06636_b200 as aims
    base = aims_synth.make_config(4, n_rad=4, n_ang=6, max_batch=100, keep_atoms=100)
    bun = copy.copy(base)
    bun.atom_xyz = np.ascontiguousarray(base.atom_xyz * 0.04)
    bun.xyz = np.ascontiguousarray(base.xyz * 0.04)
    with pytest.raises(aims.AimsError, match=r"\(-4\).*AIMS_MAX_ACTIVE_ATOMS"):
        _ctx(bun)
    # a device-side flag is reported once by synchronize and then cleared
    ok = aims_synth.make_config(1, max_batch=64)
    ctx = _ctx(ok)
    ctx.synchronize()
    ctx.synchronize()
    ctx.close()
