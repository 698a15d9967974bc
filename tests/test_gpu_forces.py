"""Parity of aims_gpu_pulay_forces (Eq. 14-18) with the CPU oracle on the same
seeded inputs, through the C ABI.  Bar: <= 1e-11 max-norm relative over the 3 n_atoms components (the same FP64 bar as
n and grad n: F is the same kind of sum in a different order), written below.  Also a property of the GPU outputs alone:
F_at = -d/dR_at [Tr(n h(R)) - Tr(q s(R))] by central differences of the library's own H and S."""
import copy

import numpy as np
import pytest

import aims_synth
from aims_synth import make_q_values
from oracle.oracle import Oracle

pytestmark = pytest.mark.gpu

TOL_F = 1e-11

CASES = {
    "cfg1_full": (1, {}),
    "cfg1_ragged37": (1, dict(max_batch=37)),
    "cfg3_coarse": (3, dict(n_rad=8, n_ang=26, max_batch=200)),
    "cfg4_toy_b500": (4, dict(n_rad=8, n_ang=38, max_batch=500, keep_atoms=40)),
    "cfg5_toy": (5, dict(n_rad=8, n_ang=26, keep_atoms=30)),
}


def _ctx(bun, **kw):
    import paper_1912_06636_b200 as aims
    return aims.aims_gpu_create(bun, device=0, **kw)


def _rel_max(a, b):
    return np.abs(a - b).max() / max(np.abs(b).max(), 1e-300)


@pytest.fixture(scope="module", params=list(CASES))
def case(request):
    cfg, kw = CASES[request.param]
    bun = aims_synth.make_config(cfg, **kw)
    ctx = _ctx(bun)
    yield request.param, bun, Oracle(bun), ctx, make_q_values(bun)
    ctx.close()


@pytest.mark.parametrize("mode", ["lda", "lda_q", "gga", "gga_q"])
def test_forces_match_oracle(case, mode):
    name, bun, orc, ctx, Q = case
    g = bun.g if mode.startswith("gga") else None
    q = Q if mode.endswith("_q") else None
    F = ctx.pulay_forces(bun.v, bun.D_values, g=g, Q=q).cpu().numpy()
    ctx.synchronize()
    ref = orc.pulay_forces(bun.v, bun.D_values, g=g, Q_values=q)
    assert F.shape == ref.shape == (bun.n_atoms, 3)
    assert _rel_max(F, ref) <= TOL_F


@pytest.mark.parametrize("mode", ["lda", "gga_q"])
def test_forces_with_kinetic_operator_match_oracle(case, mode):
    """Rows f1 + f2: h_KS phi_j of Eq. 16 with -1/2 lap phi_j (aims_gpu_pulay_forces_ks)."""
    name, bun, orc, ctx, Q = case
    g = bun.g if mode.startswith("gga") else None
    q = Q if mode.endswith("_q") else None
    F = ctx.pulay_forces(bun.v, bun.D_values, g=g, Q=q, kinetic=True).cpu().numpy()
    ctx.synchronize()
    ref = orc.pulay_forces(bun.v, bun.D_values, g=g, Q_values=q, kinetic=True)
    assert _rel_max(F, ref) <= TOL_F


def test_forces_accumulate_and_subranges(case):
    name, bun, orc, ctx, Q = case
    import torch
    mid = bun.n_batches // 2
    F = torch.zeros((bun.n_atoms, 3), dtype=torch.float64, device="cuda")
    ctx.pulay_forces(bun.v, bun.D_values, g=bun.g, Q=Q, F=F, b0=0, b1=mid, accumulate=True)
    ctx.pulay_forces(bun.v, bun.D_values, g=bun.g, Q=Q, F=F, b0=mid, b1=None, accumulate=True)
    ctx.synchronize()
    ref = orc.pulay_forces(bun.v, bun.D_values, g=bun.g, Q_values=Q)
    assert _rel_max(F.cpu().numpy(), ref) <= TOL_F
    b1 = min(mid + 3, bun.n_batches)
    part = ctx.pulay_forces(bun.v, bun.D_values, g=bun.g, b0=mid, b1=b1).cpu().numpy()
    ctx.synchronize()
    refp = orc.pulay_forces(bun.v, bun.D_values, g=bun.g, batches=np.arange(mid, b1))
    assert _rel_max(part, refp) <= TOL_F
    empty = ctx.pulay_forces(bun.v, bun.D_values, b0=2, b1=2)
    ctx.synchronize()
    assert float(empty.abs().max()) == 0.0


def test_forces_bad_arguments(case):
    name, bun, orc, ctx, Q = case
    import paper_1912_06636_b200 as aims
    with pytest.raises(aims.AimsError):
        ctx.pulay_forces(bun.v, bun.D_values, b0=0, b1=bun.n_batches + 1)
    with pytest.raises(aims.AimsError):
        ctx.pulay_forces(bun.v[:-1], bun.D_values)
    with pytest.raises(aims.AimsError):
        ctx.pulay_forces(bun.v, bun.D_values, Q=Q[:-2])


def test_gpu_forces_are_the_energy_gradient_of_gpu_H_and_S():
    """Property of the GPU outputs alone: displace one atom by +-h at fixed grid, weights, D, Q, v, g and difference
    Tr(D H) - Tr(Q S) computed by the library itself."""
    bun = aims_synth.make_config(5, n_rad=10, n_ang=26, keep_atoms=8, max_batch=120)
    Q = make_q_values(bun)
    wgt = np.full(bun.n_values, 2.0)
    for a in range(bun.n_atoms):
        q = bun.row_ptr[a]
        nfa = bun.atom_fn_ptr[a + 1] - bun.atom_fn_ptr[a]
        wgt[bun.blk_off[q]: bun.blk_off[q] + nfa * bun.blk_ld[q]] = 1.0

    def energy(b):
        ctx = _ctx(b)
        H = ctx.integrate_hamiltonian(b.v, b.g).cpu().numpy()
        S = ctx.integrate_hamiltonian(np.ones(b.n_points)).cpu().numpy()
        ctx.synchronize()
        ctx.close()
        return float((wgt * (bun.D_values * H - Q * S)).sum())

    ctx = _ctx(bun)
    F = ctx.pulay_forces(bun.v, bun.D_values, g=bun.g, Q=Q).cpu().numpy()
    ctx.synchronize()
    ctx.close()
    h = 1e-4
    scale = np.abs(F).max()
    for at, c in ((0, 0), (3, 1), (7, 2)):
        bp, bm = copy.copy(bun), copy.copy(bun)
        bp.atom_xyz = bun.atom_xyz.copy()
        bm.atom_xyz = bun.atom_xyz.copy()
        bp.atom_xyz[at, c] += h
        bm.atom_xyz[at, c] -= h
        fd = -(energy(bp) - energy(bm)) / (2 * h)
        assert abs(fd - F[at, c]) <= 2e-6 * scale, (at, c, fd, F[at, c])


# ---------------------------------------------------------------------------------------------------------------------
# Pulay stress (row f1, second half; Eq. 20): aims_gpu_pulay_forces_stress
# ---------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("mode", ["lda", "lda_q", "gga", "gga_q", "gga_q_kin"])
def test_stress_and_forces_match_oracle(case, mode):
    name, bun, orc, ctx, Q = case
    g = bun.g if mode.startswith("gga") else None
    q = Q if "_q" in mode else None
    kin = mode.endswith("_kin")
    vol = 37.5
    F, sig = ctx.pulay_forces_stress(bun.v, bun.D_values, g=g, Q=q, volume=vol, kinetic=kin)
    ctx.synchronize()
    ref = orc.pulay_stress(bun.v, bun.D_values, g=g, Q_values=q, kinetic=kin, volume=vol)
    assert sig.shape == (3, 3)
    assert _rel_max(sig.cpu().numpy(), ref) <= TOL_F
    assert _rel_max(F.cpu().numpy(), orc.pulay_forces(bun.v, bun.D_values, g=g, Q_values=q, kinetic=kin)) <= TOL_F


def test_stress_only_subranges_and_accumulation(case):
    import torch
    name, bun, orc, ctx, Q = case
    mid = bun.n_batches // 2
    sig = torch.zeros((3, 3), dtype=torch.float64, device="cuda")
    F = torch.zeros((bun.n_atoms, 3), dtype=torch.float64, device="cuda")
    ctx.pulay_forces_stress(bun.v, bun.D_values, g=bun.g, Q=Q, F=F, sigma=sig, b0=0, b1=mid, accumulate=True)
    ctx.pulay_forces_stress(bun.v, bun.D_values, g=bun.g, Q=Q, F=None, sigma=sig, b0=mid, b1=None, accumulate=True,
                            want_forces=False)                                    # stress only: F = NULL
    ctx.synchronize()
    assert _rel_max(sig.cpu().numpy(), orc.pulay_stress(bun.v, bun.D_values, g=bun.g, Q_values=Q)) <= TOL_F
    assert _rel_max(F.cpu().numpy(), orc.pulay_forces(bun.v, bun.D_values, g=bun.g, Q_values=Q, batches=np.arange(0, mid))) <= TOL_F
    import paper_1912_06636_b200 as aims
    with pytest.raises(aims.AimsError):
        ctx.pulay_forces_stress(bun.v, bun.D_values, volume=0.0)


def test_stress_far_from_the_origin_loses_nothing():
    """The kernel sums (r_p - c) and (R_at - c) relative to a point of the batch: translating the whole system by 1000 A must
    not cost digits beyond the rounding of the translated coordinates themselves."""
    bun = aims_synth.make_config(5, n_rad=8, n_ang=26, keep_atoms=12)
    Q = make_q_values(bun)
    t = np.array([1024.0, -2048.0, 512.0])                     # exactly representable shifts
    far = copy.copy(bun)
    far.atom_xyz = np.ascontiguousarray(bun.atom_xyz + t)
    far.xyz = np.ascontiguousarray(bun.xyz + t)
    ctx = _ctx(far)
    _, sig = ctx.pulay_forces_stress(far.v, far.D_values, g=far.g, Q=Q)
    ctx.synchronize()
    ref = Oracle(far).pulay_stress(far.v, far.D_values, g=far.g, Q_values=Q)
    assert _rel_max(sig.cpu().numpy(), ref) <= TOL_F
    ctx.close()
