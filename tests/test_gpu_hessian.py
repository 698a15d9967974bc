"""Parity of aims_gpu_density_hessian with the CPU oracle on the same seeded inputs,
through the C ABI.  Bar: <= 1e-11 max-norm relative over the 6 n_points components (the same FP64 bar as n and grad n)."""
import numpy as np
import pytest

import aims_synth
from oracle.oracle import Oracle

pytestmark = pytest.mark.gpu

TOL = 1e-11

CASES = {
    "cfg1_full": (1, {}),
    "cfg1_ragged37": (1, dict(max_batch=37)),
    "cfg3_coarse": (3, dict(n_rad=8, n_ang=26, max_batch=200)),
    "cfg4_toy_b500": (4, dict(n_rad=8, n_ang=38, max_batch=500, keep_atoms=40)),
    "cfg5_toy": (5, dict(n_rad=8, n_ang=26, keep_atoms=30)),
}


@pytest.fixture(scope="module", params=list(CASES))
def case(request):
    import paper_1912_06636_b200 as aims
    cfg, kw = CASES[request.param]
    bun = aims_synth.make_config(cfg, **kw)
    ctx = aims.aims_gpu_create(bun, device=0)
    yield request.param, bun, Oracle(bun), ctx
    ctx.close()


def test_density_hessian_matches_oracle(case):
    name, bun, orc, ctx = case
    Hn = ctx.density_hessian(bun.D_values).cpu().numpy()
    ctx.synchronize()
    ref = orc.density_hessian(bun.D_values)
    assert Hn.shape == ref.shape == (6, bun.n_points)
    assert np.abs(Hn - ref).max() <= TOL * np.abs(ref).max()


def test_density_hessian_subrange_reproducible_and_trace(case):
    name, bun, orc, ctx = case
    import torch
    b0, b1 = 1, min(4, bun.n_batches)
    Hn = torch.full((6, bun.n_points), -7.0, dtype=torch.float64, device="cuda")
    ctx.density_hessian(bun.D_values, hess_n=Hn, b0=b0, b1=b1)
    ctx.synchronize()
    Hn = Hn.cpu().numpy()
    lo, hi = bun.batch_ptr[b0], bun.batch_ptr[b1]
    assert np.all(Hn[:, :lo] == -7.0) and np.all(Hn[:, hi:] == -7.0)
    ref = orc.density_hessian(bun.D_values, batches=np.arange(b0, b1))
    assert np.abs(Hn[:, lo:hi] - ref[:, lo:hi]).max() <= TOL * np.abs(ref).max()
    H1 = ctx.density_hessian(bun.D_values)
    H2 = ctx.density_hessian(bun.D_values)
    ctx.synchronize()
    assert torch.equal(H1, H2)                                               # no atomics: bitwise reproducible
    with pytest.raises(Exception):
        ctx.density_hessian(bun.D_values[:-2])
