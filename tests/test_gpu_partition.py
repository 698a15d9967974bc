"""Row f4 (partition-of-unity factor of the integration weights, Eq. 21-22, reading P5) on the GPU:
aims_gpu_partition_weights against the oracle on the same seeded inputs.  Bar: <= 1e-12 absolute (the weights lie in
[0, 1]; both sides multiply the same cell-function values in a different order), exact zeros and ones at the same places."""
import numpy as np
import pytest

import aims_synth
from oracle.oracle import Oracle

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("cfg,kw", [(1, {}), (5, dict(n_rad=10, n_ang=26, keep_atoms=60)), (4, dict(n_rad=8, n_ang=26, keep_atoms=80))])
def test_partition_weights_match_oracle(cfg, kw):
    import paper_1912_06636_b200 as aims
    bun = aims_synth.make_config(cfg, **kw)
    ctx = aims.aims_gpu_create(bun, device=0)
    r_part = bun.meta["r_part"]
    w = ctx.partition_weights(bun.xyz, bun.owner, r_part).cpu().numpy()
    ctx.synchronize()
    ref = Oracle(bun).partition_weights(bun.xyz, bun.owner, r_part)
    assert np.abs(w - ref).max() <= 1e-12
    assert np.array_equal(w == 0.0, ref == 0.0) and np.array_equal(w == 1.0, ref == 1.0)
    # a property of the GPU output alone: the weights of all owners sum to one at every point
    pts = bun.xyz[:: max(1, bun.n_points // 300)]
    tot = sum(ctx.partition_weights(pts, np.full(len(pts), a, dtype=np.int32), r_part).cpu().numpy() for a in range(bun.n_atoms))
    assert np.abs(tot - 1.0).max() <= 1e-13
    # empty input and bad arguments
    assert ctx.partition_weights(np.zeros((0, 3)), np.zeros(0, dtype=np.int32), r_part).numel() == 0
    with pytest.raises(aims.AimsError):
        ctx.partition_weights(bun.xyz[:5], bun.owner[:5], -1.0)
    ctx.close()


def test_partition_weights_candidate_overflow_is_reported_by_the_call():
    """More than 256 atoms within r_part of a point: the call itself returns AIMS_ERR_UNSUPPORTED (include/aims_gpu.h), and the
    next call with a sane radius -- another cell list in the same context buffer -- is right again."""
    import paper_1912_06636_b200 as aims
    bun = aims_synth.make_config(5, n_rad=6, n_ang=14)
    assert bun.n_atoms > 256
    ctx = aims.aims_gpu_create(bun, device=0)
    pts, own = bun.xyz[:200], bun.owner[:200]
    with pytest.raises(aims.AimsError, match="more than 256 atoms"):
        ctx.partition_weights(pts, own, 1.0e3)
    ctx.synchronize()                                  # nothing left flagged for later
    r_part = bun.meta["r_part"]
    ref = Oracle(bun).partition_weights(pts, own, r_part)
    for _ in range(2):                                 # second pass runs on the cached cell list
        w = ctx.partition_weights(pts, own, r_part).cpu().numpy()
        assert np.abs(w - ref).max() <= 1e-12
    ctx.close()
