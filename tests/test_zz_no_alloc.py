"""aims_gpu_partition_weights_noalloc: the partition-of-unity weights for programs in which a library may not allocate device
memory -- an MPI rank that shares its GPU through MPS and has spent its memory limit on its own pools, a host whose caching
allocator already owns the HBM (a raw cudaMalloc then fails although the host still has room), a loop that cannot take the
device-wide stall of cudaMalloc / cudaFree.  The call keeps its scratch (cell list of the atoms, device copy of the atom
positions, one flag word) in a fixed array inside libaims_gpu.so instead of allocating it.

What is checked: the call gives what the existing, allocating path (Context.partition_weights) gives on the same inputs, within
the bar tests/test_gpu_partition.py uses for these weights (<= 1e-12 absolute, exact zeros and ones at the same places) --
on several calls IN A ROW with different systems, because every call reuses the one array and finds the previous call's
cell list and flag still in it; that sizes beyond the array are refused with a message that names the limit; and that a call
which raised the device-side flag does not leave it raised for the next one.

This file is named to be collected last: `pytest -x` stops at the first failure, so a failure here must not hide the
parity tests.  It needs nothing from the tests before it and passes alone in a fresh process as well."""
import numpy as np
import pytest

import aims_synth

pytestmark = pytest.mark.gpu

CASES = [(5, dict(n_rad=10, n_ang=26, keep_atoms=60)), (1, {}), (4, dict(n_rad=8, n_ang=26, keep_atoms=80))]


def _same_weights(w, ref):
    assert np.abs(w - ref).max() <= 1e-12
    assert np.array_equal(w == 0.0, ref == 0.0) and np.array_equal(w == 1.0, ref == 1.0)


def test_noalloc_matches_the_allocating_path_on_calls_in_a_row():
    import torch

    import paper_1912_06636_b200 as aims
    # the existing path first, each system through its own context (this is the side that allocates)
    want = []
    for cfg, kw in CASES:
        bun = aims_synth.make_config(cfg, **kw)
        ctx = aims.aims_gpu_create(bun, device=0)
        ref = ctx.partition_weights(bun.xyz, bun.owner, bun.meta["r_part"]).cpu().numpy()
        ctx.synchronize()
        ctx.close()
        want.append((bun, ref))
    # then the no-alloc call, back to back without anything in between: a larger system, a tiny one (its cell list covers
    # only the head of what the first call left in the array), a third one, and the first again
    for bun, ref in want + want[:1]:
        dev = torch.device("cuda", 0)
        x = torch.as_tensor(bun.xyz, dtype=torch.float64).to(dev).contiguous()
        o = torch.as_tensor(bun.owner, dtype=torch.int32).to(dev).contiguous()
        out = torch.full((bun.n_points,), -7.0, dtype=torch.float64, device=dev)      # caller-owned output, poisoned
        got = aims.aims_gpu_partition_weights_noalloc(bun.atom_xyz, x, o, bun.meta["r_part"], w_part=out)
        assert got.data_ptr() == out.data_ptr()
        _same_weights(out.cpu().numpy(), ref)
    # a second radius on the same atoms changes the cell grid under the same array
    bun, _ = want[0]
    ctx = aims.aims_gpu_create(bun, device=0)
    for r_part in (3.0, 6.5):
        ref = ctx.partition_weights(bun.xyz, bun.owner, r_part).cpu().numpy()
        ctx.synchronize()
        _same_weights(aims.aims_gpu_partition_weights_noalloc(bun.atom_xyz, bun.xyz, bun.owner, r_part).cpu().numpy(), ref)
    ctx.close()
    # no points: nothing to do, no error
    assert aims.aims_gpu_partition_weights_noalloc(bun.atom_xyz, np.zeros((0, 3)), np.zeros(0, dtype=np.int32), 5.0).numel() == 0


def test_noalloc_refuses_what_the_array_cannot_hold_and_recovers():
    import ctypes

    import paper_1912_06636_b200 as aims
    from paper_1912_06636_b200 import binding
    hdr = open(binding.HEADER_PATH).read()
    max_atoms = int(hdr.split("#define AIMS_NOALLOC_MAX_ATOMS")[1].split()[0])
    max_cells = int(hdr.split("#define AIMS_NOALLOC_MAX_CELLS")[1].split()[0])
    rng = np.random.default_rng(7)
    pts = rng.uniform(-1.0, 1.0, (64, 3))
    own = np.zeros(64, dtype=np.int32)
    # too many atoms
    with pytest.raises(aims.AimsError, match="AIMS_NOALLOC_MAX_ATOMS"):
        aims.aims_gpu_partition_weights_noalloc(rng.uniform(-50, 50, (max_atoms + 1, 3)), pts, own, 4.0)
    # two atoms far apart with a tiny radius: more cells than the array holds
    far = np.array([[0.0, 0.0, 0.0], [1.0 * (max_cells + 10), 0.0, 0.0]])
    with pytest.raises(aims.AimsError, match="AIMS_NOALLOC_MAX_CELLS"):
        aims.aims_gpu_partition_weights_noalloc(far, pts, own, 1.0)
    # bad arguments are told apart from size limits
    with pytest.raises(aims.AimsError, match=r"\(-1\)"):
        aims.aims_gpu_partition_weights_noalloc(far, pts, own, -1.0)
    # the C entry also works without a message buffer
    L = aims.load_library()
    assert L.aims_gpu_partition_weights_noalloc(0, None, max_atoms + 1, far.ctypes.data_as(ctypes.c_void_p), 0, None, None, 4.0, None,
                                                None, 0) == -4
    # 300 atoms inside one radius: the device raises its flag (more than 256 candidates for a point) and the call reports it ...
    crowd = rng.uniform(-0.5, 0.5, (300, 3))
    with pytest.raises(aims.AimsError, match="more than 256 atoms"):
        aims.aims_gpu_partition_weights_noalloc(crowd, pts, own, 5.0)
    # ... and the flag is not left standing in the shared array: the next call is clean and right (two atoms, closed form:
    # on the bisecting plane both cell functions are equal, so each atom gets 1/2; next to an atom that atom gets 1)
    two = np.array([[-1.0, 0.0, 0.0], [1.0, 0.0, 0.0]])
    probe = np.array([[0.0, 0.3, -0.2], [-1.0, 0.01, 0.0], [1.0, 0.0, 0.01]])
    w = aims.aims_gpu_partition_weights_noalloc(two, probe, np.zeros(3, dtype=np.int32), 6.0).cpu().numpy()
    assert abs(w[0] - 0.5) <= 1e-15 and w[1] == 1.0 and w[2] == 0.0
