"""CPU-side checks (-m "not gpu"): the C-ABI library builds, loads and exports every symbol include/aims_gpu.h
declares (no compute calls without a GPU); the product path fails loudly without a CUDA device; the host logic that
shards batches over ranks (bench.py partition_batches) is correct; and the N > 1 data path
(per-rank partial H, Eq. 28, summed by ONE all-reduce, Eq. 29; density needs none, L312) is
exercised with world_size 2 over gloo, with the CPU oracle standing in for the per-rank kernels.
"""
import ctypes
import os
import re
import socket
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib_path():
    from paper_1912_06636_b200 import build as gpu_build
    return gpu_build.build()


def test_library_exports_every_declared_symbol(lib_path):
    with open(os.path.join(ROOT, "include", "aims_gpu.h")) as f:
        text = f.read()
    declared = sorted(set(re.findall(r"\b(aims_gpu_[a-z0-9_]+)\s*\(", text)))
    assert {"aims_gpu_create", "aims_gpu_destroy", "aims_gpu_eval_basis", "aims_gpu_integrate_hamiltonian",
            "aims_gpu_update_density"} <= set(declared)
    lib = ctypes.CDLL(lib_path)
    for name in declared:
        assert hasattr(lib, name), "libaims_gpu.so does not export %s" % name
    # the binding checks the same list when it loads
    import paper_1912_06636_b200 as aims
    assert aims.exported_symbols() == declared
    aims.load_library()


def test_boundary_has_no_torch_or_cxx_types(lib_path):
    """extern "C", plain pointers and sizes: the exported names are unmangled and the header compiles as C."""
    out = subprocess.run(["nm", "-D", "--defined-only", lib_path], capture_output=True, text=True, check=True).stdout
    names = [ln.split()[-1] for ln in out.splitlines() if " T " in ln]
    assert any(n == "aims_gpu_create" for n in names)
    src = "#include \"aims_gpu.h\"\nint main(void){aims_basis_desc b; aims_grid_desc g; aims_bsr_desc p; (void)b;(void)g;(void)p; return AIMS_OK;}\n"
    r = subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), "-x", "c", "-", "-o",
                        "/dev/null"], input=src, text=True, capture_output=True)
    assert r.returncode == 0, r.stderr


def test_library_contains_sm100a_fp64_tensor_code(lib_path):
    """The contraction kernels are DMMA (FP64 tensor pipe) SASS for sm_100a -- evidence that no other arch is built."""
    r = subprocess.run(["cuobjdump", "-lelf", lib_path], capture_output=True, text=True)
    if r.returncode != 0:
        pytest.skip("cuobjdump unavailable")
    assert "sm_100a" in r.stdout and "sm_90" not in r.stdout and "sm_80" not in r.stdout


def test_product_path_fails_loudly_without_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    import aims_synth
    import paper_1912_06636_b200 as aims
    bun = aims_synth.make_config(1, n_rad=4, n_ang=6)
    with pytest.raises(aims.AimsError):
        aims.aims_gpu_create(bun)


def test_product_does_not_import_oracle():
    """The product package and the input generators never import, read or run anything under oracle/."""
    for pkg in ("paper_1912_06636_b200", "aims_synth"):
        for dirpath, _, files in os.walk(os.path.join(ROOT, pkg)):
            for fn in files:
                if fn.endswith((".py", ".cu", ".cuh", ".c", ".h")):
                    with open(os.path.join(dirpath, fn)) as f:
                        text = f.read()
                    assert not re.search(r"^\s*(from|import)\s+oracle\b", text, re.M), fn
                    assert "aims_oracle" not in text, fn
    with open(os.path.join(ROOT, "oracle", "aims_oracle.c")) as f:
        text = f.read()
    assert "#include \"aims_gpu.h\"" not in text and "common.cuh" not in text


# ------------------------------------------------------------------------------------------- sharding host logic
def _partition():
    from paper_1912_06636_b200.sharding import partition_batches
    return partition_batches


def test_slice_bundle_keeps_exactly_the_ranks_own_batches():
    import aims_synth
    from paper_1912_06636_b200.sharding import first_phase_range, slice_bundle
    bun = aims_synth.make_config(1, n_rad=12, n_ang=26, max_batch=40)
    nb = bun.n_batches
    covered = 0
    for r in range(3):
        b0, b1 = first_phase_range(nb, r, 3)
        s, lo, hi = slice_bundle(bun, b0, b1)
        assert s.batch_ptr[0] == 0 and s.batch_ptr[-1] == s.n_points == hi - lo and s.n_batches == b1 - b0
        assert np.array_equal(s.xyz, bun.xyz[lo:hi]) and np.array_equal(s.w, bun.w[lo:hi])
        assert np.array_equal(s.v, bun.v[lo:hi]) and np.array_equal(s.g, bun.g[:, lo:hi])
        assert np.array_equal(np.diff(s.batch_ptr), np.diff(bun.batch_ptr[b0:b1 + 1]))
        assert s.D_values is bun.D_values and s.n_values == bun.n_values           # global objects are shared, not cut
        covered += s.n_points
    assert covered == bun.n_points
    # per-point fields the slicer has never heard of are cut as well (by shape, not by name); global ones are not, even when a
    # dimension coincides with the number of points
    import copy
    b2 = copy.copy(bun)
    b2.xi = np.arange(bun.n_points, dtype=np.float64)                     # [n]
    b2.hess = np.arange(6 * bun.n_points, dtype=np.float64).reshape(6, -1)  # [6][n]
    b2.D_values = np.zeros(bun.n_points)                                  # global, size coincides
    s, lo, hi = slice_bundle(b2, 1, nb - 1)
    assert np.array_equal(s.xi, b2.xi[lo:hi]) and np.array_equal(s.hess, b2.hess[:, lo:hi]) and s.D_values is b2.D_values
    per = aims_synth.make_periodic(n_rad=10, n_ang=14)
    s, lo, hi = slice_bundle(per, 1, per.n_batches)
    assert np.array_equal(s.xyz_unwrapped, per.xyz_unwrapped[lo:hi]) and s.atom_T is per.atom_T and s.frac is per.frac


def test_partition_batches_is_a_contiguous_cover_and_balanced():
    part = _partition()
    rng = np.random.default_rng(3)
    for nb, n_parts in [(1, 1), (5, 2), (7, 8), (1000, 2), (1000, 4), (39638, 8), (0, 2)]:
        cost = rng.uniform(0.0, 1.0, nb) ** 3
        rs = part(cost, n_parts)
        assert len(rs) == n_parts and rs[0][0] == 0 and rs[-1][1] == nb
        for (a0, a1), (b0, b1) in zip(rs[:-1], rs[1:]):
            assert a1 == b0 and a0 <= a1
        if nb >= 1000:
            loads = np.array([cost[a:b].sum() for a, b in rs])
            assert loads.max() <= loads.mean() + cost.max() + 1e-12     # off by at most one batch
    assert part(np.zeros(4), 2)[-1][1] == 4


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


_WORKER = r"""
import os, sys
import numpy as np
import torch, torch.distributed as dist
sys.path.insert(0, %(root)r)
import aims_synth
from paper_1912_06636_b200.sharding import first_phase_range, partition_batches, slice_bundle
from oracle.oracle import Oracle
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo", rank=rank, world_size=world)
full = aims_synth.make_config(1, n_rad=12, n_ang=26, max_batch=40)
# 1. cost probe on an equal-count slice (the per-rank "library" in this CPU test is the oracle; on a GPU it is aims_gpu_batch_nnz)
p0, p1 = first_phase_range(full.n_batches, rank, world)
probe, _, _ = slice_bundle(full, p0, p1)
op = Oracle(probe)
nnz = torch.zeros(full.n_batches, dtype=torch.int32)
nnz[p0:p1] = torch.tensor([len(op.batch_nnz(b)[0]) for b in range(probe.n_batches)], dtype=torch.int32)
dist.all_reduce(nnz)                                                             # 2. one tiny all-reduce
cost = np.diff(full.batch_ptr) * nnz.numpy().astype(np.float64) ** 2
b0, b1 = partition_batches(cost, world)[rank]                                    # 3. balanced contiguous ranges
mine, lo, hi = slice_bundle(full, b0, b1)                                        # this rank knows only its own batches
assert mine.n_points == hi - lo < full.n_points
orc = Oracle(mine)
H = torch.from_numpy(orc.integrate_hamiltonian(mine.v, mine.g))                  # Eq. 28: this rank's partial sum
dist.all_reduce(H)                                                               # Eq. 29: the only communication step
n, gn = orc.update_density(mine.D_values, want_grad=True)                        # L312: no synchronisation needed
n_all = torch.zeros(full.n_points, dtype=torch.float64)
n_all[lo:hi] = torch.from_numpy(n)
dist.all_reduce(n_all)                                                           # (only to compare; a rank keeps its own points)
# widened rows: forces and stress are partial sums like H; the density Hessian shards like n
Q = aims_synth.make_q_values(mine)
F = torch.from_numpy(orc.pulay_forces(mine.v, mine.D_values, g=mine.g, Q_values=Q, kinetic=True))
sg = torch.from_numpy(orc.pulay_stress(mine.v, mine.D_values, g=mine.g, Q_values=Q))
dist.all_reduce(F)
dist.all_reduce(sg)
hn_all = torch.zeros((6, full.n_points), dtype=torch.float64)
hn_all[:, lo:hi] = torch.from_numpy(orc.density_hessian(mine.D_values))
dist.all_reduce(hn_all)
if rank == 0:
    of = Oracle(full)
    F_ref = of.pulay_forces(full.v, full.D_values, g=full.g, Q_values=Q, kinetic=True)
    assert np.abs(F.numpy() - F_ref).max() <= 1e-13 * np.abs(F_ref).max()
    s_ref = of.pulay_stress(full.v, full.D_values, g=full.g, Q_values=Q)
    assert np.abs(sg.numpy() - s_ref).max() <= 1e-13 * np.abs(s_ref).max()
    assert np.array_equal(hn_all.numpy(), of.density_hessian(full.D_values))
    H_ref = of.integrate_hamiltonian(full.v, full.g)
    n_ref, _ = of.update_density(full.D_values, want_grad=True)
    eH = np.linalg.norm(H.numpy() - H_ref) / np.linalg.norm(H_ref)
    assert eH < 1e-13, eH
    assert np.array_equal(n_all.numpy(), n_ref)   # disjoint point ranges: bitwise the single-rank result
    print("OK", b0, b1, eH)
dist.destroy_process_group()
"""


def test_two_rank_gloo_partial_sums_equal_single_rank(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(_WORKER % {"root": ROOT})
    port = _free_port()
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port),
                   OMP_NUM_THREADS="2")
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.STDOUT, text=True))
    outs = [p.communicate(timeout=300)[0] for p in procs]
    assert all(p.returncode == 0 for p in procs), "\n".join(outs)
    assert "OK" in outs[0]


def test_periodic_images_rejects_unwrapped_fractional_coordinates():
    """aims_gpu_periodic_images runs on the host (no device needed).  Its enumeration box is sized for cell atoms inside the
    cell, so fractional coordinates outside [0, 1) are refused instead of silently losing images (include/aims_gpu.h); the
    same atom wrapped into the cell is accepted and gives the oracle's list."""
    import numpy as np

    import paper_1912_06636_b200 as aims
    from oracle.periodic import periodic_images
    lat = np.array([[4.0, 0.0, 0.0], [1.0, 5.0, 0.0], [0.0, 0.5, 6.0]])
    for bad in ([1.0, 0.5, 0.5], [0.2, -1e-9, 0.5], [0.2, 0.5, 1.5], [np.nan, 0.5, 0.5]):
        with pytest.raises(aims.AimsError):
            aims.aims_gpu_periodic_images(lat, np.array([[0.1, 0.2, 0.3], bad]), 3.0)
    frac = np.array([[0.1, 0.2, 0.3], [0.0, 0.999999, 0.5]])
    home, n = aims.aims_gpu_periodic_images(lat, frac, 3.0)
    home_ref, n_ref = periodic_images(lat, frac, 3.0)
    assert np.array_equal(home, home_ref) and np.array_equal(n, n_ref)


def test_product_library_reports_no_build_switches_and_ignores_the_environment(monkeypatch):
    """The binding loads the product library only: AIMS_GPU_LIB (a round-2 override) no longer redirects it, the product build
    reports "" from aims_gpu_build_flags(), and asking for another path once a library is loaded is an error, not a swap."""
    import paper_1912_06636_b200 as aims
    from paper_1912_06636_b200 import binding
    monkeypatch.setenv("AIMS_GPU_LIB", "/nonexistent/libaims_gpu_probe.so")
    L = aims.load_library()
    assert L._aims_path == binding.LIB_PATH and L._aims_build_flags == ""
    assert "AIMS_GPU_LIB" not in open(binding.__file__).read()
    with pytest.raises(aims.AimsError):
        aims.load_library("/nonexistent/libaims_gpu_probe.so", allow_probe=True)


def test_bench_gpus_2_starts_two_ranks_with_distinct_local_ranks():
    """`python bench.py --gpus N` (the form the driver uses at N = 1) must be a real N-rank run for N > 1: outside torchrun it
    starts the ranks itself through torch.distributed.run on 127.0.0.1.  --launch-dry-run goes through exactly that launch and has
    every rank report who it is instead of touching CUDA, so the path is checked here without GPUs.  A launcher that started a
    different number of ranks than --gpus says is refused, and without enough devices a real run refuses instead of shrinking."""
    import json
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "LOCAL_RANK", "WORLD_SIZE", "MASTER_ADDR", "MASTER_PORT")}
    out = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--launch-dry-run"], env=env, cwd=root,
                         capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stderr[-2000:]
    ranks = [json.loads(line) for line in out.stdout.splitlines() if line.startswith("{")]
    assert len(ranks) == 2 and all(r["launch_dry_run"] and r["world_size"] == 2 for r in ranks)
    assert sorted(r["local_rank"] for r in ranks) == [0, 1] and sorted(r["rank"] for r in ranks) == [0, 1]
    assert len({r["pid"] for r in ranks}) == 2 and len({r["master"] for r in ranks}) == 1 and ranks[0]["master"].startswith("127.0.0.1:")
    # WORLD_SIZE from a launcher that disagrees with --gpus
    bad = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--launch-dry-run"],
                         env=dict(env, WORLD_SIZE="1", RANK="0", LOCAL_RANK="0"), cwd=root, capture_output=True, text=True, timeout=300)
    assert bad.returncode != 0 and "WORLD_SIZE=1" in bad.stderr
    # a real 2-GPU run on a machine with fewer than two devices refuses loudly (this container has none)
    import torch
    if torch.cuda.device_count() < 2:
        real = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--steps", "1"], env=env, cwd=root,
                              capture_output=True, text=True, timeout=300)
        assert real.returncode != 0 and "refusing" in real.stderr


def test_product_library_holds_no_experiment_kernels(lib_path):
    """The shipped library contains the product only: the measured-and-rejected density variants, the matrix expansion that
    served one of them and the DMMA operand-pattern probes exist in probe builds (build.py --define ... --tag ...) and nowhere else."""
    import subprocess
    out = subprocess.run(["cuobjdump", "-sass", lib_path], capture_output=True, text=True, timeout=600).stdout
    funcs = [line for line in out.splitlines() if "Function :" in line]
    assert any("k_density" in f for f in funcs) and any("k_hamiltonian" in f for f in funcs)
    for name in ("k_density2", "k_density_b", "k_expand_matrix", "k_dmma_probe"):
        assert not any(name in f for f in funcs), name
