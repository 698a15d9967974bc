#!/usr/bin/env python
"""bench.py -- grid points/s for H integration + density update (FP64) on the 375-atom Bi2Se3-shaped slab.

One "step" = one pass of the whole hot path over the whole grid: aims_gpu_integrate_hamiltonian (GGA) followed by
aims_gpu_update_density (with grad n), each including its own culling and basis evaluation.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 1..5] [--path scf|forces]

--path forces times the widened row f1 instead: one step = one aims_gpu_pulay_forces (GGA term and the
energy-weighted density matrix) over the whole grid; it is a separate line, not the headline metric.

N > 1: under torchrun (the driver's form) the ranks come from the launcher; a bare `python bench.py --gpus N` starts the N ranks
itself through torch.distributed.run on 127.0.0.1 and refuses if fewer than N devices are visible (--launch-dry-run checks that
launch without GPUs).  Contiguous batch ranges balanced by n_p*nnz^2 are sharded over the ranks; each rank adds its
partial H (Eq. 28) and the partial sums are combined by ONE NCCL all-reduce (Eq. 29, "the only communication
step"); the density needs none (L312).  Total work is fixed -> "scaling": "strong".

--impl reference times the CPU oracle (oracle/) on a bounded seeded sample of the same workload (rank 0 only).
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "grid points/s for H integration + density update (FP64); % of FP64 peak"
UNIT = "points/s"
# FP64 peak of the B200 tensor pipe from unit counts and clocks: 148 SMs x 64 FMA/clk x 2 x
# 1.965 GHz; the DMMA-chain probe (aims_gpu_fp64_peak) measures 37.2 TFLOP/s on this pool, i.e. exactly this number.
FP64_PEAK_NOMINAL_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12

WORKLOADS = {
    1: "config1: 3-atom molecule, 13,200 points, batches <=128, GGA",
    2: "config2: 64-atom Si-like cluster, 1,159,680 points, batches <=200, LDA",
    3: "config3: 64-atom Si-like cluster, 1,159,680 points, batches <=200, GGA",
    4: "config4: 200-atom two-species slab, 3,624,000 points, batches <=200, GGA",
    5: "config5: 375-atom Bi2Se3-shaped slab (3 QL x 5x5), 7,927,500 points, batches <=200, GGA",
    # not a BASELINE.json config: the periodic workload shaped like the paper's main benchmark, row f3
    6: "periodic: 54-atom diamond-Si supercell (3x3x3 primitive cells) + 505 periodic images, config-2 basis, 978,480 points, "
       "batches <=200, GGA; H^uc integration, Bloch sums at Gamma and one k, density update",
}


def make_workload(args):
    import aims_synth
    if args.config == 6:
        return aims_synth.make_periodic_si(n_rad=args.n_rad or 60, n_ang=args.n_ang or 302, max_batch=args.max_batch or 200)
    return aims_synth.make_config(args.config, n_rad=args.n_rad, n_ang=args.n_ang, max_batch=args.max_batch)


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=5)
    ap.add_argument("--max-batch", type=int, default=None)
    ap.add_argument("--n-rad", type=int, default=None, help="debug: coarser grid (not the benchmark workload)")
    ap.add_argument("--n-ang", type=int, default=None)
    ap.add_argument("--cpu-sample-batches", type=int, default=96)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--workspace-gib", type=float, default=0.0, help="Phi-plane workspace of the context (0 = library default, 24 GiB)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--launch-dry-run", action="store_true",
                    help="start the ranks exactly as a real run would, have each print its RANK / LOCAL_RANK / WORLD_SIZE and exit "
                         "(no CUDA, no workload): the launch path can be checked on a machine without GPUs")
    ap.add_argument("--lib", default=None, help="measure with a probe build of the library (build.py --define ... --tag ...); its "
                    "switches are recorded in the JSON line under build_flags, and such a line is not a bench value")
    ap.add_argument("--path", default="scf", choices=["scf", "forces", "stress", "hessian", "setup"])
    ap.add_argument("--deterministic", action="store_true",
                    help="ordered (bitwise reproducible) scatter into H: aims_gpu_set_deterministic")
    ap.add_argument("--kinetic", action="store_true",
                    help="scf path with the full h_KS phi (kinetic term, row f2): a separate line, not the headline metric")
    return ap.parse_args()


from paper_1912_06636_b200.sharding import first_phase_range, partition_batches, slice_bundle  # noqa: E402


class ClockSampler:
    """nvidia-smi clocks and throttle reasons sampled DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.rows = []
        self.proc = None
        self.idx = gpu_index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.idx), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), [x.strip() for x in line.split(",")]))

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        rows = [r for (t, r) in self.rows if t0 <= t <= t1 + 0.3] or [r for (_, r) in self.rows]
        sm, smax, reasons = [], [], set()
        for r in rows:
            try:
                sm.append(float(r[1]))
                smax.append(float(r[2]))
            except Exception:
                continue
            for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[5:9]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(smax)), "reasons": sorted(reasons),
                "samples": len(sm)}


def sample_batches(n_batches, k, seed=20191206):
    rng = np.random.default_rng(seed)
    return np.sort(rng.choice(n_batches, size=min(k, n_batches), replace=False)).astype(np.int32)


def time_oracle(bun, batches, gga, repeats=1, forces_q=None, kinetic=False, hessian=False, stress=False):
    """Oracle as it stands on the host cores: H integration + density update (or, with forces_q, the Pulay forces) on
    the listed batches."""
    from oracle import oracle as orc
    o = orc.Oracle(bun)
    pts = int(sum(bun.batch_ptr[b + 1] - bun.batch_ptr[b] for b in batches))
    best = None
    for _ in range(repeats):
        t0 = time.perf_counter()
        if hessian:
            o.density_hessian(bun.D_values, batches=batches)
        elif forces_q is not None:
            o.pulay_forces(bun.v, bun.D_values, g=bun.g if gga else None, Q_values=forces_q, batches=batches)
            if stress:
                o.pulay_stress(bun.v, bun.D_values, g=bun.g if gga else None, Q_values=forces_q, batches=batches)
        else:
            if kinetic:
                o.integrate_hamiltonian_ks(bun.v, bun.g if gga else None, kinetic=True, batches=batches)
            else:
                o.integrate_hamiltonian(bun.v, bun.g if gga else None, batches=batches)
            o.update_density(bun.D_values, want_grad=gga, batches=batches)
        dt = time.perf_counter() - t0
        best = dt if best is None else min(best, dt)
    return pts, best, orc.num_threads()


def time_blas_baseline(bun, batches, gga):
    """Paper-style CPU path (Fig. 6 CPU column, PAPER.md L319-329 / L353-363): per-batch DSYR2K / DSYMM-shaped products
    through numpy's BLAS on the host cores (oracle/blas_baseline.py), same batches as the oracle sample."""
    from oracle.blas_baseline import BlasBaseline
    bl = BlasBaseline(bun)
    Dd = bl.dense(bun.D_values)                              # set-up (the paper's loops start from the sparse n_ij too)
    Hd = np.zeros((bl.nb, bl.nb))
    pts = int(sum(bun.batch_ptr[b + 1] - bun.batch_ptr[b] for b in batches))
    t0 = time.perf_counter()
    bl.hamiltonian_dense(bun.v, bun.g if gga else None, batches=batches, out=Hd)
    bl.density(Dd, want_grad=gga, batches=batches)
    return pts, time.perf_counter() - t0


def kernel_sources_sha():
    """sha256 over the CUDA sources: profiles/*_traffic.txt records the hash its ncu capture was taken at."""
    import hashlib
    d = os.path.join(ROOT, "paper_1912_06636_b200", "csrc")
    h = hashlib.sha256()
    for f in sorted(os.listdir(d)):
        if f.endswith((".cu", ".cuh")):
            with open(os.path.join(d, f), "rb") as fh:
                h.update(f.encode() + b"\0" + fh.read())
    return h.hexdigest()[:16]


def committed_traffic(kernel, workload_key):
    """DRAM bytes per launch of `kernel` from the committed `ncu --set full` summary (profiles/r03_traffic.txt, one JSON
    object), or (None, why) when the capture was taken from other kernel sources than the ones this run loaded."""
    path = os.path.join(ROOT, "profiles", "r03_traffic.txt")
    try:
        with open(path) as f:
            rec = json.load(f)
    except Exception:
        return None, "no committed ncu capture (profiles/r03_traffic.txt)"
    if rec.get("kernel_sources_sha") != kernel_sources_sha():
        return None, "committed ncu capture was taken at kernel sources %s, this run has %s" % (
            rec.get("kernel_sources_sha"), kernel_sources_sha())
    val = rec.get("traffic", {}).get(workload_key, {}).get(kernel)
    if val is None:
        return None, "no capture of %s for %s in profiles/r03_traffic.txt" % (kernel, workload_key)
    return float(val), "dram__bytes_read.sum + dram__bytes_write.sum of one launch, %s (commit %s)" % (
        rec.get("source", "profiles/r03_traffic.txt"), rec.get("commit"))


def run_setup_path(args, aims, torch, ctx, bun, stream, workload, n_points_total, world, rank):
    """--path setup (row f4 of SURVEY.md 8(f)): one step = the partition-of-unity factor of every grid point
    (aims_gpu_partition_weights, Eq. 21-22) + the cut-plane batching of the whole grid (aims_gpu_batch_points, L210-218),
    inputs resident on the device.  Memory / latency-bound set-up work, outside the hot path: a separate line, no FP64 roofline."""
    import torch.distributed as dist
    r_part = float(bun.meta["r_part"])
    max_batch = int(bun.meta["max_batch"])
    with torch.cuda.stream(stream):
        xyz = torch.as_tensor(bun.xyz).to("cuda")
        owner = torch.as_tensor(bun.owner.astype(np.int32)).to("cuda")
    stream.synchronize()

    def step():
        with torch.cuda.stream(stream):
            w = ctx.partition_weights(xyz, owner, r_part)
        order, ptr = aims.aims_gpu_batch_points(xyz, max_batch, device=stream.device.index, stream=stream)
        return w, order, ptr

    for _ in range(max(args.warmup, 3)):
        step()
    stream.synchronize()
    sampler = ClockSampler(stream.device.index)
    sampler.start()
    time.sleep(0.3)
    t_part = t_batch = 0.0
    e = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
    tw0 = time.time()
    for _ in range(args.steps):
        e[0].record(stream)
        with torch.cuda.stream(stream):
            ctx.partition_weights(xyz, owner, r_part)
        e[1].record(stream)
        order, ptr = aims.aims_gpu_batch_points(xyz, max_batch, device=stream.device.index, stream=stream)
        e[2].record(stream)
        stream.synchronize()
        t_part += e[0].elapsed_time(e[1])
        t_batch += e[1].elapsed_time(e[2])
    tw1 = time.time()
    clocks = sampler.stop(tw0, tw1)
    ms_step = (t_part + t_batch) / args.steps
    if world > 1:
        t = torch.tensor([ms_step], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms_step = float(t.item())
    out = {"metric": "grid points/s for the GPU-side grid set-up (partition weights + cut-plane batching)", "value": n_points_total / (ms_step * 1e-3),
           "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms_step,
           "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": {"workload": workload + "; set-up path", "n_points": n_points_total, "n_atoms": int(bun.n_atoms), "r_part": r_part,
                      "max_batch": max_batch, "n_batches_found": int(len(ptr) - 1)},
           "clocks": clocks, "gpu_launches": None,
           "kernels": {"aims_gpu_partition_weights": {"ms_per_step": t_part / args.steps, "points_per_s": n_points_total / (t_part / args.steps * 1e-3)},
                       "aims_gpu_batch_points": {"ms_per_step": t_batch / args.steps, "points_per_s": n_points_total / (t_batch / args.steps * 1e-3)}},
           "e2e": None, "roofline": None, "cpu_baseline": None}
    if rank == 0:
        print(json.dumps(out))
    ctx.close()
    if world > 1:
        dist.destroy_process_group()
    return 0


def run_reference(args, bun, gga, workload, metric, forces_q=None, hessian=False, stress=False):
    """--impl reference: the CPU oracle, rank 0 only, a bounded sample per step."""
    per_step = max(4, args.cpu_sample_batches // 4)
    times, pts_step = [], 0
    for s in range(args.warmup + args.steps):
        sel = sample_batches(bun.n_batches, per_step, seed=1000 + s)
        pts, dt, cores = time_oracle(bun, sel, gga, forces_q=forces_q, kinetic=args.kinetic and forces_q is None, hessian=hessian, stress=stress)
        if s >= args.warmup:
            times.append(dt)
            pts_step += pts
    total = sum(times)
    val = pts_step / total
    sample = "%d seeded batches per step (about %d points) of %s" % (per_step, pts_step // max(args.steps, 1), workload)
    out = {"impl": "reference", "metric": metric, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": 1e3 * total / max(args.steps, 1), "higher_is_better": True,
           "scaling": "strong", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": {"workload": workload, "sample": sample},
           "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
           "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out))


def self_launch(args):
    """`python bench.py --gpus N` with N > 1 outside torchrun: start the N ranks here, one per GPU of this node, through the same
    launcher the driver uses (torch.distributed.run, rendezvous on 127.0.0.1), and return its exit code.  Rank 0 of the children
    prints the one JSON line.  Refuses when fewer than N devices are visible -- it never falls back to fewer ranks."""
    import socket
    import subprocess
    if not args.launch_dry_run:
        import torch
        have = torch.cuda.device_count() if torch.cuda.is_available() else 0
        if have < args.gpus:
            raise SystemExit("bench.py: --gpus %d but %d CUDA device(s) visible; refusing to run fewer ranks than asked for" % (args.gpus, have))
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus), "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def main():
    args = parse()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ and (args.impl != "reference" or args.launch_dry_run):
        return self_launch(args)
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if world != max(args.gpus, 1):
        raise SystemExit("bench.py: --gpus %d but the launcher started WORLD_SIZE=%d ranks" % (args.gpus, world))
    if args.launch_dry_run:
        print(json.dumps({"launch_dry_run": True, "rank": rank, "local_rank": local_rank, "world_size": world, "pid": os.getpid(),
                          "master": "%s:%s" % (os.environ.get("MASTER_ADDR"), os.environ.get("MASTER_PORT"))}), flush=True)
        return 0
    gga = args.config != 2
    workload = WORKLOADS[args.config]
    if args.max_batch:
        workload += " (max batch %d)" % args.max_batch
    if args.n_rad or args.n_ang:
        workload += " [DEBUG GRID n_rad=%s n_ang=%s: not the benchmark workload]" % (args.n_rad, args.n_ang)

    stress = args.path == "stress"                       # Pulay forces AND stress in one pass (row f1, "SCF+F+sigma")
    forces = args.path == "forces" or stress
    hessian = args.path == "hessian"
    metric = METRIC if not forces else "grid points/s for the Pulay-force pass (FP64); % of FP64 peak"
    if stress:
        metric = "grid points/s for the Pulay force + stress pass (FP64); % of FP64 peak"
    if hessian:
        metric = "grid points/s for the density-Hessian pass (FP64); % of FP64 peak"
    if args.kinetic and not forces and not hessian:
        metric = "grid points/s for H integration with the kinetic term + density update (FP64); % of FP64 peak"
    kin = bool(args.kinetic)

    import aims_synth
    if args.impl == "reference":
        if rank != 0:
            return 0
        bun = make_workload(args)
        if hessian:
            args.cpu_sample_batches = min(args.cpu_sample_batches, 32)
        run_reference(args, bun, gga, workload, metric, forces_q=aims_synth.make_q_values(bun) if forces else None,
                      hessian=hessian, stress=stress)
        return 0

    import torch
    import torch.distributed as dist
    import paper_1912_06636_b200 as aims
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    build_flags = aims.load_library(args.lib, allow_probe=args.lib is not None)._aims_build_flags
    if torch.cuda.device_count() <= local_rank:
        raise SystemExit("bench.py: rank %d wants cuda:%d but %d device(s) are visible" % (rank, local_rank, torch.cuda.device_count()))
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    t_gen = time.time()
    # synthetic input generation (not the product): every rank generates the system, then keeps only its own batches
    full = make_workload(args)
    t_gen = time.time() - t_gen
    periodic = args.config == 6
    if periodic:
        metric = "grid points/s for H^uc integration + Bloch sums + density update on a periodic cell (FP64); % of FP64 peak"
    n_points_total, n_batches_total = full.n_points, full.n_batches
    stream = torch.cuda.Stream(device=local_rank)
    t_create = time.time()
    npb_all = np.diff(full.batch_ptr).astype(np.float64)
    if world == 1:
        bun = full
        ctx = aims.aims_gpu_create(bun, device=local_rank, stream=stream, workspace_bytes=int(args.workspace_gib * 2 ** 30))
        nnz_all = ctx.batch_nnz().astype(np.float64)
        g0, g1 = 0, full.n_batches
    else:
        # "at no time does any process know the full grid" -- a rank's context holds its own batches only.
        # 1. cost probe on an equal-count slice  2. one tiny all-reduce of |nnz(B)|  3. balanced contiguous ranges
        p0, p1 = first_phase_range(full.n_batches, rank, world)
        probe_bun, _, _ = slice_bundle(full, p0, p1)
        probe = aims.aims_gpu_create(probe_bun, device=local_rank, stream=stream, workspace_bytes=1)
        nnz_t = torch.zeros(full.n_batches, dtype=torch.int32, device="cuda")
        nnz_t[p0:p1] = torch.as_tensor(probe.batch_nnz()).cuda()
        probe.close()
        dist.all_reduce(nnz_t)
        nnz_all = nnz_t.cpu().numpy().astype(np.float64)
        g0, g1 = partition_batches(npb_all * nnz_all * nnz_all, world)[rank]
        bun, _, _ = slice_bundle(full, g0, g1)
        ctx = aims.aims_gpu_create(bun, device=local_rank, stream=stream, workspace_bytes=int(args.workspace_gib * 2 ** 30))
    del full
    t_create = time.time() - t_create
    if args.deterministic:
        ctx.set_deterministic(True)
    st = ctx.stats()
    nnz = nnz_all[g0:g1]                           # this rank's batches; b0, b1 index the rank's own context
    npb = npb_all[g0:g1]
    b0, b1 = 0, bun.n_batches
    my_points = int(bun.n_points)
    syr2k = gga or bool(args.kinetic)            # Q not proportional to P: one full product, symmetrised
    flops_h = float(((2.0 if syr2k else 1.0) * npb * nnz * (nnz + (0.0 if syr2k else 1.0)))[b0:b1].sum())
    flops_n = float((2.0 * npb * nnz * nnz)[b0:b1].sum())
    # Pulay forces: the DSYMM-shaped products q_b Phi, n_b L and (GGA) n_b Phi, 2 n_p nnz^2 each
    flops_f = (3.0 if gga else 2.0) * flops_n
    flops_x = 4.0 * flops_n                      # density Hessian: n_b Phi and n_b d_e Phi, e = x, y, z
    Qh = aims_synth.make_q_values(bun) if forces else None

    with torch.cuda.stream(stream):
        v = torch.as_tensor(bun.v).to("cuda", non_blocking=False)
        g = torch.as_tensor(bun.g).to("cuda") if gga else None
        D = torch.as_tensor(bun.D_values).to("cuda")
        H = torch.empty(bun.n_values, dtype=torch.float64, device="cuda")
        n = torch.zeros(bun.n_points, dtype=torch.float64, device="cuda")
        gn = torch.zeros((3, bun.n_points), dtype=torch.float64, device="cuda") if gga else None
        Q = torch.as_tensor(Qh).to("cuda") if forces else None
        F = torch.zeros((bun.n_atoms, 3), dtype=torch.float64, device="cuda")
        SG = torch.zeros((3, 3), dtype=torch.float64, device="cuda")
        Hn = torch.zeros((6, bun.n_points), dtype=torch.float64, device="cuda") if hessian else None
        if periodic:
            nhb = int(bun.atom_fn_ptr[bun.n_home])
            kpts = [np.zeros(3), np.array([0.11, -0.07, 0.05])]
    stream.synchronize()

    def step():
        with torch.cuda.stream(stream):
            if hessian:
                ctx.density_hessian(D, hess_n=Hn, b0=b0, b1=b1)
                return
            if forces:
                if stress:
                    ctx.pulay_forces_stress(v, D, g=g, Q=Q, volume=1.0, F=F, sigma=SG, b0=b0, b1=b1, accumulate=False)
                else:
                    ctx.pulay_forces(v, D, g=g, Q=Q, F=F, b0=b0, b1=b1, accumulate=False)
                if world > 1:
                    dist.all_reduce(F)
                    if stress:
                        dist.all_reduce(SG)
                return
            ctx.integrate_hamiltonian(v, g, H=H, b0=b0, b1=b1, accumulate=False, kinetic=kin)
            if world > 1:
                dist.all_reduce(H)                        # Eq. 29: the only communication step
            if periodic:                                  # Eq. 7 in Eq. 11: h_ij(k) from the real-space matrix h^uc
                for kq in kpts:
                    ctx.bloch_fold(H, bun.atom_home, bun.atom_T, bun.n_home, kq, nhb)
            ctx.update_density(D, want_grad=gga, n=n, grad_n=gn, b0=b0, b1=b1)

    def barrier():
        stream.synchronize()
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()

    if args.path == "setup":
        return run_setup_path(args, aims, torch, ctx, bun, stream, workload, n_points_total, world, rank)
    peak_measured = ctx.fp64_peak(200.0)
    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    ctx.synchronize()

    # ---- timed region: exactly K steps, CUDA events on the launching stream, clocks sampled meanwhile
    sampler = ClockSampler(local_rank)
    sampler.start()
    time.sleep(0.3)
    ctx.timing_enable(True)
    launches0 = ctx.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    tw0 = time.time()
    e0.record(stream)
    for _ in range(args.steps):
        step()
    e1.record(stream)
    barrier()
    tw1 = time.time()
    ms_total = e0.elapsed_time(e1)
    kern = ctx.timing_read()
    ctx.timing_enable(False)
    launches = ctx.launch_count() - launches0
    clocks = sampler.stop(tw0, tw1)
    if world > 1:
        t = torch.tensor([ms_total], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms_total = float(t.item())
        lt = torch.tensor([launches], dtype=torch.int64, device="cuda")
        dist.all_reduce(lt)
        launches = int(lt.item())
    ms_step = ms_total / args.steps
    value = n_points_total / (ms_step * 1e-3)

    # ---- e2e: same step through the binding with pinned HOST buffers, copies inside the timed region
    e2e = None
    if not args.no_e2e:
        hb, dv = ctx.make_host_buffers(gga)
        hb["v"].copy_(torch.as_tensor(bun.v))
        hb["D"].copy_(torch.as_tensor(bun.D_values))
        if gga:
            hb["g"].copy_(torch.as_tensor(bun.g))
        if forces:
            hb["Q"] = torch.empty(bun.n_values, dtype=torch.float64, pin_memory=True)
            hb["Q"].copy_(torch.as_tensor(Qh))
            hb["F"] = torch.empty((bun.n_atoms, 3), dtype=torch.float64, pin_memory=True)
            dv["Q"], dv["F"] = torch.empty_like(Q), torch.empty_like(F)
            hb["SG"] = torch.empty((3, 3), dtype=torch.float64, pin_memory=True)
            dv["SG"] = torch.empty_like(SG)

        if hessian:
            hb["Hn"] = torch.empty((6, bun.n_points), dtype=torch.float64, pin_memory=True)
            dv["Hn"] = torch.empty_like(Hn)

        def step_e2e():
            with torch.cuda.stream(stream):
                if hessian:
                    dv["D"].copy_(hb["D"], non_blocking=True)
                    ctx.density_hessian(dv["D"], hess_n=dv["Hn"], b0=b0, b1=b1)
                    lo, hi = int(bun.batch_ptr[b0]), int(bun.batch_ptr[b1])
                    hb["Hn"][:, lo:hi].copy_(dv["Hn"][:, lo:hi], non_blocking=True)
                    return
                dv["v"].copy_(hb["v"], non_blocking=True)
                if forces:
                    dv["D"].copy_(hb["D"], non_blocking=True)
                if gga:
                    dv["g"].copy_(hb["g"], non_blocking=True)
                if forces:
                    dv["Q"].copy_(hb["Q"], non_blocking=True)
                    if stress:
                        ctx.pulay_forces_stress(dv["v"], dv["D"], g=dv["g"] if gga else None, Q=dv["Q"], volume=1.0,
                                                F=dv["F"], sigma=dv["SG"], b0=b0, b1=b1)
                    else:
                        ctx.pulay_forces(dv["v"], dv["D"], g=dv["g"] if gga else None, Q=dv["Q"], F=dv["F"], b0=b0, b1=b1)
                    if world > 1:
                        dist.all_reduce(dv["F"])
                        if stress:
                            dist.all_reduce(dv["SG"])
                    hb["F"].copy_(dv["F"], non_blocking=True)
                    if stress:
                        hb["SG"].copy_(dv["SG"], non_blocking=True)
                    return
                # v, g precede the integration; D (needed by the density update only) comes in and H goes out on a second
                # stream while the other call computes -- the copy engines are idle otherwise
                stream.wait_event(ev["h_out"])                     # the previous step's H has left the device
                ctx.integrate_hamiltonian(dv["v"], dv["g"] if gga else None, H=dv["H"], b0=b0, b1=b1, accumulate=False,
                                          kinetic=kin)
                if world > 1:
                    dist.all_reduce(dv["H"])
                ev["h_done"].record(stream)
            with torch.cuda.stream(copy_stream):
                copy_stream.wait_event(ev["n_done"])               # the previous step's density update has read D
                dv["D"].copy_(hb["D"], non_blocking=True)
                ev["d_in"].record(copy_stream)
                copy_stream.wait_event(ev["h_done"])
                hb["H"].copy_(dv["H"], non_blocking=True)
                ev["h_out"].record(copy_stream)
            with torch.cuda.stream(stream):
                stream.wait_event(ev["d_in"])
                ctx.update_density(dv["D"], want_grad=gga, n=dv["n"], grad_n=dv.get("grad_n"), b0=b0, b1=b1)
                ev["n_done"].record(stream)
                lo, hi = int(bun.batch_ptr[b0]), int(bun.batch_ptr[b1])
                hb["n"][lo:hi].copy_(dv["n"][lo:hi], non_blocking=True)
                if gga:
                    hb["grad_n"][:, lo:hi].copy_(dv["grad_n"][:, lo:hi], non_blocking=True)
        copy_stream = torch.cuda.Stream(device=local_rank)
        ev = {k: torch.cuda.Event() for k in ("h_done", "h_out", "d_in", "n_done")}
        for k in ("h_out", "n_done"):
            ev[k].record(stream)
        step_e2e()
        barrier()
        k2 = max(2, min(args.steps, 3))
        f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        f0.record(stream)
        for _ in range(k2):
            step_e2e()
        stream.wait_event(ev["h_out"])                             # the last H copy (second stream) is inside the timed region
        f1.record(stream)
        barrier()
        ms_e = f0.elapsed_time(f1) / k2
        if world > 1:
            t = torch.tensor([ms_e], dtype=torch.float64, device="cuda")
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            ms_e = float(t.item())
        h2d = 8 * (bun.n_points + bun.n_values + (3 * bun.n_points if gga else 0))
        d2h = 8 * (bun.n_values + my_points * (4 if gga else 1))
        if forces:
            h2d, d2h = h2d + 8 * bun.n_values, 8 * (3 * bun.n_atoms + (9 if stress else 0))
        if hessian:
            h2d, d2h = 8 * bun.n_values, 8 * 6 * my_points
        e2e = {"value": n_points_total / (ms_e * 1e-3), "unit": UNIT, "h2d_bytes_per_step": int(h2d),
               "d2h_bytes_per_step": int(d2h), "ms_per_step": ms_e}
        # the end-to-end outputs are the same numbers as the device-resident ones
        if hessian:
            assert torch.equal(hb["Hn"][:, int(bun.batch_ptr[b0]):int(bun.batch_ptr[b1])],
                               Hn[:, int(bun.batch_ptr[b0]):int(bun.batch_ptr[b1])].cpu())
        elif forces:
            assert torch.allclose(hb["F"], F.cpu(), rtol=0, atol=1e-10 * float(F.abs().max()))   # atomics: rounding only
        else:
            assert torch.equal(hb["n"][int(bun.batch_ptr[b0]):int(bun.batch_ptr[b1])],
                               n[int(bun.batch_ptr[b0]):int(bun.batch_ptr[b1])].cpu())

    # ---- roofline of the dominant kernel (FP64 tensor pipe), live CUDA-event durations from the timed region
    if hessian:                                  # the library times k_density_hessian in the k_forces slot
        kern = dict(kern)
        kern["k_density_hessian"] = kern["k_forces"]
    kflops = ({"k_density_hessian": flops_x} if hessian else {"k_forces": flops_f} if forces
              else {"k_hamiltonian": flops_h, "k_density": flops_n})
    dom = max(kflops, key=lambda k: kern[k][0])
    kd = {}
    for k in (("k_cull", "k_eval", "k_density_hessian") if hessian else ("k_cull", "k_eval", "k_forces") if forces
              else ("k_cull", "k_eval", "k_hamiltonian", "k_density")):
        ms, ln = kern[k]
        kd[k] = {"ms_per_step": ms / args.steps, "launches_per_step": ln / args.steps}
        if k in kflops and ms > 0:
            kd[k]["tflops"] = kflops[k] * args.steps / (ms * 1e-3) / 1e12
    dom_ms, dom_ln = kern[dom]
    achieved = kflops[dom] * args.steps / (dom_ms * 1e-3) / 1e12
    roofline = {"bound": "tensor", "kernel": dom, "achieved": achieved, "peak": FP64_PEAK_NOMINAL_TFLOPS,
                "unit": "TFLOP/s", "frac": achieved / FP64_PEAK_NOMINAL_TFLOPS, "traffic": None,
                "peak_source": "FP64 DMMA pipe: 148 SM x 64 FMA/clk x 2 x 1.965 GHz (unit counts x max clock); the "
                               "in-run DMMA-chain probe measured %.2f TFLOP/s" % peak_measured,
                "peak_measured_probe": peak_measured, "frac_of_measured_probe": achieved / peak_measured,
                "avg_launch_ms": dom_ms / max(dom_ln, 1), "algorithmic_flops_per_step": kflops[dom],
                "share_of_step": dom_ms / ms_total}
    total_tflops = (flops_x if hessian else flops_f if forces else flops_h + flops_n) / (ms_step * 1e-3) / 1e12
    # DRAM traffic per launch of the dominant kernel: read from the committed `ncu --set full` summary, and only if that
    # capture was taken from the kernel sources this run loaded (otherwise null, with the reason)
    wkey = "config%d%s" % (args.config, "" if not (args.max_batch or args.n_rad or args.n_ang) else "_variant")
    if world == 1:
        roofline["traffic"], roofline["traffic_note"] = committed_traffic(dom, wkey)
        roofline_eval_traffic = committed_traffic("k_eval", wkey)
    roofline["algorithmic_bytes_note"] = ("compulsory HBM bytes of the dominant contraction are ~1 GB per step (points, v, g, D, H, "
                                          "n, grad n); it is bound by the FP64 tensor pipe, so `achieved` is in flops")
    # second roofline: the HBM-bound evaluation kernel (algorithmic bytes = 8 B x planes x padded rows x padded points)
    pad = lambda a, m: np.ceil(a / m) * m                                   # noqa: E731
    pl_h, pl_d = 2.0, (4.0 if gga else 1.0)
    if hessian:
        eval_bytes = 8.0 * float((10.0 * pad(nnz, 16) * pad(npb, 8))[b0:b1].sum())
    elif forces:
        eval_bytes = 8.0 * float(((8.0 if gga else 5.0) * pad(nnz, 16) * pad(npb, 8))[b0:b1].sum())
    else:
        eval_bytes = 8.0 * float((pl_h * pad(nnz, 8) * pad(npb, 8) + pl_d * pad(nnz, 16) * pad(npb, 8))[b0:b1].sum())
    hbm_peak, hbm_src = 6561.9, "fallback: this pool's measured copy bandwidth recorded in DESIGN.md"
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            hbm_peak, hbm_src = float(json.load(f)["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs (burst copy bandwidth)"
    except Exception:
        pass
    ev_ms, ev_ln = kern["k_eval"]
    ev_gbs = eval_bytes * args.steps / (ev_ms * 1e-3) / 1e9 if ev_ms > 0 else 0.0
    if world != 1:
        roofline_eval_traffic = (None, "single-GPU capture only")
    roofline_eval = {"bound": "hbm", "kernel": "k_eval", "achieved": ev_gbs, "peak": hbm_peak, "unit": "GB/s",
                     "frac": ev_gbs / hbm_peak, "peak_source": hbm_src, "algorithmic_bytes_per_step": eval_bytes,
                     "avg_launch_ms": ev_ms / max(ev_ln, 1), "share_of_step": ev_ms / ms_total,
                     "traffic": roofline_eval_traffic[0], "traffic_note": roofline_eval_traffic[1]}

    out = {"metric": metric, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
           "ms_per_step": ms_step, "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f64",
           "data": "synthetic",
           "config": {"workload": workload, "n_points": n_points_total, "n_batches": n_batches_total, "n_basis": bun.n_basis,
                      "mean_nnz": float(nnz_all.mean()) if len(nnz_all) else 0.0, "max_nnz": int(nnz_all.max(initial=0)),
                      # workload metric of the paper, Eq. 31: #B x <|B|> x <nnz>^2, and the exact sum it models
                      "eq31_ops": float(len(nnz_all) * npb_all.mean() * nnz_all.mean() ** 2) if len(nnz_all) else 0.0,
                      "sum_np_nnz2": float((npb_all * nnz_all * nnz_all).sum()),
                      "ms_per_eq31_gops": (ms_step / (len(nnz_all) * npb_all.mean() * nnz_all.mean() ** 2 * 1e-9)) if len(nnz_all) else None,
                      "sharding": ("none" if world == 1 else "each rank's context holds only its own contiguous batch range "
                                   "(balanced by n_p*nnz^2); one NCCL all-reduce of H per step, none for n"),
                      "deterministic_H": bool(args.deterministic),
                      "max_active_atoms": st["max_active_atoms"], "parallelism": "batch-range x%d" % world,
                      "l2": "inputs larger than L2: each step streams %.1f GB of Phi planes plus a %.2f GB H and D"
                            % (1e-9 * eval_bytes, 8e-9 * bun.n_values)},
           "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline,
           "roofline_eval": roofline_eval, "fp64_tflops_step": total_tflops, "fp64_frac_of_peak_step": total_tflops / FP64_PEAK_NOMINAL_TFLOPS,
           "kernels": kd, "setup_s": {"generate_inputs": t_gen, "create_ctx": t_create}, "build_flags": build_flags}

    # ---- CPU baseline: the oracle on a bounded seeded sample, rank 0 at N=1 only
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        sel = sample_batches(bun.n_batches, args.cpu_sample_batches)
        if hessian:
            sel = sel[:32]
        pts, dt, cores = time_oracle(bun, sel, gga, forces_q=Qh, kinetic=kin and not forces and not hessian, hessian=hessian, stress=stress)
        out["cpu_baseline"] = {"value": pts / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
                               "sample": "%d seeded batches (%d points) of the same workload, %.1f s" % (len(sel), pts, dt)}
        if not forces and not hessian and not kin:
            # second, fairer CPU number: the paper's own CPU path, per-batch BLAS through numpy
            pts2, dt2 = time_blas_baseline(bun, sel, gga)
            out["cpu_baseline_blas"] = {"value": pts2 / dt2, "unit": UNIT, "cores": cores, "kind": "per-batch BLAS (numpy dgemm), Fig. 6 CPU column",
                                        "sample": "%d seeded batches (%d points) of the same workload, %.1f s" % (len(sel), pts2, dt2)}
    else:
        out["cpu_baseline"] = None
    if rank == 0:
        print(json.dumps(out))
    ctx.close()
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
