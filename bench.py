#!/usr/bin/env python
"""bench.py -- throughput of the fused DVM step on B200 (one JSON line on stdout).

metric: phase-space cell updates per second (N_kinetic * Nv * steps / time), BASELINE.json.
Workload (N=1): the configuration the north-star target is stated on -- the ~1.0e6-leaf periodic
octree with a 24^3 velocity grid, fp32 storage, fp64 moment accumulation (BASELINE.json configs[3],
SURVEY.md 8(d) row 4); both f buffers (2 x 55.8 GB) resident in HBM.  Synthetic, seeded inputs.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload config4|config4_lit|config4_small|config2|config3|config5|lbm19|lbm27|lbm19_f32|lbm19_small]
    python bench.py --impl reference ...      # the CPU oracle on a bounded sample of the same workload
    python bench.py --emulate-ranks R ...     # 1 GPU: the workload cut into R ranks with the ghost exchange
    torchrun ... bench.py --gpus N --partition  # one partitioned problem over N GPUs (NCCL ghost exchange)
    ... --fused-exchange                      # with either of the two: the step kernel writes the peers' ghost cells itself

N > 1 runs N independent replicas by default (the path is one GPU by the north star).
"""
import argparse
import json
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "phase-space cell updates/s per DVM step"
UNIT = "updates/s"


def make_case(workload: str):
    from paper_1503_00707_b200 import inputs
    if workload == "config4":
        return inputs.config4()
    if workload == "config4_lit":
        return inputs.config4(target_leaves=None)
    if workload == "config4_small":      # the same recipe one level coarser (ncu captures, quick looks)
        return inputs.config4(base=5, lmax=7, target_leaves=125_000, side_scale=2.0)
    if workload == "config2":
        return inputs.config2()
    if workload == "config3":
        return inputs.config3(lmax=8)
    if workload == "config5":
        return inputs.config5(lmax=8)
    raise SystemExit(f"unknown workload {workload}")


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json, copy bandwidth)"
    return 6650.0, "fallback (B200_PROFILING.md)"


def ncu_traffic_ratio(workload: str):
    """DRAM bytes per algorithmic byte of the step kernel from the committed ncu capture of exactly this workload
    (profiles/step_kernel_traffic.csv), or None if there is no such row."""
    path = os.path.join(ROOT, "profiles", "step_kernel_traffic.csv")
    if not os.path.exists(path):
        return None
    with open(path) as fh:
        for line in fh:
            if line.startswith("#") or not line.strip():
                continue
            w, storage, alg, rd, wr = line.strip().split(",")[:5]
            if w == workload:
                return (float(rd) + float(wr)) / float(alg)
    return None


def oracle_sample(case, n_sample: int):
    """A bounded sample of the workload for the CPU oracle: the window made of the first n_sample kinetic leaves in
    Morton order plus the non-kinetic leaves among them (missing neighbours at the window edge become zero-gradient
    ghosts).  Computed here with numpy: this leg never loads the CUDA library."""
    from paper_1503_00707_b200 import inputs
    order = inputs.morton_order(case.level, case.ijk)
    kin_pos = np.nonzero(case.kind[order] == inputs.CELL_KINETIC)[0]
    last = kin_pos[min(n_sample, kin_pos.size) - 1]
    return inputs.sub_case(case, np.sort(order[:last + 1]), case.name + "_sample")


def time_oracle(case, n_sample: int, steps: int, warmup: int, one_thread_leaves: int = 0):
    """The oracle as it stands (fp64, OpenMP over cells) on a Morton window of the workload: all cores, `steps` steps
    (>= 3 by BASELINE.md section 3); optionally also with 1 thread on a smaller window."""
    from oracle import dvm_oracle
    from paper_1503_00707_b200 import inputs

    def run(n_leaves, n_threads, k, w):
        sub = oracle_sample(case, n_leaves)
        dvm_oracle.set_threads(n_threads)
        o = dvm_oracle.Oracle(sub, window=True)     # neighbour-table build: outside the timed region
        f = inputs.initial_f(sub)
        for _ in range(w):
            f = o.step(f, case.dt)
        t0 = time.perf_counter()
        for _ in range(k):
            f = o.step(f, case.dt)
        t = time.perf_counter() - t0
        return o.n_kinetic * sub.Nv * k / t, t, o.n_kinetic

    cores = os.cpu_count() or dvm_oracle.threads()
    cores = min(cores, dvm_oracle.threads()) if dvm_oracle.threads() > 1 else cores
    steps = max(3, steps)
    value, t, n_kin = run(n_sample, cores, steps, warmup)
    out = {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
           "sample": f"window of the first {n_kin} Morton-ordered kinetic leaves of {case.name}, {steps} steps "
                     f"(fp64, OpenMP over cells, {cores} threads)", "seconds": t}
    if one_thread_leaves:
        v1, t1, n1 = run(one_thread_leaves, 1, steps, 0)
        out["value_1_thread"] = v1
        out["sample_1_thread"] = f"first {n1} Morton-ordered kinetic leaves, {steps} steps, 1 thread"
        out["seconds"] = t + t1
        dvm_oracle.set_threads(cores)
    return out, t / steps


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    case = make_case(args.workload)
    n_sample = args.oracle_leaves or 4096
    base, sec = time_oracle(case, n_sample, args.steps, args.warmup, one_thread_leaves=max(64, n_sample // 16))
    keys = ("value", "unit", "cores", "kind", "sample", "value_1_thread", "sample_1_thread")
    line = {"impl": "reference", "metric": METRIC, "value": base["value"], "unit": UNIT, "n_gpus": args.gpus,
            "steps": max(3, args.steps), "warmup": args.warmup, "ms_per_step": sec * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(case, args),
            "cpu_baseline": {k: base[k] for k in keys if k in base},
            "e2e": {"value": base["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def aggregate_over_ranks(ms_local: float, units_local: float, device=None):
    """Whole-job figures of N independent replicas: the slowest rank's device time and the
    units all ranks processed.  Works on any initialised process group (nccl on the GPU box, gloo in the CPU test);
    without one it returns its arguments."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return ms_local, units_local
    t = torch.tensor([ms_local], dtype=torch.float64, device=device)
    u = torch.tensor([units_local], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def sustained_copy_gbs(torch, dev, seconds=1.0):
    """Read + write bytes per second of b.copy_(a) over 2 x 2 GiB (the recipe behind MEASURED_PEAKS.json's hbm_gbs), best of
    the first ten copies and the mean over about `seconds` of back-to-back copies, on torch's current stream."""
    n = 1 << 30
    a = torch.empty(n, dtype=torch.int16, device=dev).zero_()
    b = torch.empty_like(a)
    for _ in range(3):
        b.copy_(a)
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(11)]
    ev[0].record()
    for i in range(10):
        b.copy_(a)
        ev[i + 1].record()
    torch.cuda.synchronize(dev)
    burst_ms = min(ev[i].elapsed_time(ev[i + 1]) for i in range(10))
    reps = max(10, int(seconds * 1e3 / burst_ms))
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(reps):
        b.copy_(a)
    e1.record()
    torch.cuda.synchronize(dev)
    bytes_per_copy = 2.0 * n * 2
    out = {"burst_GBs": bytes_per_copy / (burst_ms * 1e-3) / 1e9,
           "sustained_GBs": bytes_per_copy * reps / (e0.elapsed_time(e1) * 1e-3) / 1e9, "sustained_copies": reps,
           "what": "torch b.copy_(a), 2 GiB read + 2 GiB written per copy, after the timed steps"}
    del a, b
    return out


def run_partitioned(args):
    """The partitioned step (include/ufs_dvm.h "Partitioned mesh"): the workload cut along the
    N-order curve into equal-weight ranks, ghost chunks exchanged before every step.  Under torchrun every process is
    one rank (NCCL send / recv, strong scaling of ONE problem); with --emulate-ranks R the R ranks live on one GPU and
    one stream and the transfer is a device copy, which measures what the exchange costs besides the wire."""
    import torch
    import torch.distributed as dist
    from paper_1503_00707_b200 import binding as B
    from paper_1503_00707_b200 import harness
    from paper_1503_00707_b200.partition import (RankStepper, exchange_distributed, exchange_local, setup_push_distributed,
                                                 setup_push_local, step_pushed_distributed, step_pushed_local)
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the DVM step has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    emulate = args.emulate_ranks if world == 1 else 0
    n_ranks = emulate if emulate else world
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    case = make_case(args.workload)
    desc, keep = B.make_desc(case)
    rol = B.ufs_dvm_partition(desc, n_ranks, 1.0, 0.0)
    mine = list(range(n_ranks)) if emulate else [rank]
    fused = args.fused_exchange
    ranks = [RankStepper(case, rol, r, n_ranks, device=dev, symmetric=fused and not emulate) for r in mine]
    for st in ranks:
        harness.fill_initial_f_device(st, case)
    stream = ranks[0].stream
    if fused:
        setup_push_local(ranks) if emulate else setup_push_distributed(ranks[0])

    def exchange():
        if emulate:
            exchange_local(ranks)
        else:
            exchange_distributed(ranks[0])

    def step(k):
        for _ in range(k):
            if fused:          # the step kernel writes the peers' ghost slabs itself; what is left is the ghost sums
                step_pushed_local(ranks, case.dt) if emulate else step_pushed_distributed(ranks[0], case.dt)
            else:
                exchange()
                for st in ranks:
                    st.step(case.dt, 1)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    if fused:
        exchange()             # the ghosts of the very first step
    step(args.warmup)
    barrier()
    launches0 = sum(B.ufs_dvm_launch_count(st.h) for st in ranks)
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
    for st in ranks:
        B.ufs_dvm_profile(st.h, True)          # events around each rank's k_tiles launch
    with harness.ClockSampler(index=torch.cuda.current_device()) as clk:
        ev[0].record(stream)
        step(args.steps)
        ev[1].record(stream)
        barrier()
    launches = sum(B.ufs_dvm_launch_count(st.h) for st in ranks) - launches0
    kernel_ms = 0.0                             # per step: the ranks' streaming kernels one after the other (this process)
    for st in ranks:
        kernel_ms += B.ufs_dvm_kernel_ms(st.h)[0]
        B.ufs_dvm_profile(st.h, False)
    ev[2].record(stream)                       # the exchange alone (pack, transfer, unpack, ghost sums)
    for _ in range(args.steps):
        if fused:
            for st in ranks:
                st.halo_done()
        else:
            exchange()
    ev[3].record(stream)
    barrier()
    for st in ranks:
        st.sync()
    ms, ms_x = ev[0].elapsed_time(ev[1]), ev[2].elapsed_time(ev[3])
    n_inner = sum(st.n_inner for st in ranks)
    ms, units = aggregate_over_ranks(ms, float(n_inner * case.Nv * args.steps), dev)
    ms_x, _ = aggregate_over_ranks(ms_x, 0.0, dev)
    sent = sum(st.halo_bytes()[0] for st in ranks)
    ghosts = sum(st.n_ghost for st in ranks)
    elem = 4 if case.storage == 1 else 8
    cfg = workload_config(case, args)
    if fused:
        cfg["parallelism"] = (f"{n_ranks} ranks emulated on 1 GPU, one stream; fused exchange: k_tiles stores the boundary cells "
                              "into the peers' ghost slabs" if emulate
                              else f"{n_ranks} ranks, one GPU each; fused exchange: k_tiles stores the boundary cells into the "
                                   "peers' ghost slabs over NVLink (symmetric memory), one stream barrier per step")
    else:
        cfg["parallelism"] = (f"{n_ranks} ranks emulated on 1 GPU, one stream (device copy instead of NCCL)" if emulate
                              else f"{n_ranks} ranks, one GPU each, NCCL send/recv of the packed ghost chunks")
    line = {"metric": METRIC, "value": units / (ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
            "scaling": "strong" if world > 1 else "weak", "vs_baseline": None,
            "dtype": "f32" if case.storage == 1 else "f64", "data": "synthetic", "config": cfg, "clocks": clk.summary(),
            "e2e": None, "gpu_launches": launches,
            "halo": {"ranks": n_ranks, "inner_cells_this_process": n_inner, "ghost_cells_this_process": ghosts,
                     "ghost_fraction": ghosts / max(n_inner, 1), "sent_bytes_per_step_this_process": sent,
                     "sent_fraction_of_f": sent / max(n_inner * case.Nv * elem, 1),
                     "exchange_ms_per_step": ms_x / args.steps, "exchange_share_of_step": ms_x / ms,
                     "streaming_kernel_ms_per_step_this_process": kernel_ms}}
    if rank == 0:
        print(json.dumps(line), flush=True)
    for st in ranks:
        st.close()
    if world > 1:
        dist.destroy_process_group()


def run_lbm(args):
    """The lattice-Boltzmann variant (include/ufs_lbm.h; Table 1: ~1M cells): D3Q19 / D3Q27 on the
    config-4 octree (1 009 261 leaves, periodic), one kernel per step.  A "phase-space cell" is (leaf, lattice velocity);
    algorithmic bytes = one read and one write of f = 2 * Q * sizeof(storage) per leaf."""
    import torch
    from paper_1503_00707_b200 import harness, inputs
    from paper_1503_00707_b200 import lbm as K
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the LBM step has no CPU fallback")
    q = 27 if "27" in args.workload else 19
    tree = inputs.config4(base=5, lmax=7, target_leaves=125_000, side_scale=2.0) if args.workload.endswith("_small") else inputs.config4()
    case = inputs.lbm_case(tree, q, storage=inputs.STORE_F32 if "f32" in args.workload else inputs.STORE_F64)
    dev = torch.device("cuda", 0)
    st = K.LbmStepper(case, device=dev)
    # f(t=0): every cell at rest with its density, w_i rho (weights from the library's layout call)
    rho = torch.as_tensor(case.prim0[st.cell_of_row, 0], device=dev)
    st.f[K.ufs_lbm_current(st.h)].copy_((torch.as_tensor(st.w, device=dev)[:, None] * rho[None, :]).to(st.dtype))   # [Q, n]
    n, elem, dt = st.n_cells, (4 if st.storage == 1 else 8), case.dt
    st.step(dt, args.warmup)
    torch.cuda.synchronize(dev)
    l0 = K.ufs_lbm_launch_count(st.h)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with harness.ClockSampler(index=0) as clk:
        ev0.record(st.stream)
        st.step(dt, args.steps)
        ev1.record(st.stream)
        torch.cuda.synchronize(dev)
    st.sync()
    ms = ev0.elapsed_time(ev1)
    launches = K.ufs_lbm_launch_count(st.h) - l0
    peak, peak_src = peaks()
    alg = 2.0 * n * q * elem
    rec_bytes = 32.0 * n
    achieved = alg / (ms * 1e-3 / args.steps) / 1e9
    line = {"metric": METRIC, "value": n * q * args.steps / (ms * 1e-3), "unit": UNIT, "n_gpus": 1, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"{args.workload}: D3Q{q} on the config-4 octree, {n} cells (levels {int(case.level.min())}-{int(case.level.max())}), "
                                   f"omega = dt/tau = {case.meta['omega']}, CFL {case.cfl}",
                       "storage": "fp32" if st.storage == 1 else "fp64",
                       "l2": "f buffers (2 x %.0f MB) exceed L2 for the full-size tree" % (n * q * elem / 1e6), "parallelism": "1 GPU"},
            "clocks": clk.summary(), "e2e": None, "gpu_launches": launches,
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": None,
                         "peak_source": peak_src, "kernel": "k_lbm_step", "kernel_ms": ms / args.steps,
                         "algorithmic_bytes_per_launch": alg, "cell_record_bytes_per_launch": rec_bytes,
                         "frac_with_cell_records": (alg + rec_bytes) / (ms * 1e-3 / args.steps) / 1e9 / peak}}
    st.close()
    if not args.no_cpu_baseline:
        from oracle import dvm_oracle, lbm_oracle
        sub = oracle_sample(case, args.oracle_leaves or 32768)
        sub.meta = case.meta
        o = lbm_oracle.LbmOracle(sub, inputs.lbm_tau(case), window=True)
        f = lbm_oracle.initial_f(sub)
        t0 = time.perf_counter()
        f = o.step(f, dt, 3)
        t = time.perf_counter() - t0
        line["cpu_baseline"] = {"value": o.n * q * 3 / t, "unit": UNIT, "cores": dvm_oracle.threads(), "kind": "oracle",
                                "sample": f"first {o.n} Morton-ordered cells, 3 steps (C transport over cells + numpy collision)"}
    print(json.dumps(line), flush=True)


def workload_config(case, args):
    return {"workload": f"{args.workload}: {case.name}, {int((case.kind == 0).sum())} kinetic leaves "
                        f"(levels {int(case.level.min())}-{int(case.level.max())}), velocity grid "
                        f"{case.nv[0]}x{case.nv[1]}x{case.nv[2]} on [{case.vmin[0]},{case.vmax[0]}]^3, Kn {case.kn}, CFL {case.cfl}",
            "storage": "fp32" if case.storage == 1 else "fp64",
            "l2": "inputs larger than L2 (f buffers far exceed 126 MB); no flush needed",
            "parallelism": "1 GPU" if args.gpus == 1 else f"{args.gpus} independent replicas"}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="config4")
    ap.add_argument("--oracle-leaves", type=int, default=0, help="size of the CPU-oracle sample (0 = default)")
    ap.add_argument("--kn", type=float, default=None, help="override the Knudsen number (inf = collisions off)")
    ap.add_argument("--partition", action="store_true",
                    help="N > 1: one partitioned problem over the ranks (ghost exchange) instead of N replicas")
    ap.add_argument("--emulate-ranks", type=int, default=0,
                    help="1 GPU: cut the workload into R ranks on this GPU and step them with the ghost exchange")
    ap.add_argument("--fused-exchange", action="store_true",
                    help="partitioned step: the step kernel writes the peers' ghost slabs itself (ufs_dvm_halo_push_setup)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-copy-context", action="store_true", help="skip the plain-copy bandwidth measured beside the roofline")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.workload.startswith("lbm"):
        return run_lbm(args)
    if args.emulate_ranks > 1 or (args.partition and int(os.environ.get("WORLD_SIZE", "1")) > 1):
        return run_partitioned(args)

    import torch
    import torch.distributed as dist
    from paper_1503_00707_b200 import binding as B
    from paper_1503_00707_b200 import harness

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the DVM step has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    case = make_case(args.workload)
    if args.kn is not None:
        case.kn = args.kn
    st = B.DvmStepper(case, device=dev)
    harness.fill_initial_f_device(st, case)
    torch.cuda.synchronize(dev)
    n_kin, Nv = st.n_kinetic, st.Nv
    elem = 4 if case.storage == 1 else 8
    dt = case.dt
    info = B.ufs_dvm_kernel_info(st.h)
    kernel_name = B.ufs_dvm_kernel_name(st.h)

    # ---- end-to-end leg first (it restarts from f0): host buffers through ufs_dvm_run_host ----
    e2e = None
    if not args.no_e2e:
        try:
            host_in = torch.empty((n_kin, Nv), dtype=st.dtype, pin_memory=True)
            host_in.copy_(st.f[B.ufs_dvm_current(st.h)])
            mom_host = torch.empty((5, n_kin), dtype=torch.float64, pin_memory=True)
            B.ufs_dvm_run_host(st.h, host_in.data_ptr(), None, st.mom.data_ptr(), mom_host.data_ptr(), dt, 1)  # warm
            barrier()
            t0 = time.perf_counter()
            B.ufs_dvm_run_host(st.h, host_in.data_ptr(), None, st.mom.data_ptr(), mom_host.data_ptr(), dt, args.steps)
            torch.cuda.synchronize(dev)
            t_e2e = time.perf_counter() - t0
            t_e2e, units_e2e = aggregate_over_ranks(t_e2e, float(n_kin * Nv * args.steps), dev)
            e2e = {"value": units_e2e / t_e2e, "unit": UNIT,
                   "h2d_bytes_per_step": n_kin * Nv * elem / args.steps, "d2h_bytes_per_step": n_kin * 40 / args.steps,
                   "seconds": t_e2e,
                   "what": "ufs_dvm_run_host: pinned host f -> device, K steps, moments, moments -> host"}
            del host_in
        except Exception as ex:  # host memory too small for a pinned copy of f, etc.
            e2e = {"value": None, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0,
                   "unavailable": f"{type(ex).__name__}: {ex}"[:200]}
        harness.fill_initial_f_device(st, case)
        torch.cuda.synchronize(dev)

    # ---- device-resident timing: W warm-up steps, then exactly K steps between CUDA events ----
    st.step(dt, args.warmup)
    barrier()
    launches0 = B.ufs_dvm_launch_count(st.h)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    B.ufs_dvm_profile(st.h, True)               # the library brackets the main kernel of each step with events
    with harness.ClockSampler(index=torch.cuda.current_device()) as clk:
        ev0.record(st.stream)
        st.step(dt, args.steps)
        ev1.record(st.stream)
        barrier()
    ms = ev0.elapsed_time(ev1)
    kernel_ms, kernel_n = B.ufs_dvm_kernel_ms(st.h)
    B.ufs_dvm_profile(st.h, False)
    launches = B.ufs_dvm_launch_count(st.h) - launches0
    st.sync()                                   # raises on a sticky CUDA / Newton error
    ms_local = ms
    ms, updates_all = aggregate_over_ranks(ms, float(n_kin * Nv * args.steps), dev)
    value = updates_all / (ms * 1e-3)

    # ---- context for the roofline: what a plain device copy sustains on this box right now (MEASURED_PEAKS.json holds the
    # burst figure, best of ten copies on a cool device; a long step runs under the power cap)
    copy_ctx = None
    if rank == 0 and not args.no_copy_context:
        try:
            copy_ctx = sustained_copy_gbs(torch, dev)
        except Exception as ex:  # not enough free device memory beside f, etc.
            copy_ctx = {"unavailable": f"{type(ex).__name__}: {ex}"[:160]}

    # ---- roofline of the dominant kernel (the streaming pass over f): its own launches, timed by events ----
    peak, peak_src = peaks()
    alg_bytes_per_launch = 2.0 * n_kin * Nv * elem          # 1 read + 1 write of f per phase-space cell
    if kernel_n == 0:                                       # more steps than event pairs: fall back to the step time
        kernel_ms = ms / args.steps
    achieved = alg_bytes_per_launch / (kernel_ms * 1e-3) / 1e9
    ratio = ncu_traffic_ratio(args.workload)
    roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": None if ratio is None else ratio * alg_bytes_per_launch,
                "traffic_source": None if ratio is None else f"profiles/step_kernel_traffic.csv row '{args.workload}': ncu dram bytes per algorithmic byte x this launch's algorithmic bytes",
                "peak_source": peak_src, "kernel": kernel_name, "kernel_ms": kernel_ms, "kernel_launches_timed": kernel_n,
                "kernel_share_of_step": kernel_ms / (ms_local / args.steps),
                "algorithmic_bytes_per_launch": alg_bytes_per_launch,
                "whole_step_GBs": alg_bytes_per_launch / (ms * 1e-3 / args.steps) / 1e9,
                "frac_of_8TBs_nominal": achieved / 8000.0}
    if copy_ctx is not None:
        roofline["copy_on_this_box"] = copy_ctx
        if copy_ctx.get("sustained_GBs"):
            roofline["frac_of_sustained_copy"] = achieved / copy_ctx["sustained_GBs"]

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32" if case.storage == 1 else "f64", "data": "synthetic",
            "config": workload_config(case, args), "clocks": clk.summary(), "e2e": e2e, "gpu_launches": launches,
            "roofline": roofline, "kernel": info}

    if rank == 0 and not args.no_cpu_baseline and world == 1:
        st.close(); del st
        torch.cuda.empty_cache()
        n_or = args.oracle_leaves or 16384
        base, _ = time_oracle(case, n_or, 3, 0, one_thread_leaves=n_or // 16)
        keys = ("value", "unit", "cores", "kind", "sample", "value_1_thread", "sample_1_thread")
        line["cpu_baseline"] = {k: base[k] for k in keys if k in base}
    if rank == 0:
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
