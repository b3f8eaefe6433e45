"""bench.py -- one "step" = one pass of the whole NOLSM hot path (a0 neighbour
lists, a1 gather, a2 S^-1, a3 operator, a4 sign iteration, a5-a6 density columns + write-back, a7
electron count) over one seeded synthetic water-like system, at fixed mu = -0.85 (one N(mu) evaluation).

    python bench.py --gpus 1 --steps 3 --warmup 3                      # the CUDA path
    python bench.py --impl reference --steps 1 --warmup 0              # the FP64 oracle on the host cores
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 \
        --master-port P bench.py --gpus N ...                          # N independent replicas (weak scaling)

Workload at N=1: BASELINE.json configs[2] ("w32768": 32,768 molecules, cutoff 10 A, FP16 operands /
FP32 accumulate, tol 1e-2) -- the configuration north_star quotes the target on; it fits one GPU with
the dense submatrices streamed through a 24 GiB workspace.  `--workload w4096` runs configs[1] (FP32).
Prints ONE JSON line (rank 0).  No file under /root/reference is read; all inputs are generated here.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

MU = -0.85
WORKLOADS = {          # name -> (precision, description)
    "tiny32": (0, "configs[0]"),
    "w4096": (1, "configs[1]: 4096 molecules, 8 A, all-FP32"),
    "w32768": (0, "configs[2]: 32768 molecules, 10 A, FP16 operands / FP32 accumulate"),
    "w262144": (0, "configs[3]: 262144 molecules, 12 A, FP16/FP32, streamed"),
}
DATASHEET_FP16_TFLOPS = 2250.0
# dram__bytes_read.sum + dram__bytes_write.sum of ONE sign-iteration launch of k_chain: an ncu CONSTANT from the
# `ncu --set full` capture named here (bench.py cannot read DRAM counters itself); None where no capture exists
NCU_TRAFFIC = {"w32768": 55.2e9}   # per batch: iteration 0 (4.35 + 3.24 GB) + the other iterations (26.83 + 20.76 GB), end-of-round capture
NCU_TRAFFIC_SOURCE = "profiles/r2_k_chain_sign_w32768.md"
METRIC = "molecules/s per NOLSM step (sign-iteration TFLOP/s in roofline.achieved)"


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            d = json.load(f)
        return {"hbm_gbs": d.get("hbm_gbs", 6650.0), "tflops_burst": d.get("bf16_tflops", 1590.0),
                "tflops_sustained": d.get("bf16_tflops_sustained", 1400.0), "source": "measured"}
    return {"hbm_gbs": 6650.0, "tflops_burst": 1590.0, "tflops_sustained": 1400.0, "source": "fallback"}


# ------------------------------------------------------------------------------------------------
# CPU baseline: the oracle as it stands, one submatrix per process, single-threaded BLAS inside
# ------------------------------------------------------------------------------------------------
_SYSTEM = None


def _oracle_one(j):
    import oracle.nolsm_oracle as orc
    s = _SYSTEM
    sol = orc.solve_molecule(s.row_ptr, s.col_idx, s.h_val, s.s_val, int(j))
    cols = sol.density_columns(MU)
    return sol.population(MU), float(abs(cols).max())


def time_oracle(system, n_sample, cores):
    """Oracle on `n_sample` molecules spread over the system; returns (molecules/s, seconds)."""
    import multiprocessing as mp
    import numpy as np
    from threadpoolctl import threadpool_limits
    import oracle.nolsm_oracle  # noqa: F401  (loads LAPACK in the parent so the thread limit below reaches it)
    global _SYSTEM
    _SYSTEM = system
    mols = np.linspace(0, system.n_mol - 1, n_sample).astype(int).tolist()
    with threadpool_limits(limits=1):
        if cores > 1:
            ctx = mp.get_context("fork")   # CUDA is not initialised yet in this process
            with ctx.Pool(cores) as pool:
                pool.map(_oracle_one, mols[:cores])          # start-up outside the timed region
                t0 = time.perf_counter()
                pool.map(_oracle_one, mols, chunksize=1)
                dt = time.perf_counter() - t0
        else:
            t0 = time.perf_counter()
            for j in mols:
                _oracle_one(j)
            dt = time.perf_counter() - t0
    return n_sample / dt, dt


def oracle_sample_size(system, cores):
    """About 10-30 s of CPU work: LAPACK dsygvd + projector is ~0.5 ns * n^3 per submatrix per core."""
    import numpy as np
    n = 6.0 * float(np.diff(system.row_ptr).mean())
    per = max(5e-10 * n ** 3, 1e-3)
    return int(max(cores, min(system.n_mol, round(15.0 * cores / per))))


# ------------------------------------------------------------------------------------------------
# clocks during the timed region
# ------------------------------------------------------------------------------------------------
class ClockSampler:
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.FIELDS,
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        self.thread.join(timeout=2)
        sm, smax, reasons, power = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            if len(r) < 7:
                continue
            try:
                sm.append(float(r[0])); smax.append(float(r[1])); power.append(float(r[2]))
            except ValueError:
                continue
            for name, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "power_w_max": max(power) if power else None, "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------------------
# N > 1: independent replicas -- the only cross-rank step is the max of the times
# ------------------------------------------------------------------------------------------------
def max_over_ranks(ms, device="cpu"):
    """Max over the ranks of a per-rank time (all-reduce MAX; identity without a process group)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(ms)
    t = torch.tensor([float(ms)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_value(world, n_mol, ms_step):
    """Whole-job molecules/s: every rank processes its own replica of n_mol molecules per step."""
    return world * n_mol / (ms_step * 1e-3)


# ------------------------------------------------------------------------------------------------
# the two arms
# ------------------------------------------------------------------------------------------------
def run_reference(args, system, rank):
    """--impl reference: the FP64 oracle (the only 'reference implementation' this tier has), on the
    host cores, each step a bounded sample of the workload."""
    if rank != 0:
        return None
    cores = os.cpu_count() or 1
    n_sample = oracle_sample_size(system, cores)
    for _ in range(args.warmup):
        time_oracle(system, max(cores, n_sample // 8), cores)
    t0 = time.perf_counter()
    rates = [time_oracle(system, n_sample, cores)[0] for _ in range(args.steps)]
    total = time.perf_counter() - t0
    value = len(rates) / sum(1.0 / r for r in rates)
    sample = f"{n_sample} of {system.n_mol} molecules per step, evenly spaced ids; one submatrix per process, 1 BLAS thread each"
    return {"impl": "reference", "metric": METRIC, "value": value, "unit": "molecules/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total / max(args.steps, 1),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": args.workload, "mu": MU, "note": "FP64 oracle (generalized eigensolve per submatrix)"},
            "cpu_baseline": {"value": value, "unit": "molecules/s", "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": "molecules/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}


def run_native(args, system, rank, world, local_rank):
    import numpy as np
    # CPU baseline first: it forks, which must happen before CUDA is initialised in this process
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cores = os.cpu_count() or 1
        n_sample = oracle_sample_size(system, cores)
        rate, dt = time_oracle(system, n_sample, cores)
        cpu = {"value": rate, "unit": "molecules/s", "cores": cores, "kind": "oracle",
               "sample": f"{n_sample} of {system.n_mol} molecules (evenly spaced ids) in {dt:.1f} s; "
                         "one submatrix per process, 1 BLAS thread each; FP64 dsygvd + projector + population"}
    import torch
    import paper_2104_08245_b200 as nolsm
    nolsm.load_library()   # fails loudly when libnolsm.so is missing: there is no fallback
    if not torch.cuda.is_available():
        raise SystemExit("bench.py (native arm) needs a CUDA device; there is no CPU fallback")
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    precision = WORKLOADS[args.workload][0] if args.precision < 0 else args.precision
    cfg = nolsm.Config(precision=precision, workspace_bytes=int(args.workspace_gib * (1 << 30)), group=args.group,
                       flags=args.flags, cache_bytes=-1 if args.no_cache else 0, gap_hint=args.gap_hint)
    ctx = nolsm.Context(cfg)
    dev = torch.device("cuda", local_rank)
    pos = torch.as_tensor(system.pos_q).to(dev)
    h_val = torch.as_tensor(system.h_val).to(dev)
    s_val = torch.as_tensor(system.s_val).to(dev)
    mu_lo, mu_hi = 2 * MU, 0.0        # one evaluation at the midpoint mu = -0.85
    if args.elements != "gathered":   # T_j(H), T_j(S) evaluated on the device from the positions
        import nolsm_inputs as gi
        ctx.set_model(pos, eval_fp32=args.elements == "generated-fp32", **gi.model_parameters(system))

    def step():
        rp, ci = ctx.build_neighbours(pos, system.box_q, system.rc_q, cap=system.nnzb)
        H = nolsm.BlockSparse(rp, ci, h_val)
        S = nolsm.BlockSparse(rp, ci, s_val)
        D = nolsm.BlockSparse(rp, ci, step.d_val)
        return ctx.solve_mu(H, S, system.n_electrons, mu_lo, mu_hi, tol_ne_per_mol=-1.0, max_steps=args.mu_steps, D=D)

    step.d_val = torch.empty_like(s_val)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        step()
    barrier()
    sampler = ClockSampler(local_rank)
    sampler.start()
    l0 = ctx.launch_count
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    agg = {"ms_gather": 0.0, "ms_prepare": 0.0, "ms_sign": 0.0, "ms_density": 0.0, "flops_sign": 0.0,
           "flops_sign_padded": 0.0, "flops_prepare": 0.0, "ms_chain": 0.0, "chain_launches": 0}
    ev0.record()
    last = None
    for _ in range(args.steps):
        mu, ne, D, st = step()
        last = (mu, ne, st)
        for k in ("ms_gather", "ms_prepare", "ms_sign", "ms_density", "ms_chain", "chain_launches"):
            agg[k] += getattr(st, k)
        agg["flops_sign"] += st.flops_sign_total
        agg["flops_sign_padded"] += st.last.flops_sign_padded
        agg["flops_prepare"] += st.flops_prepare_total
    ev1.record()
    barrier()
    clocks = sampler.stop()
    launches = ctx.launch_count - l0
    ms = max_over_ranks(ev0.elapsed_time(ev1), dev)
    mu, ne, st = last
    ms_step = ms / args.steps
    value = job_value(world, system.n_mol, ms_step)

    # end to end through the host-buffer entry (transfers inside the timed region)
    e2e = None
    if not args.no_e2e:
        hp = [torch.as_tensor(x).contiguous().pin_memory() for x in
              (system.row_ptr, system.col_idx, system.h_val.reshape(-1), system.s_val.reshape(-1))]
        d_host = torch.empty(system.nnzb * 36, dtype=torch.float32).pin_memory()
        ctx.solve_mu_host(hp[0], hp[1], hp[2], hp[3], d_host, system.n_electrons, mu_lo, mu_hi, -1.0, 1)  # warm-up
        barrier()
        t0 = time.perf_counter()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        reps = max(5, args.steps)
        pos_host = torch.as_tensor(system.pos_q).contiguous().pin_memory()
        for _ in range(reps):
            # a0 inside the timed region too: positions host -> device, neighbour lists rebuilt on the device
            # (bit-identical to the host pattern the call below is given, tests/test_gpu_parity.py)
            ctx.build_neighbours(pos_host.to(dev, non_blocking=True), system.box_q, system.rc_q, cap=system.nnzb)
            _, ne_h, _, h2d, d2h = ctx.solve_mu_host(hp[0], hp[1], hp[2], hp[3], d_host, system.n_electrons,
                                                     mu_lo, mu_hi, -1.0, 1)
            h2d += pos_host.numel() * 4
        e1.record()
        barrier()
        ms_e = max_over_ranks(max(e0.elapsed_time(e1), 1e3 * (time.perf_counter() - t0)) / reps, dev)
        e2e = {"value": job_value(world, system.n_mol, ms_e), "unit": "molecules/s", "h2d_bytes_per_step": h2d,
               "d2h_bytes_per_step": d2h, "ms_per_step": ms_e, "n_electrons": ne_h,
               "reps": reps,
               "note": "per step: positions pinned host->device + nolsm_build_neighbours (a0), then "
                       "nolsm_solve_mu_host: pattern+H+S pinned host->device, a1-a7, D device->host"}
    if dist is not None:
        dist.destroy_process_group()
    if rank != 0:
        return None
    peaks = measured_peaks()
    # dominant kernel: k_chain running the sign iteration (Eq. 9-10) of one batch, all iterations in
    # one launch; timed with CUDA events on the library's stream around every such launch
    ms_kernel = agg["ms_chain"] if agg["ms_chain"] > 0 else agg["ms_sign"]
    sign_tflops = agg["flops_sign"] / max(ms_kernel, 1e-9) * 1e-9
    n_launch = max(int(agg["chain_launches"]), 1)
    out = {
        "metric": METRIC, "value": value, "unit": "molecules/s", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f16 operands / f32 accumulate" if precision == 0 else "f32 (split f16 operands)",
        "data": "synthetic",
        "config": {"workload": args.workload, "description": WORKLOADS[args.workload][1], "n_mol": system.n_mol,
                   "cutoff_A": system.cutoff, "mu": MU, "seed": system.seed, "nnz_blocks": system.nnzb,
                   "mean_submatrix_dim": 6.0 * system.nnzb / system.n_mol, "tol": 1e-2 if precision == 0 else 1e-5,
                   "workspace_gib": args.workspace_gib, "batches": st.n_batches, "replicas": world,
                   "group": args.group, "engine_flags": args.flags, "elements": args.elements, "mu_steps": args.mu_steps, "gap_hint": args.gap_hint,
                   "l2": "inputs larger than L2 (block stores 3 x %.0f MB, dense workspace %.0f GiB)" %
                         (system.nnzb * 144 / 1e6, args.workspace_gib)},
        "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches),
        "roofline": {"bound": "tensor",
                     "kernel": "k_chain, sign iteration of one batch (Eq. 9-10: iteration 0 with the rescale in one launch, all others in a second one; per launch = per batch)",
                     "achieved": sign_tflops, "peak": peaks["tflops_sustained"], "unit": "TFLOP/s",
                     "frac": sign_tflops / peaks["tflops_sustained"], "traffic": NCU_TRAFFIC.get(args.workload),
                     "traffic_source": "ncu constant, " + NCU_TRAFFIC_SOURCE,
                     "peak_source": peaks["source"] + " bf16_tflops_sustained (kernel timed inside a long step); "
                                    "FP32 mode issues 3 FP16 MMAs per product, so its bound is peak / 3"
                                    if precision == 1 else
                                    peaks["source"] + " bf16_tflops_sustained (kernel timed inside a long step)",
                     "frac_of_datasheet_fp16": sign_tflops / DATASHEET_FP16_TFLOPS,
                     "flops": "2 n^3 per executed sign-iteration GEMM, true n (PAPER.md:246)",
                     "flops_per_launch": agg["flops_sign"] / n_launch, "launches": n_launch,
                     "avg_launch_ms": ms_kernel / n_launch,
                     "achieved_padded": agg["flops_sign_padded"] / max(ms_kernel, 1e-9) * 1e-9,
                     "achieved_whole_sign_stage": agg["flops_sign"] / max(agg["ms_sign"], 1e-9) * 1e-9},
        # the other tensor-bound stage: a2 + a3 (Eq. 15-17, S^-1 = Z^2, refinement, B = S^-1 H), CUDA-event time of
        # the whole stage (its products, norm bounds and element-wise passes) per step
        "roofline_prepare": {"bound": "tensor", "kernel": "k_chain, prepare launches (Eq. 15-17 chain, Z^2, refinement, B)",
                             "achieved": agg["flops_prepare"] / max(agg["ms_prepare"], 1e-9) * 1e-9,
                             "peak": peaks["tflops_sustained"], "unit": "TFLOP/s",
                             "frac": agg["flops_prepare"] / max(agg["ms_prepare"], 1e-9) * 1e-9 / peaks["tflops_sustained"],
                             "flops": "2 n^3 per product (a split-operand product counts once, but runs 3 FP16 MMAs)",
                             "ms_per_step": agg["ms_prepare"] / args.steps, "traffic": None},
        "cpu_baseline": cpu,
        "detail": {"sign_tflops": sign_tflops, "ms_gather": agg["ms_gather"] / args.steps,
                   "ms_prepare": agg["ms_prepare"] / args.steps, "ms_sign": agg["ms_sign"] / args.steps,
                   "ms_density": agg["ms_density"] / args.steps,
                   "prepare_tflops": agg["flops_prepare"] / max(agg["ms_prepare"], 1e-9) * 1e-9,
                   "sign_iter_min": st.last.iter_min, "sign_iter_max": st.last.iter_max,
                   "n_unconverged": st.last.n_unconverged, "worst_residual": st.last.worst_residual,
                   "n_electrons": ne, "n_electrons_diag": st.ne_diag, "n_electrons_target": system.n_electrons},
    }
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="native", choices=["native", "reference"])
    ap.add_argument("--workload", default="w32768", choices=sorted(WORKLOADS))
    ap.add_argument("--precision", type=int, default=-1, help="0 = FP16/FP32, 1 = FP32 (default: the workload's)")
    ap.add_argument("--workspace-gib", type=float, default=24.0)
    ap.add_argument("--group", type=int, default=0, help="window: submatrices in flight together (0: from the L2 size)")
    ap.add_argument("--flags", type=int, default=0, help="NOLSM_FLAG_* bits (2: pair engine, 8: single-CTA engine, 16: unit scaling, 32: third-order iteration, "
                         "64: no a-priori stop of Eq. 15-17, 128: symmetric Loewdin form, FP32 workloads only, "
                         "256: no rescaled first sign iteration)")
    ap.add_argument("--elements", default="gathered", choices=["gathered", "generated", "generated-fp32"],
                    help="submatrix elements gathered from the block stores (the north_star path) or evaluated "
                         "on the device from the positions (nolsm_set_model; -fp32: FP32 + SFU as in PAPER.md:202)")
    ap.add_argument("--mu-steps", type=int, default=1,
                    help="N(mu) evaluations per step (default 1 = the headline step; 5 = BASELINE configs[1]'s bisection)")
    ap.add_argument("--gap-hint", type=float, default=0.0,
                    help="nolsm_config.gap_hint: lower bound on |lambda - mu| (the generator's gap gives 0.15 at "
                         "mu = -0.85); > 0 starts the sign iteration with scaled steps.  Default 0: plain Eq. 9")
    ap.add_argument("--no-cache", action="store_true", help="nolsm_config.cache_bytes = -1 (only matters for --mu-steps > 1)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference" and rank != 0:
        return 0
    import nolsm_inputs as gi
    n_mol, cutoff = gi.CONFIGS[args.workload]
    system = gi.make_water_system(n_mol, cutoff)
    if args.impl == "reference":
        out = run_reference(args, system, rank)
    else:
        out = run_native(args, system, rank, world, local_rank)
    if out is not None:
        print(json.dumps(out), flush=True)
    return 0


if __name__ == "__main__":
    sys.exit(main())
