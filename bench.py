#!/usr/bin/env python
"""bench.py -- headline benchmark of the generalized -> standard reduction + back-transform.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config I] [--impl ours|reference]

One "step" = one pass of the whole hot path (gs_cholesky, gs_invert_triangular, gs_to_standard,
gs_backtransform: PAPER.md:61-67) over one seeded synthetic pencil of BASELINE.json `configs[2]`
(N = 16384 real FP64, nev = 4096).  Metric: FP64 TFLOP/s with the nominal flop counts of
BASELINE.json (N^3/3 + N^3/3 + N^3 + N^2 nev).  Prints ONE JSON line (rank 0).

N > 1 GPUs: the path does not shard (replicas only) -- every rank reduces its
own independent pencil (different seed; the paper's "trivial parallelism" over k-points / spin
channels), no data-path collective; value = all ranks' flops / max-over-ranks time.

`--impl reference` times the CPU oracle (oracle/, as it stands) on the host cores on a bounded
sample of the same workload; it is the reference arm of the contract for this tier.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "FP64 TFLOP/s of Cholesky+invert+transform+backtransform at N=16384; % FP64 peak"
UNIT = "TFLOP/s"
STAGES = ("cholesky", "invert", "to_standard", "backtransform")


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=2, help="index into BASELINE.json configs (default 2 = headline)")
    ap.add_argument("--n", type=int, default=0, help="context runs only: a real pencil of this order instead of a BASELINE config "
                                                     "(e.g. 40960 = the size of the paper's Table 1, PAPER.md:136)")
    ap.add_argument("--nev", type=int, default=0, help="with --n: number of eigenvectors (default n / 4)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--cpu-sample", type=int, default=4096, help="order of the leading block the oracle is timed on")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-checks", action="store_true")
    ap.add_argument("--no-evp", action="store_true", help="skip the standard-eigensolver block (NEXT-4, outside the metric)")
    ap.add_argument("--batch", type=int, default=0, help="NEXT-2: K independent pencils in flight on one GPU (not the headline)")
    ap.add_argument("--batch-n", type=int, default=2048)
    ap.add_argument("--sharded", action="store_true",
                    help="NEXT-3: ONE pencil over all ranks (steps 2-4 by column ranges, one exchange); strong scaling, not the headline mode")
    ap.add_argument("--exchange", default="push", choices=["push", "collective"],
                    help="--sharded: slabs stored into the peers' buffers from the kernel epilogues (push) or NCCL broadcasts after the kernels")
    ap.add_argument("--shard-sync", default="host", choices=["host", "device"],
                    help="--sharded with the push exchange: order producing and consuming launches by host barriers or by device-side flags")
    ap.add_argument("--shard-chol-mode", default="leading", choices=["leading", "sharded"],
                    help="--sharded: step 1 per rank on the leading block it needs, or over the ranks (gs_cholesky_sharded; needs --exchange push --shard-sync device)")
    ap.add_argument("--shard-shares", type=int, default=0,
                    help="NEXT-3: time, on ONE GPU and one after the other, the share each of R ranks would run (not the headline)")
    ap.add_argument("--batch-complex", action="store_true")
    ap.add_argument("--shard-chol", type=int, default=0,
                    help="NEXT-3: gs_cholesky_sharded with R ranks emulated on ONE GPU (R plans, R streams) and the model projection")
    return ap.parse_args()


# ------------------------------------------------------------------------------------------------
# clocks: sample SM clock and throttle reasons DURING the timed region (NVML, background thread)
# ------------------------------------------------------------------------------------------------
class ClockSampler:
    REASONS = {
        0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap",
        0x80: "hw_power_brake", 0x2: "applications_clocks_setting", 0x100: "display_clock_setting",
    }

    def __init__(self, index: int):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thread = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self._nv = pynvml
            self._h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self._nv = None

    def _run(self):
        nv = self._nv
        while not self._stop.is_set():
            try:
                self.samples.append(float(nv.nvmlDeviceGetClockInfo(self._h, nv.NVML_CLOCK_SM)))
                mask = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self._h))
                for bit, name in self.REASONS.items():
                    if mask & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            self._stop.wait(0.05)

    def start(self):
        if self._nv is not None:
            self._thread = threading.Thread(target=self._run, daemon=True)
            self._thread.start()

    def stop(self) -> dict:
        self._stop.set()
        if self._thread is not None:
            self._thread.join()
        s = sorted(self.samples)
        return {"sm_mhz": s[len(s) // 2] if s else None, "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(s)}


# ------------------------------------------------------------------------------------------------
# CPU oracle timing (reported baseline / reference arm).  The oracle is timed as it stands.
# ------------------------------------------------------------------------------------------------
def oracle_step(k: int, inputs=None):
    """One pass of the oracle's four stages on the BASELINE recipe at order k, nev = k/4.
    Returns (seconds, per-stage seconds, inputs)."""
    import oracle
    from paper_2502_02460_b200 import workloads as wl

    if inputs is None:
        p = wl.make_pencil(k, wl.scaled_box(k), wl.BASE_SEED + 1)   # configs[1]'s seed when k = 4096
        inputs = (p.H.numpy(), p.S.numpy(), wl.dense_rhs(k, k // 4, 1).numpy())
    H, S, Ct = inputs
    t0 = time.perf_counter()
    U = oracle.cholesky(S)
    t1 = time.perf_counter()
    V = oracle.invert_upper(U)
    t2 = time.perf_counter()
    oracle.to_standard(H, V)
    t3 = time.perf_counter()
    oracle.backtransform(V, Ct)
    t4 = time.perf_counter()
    return t4 - t0, dict(zip(STAGES, (t1 - t0, t2 - t1, t3 - t2, t4 - t3))), inputs


def _one_thread_oracle(k: int):
    """The same oracle on ONE host thread (OMP_NUM_THREADS=1 in a child process), at a smaller order so that it
    stays within seconds.  Returns {"value", "sample_N", "seconds"} or None."""
    import subprocess
    code = ("import json, bench; sec, st, _ = bench.oracle_step(%d); "
            "print(json.dumps({'seconds': sec}))" % k)
    try:
        env = dict(os.environ, OMP_NUM_THREADS="1", CUDA_VISIBLE_DEVICES="")
        out = subprocess.run([sys.executable, "-c", code], cwd=ROOT, env=env, capture_output=True, text=True, timeout=300)
        sec = json.loads(out.stdout.strip().splitlines()[-1])["seconds"]
    except Exception:
        return None
    from paper_2502_02460_b200 import workloads as wl
    return {"value": wl.nominal_flops(k, k // 4)["total"] / sec / 1e12, "unit": UNIT, "cores": 1, "sample_N": k, "seconds": sec}


def cpu_baseline(k: int) -> dict:
    import oracle
    from paper_2502_02460_b200 import workloads as wl

    sec, stages, _ = oracle_step(k)
    fl = wl.nominal_flops(k, k // 4)["total"]
    return {"value": fl / sec / 1e12, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
            "sample": f"one pass of the four oracle stages on the BASELINE recipe at N={k}, nev={k // 4} "
                      f"(configs[1] size; the full N=16384 oracle would take hours)",
            "seconds": sec, "stage_seconds": stages,
            "one_thread": _one_thread_oracle(min(k, 1536))}


def run_reference(args):
    """Reference arm: the CPU oracle on the host cores, rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    import oracle
    from paper_2502_02460_b200 import workloads as wl

    # size the per-step sample so that the whole (warmup + steps) run ends within ~3 minutes:
    # probe the oracle's rate at N=1024, then take the largest order whose predicted cost fits
    probe_sec, _, _ = oracle_step(1024)
    k = 1024
    for cand in (args.cpu_sample, 3072, 2048):
        if cand <= args.cpu_sample and probe_sec * (cand / 1024.0) ** 3 * (args.steps + args.warmup) <= 180.0:
            k = cand
            break
    fl = wl.nominal_flops(k, k // 4)["total"]
    inputs = None
    warm = args.warmup
    for _ in range(warm):
        _, _, inputs = oracle_step(k, inputs)
    total = 0.0
    for _ in range(args.steps):
        sec, _, inputs = oracle_step(k, inputs)
        total += sec
    value = fl * args.steps / total / 1e12
    cfg = wl.CONFIGS[args.config]
    sample = (f"each step = one pass of the four oracle stages on the BASELINE recipe at N={k}, nev={k // 4} "
              f"(bounded sample of {cfg.name}); warm-up passes run: {warm}")
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": total / args.steps * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": cfg.name, "sample_N": k, "sample_nev": k // 4},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


# ------------------------------------------------------------------------------------------------
# the CUDA path
# ------------------------------------------------------------------------------------------------
def _measured_peaks() -> dict:
    try:
        return json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        return {}


TRAFFIC_FILE = os.path.join("profiles", "dominant_kernel_traffic.json")


def _ncu_traffic(label: str):
    """Per-launch DRAM bytes of the dominant kernel from the committed ncu capture (profiles/), or None."""
    try:
        d = json.load(open(os.path.join(ROOT, TRAFFIC_FILE)))
        return d.get(label)
    except Exception:
        return None


def _traffic_source() -> dict:
    """Where `roofline.traffic` comes from: the committed file, its git blob id (so that a stale capture is visible
    in the bench line: the id changes only when the capture is regenerated) and the capture it was made from."""
    import hashlib
    try:
        raw = open(os.path.join(ROOT, TRAFFIC_FILE), "rb").read()
        blob = hashlib.sha1(b"blob %d\0" % len(raw) + raw).hexdigest()
        return {"file": TRAFFIC_FILE, "git_blob": blob, "capture": json.loads(raw).get("_source")}
    except Exception:
        return {"file": TRAFFIC_FILE, "git_blob": None}


def _nvml_index(local_rank: int) -> int:
    vis = os.environ.get("CUDA_VISIBLE_DEVICES", "")
    ids = [v for v in vis.split(",") if v.strip()]
    if local_rank < len(ids) and ids[local_rank].strip().isdigit():
        return int(ids[local_rank])
    return local_rank


def run_ours(args):
    import torch

    from paper_2502_02460_b200 import gs
    from paper_2502_02460_b200 import workloads as wl

    from paper_2502_02460_b200 import replicas

    info = replicas.rank_info()
    rank, world, local_rank = info.rank, info.world, info.local_rank
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    replicas.init(info, "nccl", dev)

    def barrier():
        replicas.barrier(info)

    def max_over_ranks(x: float) -> float:
        return replicas.max_over_ranks(info, x, dev)

    cfg = wl.CONFIGS[args.config]
    if args.n > 0:      # a context run at another size (same recipe, box scaled like configs 1-4): never the headline
        cfg = wl.Config(9, args.n, args.nev if args.nev > 0 else args.n // 4, False, wl.scaled_box(args.n))
    N, nev = cfg.N, cfg.nev
    cplx = cfg.complex
    tdt = torch.complex128 if cplx else torch.float64
    flops = wl.nominal_flops(N, nev, cplx)     # complex: real-equivalent = 4x the real formulas

    # every rank reduces its own independent pencil (replicas; different seed per rank)
    pencil = wl.make_pencil(N, cfg.box, replicas.replica_seed(cfg.seed, rank), complex=cplx, device=dev)
    H, S0 = pencil.H, pencil.S
    U = wl.colmajor_empty(N, N, dtype=tdt, device=dev)
    V = wl.colmajor_empty(N, N, dtype=tdt, device=dev)
    Ht = wl.colmajor_zeros(N, N, dtype=tdt, device=dev)
    Ct = wl.dense_rhs(N, nev, seed=rank, complex=cplx, device=dev)
    C = wl.colmajor_empty(N, nev, dtype=tdt, device=dev)
    plan = gs.Plan(N, nev, dtype=gs.GS_COMPLEX128 if cplx else gs.GS_REAL64, device=dev)

    # FP64 roofline denominator, measured on this device right now (MEASURED_PEAKS.json has no FP64 entry)
    dmma_sus, dmma_burst = gs.measure_fp64_peak(0, 1.0)
    dfma_sus, dfma_burst = gs.measure_fp64_peak(1, 0.5)
    fp64_peak = max(dmma_sus, dfma_sus)

    nvtx = torch.cuda.nvtx

    def one_step(ev=None):
        """The four ABI calls; NVTX ranges name the stages for `ncu --nvtx --nvtx-include "<stage>/"`."""
        U.copy_(S0)                       # restore S (outside the per-step events)
        if ev is not None:
            ev[0].record()
        nvtx.range_push("cholesky")
        plan.cholesky(U)
        nvtx.range_pop()
        if ev is not None:
            ev[1].record()
        nvtx.range_push("invert")
        plan.invert_triangular(U, V)
        nvtx.range_pop()
        if ev is not None:
            ev[2].record()
        nvtx.range_push("to_standard")
        plan.to_standard(H, V, Ht)
        nvtx.range_pop()
        if ev is not None:
            ev[3].record()
        nvtx.range_push("backtransform")
        plan.backtransform(V, Ct, C)
        nvtx.range_pop()
        if ev is not None:
            ev[4].record()

    for _ in range(args.warmup):
        one_step()
    plan.last_info()
    torch.cuda.synchronize()
    barrier()

    sampler = ClockSampler(_nvml_index(local_rank))
    events = [[torch.cuda.Event(enable_timing=True) for _ in range(5)] for _ in range(args.steps)]
    plan.set_timing(2)                    # CUDA events around the dominant kernel only (2 events / step)
    launches0 = plan.launch_count()
    sampler.start()
    wall0 = time.perf_counter()
    for k in range(args.steps):
        one_step(events[k])
    plan.last_info()                      # synchronises the stream, raises on numerical failure
    torch.cuda.synchronize()
    wall1 = time.perf_counter()
    clocks = sampler.stop()
    barrier()
    launches = plan.launch_count() - launches0
    dom = plan.launch_times().get("to_standard.syr2k", (0, 0.0))
    plan.set_timing(0)

    stage_ms = [sum(e[i].elapsed_time(e[i + 1]) for e in events) / args.steps for i in range(4)]
    step_ms = max_over_ranks(sum(stage_ms))
    value = replicas.aggregate_throughput(info, flops["total"], step_ms)

    # per-kernel device times: one extra (untimed) step with events around every launch
    plan.set_timing(1)
    one_step()
    plan.last_info()
    kernels = {k: {"launches": n, "ms": round(ms, 3)} for k, (n, ms) in plan.launch_times().items()}
    plan.set_timing(0)

    # roofline of the dominant kernel: the SYR2K-shaped launch of gs_to_standard (2N^3/3 flop of the
    # nominal 2.67 N^3-ish path: the largest single launch), timed live with CUDA events above
    dom_flop = (4.0 if cplx else 1.0) * 2.0 * float(N) ** 3 / 3.0
    dom_ms = dom[1] / max(dom[0], 1)
    achieved = dom_flop / (dom_ms * 1e-3) / 1e12 if dom_ms > 0 else None
    mp = _measured_peaks()
    roofline = {
        "bound": "tensor", "kernel": ("ctile_engine_kernel<TN>" if cplx else "tile64_engine_kernel<TN> (64x64 CTA tiles, 4 per logical tile)") + " as to_standard.syr2k (FP64 DMMA)",
        "achieved": achieved, "peak": fp64_peak, "unit": "TFLOP/s",
        "frac": (achieved / fp64_peak) if achieved else None,
        "traffic": _ncu_traffic("to_standard.syr2k.complex" if cplx else "to_standard.syr2k") if N == (8192 if cplx else 16384) else None,
        "traffic_source": _traffic_source(),
        "algorithmic_flop_per_launch": dom_flop, "launch_ms": dom_ms, "launches_timed": dom[0],
        "peak_source": "measured live on this device: sustained mma.sync.m8n8k4.f64 (DMMA) microbenchmark "
                       "(libgs_peak.so); MEASURED_PEAKS.json has no FP64 entry",
        "peaks": {"dmma_sustained": dmma_sus, "dmma_burst": dmma_burst, "dfma_sustained": dfma_sus,
                  "dfma_burst": dfma_burst,
                  "bf16_measured_x_nominal_ratio": (mp.get("bf16_tflops_sustained", 0.0) * 40.0 / 2250.0) or None,
                  "hbm_gbs_measured": mp.get("hbm_gbs")},
    }

    # NEXT-1 (outside the metric): the density matrix P = sum_l f_l c*_l c_l over the nev columns of C
    # (PAPER.md:77), a weighted SYRK / HERK on the same tile engine; nominal N^2 nev flop (one triangle)
    focc = torch.full((nev,), 2.0, dtype=torch.float64, device=dev)
    plan.density_matrix(C, focc, Ht)
    ev_d = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
    ev_d[0].record()
    for _ in range(3):
        plan.density_matrix(C, focc, Ht)
    ev_d[1].record()
    plan.last_info()
    dens_ms = ev_d[0].elapsed_time(ev_d[1]) / 3.0
    dens_flop = (4.0 if cplx else 1.0) * float(N) ** 2 * nev
    next_stages = {"density_matrix": {"ms": round(dens_ms, 3), "tflops": dens_flop / (dens_ms * 1e-3) / 1e12,
                                      "frac_of_fp64_peak": dens_flop / (dens_ms * 1e-3) / 1e12 / fp64_peak,
                                      "nominal_flop": dens_flop}}
    plan.to_standard(H, V, Ht)            # restore H~ for the checks below
    plan.last_info()

    # NEXT-4 (outside the metric): the standard eigenproblem H~ C~ = C~ eps between step 3 and the back-transformation
    # (Table 1 "Tridiag. / Solve / Back"), and the WHOLE generalized solve as one chain
    if not args.no_evp:
        next_stages["standard_evp"] = standard_evp_block(plan, H, S0, U, V, Ht, C, N, nev, cplx, fp64_peak, _measured_peaks().get("hbm_gbs"))
        plan.to_standard(H, V, Ht)        # (the eigensolver destroyed H~)
        plan.last_info()

    stages = {}
    for name, ms in zip(STAGES, stage_ms):
        stages[name] = {"ms": round(ms, 3), "tflops": flops[name] / (ms * 1e-3) / 1e12,
                        "frac_of_fp64_peak": flops[name] / (ms * 1e-3) / 1e12 / fp64_peak}

    # ---- checks (off the timed region, plain torch FP64 on the device) ----
    checks = None
    if not args.no_checks and rank == 0:
        Ut = torch.triu(U)
        checks = {
            "chol_resid_fro": ((Ut.conj().t() @ Ut - S0).norm() / S0.norm()).item(),
            "lower_U_max": torch.tril(U, -1).abs().max().item(),
            "lower_Uinv_max": torch.tril(V, -1).abs().max().item(),
        }
        R = Ut @ V
        R.diagonal().sub_(1.0)
        checks["U_Uinv_minus_I_fro_over_sqrtN"] = R.norm().item() / N ** 0.5
        del R
        Href = V.conj().t() @ (H @ V)
        checks["Htilde_rel_fro_vs_torch"] = (torch.triu(Ht - Href).norm() / torch.triu(Href).norm()).item()
        del Href
        Cref = V @ Ct
        checks["C_rel_fro_vs_torch"] = ((C - Cref).norm() / Cref.norm()).item()
        del Cref, Ut
        checks["ok"] = bool(checks["chol_resid_fro"] < 1e-13 and checks["U_Uinv_minus_I_fro_over_sqrtN"] < 1e-11 and
                            checks["Htilde_rel_fro_vs_torch"] < 1e-11 and checks["C_rel_fro_vs_torch"] < 1e-11 and
                            checks["lower_U_max"] == 0.0 and checks["lower_Uinv_max"] == 0.0)

    # ---- end to end through the host-buffer C ABI calls (pinned host memory, copies inside the timing) ----
    e2e = None
    if not args.no_e2e:
        del U, Ht, C
        torch.cuda.empty_cache()
        hH = torch.empty((N, N), dtype=tdt).pin_memory()
        hS = torch.empty((N, N), dtype=tdt).pin_memory()
        hHt = torch.empty((N, N), dtype=tdt).pin_memory()
        hCt = torch.empty((nev, N), dtype=tdt).pin_memory()
        hC = torch.empty((nev, N), dtype=tdt).pin_memory()
        hH.copy_(H.t())           # buffers hold the column-major images
        hS.copy_(S0.t())
        hCt.copy_(Ct.t())
        scratch = torch.empty(plan.host_scratch_bytes(), dtype=torch.uint8, device=dev)
        e2e_steps = max(1, min(args.steps, 3))

        def e2e_step():
            plan.reduce_host(hH, hS, None, None, hHt, scratch)
            plan.backtransform_host(hCt, hC, scratch)

        e2e_step()
        torch.cuda.synchronize()
        barrier()
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            e2e_step()
        torch.cuda.synchronize()
        t1 = time.perf_counter()
        barrier()
        e2e_sec = max_over_ranks((t1 - t0) / e2e_steps)
        esz = 16 if cplx else 8
        e2e = {"value": world * flops["total"] / e2e_sec / 1e12, "unit": UNIT,
               "h2d_bytes_per_step": plan.reduce_host_h2d_bytes() + N * nev * esz, "d2h_bytes_per_step": plan.reduce_host_d2h_bytes() + N * nev * esz,
               "ms_per_step": e2e_sec * 1e3, "steps": e2e_steps,
               "api": "gs_reduce_host + gs_backtransform_host (pinned host buffers in, H~ and C out)"}
        if checks is not None:
            # the host-buffer path must reproduce the device-buffer path bit for bit (same kernels, same order)
            plan.to_standard(H, V, Ht2 := wl.colmajor_zeros(N, N, dtype=tdt, device=dev))
            plan.last_info()
            checks["e2e_Htilde_equals_device_path"] = bool(torch.equal(torch.triu(hHt.t().to(dev)), torch.triu(Ht2)))
            del Ht2
            Cref = V @ Ct
            checks["e2e_C_rel_fro_vs_torch"] = ((hC.t().to(dev) - Cref).norm() / Cref.norm()).item()
            del Cref
            checks["ok"] = bool(checks["ok"] and checks["e2e_Htilde_equals_device_path"] and checks["e2e_C_rel_fro_vs_torch"] < 1e-11)
        del scratch, hH, hS, hHt, hCt, hC

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu = cpu_baseline(args.cpu_sample)

    if rank == 0:
        print(json.dumps({
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": step_ms, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "c128 (FP64 arithmetic)" if cplx else "f64", "data": "synthetic",
            "config": {"workload": cfg.name, "N": N, "nev": nev, "seed": cfg.seed,
                       "recipe": ("BASELINE.json configs[%d]: Gaussian-overlap S, H = -S(1+0.1g)+diag" % cfg.index) if args.n <= 0 else
                                 "CONTEXT RUN, not a BASELINE config: the same recipe at N=%d (Table 1's size is 40960, PAPER.md:136)" % N,
                       "parallelism": "replicas x%d (one independent pencil per GPU)" % world,
                       "cache": "inputs_larger_than_L2 (each matrix %.1f GiB vs 126 MB L2)" % (N * N * (16 if cplx else 8) / 2 ** 30),
                       "timing": "CUDA events per step on the launching stream; S restored between steps outside the events"},
            "frac_of_fp64_peak": value / world / fp64_peak, "fp64_peak_tflops": fp64_peak,
            "stages": stages, "next_stages": next_stages, "roofline": roofline, "kernels": kernels, "cpu_baseline": cpu, "e2e": e2e,
            "gpu_launches": launches, "clocks": clocks, "checks": checks,
            "wall_s_timed_region": wall1 - wall0,
            "paper_context": "PAPER.md:133 Table 1 (ELPA 2024.05, NCCL, 4x A100-40GB, N=40960, nev=N): Cholesky 2.3 s, "
                             "Invert 1.8 s, Multiply 18.8 s, Backtr. 6.8 s = 29.7 s, i.e. ~6.2 TFLOP/s on 4 GPUs (context only)",
        }))
    replicas.finalize(info)


def standard_evp_block(plan, H, S0, U, V, Ht, C, N, nev, cplx, fp64_peak, hbm_gbs):
    """Times the three stages of the standard eigensolver on the H~ the path just formed, then the whole generalized
    solve (steps 1-3, eigensolver, back-transformation) as one chain; checks the acceptance metrics on the result."""
    import torch
    from paper_2502_02460_b200 import metrics as M

    plan.ensure_evp_workspace()
    C = torch.empty_like(C)               # (the caller's C keeps the back-transform of its own C~ for the checks)
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
    A = Ht.clone()
    plan.evp_tridiagonalize(A)            # warm-up (module load, workspace touch)
    A.copy_(Ht)
    ev[0].record()
    d, e, tau = plan.evp_tridiagonalize(A)
    ev[1].record()
    eps, Z = plan.evp_tridiag_solve(d, e)
    ev[2].record()
    Ct = plan.evp_backtransform(A, Z)
    ev[3].record()
    plan.last_info()
    t_tri, t_solve, t_back = (ev[i].elapsed_time(ev[i + 1]) for i in range(3))
    f = 4.0 if cplx else 1.0
    es = 16 if cplx else 8
    tri_bytes = 4.0 * float(N) ** 3 / 3.0 * (es / 8.0)       # one triangle of the leading block per step: sum_m 4 m^2 (x2 complex)
    back_flop = f * 2.0 * float(N) ** 2 * nev
    her2k_flop = f * 2.0 * float(N) ** 3 / 3.0
    # eigenvalues only: bisection on (d, e) instead of Solve and Back
    evb = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
    plan.evp_tridiag_eigenvalues(d, e, count=nev)                # warm-up (loads the kernel)
    evb[0].record()
    lam = plan.evp_tridiag_eigenvalues(d, e, count=nev)
    evb[1].record()
    plan.last_info()
    t_bisect = evb[0].elapsed_time(evb[1])
    bisect_diff = float((lam - eps).abs().max() / max(1.0, float(eps.abs().max())))
    # per-label device times of one more pass
    A.copy_(Ht)
    plan.set_timing(1)
    d, e, tau = plan.evp_tridiagonalize(A)
    eps, Z = plan.evp_tridiag_solve(d, e)
    Ct = plan.evp_backtransform(A, Z)
    plan.last_info()
    kern = {k: {"launches": n, "ms": round(ms, 3)} for k, (n, ms) in plan.launch_times().items() if k.startswith("evp.")}
    plan.set_timing(0)
    out = {
        "method": "one-stage Householder tridiagonalisation (ELPA1 route, PAPER.md:120) / divide and conquer / compact-WY back-transformation",
        "tridiag": {"ms": round(t_tri, 3), "bound": "hbm", "algorithmic_bytes": tri_bytes,
                    "achieved_gbs": tri_bytes / (t_tri * 1e-3) / 1e9,
                    "frac_of_hbm": (tri_bytes / (t_tri * 1e-3) / 1e9 / hbm_gbs) if hbm_gbs else None, "hbm_gbs_peak": hbm_gbs,
                    "her2k_tflops": (her2k_flop / (kern["evp.tridiag.her2k"]["ms"] * 1e-3) / 1e12) if "evp.tridiag.her2k" in kern else None},
        "solve": {"ms": round(t_solve, 3), "bound": "tensor (block products) + latency (secular equation, deflation)",
                  "gemm_ms": kern.get("evp.solve.gemm", {}).get("ms")},
        "back": {"ms": round(t_back, 3), "bound": "tensor", "nominal_flop": back_flop,
                 "tflops": back_flop / (t_back * 1e-3) / 1e12, "frac_of_fp64_peak": back_flop / (t_back * 1e-3) / 1e12 / fp64_peak},
        "eigenvalues_only": {"bisect_ms": round(t_bisect, 3), "total_ms": round(t_tri + t_bisect, 3), "bound": "latency (one dependent FMA per row and count)",
                             "max_diff_to_solve_rel": bisect_diff},
        "total_ms": round(t_tri + t_solve + t_back, 3), "kernels": kern,
    }
    # the whole generalized solve, one chain on one stream
    evc = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
    U.copy_(S0)
    evc[0].record()
    plan.cholesky(U)
    plan.invert_triangular(U, V)
    plan.to_standard(H, V, Ht)
    eps, Ct = plan.standard_eigh(Ht)
    plan.backtransform(V, Ct, C)
    evc[1].record()
    plan.last_info()
    out["generalized_solve_ms"] = round(evc[0].elapsed_time(evc[1]), 3)
    out["checks"] = {"eig_residual": M.eig_residual(H, S0, C, eps), "s_orthonormality": M.s_orthonormality(S0, C),
                     "tolerances": {"eig_residual": M.TOL_RESIDUAL, "s_orthonormality": M.TOL_SORTH}}
    out["checks"]["ok"] = bool(out["checks"]["eig_residual"] <= M.TOL_RESIDUAL and out["checks"]["s_orthonormality"] <= M.TOL_SORTH)
    out["paper_context"] = ("PAPER.md:133 Table 1 (ELPA 2024.05, NCCL, 4x A100-40GB, N=40960, nev=N): Tridiag. 49.5 s, Solve 40.1 s, "
                            "Back 14.6 s; whole generalized solve 134 s (context only)")
    del A, Z, Ct
    return out


def run_batch(args):
    """NEXT-2: K mid-size pencils concurrently on K streams vs one after the other."""
    import torch

    from paper_2502_02460_b200 import workloads as wl
    from paper_2502_02460_b200.batch import Batch

    torch.cuda.set_device(0)
    K, N, cplx = args.batch, args.batch_n, args.batch_complex
    nev = N // 4
    flops = wl.nominal_flops(N, nev, cplx)["total"]
    pens = [wl.make_pencil(N, wl.scaled_box(N), wl.BASE_SEED + 700 + k, complex=cplx, device="cuda") for k in range(K)]
    b = Batch(K, N, nev, complex=cplx)
    U, V, Ht, C = b.alloc(), b.alloc(), b.alloc(zeros=True), b.alloc(cols=nev)
    Ct = [wl.dense_rhs(N, nev, seed=k, complex=cplx, device="cuda") for k in range(K)]
    H, S = [p.H for p in pens], [p.S for p in pens]

    def concurrent():
        b.reduce(H, S, U, V, Ht)
        b.backtransform(V, Ct, C)

    def sequential():
        for k in range(K):
            U[k].copy_(S[k])
            b.plans[k].cholesky(U[k])
            b.plans[k].invert_triangular(U[k], V[k])
            b.plans[k].to_standard(H[k], V[k], Ht[k])
            b.plans[k].backtransform(V[k], Ct[k], C[k])

    out = {}
    for name, fn in (("sequential", sequential), ("concurrent", concurrent)):
        for _ in range(max(1, args.warmup)):
            fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(args.steps):
            fn()
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / args.steps
        out[name] = {"ms_per_batch": ms, "tflops": K * flops / (ms * 1e-3) / 1e12}
    assert b.last_info() == [0] * K
    print(json.dumps({"metric": "FP64 TFLOP/s of K independent reductions in flight (NEXT-2, not the headline)",
                      "unit": UNIT, "value": out["concurrent"]["tflops"], "n_gpus": 1, "steps": args.steps, "warmup": args.warmup,
                      "config": {"workload": f"batch_K{K}_N{N}_{'c128' if cplx else 'f64'}_nev{nev}"}, "dtype": "c128" if cplx else "f64",
                      "data": "synthetic", "detail": out}))


def run_sharded(args):
    """NEXT-3 under torchrun: every rank holds the SAME pencil; step 1 replicated, steps 2-4 by column ranges
    with one exchange of the U^-1 and G slabs (NCCL broadcasts over NVLink), C gathered at the end."""
    import torch

    from paper_2502_02460_b200 import gs, metrics as M, replicas, sharded
    from paper_2502_02460_b200 import workloads as wl

    info = replicas.rank_info()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    torch.cuda.set_device(info.local_rank)
    dev = torch.device("cuda", info.local_rank)
    replicas.init(info, "nccl", dev)
    cfg = wl.CONFIGS[args.config]
    N, nev, cplx = cfg.N, cfg.nev, cfg.complex
    pen = wl.make_pencil(N, cfg.box, cfg.seed, complex=cplx, device=dev)      # the same on every rank
    plan = gs.Plan(N, nev, dtype=gs.GS_COMPLEX128 if cplx else gs.GS_REAL64, device=dev)
    drv = sharded.ShardedReduction(plan, info.rank, info.world, exchange=args.exchange, sync=args.shard_sync, chol=args.shard_chol_mode)
    bufs = drv.alloc(pen.H)
    Ct = wl.dense_rhs(N, nev, seed=0, complex=cplx, device=dev)
    C = bufs.C if drv.push else wl.colmajor_empty(N, nev, dtype=pen.H.dtype, device=dev)

    def step():
        res = drv.reduce(pen.H, pen.S, out=bufs)
        drv.backtransform(res.Uinv, Ct, out=C)

    for _ in range(max(3, args.warmup)):
        step()
    replicas.barrier(info)
    torch.cuda.synchronize()
    l0 = plan.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    torch.cuda.synchronize()
    replicas.barrier(info)
    ms = replicas.max_over_ranks(info, e0.elapsed_time(e1) / args.steps, dev)
    launches = plan.launch_count() - l0
    Ht = drv.gather_htilde(bufs)
    checks = None
    if info.rank == 0 and not args.no_checks:      # against the whole-matrix calls on this rank
        V1 = wl.colmajor_empty(N, N, dtype=pen.H.dtype, device=dev)
        plan.invert_triangular(bufs.U, V1)
        plan.to_standard(pen.H, V1, bufs.G)        # G is free now; upper triangle of H~ by the one-GPU path
        plan.last_info()
        checks = {"Uinv_rel_fro_vs_one_gpu_path": M.rel_frob_upper(bufs.Uinv, V1),
                  "Htilde_rel_fro_vs_one_gpu_path": M.rel_frob_upper(Ht, bufs.G)}
        checks["ok"] = bool(max(checks.values()) <= M.TOL_FROB)
    flops = wl.nominal_flops(N, nev, cplx)["total"]
    if info.rank == 0:
        print(json.dumps({"metric": METRIC, "value": flops / (ms * 1e-3) / 1e12, "unit": UNIT, "n_gpus": info.world,
                          "steps": args.steps, "warmup": max(3, args.warmup), "ms_per_step": ms, "higher_is_better": True,
                          "scaling": "strong", "vs_baseline": None, "dtype": "c128 (FP64 arithmetic)" if cplx else "f64",
                          "data": "synthetic",
                          "config": {"workload": cfg.name, "N": N, "nev": nev, "seed": cfg.seed,
                                     "parallelism": f"sharded x{info.world}: step 1 " +
                                                    ("over the ranks (gs_cholesky_sharded)" if drv.chol_sharded else "per rank on the leading block it needs") +
                                                    ", steps 2-4 by column ranges, one exchange of the U^-1 and G slabs (NEXT-3)",
                                     "sync": "device-side flags" if drv.device_sync else "host barriers",
                                     "exchange": ("push: fused into the kernel epilogues over peer memory" if drv.push else
                                                  "collective: broadcasts after the kernels" if info.world > 1 else "none (one rank)"),
                                     "column_ranges": drv.ranges},
                          "gpu_launches": launches, "checks": checks}))
    drv.close()
    replicas.finalize(info)


def run_shard_chol(args):
    """NEXT-3, step 1 over R ranks (gs_cholesky_sharded), on ONE GPU: (a) the look-ahead factorisation of the contract
    path, (b) the same entry point with one rank (no look-ahead, one stream), (c) R emulated ranks = R plans on R streams
    sharing the device (correctness and the total work incl. the copies -- NOT a parallel time), (d) the serial part:
    the owner's diagonal-block chain, timed as a one-rank factorisation of one panel plus one block, times the number of
    panels.  Projection at R GPUs, compute only: between chain + (one-rank time - chain) / R (nothing overlaps the chains)
    and one panel + max(the other chains, the rest / R) (the look-ahead hides the shorter of the two completely)."""
    import torch

    from paper_2502_02460_b200 import gs
    from paper_2502_02460_b200 import workloads as wl

    torch.cuda.set_device(0)
    R = args.shard_chol
    cfg = wl.CONFIGS[args.config]
    N, cplx = cfg.N, cfg.complex
    pen = wl.make_config(cfg, device="cuda")
    dtc = gs.GS_COMPLEX128 if cplx else gs.GS_REAL64

    def timed(fn, prep):
        ts = []
        for it in range(args.warmup + args.steps):
            prep()
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            fn()
            e1.record()
            torch.cuda.synchronize()
            if it >= args.warmup:
                ts.append(e0.elapsed_time(e1))
        return sum(ts) / len(ts)

    plan = gs.Plan(N, 0, dtype=dtc)
    U = wl.colmajor_empty(N, N, dtype=pen.S.dtype, device="cuda")
    t_look = timed(lambda: plan.cholesky(U), lambda: U.copy_(pen.S))
    t_one = timed(lambda: plan.cholesky_sharded(U, 0, 1), lambda: U.copy_(pen.S))
    plan.last_info()
    U_ref = U.clone()
    panel = plan.block * 8
    npanels = (N + panel - 1) // panel
    Np = min(N, panel + plan.block)
    pp = gs.Plan(Np, 0, dtype=dtc)
    Sp = wl.to_colmajor(pen.S[:Np, :Np].contiguous())
    Up = torch.empty_like(Sp)
    t_panel = timed(lambda: pp.cholesky_sharded(Up, 0, 1), lambda: Up.copy_(Sp))
    pp.last_info()
    pp.close()
    plans = [plan] + [gs.Plan(N, 0, dtype=dtc) for _ in range(R - 1)]
    streams = [torch.cuda.Stream() for _ in range(R)]
    Us = [U] + [wl.colmajor_empty(N, N, dtype=pen.S.dtype, device="cuda") for _ in range(R - 1)]
    flags = [torch.zeros(R, dtype=torch.int32, device="cuda") for _ in range(R)]
    nep = plan.cholesky_sharded_epochs()
    state = {"epoch": 0}

    def prep():
        for x in Us:
            x.copy_(pen.S)

    def emul():
        # one host thread per emulated rank (as one process per GPU would be): a rank's stream blocks on its waits, and a
        # single thread that filled one stream's launch queue could never get to enqueue the rank it is waiting for
        import threading
        ev = torch.cuda.Event()
        ev.record()

        def rank_program(r):
            torch.cuda.set_device(0)
            streams[r].wait_event(ev)
            plans[r].cholesky_sharded(Us[r], r, R, [x.data_ptr() for x in Us], [pl.workspace.data_ptr() for pl in plans],
                                      [f.data_ptr() for f in flags], epoch0=state["epoch"], stream=streams[r])
        th = [threading.Thread(target=rank_program, args=(r,)) for r in range(R)]
        for t in th:
            t.start()
        for t in th:
            t.join()
        state["epoch"] += nep
        for st in streams:
            torch.cuda.current_stream().wait_stream(st)
    t_emul = timed(emul, prep) if R > 1 else t_one
    for pl in plans:
        pl.last_info()
    same = all(bool(torch.equal(x, Us[0])) for x in Us)
    err = float((torch.triu(Us[0]) - torch.triu(U_ref)).norm() / torch.triu(U_ref).norm())
    t_chain = min(npanels * t_panel, t_one)
    t_proj = t_chain + (t_one - t_chain) / R                 # no overlap of the chains with anything
    t_proj_overlap = t_panel + max(t_chain - t_panel, (t_one - t_chain) / R)   # the look-ahead hides whichever is shorter
    flop = wl.nominal_flops(N, 0, cplx)["cholesky"]
    print(json.dumps({"metric": "step 1 (Cholesky) over R ranks, gs_cholesky_sharded, emulated on one GPU + model projection (NEXT-3, not the headline)",
                      "unit": "ms", "n_gpus": 1, "ranks": R, "steps": args.steps, "warmup": args.warmup, "dtype": "c128" if cplx else "f64",
                      "data": "synthetic", "config": {"workload": f"shard_chol_R{R}_{cfg.name}"},
                      "value": t_proj,
                      "detail": {"cholesky_lookahead_ms": t_look, "sharded_one_rank_ms": t_one, "emulated_R_ranks_on_one_gpu_ms": t_emul,
                                 "one_panel_ms": t_panel, "panels": npanels, "chain_ms": t_chain,
                                 "projected_R_gpus_ms": t_proj, "projected_tflops": flop / (t_proj * 1e-3) / 1e12,
                                 "projected_R_gpus_full_overlap_ms": t_proj_overlap,
                                 "all_ranks_bit_identical": same, "rel_frob_vs_one_rank": err,
                                 "note": "projections: the owners' diagonal-block chains (serial) + the rest / R, and with the look-ahead hiding the shorter of the two; copies over NVLink and flag latency not included"}}))
    assert same and err <= 1e-12


def run_shard_shares(args):
    """NEXT-3: the column-range calls of every one of R ranks, timed on ONE GPU one rank
    after the other.  No multi-GPU hardware is available to this run, so the exchange is not timed: the
    line reports what each rank would compute -- its leading-block Cholesky and its column ranges of steps 2-4
    (max over ranks = the step's compute time at R GPUs) -- and the bytes the one exchange step moves."""
    import torch

    from paper_2502_02460_b200 import gs, sharded
    from paper_2502_02460_b200 import workloads as wl

    torch.cuda.set_device(0)
    R = args.shard_shares
    cfg = wl.CONFIGS[args.config]
    N, nev, cplx = cfg.N, cfg.nev, cfg.complex
    pen = wl.make_config(cfg, device="cuda")
    dt = pen.H.dtype
    plan = gs.Plan(N, nev, dtype=gs.GS_COMPLEX128 if cplx else gs.GS_REAL64)
    U, V, G, Ht = (wl.colmajor_empty(N, N, dtype=dt, device="cuda") for _ in range(4))
    Ct = wl.dense_rhs(N, nev, seed=3, complex=cplx, device="cuda")
    C = wl.colmajor_empty(N, nev, dtype=dt, device="cuda")
    ranges = sharded.column_ranges(N, R, plan.block)
    eig = sharded.even_ranges(nev, R, 2)

    def timed(fn):
        for _ in range(max(1, args.warmup)):
            fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(args.steps):
            fn()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / args.steps

    def chol(ncols):
        U.copy_(pen.S)
        plan.cholesky_leading(U, ncols)
    t_copy = timed(lambda: U.copy_(pen.S))
    t_chol = timed(lambda: chol(N)) - t_copy     # leaves all of U
    plan.invert_triangular(U, V)           # complete V, G for the step-3 shares
    for c0, c1 in ranges:
        plan.to_standard_g_cols(pen.H, V, G, c0, c1 - c0)
    ranks = []
    Us = wl.colmajor_empty(N, N, dtype=dt, device="cuda")
    Vr = wl.colmajor_empty(N, N, dtype=dt, device="cuda")

    def chol_lead(ncols):
        Us.copy_(pen.S)
        plan.cholesky_leading(Us, ncols)
    for r, ((c0, c1), (k0, k1)) in enumerate(zip(ranges, eig)):
        w = c1 - c0
        def ranged(name, fn):       # NVTX range per stage and rank: `ncu --nvtx --nvtx-include "shard.<stage>.r<rank>/"`
            def run():
                torch.cuda.nvtx.range_push(f"shard.{name}.r{r}")
                fn()
                torch.cuda.nvtx.range_pop()
            return run
        t = {"cols": [c0, c1], "eig_cols": [k0, k1],
             "cholesky_leading": (timed(ranged("cholesky", lambda: chol_lead(c1))) - t_copy) if w > 0 else 0.0,
             "invert": timed(ranged("invert", lambda: plan.invert_triangular_cols(U, Vr, c0, w))),
             "g": timed(ranged("g", lambda: plan.to_standard_g_cols(pen.H, V, G, c0, w))),
             "syr2k": timed(ranged("syr2k", lambda: plan.to_standard_cols(V, G, Ht, c0, w))),
             "backtransform": timed(ranged("back", lambda: plan.backtransform_cols(V, Ct, C, k0, k1 - k0)))}
        t["sum_ms"] = t["cholesky_leading"] + t["invert"] + t["g"] + t["syr2k"] + t["backtransform"]
        ranks.append(t)
    plan.last_info()
    es = 16 if cplx else 8
    total_ms = max(t["sum_ms"] for t in ranks)
    flops = wl.nominal_flops(N, nev, cplx)["total"]
    print(json.dumps({"metric": "FP64 TFLOP/s of the column-sharded path at R ranks, compute only, projected from one GPU (NEXT-3, not the headline)",
                      "unit": UNIT, "value": flops / (total_ms * 1e-3) / 1e12, "n_gpus": 1, "ranks_projected": R,
                      "steps": args.steps, "warmup": args.warmup, "dtype": "c128" if cplx else "f64", "data": "synthetic",
                      "config": {"workload": f"shard_R{R}_{cfg.name}"},
                      "detail": {"cholesky_whole_ms": t_chol, "step_ms": total_ms,
                                 "sum_over_ranks_ms": sum(t["sum_ms"] for t in ranks),
                                 "chol_weight": sharded.CHOL_WEIGHT,
                                 "exchange_bytes_per_rank_received": 2 * N * N * es, "exchange": "not timed (one GPU)",
                                 "ranks": ranks}}))


def main():
    args = parse_args()
    if args.batch > 0:
        run_batch(args)
        return
    if args.shard_shares > 0:
        run_shard_shares(args)
        return
    if args.shard_chol > 0:
        run_shard_chol(args)
        return
    if args.sharded and args.impl == "ours":
        run_sharded(args)
        return
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
