#!/usr/bin/env python
"""bench.py -- LB-CNN kernel-selection inner loop on B200: candidates/s through expand + fit + score.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload mnist] [--impl cuda|reference]

A "step" is ONE pass of the whole hot path over one batch
of synthetic input: one lbcnn_search_candidates call that expands the train and test sets through the
binary-conv layers for every candidate kernel set of the workload, fits the ELM output layer per
candidate, scores the held-out set and picks best / worst.  Default workload =
BASELINE.json configs[1] ("MNIST-shaped reduced-subset search": N_train 20000, N_test 10000, 64 candidates).

One JSON line on stdout (rank 0):
  value        candidates/s, inputs resident in HBM, CUDA events on the launching stream, max over ranks
  e2e          the same metric through lbcnn_search_candidates_host: HOST (pinned) buffers, host<->device
               copies inside the timed region
  roofline     dominant kernel of the step: algorithmic work / its CUDA-event time in the timed region
  cpu_baseline the oracle (oracle/, as it stands) on this box's host cores on a bounded sample
  gpu_launches kernels liblbcnn enqueued inside the timed region (counted by the library)

--impl reference times the oracle itself (this tier's reference arm): each step = `--ref-cands` candidate(s)
of the same workload at full N on the host cores.

Multi-GPU (torchrun, one rank per GPU): candidates are independent, the path has no exchange step, so every
rank searches its OWN batch of n_cand candidate kernel sets on the same images ("replicas only", weak
scaling); the only collectives are the timing barrier and the max over ranks.
"""
from __future__ import annotations

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

# cpu_baseline sample per workload: (candidates, N_train, N_test), sized for about 10-30 s of host work
CPU_SAMPLE = {"tiny_mnist": (8, 2000, 500), "mnist": (10, 20000, 10000), "orl": (32, 280, 120),
              "gtsrb": (1, 3000, 1263), "vggface": (1, 1000, 250)}

METRIC = "ELM candidate kernel-sets evaluated/sec (expand+fit+score); % HBM & tensor roofline"
UNIT = "candidates/s"


def _peaks():
    """measured roofline denominators (driver-written MEASURED_PEAKS.json), else the profiling guide's fallback."""
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return dict(hbm_gbs=float(d["hbm_gbs"]), bf16_burst=float(d["bf16_tflops"]),
                    bf16_sustained=float(d.get("bf16_tflops_sustained", d["bf16_tflops"])), source="measured")
    return dict(hbm_gbs=6650.0, bf16_burst=1590.0, bf16_sustained=1400.0, source="fallback")


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (profiling guide's clocks line)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for ln in self.proc.stdout:
            self.lines.append(ln.strip())

    def stop(self):
        if self.proc is None:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["nvidia-smi unavailable"])
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1])); mx.append(float(f[2]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["no samples"])
        sm.sort()
        return dict(sm_mhz=sm[len(sm) // 2], sm_max_mhz=max(mx), reasons=sorted(reasons), samples=len(sm))


def _phase_rooflines(w, F, n_cand, phase_ms, steps, peaks, sustained: bool):
    """Algorithmic work per step for each phase (SURVEY.md 8(d) / DESIGN.md "Rooflines") over its measured
    CUDA-event time per step.  Returns {phase: roofline-dict}."""
    N, Nte, c = w.n_train, w.n_test, w.n_classes
    px = w.in_h * w.in_w * w.in_c
    primal = F < N
    dim = F if primal else N
    hbm = peaks["hbm_gbs"]
    # fp32-accurate tensor peak: TF32 dense = bf16 / 2 (guide's nominal ratio 1.1 / 2.25 PF), three TF32 passes
    bf16 = peaks["bf16_sustained"] if sustained else peaks["bf16_burst"]
    tens = bf16 / 2.0 / 3.0
    work = {
        # H written once (4 F bytes per image per candidate) + every image read once per launch
        "expand": ("hbm", "GB/s", hbm, (n_cand * (N + Nte) * F * 4.0 + (N + Nte) * px) / 1e9),
        # symmetric half of the Gram: N dim (dim + 1) flop per candidate (primal), F N (N + 1) (dual)
        "gram": ("tensor", "TFLOP/s", tens, n_cand * (float(N) * F * (F + 1) if primal else float(F) * N * (N + 1)) / 1e12),
        "rhs": ("hbm", "GB/s", hbm, (n_cand * float(N) * F * 4.0 if primal else n_cand * float(N) * c * 8.0) / 1e9),
        # Cholesky dim^3/3 + two triangular solves with c right-hand sides 2 dim^2 c (+ dual back-projection 2 N F c)
        "solve": ("tensor", "TFLOP/s", tens,
                  n_cand * (dim ** 3 / 3.0 + 2.0 * dim * dim * c + (0 if primal else 2.0 * N * F * c)) / 1e12),
        # test features read once + W
        "score": ("hbm", "GB/s", hbm, n_cand * (float(Nte) * F * 4.0 + F * c * 4.0) / 1e9),
    }
    out = {}
    for ph, (bound, unit, peak, amount) in work.items():
        ms = phase_ms.get(ph, (0.0, 0))[0] / max(steps, 1)
        if ms <= 0:
            continue
        ach = amount / (ms * 1e-3)
        out[ph] = dict(bound=bound, achieved=round(ach, 3), peak=round(peak, 1), unit=unit, frac=round(ach / peak, 4),
                       traffic=None, ms_per_step=round(ms, 4), work_per_step=round(amount, 4))
    return out


def _oracle_sample(w, trx, try_, tex, tey, n_cand_sample: int, first: int = 0):
    """time the oracle's search loop (as it stands) on `n_cand_sample` candidates of the workload at full N."""
    from oracle import oracle as orc
    from paper_2106_15350_b200 import synth
    ker = synth.make_kernels(w, n_cand_sample, first=first)
    oa = orc.make_arch(w.in_h, w.in_w, w.in_c, w.layers)
    t0 = time.perf_counter()
    r = orc.search(oa, trx, try_, tex, tey, w.n_classes, w.C, ker, feature_scale=w.feature_scale)
    dt = time.perf_counter() - t0
    return dt, r, orc.n_threads()


def run_reference(args):
    """--impl reference: the oracle on the host cores (rank 0 only; other ranks exit 0 without work)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return 0
    from oracle import oracle as orc
    from paper_2106_15350_b200 import synth
    orc.build()
    w = synth.WORKLOADS[args.workload]
    trx, try_, tex, tey = synth.make_dataset(w)
    nc = args.ref_cands
    for i in range(args.warmup):
        _oracle_sample(w, trx, try_, tex, tey, nc, first=i * nc)
    t_tot, threads = 0.0, 1
    for i in range(args.steps):
        dt, _, threads = _oracle_sample(w, trx, try_, tex, tey, nc, first=(args.warmup + i) * nc)
        t_tot += dt
    value = nc * args.steps / t_tot
    sample = "%d candidate(s) per step of workload %s at full N_train=%d N_test=%d" % (nc, w.name, w.n_train, w.n_test)
    line = dict(impl="reference", metric=METRIC, value=value, unit=UNIT, n_gpus=args.gpus, steps=args.steps,
                warmup=args.warmup, ms_per_step=1e3 * t_tot / args.steps, higher_is_better=True, scaling="weak",
                vs_baseline=None, dtype="f64", data="synthetic",
                config=_config(w, nc, "none (host)"),
                cpu_baseline=dict(value=value, unit=UNIT, cores=threads, kind="oracle", sample=sample),
                e2e=dict(value=value, unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0), gpu_launches=0)
    print(json.dumps(line), flush=True)
    return 0


def _config(w, n_cand, l2_note):
    return dict(workload="BASELINE.json configs[%d] (%s): %dx%dx%d u8, N_train=%d N_test=%d classes=%d, layers=%s, C=%g"
                % (w.config - 1, w.name, w.in_h, w.in_w, w.in_c, w.n_train, w.n_test, w.n_classes,
                   "+".join("%d@%dx%d/pool%d" % (L.n_kernels, L.ksize, L.ksize, L.pool_k) for L in w.layers), w.C),
                candidates_per_step=n_cand, parallelism="replicas only (candidates independent; no collective)",
                l2=l2_note)


def run_cuda(args):
    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_2106_15350_b200 import binding as lb
    from paper_2106_15350_b200 import replicas, synth

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: liblbcnn has no CPU path")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    lb.lib()   # raises ImportError if liblbcnn.so is not built

    w = synth.WORKLOADS[args.workload]
    if args.n_cand:
        w = synth.scaled(w, n_cand=args.n_cand)
    K = w.n_cand
    trx, try_, tex, tey = synth.make_dataset(w)
    ker = synth.make_kernels(w, K, first=replicas.first_candidate(rank, K))   # every rank searches its own K candidates
    arch = lb.arch_of(w)
    F, _ = lb.feature_dim(arch)
    dev = torch.device("cuda", local)
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    h_in = [pin(trx), pin(try_), pin(tex), pin(tey), pin(ker)]
    d_in = [t.to(dev) for t in h_in]

    h = lb.Handle(local)
    stage = lb.host_staging_bytes(arch, w.n_train, w.n_test, w.n_classes, K)
    budget = int(args.ws_gb * (1 << 30))
    ws_bytes, ws_min = lb.workspace_bytes(arch, w.n_train, w.n_test, w.n_classes, K, budget)
    h.ensure_workspace(ws_bytes + stage)
    l2_note = "inputs exceed L2: workspace %.2f GB of features/Gram streams through the 126 MB L2 every step" % (ws_bytes / 1e9)

    def step(out=None):
        return h.search_candidates(arch, d_in[0], d_in[1], d_in[2], d_in[3], w.n_classes, w.C, d_in[4], out=out)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    out = step()
    for _ in range(max(args.warmup - 1, 0)):
        step(out)
    barrier()
    # ---- timed region: device-resident inputs, CUDA events on the launching (current) stream ----
    sampler = ClockSampler(local)
    sampler.start()
    h.set_profiling(True)
    n0 = h.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record()
    for _ in range(args.steps):
        step(out)
    e1.record()
    barrier()
    ms = e0.elapsed_time(e1)
    launches = h.launch_count() - n0
    phase_ms = h.phase_times()
    h.set_profiling(False)
    clocks = sampler.stop()
    ms = replicas.max_over_ranks(ms, dev)
    acc = out["acc"].cpu().numpy()
    info = out["info"].cpu().numpy()
    if (info != 0).any() or not np.isfinite(acc).all():
        raise RuntimeError("fit failed for some candidate: info=%s" % info.tolist())

    # ---- e2e: host (pinned) buffers through lbcnn_search_candidates_host, copies inside the timed region ----
    hout = h.search_candidates_host(arch, *h_in[:4], w.n_classes, w.C, h_in[4])
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        h.search_candidates_host(arch, *h_in[:4], w.n_classes, w.C, h_in[4], out=hout)   # synchronises inside
    barrier()
    e2e_s = time.perf_counter() - t0
    e2e_s = replicas.max_over_ranks(e2e_s, dev)
    if not np.array_equal(hout["correct"].numpy(), out["correct"].cpu().numpy()):
        raise RuntimeError("host-buffer path and device-buffer path disagree")
    h2d = sum(t.numel() * t.element_size() for t in h_in)
    d2h = sum(t.numel() * t.element_size() for t in hout.values() if t is not None)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0
    peaks = _peaks()
    total_s = ms * 1e-3
    roofs = _phase_rooflines(w, F, K, phase_ms, args.steps, peaks, sustained=total_s > 2.0)
    dominant = max(roofs, key=lambda p: roofs[p]["ms_per_step"]) if roofs else None
    roofline = dict(roofs[dominant]) if dominant else None
    if roofline:
        roofline["kernel"] = dominant
        roofline["peak_source"] = "%s (%s)" % (peaks["source"],
                                               "HBM copy GB/s" if roofline["bound"] == "hbm" else
                                               "bf16 %s / 2 (TF32 nominal ratio) / 3 (3xTF32 = fp32-accurate)"
                                               % ("sustained" if total_s > 2.0 else "burst"))
        prof = os.path.join(ROOT, "profiles", "traffic_%s.txt" % w.name)   # JSON text written from the ncu capture
        if os.path.exists(prof):      # dram bytes per launch from the committed ncu --set full capture
            with open(prof) as f:
                roofline["traffic"] = json.load(f).get(dominant)
    line = dict(metric=METRIC, value=replicas.job_throughput(world, K, args.steps, total_s), unit=UNIT, n_gpus=world, steps=args.steps,
                warmup=args.warmup, ms_per_step=ms / args.steps, higher_is_better=True, scaling="weak",
                vs_baseline=None, dtype="int8 x int8 -> int32 tensor-core expander and Gram (exact), f64 Cholesky and logits, f32 features/weights",
                data="synthetic", config=_config(w, K, l2_note), clocks=clocks,
                e2e=dict(value=replicas.job_throughput(world, K, args.steps, e2e_s), unit=UNIT, h2d_bytes_per_step=h2d, d2h_bytes_per_step=d2h),
                gpu_launches=int(launches), roofline=roofline, phases=roofs,
                accuracy=dict(best=float(acc.max()), worst=float(acc.min()), best_index=int(out["best"][0].item())))
    if not args.no_cpu_baseline:
        # bounded sample (about 10-30 s of host work): (candidates, N_train, N_test) of the same workload
        nc, ntr, nte = CPU_SAMPLE.get(w.name, (1, w.n_train, w.n_test))
        if args.ref_cands_baseline:
            nc = args.ref_cands_baseline
        nc = min(nc, K)
        full = (ntr >= w.n_train and nte >= w.n_test)
        dt, r, threads = _oracle_sample(w, trx[:ntr], try_[:ntr], tex[:nte], tey[:nte], nc, first=0)
        if full:
            ok = bool(np.all(np.abs(r["acc"] - acc[:nc].astype(np.float64)) * 100.0 <= 0.2))
            sample = ("first %d of %d candidates of the same workload at full N (%.1f s); accuracies agree with the "
                      "GPU's within 0.2 pp: %s" % (nc, K, dt, ok))
        else:
            sample = ("first %d of %d candidates of the same workload on its first %d train / %d test samples "
                      "(%.1f s; the full-N oracle run would take minutes per candidate)" % (nc, K, ntr, nte, dt))
        line["cpu_baseline"] = dict(value=nc / dt, unit=UNIT, cores=threads, kind="oracle", sample=sample)
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--workload", default="mnist", choices=["tiny_mnist", "mnist", "gtsrb", "orl", "vggface"])
    ap.add_argument("--n-cand", type=int, default=0, help="override the workload's candidate count (not a bench line)")
    ap.add_argument("--ws-gb", type=float, default=100.0, help="workspace budget; candidates are chunked to fit")
    ap.add_argument("--ref-cands", type=int, default=1, help="--impl reference: candidates per step")
    ap.add_argument("--ref-cands-baseline", type=int, default=0, help="cpu_baseline sample size (candidates); 0 = per workload")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.warmup < 1 or args.steps < 1:
        ap.error("--steps and --warmup must be >= 1")
    return run_reference(args) if args.impl == "reference" else run_cuda(args)


if __name__ == "__main__":
    sys.exit(main())
