#!/usr/bin/env python
"""bench.py -- LB-CNN kernel-selection inner loop on B200: candidates/s through expand + fit + score.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload mnist] [--impl cuda|reference]

A "step" is ONE pass of the whole hot path over one batch
of synthetic input: one lbcnn_search_candidates call that expands the train and test sets through the
binary-conv layers for every candidate kernel set of the workload, fits the ELM output layer per
candidate, scores the held-out set and picks best / worst.  Default workload =
BASELINE.json configs[1] ("MNIST-shaped reduced-subset search": N_train 20000, N_test 10000, 64 candidates).

One JSON line on stdout (rank 0):
  value        candidates/s, inputs resident in HBM, CUDA events on the launching stream, max over ranks; the
               library's per-phase events are OFF in this pass
  phases       a second pass of the same steps with per-phase CUDA events ON: time, algorithmic work and roofline
               fraction of every phase, each against the peak of the pipe its kernels run on
  roofline     the phase with the largest time (`kernel`), copied from `phases`
  e2e          the same metric through lbcnn_search_candidates_host: HOST (pinned) buffers, host<->device
               copies inside the timed region
  per_config   value / ms_per_step / e2e / phases / clocks / accuracy of ALL FIVE BASELINE.json configs measured in
               this run (north_star: "candidates/sec reported for each config"); the headline stays --workload
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
              "gtsrb": (1, 3000, 1263), "vggface": (1, 1000, 250), "paper_table1": (1, 1000, 500)}

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


# B200 fp64 pipe: DMMA (mma.sync.m8n8k4.f64) 64 FMA/clk/SM x 148 SMs x 1.965 GHz x 2 (measured 64/clk)
FP64_TFLOPS = 64 * 148 * 1.965e9 * 2 / 1e12


def _phase_rooflines(w, F, n_cand, phase_ms, steps, peaks, sustained: bool, stats=None):
    """Algorithmic work per step for each phase (SURVEY.md 8(d) / DESIGN.md "Rooflines") over its measured
    CUDA-event time per step.  Every phase is divided by the peak of the pipe its kernels actually run on.
    Returns {phase: roofline-dict}."""
    N, Nte, c = w.n_train, w.n_test, w.n_classes
    px = w.in_h * w.in_w * w.in_c
    primal = F < N
    dim = F if primal else N
    hbm = peaks["hbm_gbs"]
    bf16 = peaks["bf16_sustained"] if sustained else peaks["bf16_burst"]
    which = "sustained" if sustained else "burst"
    # fp32-accurate tensor peak (north_star's Gram denominator): TF32 dense = bf16 / 2 (guide's nominal ratio
    # 1.1 / 2.25 PF), three TF32 passes.  The kernels themselves run int8 digit products: int8 dense = 2 x bf16.
    tens = bf16 / 2.0 / 3.0
    int8 = 2.0 * bf16
    stats = stats or {}
    # dual branch (F >= N), scored through the kernel trick (the driver's default): the Gram of the stacked
    # [train; test] rows also yields the cross-Gram (2 F N_te N flop), the factorisation carries c + N_te appended rows, the
    # scores are one N_te x N x c product of appended rows (fp64) -- no F x c back-projection, no pass over the test features
    kt = (not primal) and not any(o == 9 and v == 0 for o, v in OPTIONS)
    gram_flop = n_cand * (float(N) * F * (F + 1) if primal else float(F) * N * (N + 1) + (2.0 * F * Nte * N if kt else 0.0))
    solve_flop = n_cand * (dim ** 3 / 3.0 + 2.0 * dim * dim * c + (0 if primal else (float(dim) * dim * Nte if kt else 2.0 * N * F * c)))
    work = {
        # H written once (4 F bytes per image per candidate) + every image read once per launch
        "expand": ("hbm", "GB/s", hbm, (n_cand * (N + Nte) * F * 4.0 + (N + Nte) * px) / 1e9, "HBM copy GB/s"),
        # symmetric half of the Gram: N dim (dim + 1) flop per candidate (primal), F N (N + 1) (dual)
        "gram": ("tensor", "TFLOP/s", tens, gram_flop / 1e12,
                 "bf16 %s / 2 (TF32 nominal ratio) / 3 (3xTF32 = fp32-accurate)" % which),
        "rhs": ("hbm", "GB/s", hbm, (n_cand * float(N) * F * 4.0 if primal else n_cand * float(N) * c * 8.0) / 1e9,
                "HBM copy GB/s"),
        # Cholesky dim^3/3 + two triangular solves with c right-hand sides 2 dim^2 c (+ dual back-projection 2 N F c)
        "solve": ("fp64", "TFLOP/s", FP64_TFLOPS, solve_flop / 1e12,
                  "fp64 DMMA pipe: 64 FMA/clk/SM x 148 SMs x 1.965 GHz (DESIGN.md section 7)"),
        # test features read once + W
        "score": ("hbm", "GB/s", hbm, n_cand * (float(Nte) * F * 4.0 + F * c * 4.0) / 1e9, "HBM copy GB/s"),
    }
    if kt:
        work["score"] = ("fp64", "TFLOP/s", FP64_TFLOPS, n_cand * 2.0 * Nte * N * c / 1e12,
                         "fp64 DMMA pipe (kernel-trick logits: a product of the factorisation's appended rows)")
    out = {}
    for ph, (bound, unit, peak, amount, src) in work.items():
        ms = phase_ms.get(ph, (0.0, 0))[0] / max(steps, 1)
        if ms <= 0:
            continue
        ach = amount / (ms * 1e-3)
        out[ph] = dict(bound=bound, achieved=round(ach, 3), peak=round(peak, 1), unit=unit, frac=round(ach / peak, 4),
                       traffic=None, ms_per_step=round(ms, 4), work_per_step=round(amount, 4),
                       peak_source="%s (%s)" % (peaks["source"], src))
    # Phases whose kernels run on the int8 tensor pipe are rated against THAT pipe (kernel-counted int8 multiply-adds,
    # tile padding included, x 2 / phase time against int8 dense = 2 x bf16), so no fraction can exceed 1; the
    # useful-work figure against the convention peak (north_star's "fp32-accurate tensor-pipe peak" for the Gram, the fp64
    # pipe for the solve) is kept beside it as `useful`.
    for ph, key, note in (("gram", "gram_int8_tmac_per_step", "gram_tc_kernel digit products (split pass included in the time)"),
                          ("solve", "solve_int8_tmac_per_step", "trailing updates' digit products (fp64 panels, substitutions and "
                           "splits included in the time)")):
        if ph in out and stats.get(key):
            o = out[ph]
            tops = 2.0 * stats[key] / (o["ms_per_step"] * 1e-3)
            o["useful"] = dict(bound=o["bound"], achieved=o["achieved"], peak=o["peak"], unit=o["unit"],
                               ratio=round(o["achieved"] / o["peak"], 4), peak_source=o["peak_source"],
                               note="algorithmic flop / phase time against the convention peak; above 1 means the int8 digit "
                                    "route is cheaper than that convention's arithmetic")
            o.update(bound="tensor", achieved=round(tops, 1), peak=round(int8, 1), unit="TOP/s", frac=round(tops / int8, 4),
                     peak_source="%s (int8 dense = 2 x bf16 %s)" % (peaks["source"], which), note="kernel-counted int8 MACs x 2: " + note)
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
    origin = ("BASELINE.json configs[%d]" % (w.config - 1)) if w.config <= 5 else "paper Table I shape (PAPER.md:104-113), not a BASELINE config"
    return dict(workload="%s (%s): %dx%dx%d u8, N_train=%d N_test=%d classes=%d, layers=%s, C=%g"
                % (origin, w.name, w.in_h, w.in_w, w.in_c, w.n_train, w.n_test, w.n_classes,
                   "+".join("%d@%dx%d/pool%d" % (L.n_kernels, L.ksize, L.ksize, L.pool_k) for L in w.layers), w.C),
                candidates_per_step=n_cand, parallelism="replicas only (candidates independent; no collective)",
                l2=l2_note)


def _git_head_of(paths):
    """hash of the last commit that touched `paths` (None outside a git checkout, e.g. on the GPU box's snapshot)."""
    try:
        r = subprocess.run(["git", "-C", ROOT, "log", "-1", "--format=%H", "--"] + list(paths), capture_output=True,
                           text=True, timeout=10)
        return r.stdout.strip() or None
    except Exception:
        return None


def _traffic(name, phase):
    """dram bytes per step of `phase` from the committed ncu --set full capture (profiles/traffic_<workload>.txt, JSON
    text stamped with the commit of csrc/ it was captured at).  Dropped (None) when csrc/ has changed since -- a stale
    capture must not label a newer kernel; kept when git is unavailable and the stamp cannot be checked."""
    prof = os.path.join(ROOT, "profiles", "traffic_%s.txt" % name)
    if not os.path.exists(prof):
        return None
    with open(prof) as f:
        d = json.load(f)
    head = _git_head_of(["paper_2106_15350_b200/csrc"])
    if head is not None and d.get("csrc_commit") not in (None, head):
        return None
    return d.get(phase)


def _measure(lb, replicas, synth, torch, np, dist, name, steps, warmup, ws_gb, world, rank, local, n_cand=0,
             with_e2e=True):
    """one workload: `warmup` untimed steps, `steps` timed steps with profiling OFF (value), the same number of steps
    again with per-phase events ON (phases), then the host-buffer entry (e2e).  Returns the pieces of the JSON line."""
    w = synth.WORKLOADS[name]
    if n_cand:
        w = synth.scaled(w, n_cand=n_cand)
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
    for opt, val in OPTIONS:
        h.set_option(opt, val)
    stage = lb.host_staging_bytes(arch, w.n_train, w.n_test, w.n_classes, K)
    budget = int(ws_gb * (1 << 30))
    ws_bytes, ws_min = lb.workspace_bytes(arch, w.n_train, w.n_test, w.n_classes, K, budget, handle=h)
    h.ensure_workspace(ws_bytes + stage)
    l2_note = "inputs exceed L2: workspace %.2f GB of features/Gram streams through the 126 MB L2 every step" % (ws_bytes / 1e9)
    if ws_bytes < 2 * 126e6:
        l2_note = "workspace %.3f GB; L2 flushed by writing a 256 MB buffer between timed steps" % (ws_bytes / 1e9)
        flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    else:
        flush = None

    def step(out=None):
        return h.search_candidates(arch, d_in[0], d_in[1], d_in[2], d_in[3], w.n_classes, w.C, d_in[4], out=out)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(nsteps):
        """CUDA events on the launching (current) stream around each step; the L2 flush sits between the brackets"""
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(nsteps)]
        barrier()
        for a, b in evs:
            if flush is not None:
                flush.fill_(1)
            a.record()
            step(out)
            b.record()
        barrier()
        return [a.elapsed_time(b) for a, b in evs]

    out = step()
    for _ in range(max(warmup - 2, 0)):
        step(out)
    barrier()
    # nvidia-smi needs ~100 ms to deliver its first sample: start it one warm-up step early so that short timed
    # regions (configs[0], [3]) still get samples under load
    sampler = ClockSampler(local)
    sampler.start()
    t_w = time.perf_counter()
    while True:
        step(out)
        torch.cuda.synchronize()
        if warmup < 2 or time.perf_counter() - t_w > 0.25:
            break
    barrier()
    # ---- timed region: device-resident inputs, per-phase events OFF ----
    n0 = h.launch_count()
    ms_steps = timed(steps)
    launches = h.launch_count() - n0
    clocks = sampler.stop()
    ms = replicas.max_over_ranks(sum(ms_steps), dev)
    # ---- second pass, per-phase CUDA events ON: where the time goes (not part of `value`) ----
    h.op_stats()                      # reset the device-side int8 operation counters
    h.set_profiling(True)
    timed(steps)
    phase_ms = h.phase_times()
    h.set_profiling(False)
    stats = h.op_stats()
    acc = out["acc"].cpu().numpy()
    info = out["info"].cpu().numpy()
    if (info != 0).any() or not np.isfinite(acc).all():
        raise RuntimeError("fit failed for some candidate: info=%s" % info.tolist())

    res = dict(w=w, K=K, F=F, ms=ms, ms_steps=sorted(ms_steps), launches=launches, clocks=clocks, phase_ms=phase_ms, stats=stats, acc=acc,
               best=int(out["best"][0].item()), l2_note=l2_note, data=(trx, try_, tex, tey), e2e=None)
    if with_e2e:
        # ---- e2e: host (pinned) buffers through lbcnn_search_candidates_host, copies inside the timed region ----
        hout = h.search_candidates_host(arch, *h_in[:4], w.n_classes, w.C, h_in[4])
        barrier()
        t0 = time.perf_counter()
        for _ in range(steps):
            h.search_candidates_host(arch, *h_in[:4], w.n_classes, w.C, h_in[4], out=hout)   # synchronises inside
        barrier()
        e2e_s = replicas.max_over_ranks(time.perf_counter() - t0, dev)
        if not np.array_equal(hout["correct"].numpy(), out["correct"].cpu().numpy()):
            raise RuntimeError("host-buffer path and device-buffer path disagree")
        h2d = sum(t.numel() * t.element_size() for t in h_in)
        d2h = sum(t.numel() * t.element_size() for t in hout.values() if t is not None)
        res["e2e"] = dict(value=replicas.job_throughput(world, K, steps, e2e_s), unit=UNIT, h2d_bytes_per_step=h2d,
                          d2h_bytes_per_step=d2h)
    h.close()
    del d_in, out, flush
    torch.cuda.empty_cache()
    return res


def _cpu_baseline(np, w, data, K, acc, nc_override):
    """the oracle as it stands on the host cores, on a bounded sample (about 10-30 s of host work) of workload `w`:
    CPU_SAMPLE's (candidates, N_train, N_test); `acc` = the GPU's accuracies of the same candidates (compared at full N)."""
    trx, try_, tex, tey = data
    nc, ntr, nte = CPU_SAMPLE.get(w.name, (1, w.n_train, w.n_test))
    if nc_override:
        nc = nc_override
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
    return dict(value=nc / dt, unit=UNIT, cores=threads, kind="oracle", sample=sample)


OPTIONS = []       # (option, value) pairs from --solver / --panel (measurement switches; default = the product path)

DTYPE = ("int8 x int8 -> int32 tensor-core expander, Gram and Cholesky trailing updates (exact digit products), "
         "f64 Cholesky panels and logits, f32 features/weights")


def _summary(res, steps, world, replicas, peaks):
    total_s = res["ms"] * 1e-3
    w = res["w"]
    stats = {k + "_per_step": v / float(steps) for k, v in res["stats"].items()}     # counted over the phase pass
    roofs = _phase_rooflines(w, res["F"], res["K"], res["phase_ms"], steps, peaks, sustained=total_s > 2.0, stats=stats)
    for ph in roofs:
        roofs[ph]["traffic"] = _traffic(w.name, ph)
    dominant = max(roofs, key=lambda p: roofs[p]["ms_per_step"]) if roofs else None
    roofline = dict(roofs[dominant]) if dominant else None
    if roofline:
        roofline["kernel"] = dominant
    acc = res["acc"]
    med = res["ms_steps"][len(res["ms_steps"]) // 2] if len(res["ms_steps"]) % 2 else \
        0.5 * (res["ms_steps"][len(res["ms_steps"]) // 2 - 1] + res["ms_steps"][len(res["ms_steps"]) // 2])
    return dict(value=replicas.job_throughput(world, res["K"], steps, total_s), ms_per_step=res["ms"] / steps,
                ms_per_step_median=med, e2e=res["e2e"], gpu_launches=int(res["launches"]), clocks=res["clocks"], roofline=roofline, phases=roofs,
                accuracy=dict(best=float(acc.max()), worst=float(acc.min()), best_index=res["best"]),
                config=_config(w, res["K"], res["l2_note"]))


def _extras(lb, synth, torch, np, name, peaks, local):
    """the SURVEY.md 8(f) rows built so far, measured on the bench workload (CUDA events, 3 timed repeats after 2 warm-ups):
    streamed search (8(f)-1), int8 output layer + exact integer scorer (8(f)-2), one genetic generation (8(f)-3)."""
    w = synth.WORKLOADS[name]
    K = w.n_cand
    trx, try_, tex, tey = synth.make_dataset(w)
    dev = torch.device("cuda", local)
    d = [torch.from_numpy(np.ascontiguousarray(a)).to(dev) for a in (trx, try_, tex, tey, synth.make_kernels(w, K))]
    arch = lb.arch_of(w)
    F, _ = lb.feature_dim(arch)
    h = lb.Handle(local)

    def timed(fn, reps=3, warm=2):
        for _ in range(warm):
            fn()
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(reps)]
        torch.cuda.synchronize()
        for a, b in ev:
            a.record(); fn(); b.record()
        torch.cuda.synchronize()
        return sum(a.elapsed_time(b) for a, b in ev) / reps

    out = {}
    # 8(f)-1: streamed search, 4096 samples resident at once
    rows = 4096
    full = lb.workspace_bytes(arch, w.n_train, w.n_test, w.n_classes, K, handle=h)[0]
    h.set_option(lb.OPT_STREAM_ROWS, rows)
    small = lb.workspace_bytes(arch, w.n_train, w.n_test, w.n_classes, K, handle=h)[0]
    h.ensure_workspace(small)
    res = {}
    ms = timed(lambda: res.update(h.search_candidates(arch, d[0], d[1], d[2], d[3], w.n_classes, w.C, d[4], out=res or None)))
    out["streamed_search"] = dict(stream_rows=rows, value=K / (ms * 1e-3), unit=UNIT, ms_per_step=round(ms, 3),
                                  workspace_gb=round(small / 1e9, 3), resident_workspace_gb=round(full / 1e9, 3),
                                  note="bit-identical results to the resident search (tests/test_gpu_parity.py)")
    h.set_option(lb.OPT_STREAM_ROWS, 0)
    acc = res["acc"].clone()
    h.set_workspace(None)
    # 8(f)-2: int8 output layer on the first min(K, 16) candidates' test features
    kq = min(K, 16)
    a1 = lb.arch_of(w, 1.0)
    Hte = h.expand(a1, d[2], d[4][:kq])
    Htr = h.expand(a1, d[0], d[4][:kq])
    h.ensure_workspace(lb.fit_workspace_bytes(w.n_train, F, w.n_classes, kq, lb.H_INTEGER))
    s = float(np.float32(w.feature_scale))
    W, _ = h.elm_fit(Htr, d[1], w.n_classes, w.C, h_scale=s, flags=lb.H_INTEGER)
    del Htr
    Wq, _ = h.quantize_output_layer(W, 8)
    corr = {}
    ms_q = timed(lambda: corr.update(c=h.elm_score_q(Hte, Wq, d[3], want_pred=False)[1]))
    _, corr_f = h.elm_score(Hte, W, d[3], h_scale=s, want_pred=False)
    gb = kq * (float(w.n_test) * F * 4.0 + F * w.n_classes) / 1e9
    out["score_q8"] = dict(candidates=kq, ms=round(ms_q, 4), achieved=round(gb / (ms_q * 1e-3), 1), peak=round(peaks["hbm_gbs"], 1),
                           unit="GB/s", frac=round(gb / (ms_q * 1e-3) / peaks["hbm_gbs"], 4), bound="hbm",
                           accuracy_int8=round(float(corr["c"].float().mean().item()) / w.n_test, 4),
                           accuracy_fp32=round(float(corr_f.float().mean().item()) / w.n_test, 4),
                           note="exact integer logits (lbcnn_elm_score_q), test features read once as fp32")
    # 8(f)-4: one epoch of softmax cross-entropy / Adam refinement of candidate 0's output layer on the whole training set
    Htr0 = h.expand(a1, d[0], d[4][:1])[0].contiguous()
    ref = {}
    ms_r = timed(lambda: ref.update(r=h.refine_output_layer(Htr0, d[1], W[0].contiguous(), epochs=2, batch=128, lr=1e-5, seed=1, h_scale=s)), reps=1, warm=1)
    Wr, lossr = ref["r"]
    _, corr_r = h.elm_score(Hte[:1].contiguous(), Wr[None].contiguous(), d[3], h_scale=s, want_pred=False)
    out["refine"] = dict(epochs=2, batch=128, lr=1e-5, ms_per_epoch=round(ms_r / 2.0, 2), mean_loss_per_epoch=[round(float(x), 5) for x in lossr.tolist()],
                         accuracy_elm=round(float(corr_f[0].item()) / w.n_test, 4), accuracy_after=round(float(corr_r[0].item()) / w.n_test, 4),
                         note="lbcnn_refine_output_layer (softmax cross-entropy + Adam, reading R18): %d sequential mini-batch steps of five "
                              "launches per epoch, fp64 DMMA.  The starting point is already the exact ridge optimum on the whole set, so "
                              "the first epochs of a different loss move away from it: a timing and parity line, not an accuracy claim"
                              % ((w.n_train + 127) // 128))
    del Htr0
    # 8(f)-3: one genetic generation over the K kernel sets
    ms_g = timed(lambda: h.evolve_candidates(d[4], acc, max(1, K // 8), 20000, 1, 0))
    out["evolve"] = dict(candidates=K, ms=round(ms_g, 4), note="rank + tournament + uniform crossover + mutation (lbcnn_evolve_candidates)")
    h.close()
    torch.cuda.empty_cache()
    return out


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
    if args.solver:
        OPTIONS.append((lb.OPT_SOLVER, {"auto": lb.SOLVER_AUTO, "fp64": lb.SOLVER_FP64, "mixed": lb.SOLVER_MIXED}[args.solver]))
    if args.panel:
        OPTIONS.append((lb.OPT_PANEL, args.panel))
    if args.mid_panel >= 0:
        OPTIONS.append((lb.OPT_MID_PANEL, args.mid_panel))
    if args.stream_rows > 0:
        OPTIONS.append((lb.OPT_STREAM_ROWS, args.stream_rows))
    if args.dual_trick >= 0:
        OPTIONS.append((lb.OPT_DUAL_TRICK, args.dual_trick))
    if args.scorer:
        OPTIONS.append((lb.OPT_SCORER, {"auto": lb.SCORER_AUTO, "fp64": lb.SCORER_FP64, "tensor": lb.SCORER_TENSOR}[args.scorer]))

    common = (lb, replicas, synth, torch, np, dist)
    res = _measure(*common, args.workload, args.steps, args.warmup, args.ws_gb, world, rank, local, n_cand=args.n_cand)
    peaks = _peaks()
    main = _summary(res, args.steps, world, replicas, peaks)
    # ---- the other configs of BASELINE.json (north_star: "candidates/sec reported for each config"), same process,
    #      same rules (warm-up, events, clocks), fewer timed steps; the headline stays the --workload line ----
    per_config = {}
    if not args.no_per_config and not args.n_cand:
        for name in ("tiny_mnist", "mnist", "gtsrb", "orl", "vggface"):
            if name == args.workload:
                per_config[name] = {k: main[k] for k in ("value", "ms_per_step", "ms_per_step_median", "e2e", "gpu_launches", "clocks", "phases", "accuracy", "config")}
                per_config[name]["steps"] = args.steps
                continue
            r = _measure(*common, name, args.per_config_steps, 3, args.ws_gb, world, rank, local)
            sm = _summary(r, args.per_config_steps, world, replicas, peaks)
            sm["steps"] = args.per_config_steps
            del sm["roofline"]
            if rank == 0 and world == 1 and not args.no_cpu_baseline:
                sm["cpu_baseline"] = _cpu_baseline(np, r["w"], r["data"], r["K"], r["acc"], 0)
            per_config[name] = sm

    extras = None
    if not args.no_extras and not args.n_cand and world == 1:
        extras = _extras(lb, synth, torch, np, args.workload, peaks, local)
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0
    w, K, acc = res["w"], res["K"], res["acc"]
    line = dict(metric=METRIC, value=main["value"], unit=UNIT, n_gpus=world, steps=args.steps,
                warmup=args.warmup, ms_per_step=main["ms_per_step"], higher_is_better=True, scaling="weak",
                vs_baseline=None, dtype=DTYPE, data="synthetic", config=main["config"], clocks=main["clocks"],
                e2e=main["e2e"], gpu_launches=main["gpu_launches"], roofline=main["roofline"], phases=main["phases"],
                accuracy=main["accuracy"])
    if per_config:
        line["per_config"] = per_config
    if extras:
        line["extras"] = extras
    if not args.no_cpu_baseline:
        line["cpu_baseline"] = _cpu_baseline(np, w, res["data"], K, acc, args.ref_cands_baseline)
        if w.name in per_config:
            per_config[w.name]["cpu_baseline"] = line["cpu_baseline"]
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
    ap.add_argument("--workload", default="mnist", choices=["tiny_mnist", "mnist", "gtsrb", "orl", "vggface", "paper_table1"])
    ap.add_argument("--n-cand", type=int, default=0, help="override the workload's candidate count (not a bench line)")
    ap.add_argument("--ws-gb", type=float, default=100.0, help="workspace budget; candidates are chunked to fit")
    ap.add_argument("--ref-cands", type=int, default=1, help="--impl reference: candidates per step")
    ap.add_argument("--ref-cands-baseline", type=int, default=0, help="cpu_baseline sample size (candidates); 0 = per workload")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--solver", default="", choices=["", "auto", "fp64", "mixed"], help="LBCNN_OPT_SOLVER (measurement)")
    ap.add_argument("--panel", type=int, default=0, help="LBCNN_OPT_PANEL (measurement)")
    ap.add_argument("--mid-panel", type=int, default=-1, help="LBCNN_OPT_MID_PANEL (measurement)")
    ap.add_argument("--dual-trick", type=int, default=-1, help="LBCNN_OPT_DUAL_TRICK (measurement)")
    ap.add_argument("--stream-rows", type=int, default=0, help="LBCNN_OPT_STREAM_ROWS: streamed search, samples per chunk")
    ap.add_argument("--scorer", default="", choices=["", "auto", "fp64", "tensor"], help="LBCNN_OPT_SCORER (measurement)")
    ap.add_argument("--no-extras", action="store_true", help="skip the measurements of the SURVEY.md 8(f) rows")
    ap.add_argument("--no-per-config", action="store_true", help="skip the per_config object (the other four workloads)")
    ap.add_argument("--per-config-steps", type=int, default=5, help="timed steps for each per_config workload")
    args = ap.parse_args()
    if args.warmup < 1 or args.steps < 1:
        ap.error("--steps and --warmup must be >= 1")
    return run_reference(args) if args.impl == "reference" else run_cuda(args)


if __name__ == "__main__":
    sys.exit(main())
