#!/usr/bin/env python
"""bench.py -- EM cell-updates/s of the hot path (H update + E update + source injection + Joule
accumulation + PEC masks, one em_step) on the full-package config of BASELINE.json (config 4:
1024 x 1024 x 192 cells, fp32, 16-entry material table, 256 bursty sources, Joule map output every
100 steps), plus the roofline of the dominant kernel and the CPU-oracle baseline.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--scale 1] [--impl reference]

N > 1 (torchrun): ONE problem cut into z slabs, one rank per slab (strong scaling; the halo of SURVEY.md 8(e) is
fused into the sweep as peer stores, --halo p2p uses NCCL send/recv instead); --decomp replicas runs N independent
replicas (weak scaling).  value = whole-job cell-updates / max-over-ranks device time.
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
sys.path.insert(0, ROOT)

B_MIN = {32: 57, 64: 113}     # algorithmic bytes per cell-update (DESIGN.md / SURVEY.md 8(d))
B_EONLY = {32: 45, 64: 89}    # E-only recurrence of eq. (2): 9 field words + 1 B id + 2 words of q


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--scale", type=int, default=1)
    ap.add_argument("--precision", type=int, default=0, help="0 = the config's own")
    ap.add_argument("--kernel", default="auto", choices=["auto", "split", "tma"])
    ap.add_argument("--formulation", default="leapfrog", choices=["leapfrog", "eonly"],
                    help="eonly: the paper's literal three-level recurrence of eq. (2) (state e^n, e^{n-1}; 45 B fp32 / "
                         "89 B fp64 per cell-update; fp32 leaves the 2e-5 parity bound on long runs, see DESIGN.md)")
    ap.add_argument("--force-joule-output", action="store_true",
                    help="one Joule-map output at the end of every timed repetition even when K is below the config's "
                         "cadence (default: outputs fall where the cadence puts them; their count is stated in config)")
    ap.add_argument("--dist-backend", default="nccl", choices=["nccl", "gloo"],
                    help="gloo lets several ranks share one GPU (testing the N > 1 path on a one-GPU box; peer halo only)")
    ap.add_argument("--reps", type=int, default=3, help="timed repetitions of the K steps (each after em_reset); the median is reported")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--decomp", default="slabs", choices=["slabs", "replicas"],
                    help="N > 1: ONE problem cut into z slabs (default; strong scaling; SURVEY.md 8(e); "
                         "paper_2603_07038_b200/slabs.py) or N independent replicas (weak scaling, no data plane)")
    ap.add_argument("--halo", default="peer", choices=["peer", "p2p"],
                    help="slabs: halo stores fused into the sweep over a CUDA IPC / NVLink peer mapping + one tiny all-reduce "
                         "per step (default), or pack kernel -> NCCL send/recv -> unpack kernel")
    ap.add_argument("--thermal-nodal", action="store_true",
                    help="--thermal with theta on the mesh NODES (the paper's placement, em_grid.thermal = EM_THERMAL_NODE; split kernels)")
    ap.add_argument("--thermal", action="store_true",
                    help="two-way EM-thermal coupling (PAPER.md eq. (4)-(6)) with the handbook-order thermal table")
    ap.add_argument("--cpu-seconds", type=float, default=15.0)
    args = ap.parse_args()
    if args.thermal_nodal:
        args.thermal = True
    return args


# ------------------------------------------------------------------------------------------------
class ClockSampler(threading.Thread):
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index = index; self.samples = []; self.stop_flag = False

    def run(self):
        while not self.stop_flag:
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                      "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=5).stdout
                parts = [x.strip() for x in out.strip().split(",")]
                if len(parts) >= 7:
                    self.samples.append(parts)
            except Exception:
                pass
            time.sleep(0.2)

    def summary(self):
        sm = sorted(float(s[0]) for s in self.samples if s[0].replace(".", "").isdigit())
        mx = [float(s[1]) for s in self.samples if s[1].replace(".", "").isdigit()]
        reasons = set()
        for s in self.samples:
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), s[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(self.samples)}


def measured_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def ncu_traffic(kernel_name: str, cells: int):
    """dram bytes per launch of the dominant kernel from the committed ncu summary, if any."""
    for name in ("r2_traffic.txt", "r1_traffic.txt"):            # JSON text written from the ncu summary beside it
        try:
            with open(os.path.join(ROOT, "profiles", name)) as f:
                t = json.load(f)
            ent = t.get(kernel_name)
            if ent and ent.get("cells") == cells:
                return float(ent["dram_bytes_per_launch"])
        except Exception:
            pass
    return None


def make_problem(args):
    import workloads as W
    kw = {}
    if args.config in (4, 5):
        kw["steps"] = max(args.steps + args.warmup, 1000) if args.scale == 1 else args.steps + args.warmup
    elif args.config in (2, 3, 6):
        kw["steps"] = args.steps + args.warmup
    p = W.make_config(1) if args.config == 1 else W.make_config(args.config, scale=args.scale, **kw)
    if getattr(args, "thermal", False):
        p.thermal = W.thermal_table(p.table.shape[0])
        if getattr(args, "thermal_nodal", False):
            p.thermal_placement = "node"
    return p


# ------------------------------------------------------------------------------------------------
def cpu_oracle_rate(args, seconds: float):
    """The oracle as it stands, timed on the host cores on a bounded sample of the same workload."""
    import workloads as W
    from oracle import emo
    threads = emo.set_threads(os.cpu_count() or 1)
    scale = max(args.scale, 4) if args.config in (3, 4, 5) else 1
    kw = {"steps": 64} if args.config != 1 else {}
    p = W.make_config(args.config, scale=scale, **kw) if args.config != 1 else W.make_config(1)
    if getattr(args, "thermal", False):
        p.thermal = W.thermal_table(p.table.shape[0])
        if getattr(args, "thermal_nodal", False):
            p.thermal_placement = "node"
    o = emo.Oracle(p)
    o.step(1)                                        # warm the pages
    t0 = time.perf_counter(); n = 0
    while True:
        o.step(1); n += 1
        el = time.perf_counter() - t0
        if el >= seconds or n >= 60:
            break
    rate = p.n_cells * n / el
    sample = "%s at %dx%dx%d cells (scale 1/%d in x,y), %d steps, fp64%s" % (
        p.name, p.nx, p.ny, p.nz, scale, n, ", thermal coupling on" if getattr(args, "thermal", False) else "")
    # the same oracle on ONE thread (2 steps), for the single-core figure SURVEY.md 8(d) asks for
    emo.set_threads(1)
    t1 = time.perf_counter(); o.step(2)
    cpu_oracle_rate.single_thread = p.n_cells * 2 / (time.perf_counter() - t1)
    emo.set_threads(threads)
    o.close()
    return rate, threads, sample, el / n * 1e3, p


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    # bounded: K timed "steps", each = one oracle time step on the sample grid
    import workloads as W
    from oracle import emo
    threads = emo.set_threads(os.cpu_count() or 1)
    scale = max(args.scale, 4) if args.config in (3, 4, 5) else 1
    K, Wm = args.steps, args.warmup
    # keep the whole run within a few minutes: shrink further if K is large
    while args.config in (3, 4, 5) and K * (1024 // scale) ** 2 * 192 / 1.5e8 > 150 and scale < 32:
        scale *= 2
    p = W.make_config(args.config, scale=scale, steps=K + Wm) if args.config != 1 else W.make_config(1)
    o = emo.Oracle(p)
    o.step(Wm)
    t0 = time.perf_counter()
    o.step(K)
    el = time.perf_counter() - t0
    val = p.n_cells * K / el
    sample = "%s at %dx%dx%d cells (scale 1/%d in x,y), fp64 oracle" % (p.name, p.nx, p.ny, p.nz, scale)
    line = {
        "impl": "reference", "metric": "EM cell-updates/sec", "value": val, "unit": "cell-updates/s",
        "n_gpus": args.gpus, "steps": K, "warmup": Wm, "ms_per_step": el / K * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "config %d (%s), bounded sample: %s" % (args.config, p.name, sample)},
        "cpu_baseline": {"value": val, "unit": "cell-updates/s", "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": "cell-updates/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    print(json.dumps(line))


# ------------------------------------------------------------------------------------------------
def run_b200(args):
    import numpy as np
    import torch
    import paper_2603_07038_b200 as P
    from paper_2603_07038_b200.replicas import aggregate_throughput, max_over_ranks

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    dist = None
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: there is no CPU fallback for the product path")
    n_dev = torch.cuda.device_count()
    if local >= n_dev and args.dist_backend == "nccl":
        raise RuntimeError("rank %d has no GPU of its own (%d visible): one process per GPU" % (local, n_dev))
    local_dev = local % n_dev                                  # (--dist-backend gloo: ranks may share a GPU, for testing the N > 1 path)
    if world > 1:
        import torch.distributed as dist_
        dist = dist_
        if args.dist_backend == "nccl":
            dist.init_process_group("nccl", device_id=torch.device("cuda", local_dev))
        else:
            dist.init_process_group(args.dist_backend)
    torch.cuda.set_device(local_dev)
    dev = torch.device("cuda", local_dev)
    red_dev = dev if args.dist_backend == "nccl" else None     # where the timing scalars are reduced

    p = make_problem(args)
    precision = args.precision or p.precision
    kernel = {"auto": P.EM_KERNEL_AUTO, "split": P.EM_KERNEL_SPLIT, "tma": P.EM_KERNEL_TMA}[args.kernel]
    form = P.EM_FORM_EONLY if args.formulation == "eonly" else P.EM_FORM_LEAPFROG
    comps = (0, 1, 2, 6, 7, 8) if form == P.EM_FORM_EONLY else tuple(range(6))
    K, Wm = args.steps, args.warmup
    slab = None
    p_global = p
    if args.decomp == "slabs" and world > 1:
        from paper_2603_07038_b200 import slabs
        if form == P.EM_FORM_EONLY:
            raise SystemExit("the z-slab halo covers the leapfrog formulation: use --decomp replicas with --formulation eonly")
        p, meta = slabs.sub_problem(p_global, rank, world)       # this rank's extended slab (PMC on the artificial walls)
    em = P.EM(p, precision=precision, kernel=kernel, device=dev, formulation=form)
    if args.decomp == "slabs" and world > 1:
        slab = slabs.SlabRank(em, meta)
        if args.halo == "peer" and not args.thermal and form == P.EM_FORM_LEAPFROG and kernel != P.EM_KERNEL_SPLIT:
            try:
                slabs.connect_peers_dist(slab, dist)
            except Exception as exc:                             # no peer mapping between these GPUs: NCCL send/recv instead
                print("peer halo unavailable (%s): falling back to --halo p2p" % exc, file=sys.stderr)
                slab.mode = "p2p"
            modes = [None] * world                               # every rank must use the same transport
            dist.all_gather_object(modes, slab.mode)
            if any(m != "peer" for m in modes):
                if slab.mode == "peer":
                    em.em_set_peer_halo(0, 0, None); em.em_set_peer_halo(1, 0, None)
                slab.mode = "p2p"
        args.no_e2e = True                                       # the end-to-end leg is defined for whole problems
    cells = p.n_cells
    je = p.joule_every if p.joule_every else 0
    pw_map = torch.empty((p.nz, p.ny, p.nx), dtype=em.dtype, device=dev) if je else None
    q_map = torch.empty((p.nz, p.ny, p.nx), dtype=em.dtype, device=dev) if je else None

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize(dev)

    outputs = [0]

    def run_steps(n, start, force_output=False):
        """n steps with the config's Joule-map outputs (energy + power maps to device buffers) inside: every
        joule_every steps, and (force_output) once at the end if the run is too short to reach one."""
        done = 0; made = 0
        while done < n:
            nxt = n - done
            if je:
                to_out = je - ((start + done) % je)
                nxt = min(nxt, to_out)
            if slab is None:
                em.em_step(nxt)
            else:                                                # one halo exchange after every step
                slab.step(nxt, dist)
            done += nxt
            if je and (start + done) % je == 0:
                em.em_joule(pw_map, q_map, total=False); made += 1
        if je and force_output and made == 0:
            em.em_joule(pw_map, q_map, total=False); made += 1
        outputs[0] = made

    # ---- device-resident timing: W warm-up steps, then `reps` repetitions of [em_reset, K steps]; the MEDIAN repetition
    # is reported.  Every repetition contains at least one Joule-map output when the config has them.
    run_steps(Wm, 0)
    em.em_timing_enable(True)
    sampler = ClockSampler(local_dev); sampler.start()
    l0 = em.launch_count
    rep_ms = []
    for _ in range(max(args.reps, 1)):
        em.em_reset() if slab is None else slab.reset()
        barrier()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record()
        run_steps(K, 0, force_output=args.force_joule_output)
        ev1.record()
        barrier()
        rep_ms.append(max_over_ranks(ev0.elapsed_time(ev1), dist, red_dev))
    sampler.stop_flag = True
    out_ms = None
    if je:                               # one Joule-map output (energy + power maps to device buffers), timed on its own
        barrier()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record(); em.em_joule(pw_map, q_map, total=False); ev1.record()
        barrier()
        out_ms = ev0.elapsed_time(ev1)
    ms = sorted(rep_ms)[len(rep_ms) // 2]
    launches = (em.launch_count - l0) // max(args.reps, 1)
    kname, klaunch, kms = em.em_timing_read()
    em.em_timing_enable(False)
    kcells = p.n_cells
    if slab is None:
        value = aggregate_throughput(cells * K, ms * 1e-3, world)
    else:                                                        # one problem over all ranks: its own cells / max time
        cells = p_global.n_cells
        value = aggregate_throughput(cells * K, ms * 1e-3, 1)

    # ---- end to end through the C ABI with host buffers -------------------------------------------
    e2e = None
    if not args.no_e2e:
        shapes = em.shapes
        host_in = [torch.zeros(s, dtype=em.dtype).pin_memory() for s in shapes]
        rng = np.random.default_rng(7)
        host_in = [host_in[c] for c in comps]
        for c, h in zip(comps, host_in):                     # small seeded seed field, not all zeros
            h.view(-1)[:: max(1, h.numel() // 4096)] = float(rng.standard_normal()) * (1 / 376.73 if 3 <= c < 6 else 1.0)
        host_out = [torch.empty(shapes[c], dtype=em.dtype).pin_memory() for c in comps]
        host_q = torch.empty((p.nz, p.ny, p.nx), dtype=em.dtype).pin_memory()
        probes = p.probes if len(p.probes) else np.asarray([[0, 0, 1, 1]], np.int32)
        if form == P.EM_FORM_EONLY:                          # (an E-only context has no H to probe)
            probes = probes[probes[:, 0] < 3] if (probes[:, 0] < 3).any() else np.asarray([[0, 0, 1, 1]], np.int32)
        em.em_reset()
        barrier()
        t0 = time.perf_counter()
        h2d = d2h = 0
        for n, c in enumerate(comps):
            em.em_set_field(c, host_in[n].numpy()); h2d += host_in[n].numel() * host_in[n].element_size()
        done = 0
        while done < K:
            nxt = min(K - done, (je - (done % je)) if je else 64)
            em.em_step(nxt); done += nxt
            vals = em.em_probe(probes); d2h += vals.nbytes     # per-chunk read of the run's observable
            if je and done % je == 0:
                em.em_joule(pw_map, q_map, total=False)
                host_q.copy_(q_map, non_blocking=False); d2h += host_q.numel() * host_q.element_size()
        for n, c in enumerate(comps):
            em.em_get_field(c, host_out[n].numpy()); d2h += host_out[n].numel() * host_out[n].element_size()
        tot = em.em_joule(None, None, total=True); d2h += 8
        torch.cuda.synchronize(dev)
        el = time.perf_counter() - t0
        el = max_over_ranks(el, dist, red_dev)
        e2e = {"value": aggregate_throughput(cells * K, el, world), "unit": "cell-updates/s", "h2d_bytes_per_step": h2d / K,
               "d2h_bytes_per_step": d2h / K,
               "what": "em_set_field x6 from pinned host, %d x em_step with em_probe reads%s, em_get_field x6 + Joule total to host"
                       % (K, " and Joule maps to host every %d steps" % je if je else "")}
        del host_in, host_out, host_q

    q_total = slab.joule_total(dist) if slab is not None else None     # all-reduce of the owned layers' Joule totals
    if rank != 0:
        em.close()
        if dist is not None:
            dist.destroy_process_group()
        return

    peak, peak_src = measured_peak()
    bmin = B_EONLY[precision] if form == P.EM_FORM_EONLY else B_MIN[precision]
    if args.thermal:                 # + theta read/write + sigma(T) read/write per cell-update
        bmin += 4 * (precision // 8)
    avg_ms = kms / max(klaunch, 1)
    achieved = bmin * kcells / (avg_ms * 1e-3) / 1e9 if klaunch else None
    if kname.startswith("k_split") or args.thermal:
        # split strategy (and the thermal coupling that runs on it): the step is several kernels, each moving only
        # part of B_min, so the honest roofline figure is the whole step's, not one kernel's
        step_ms = ms / K
        achieved = bmin * kcells / (step_ms * 1e-3) / 1e9
        avg_ms = step_ms
        if kname.startswith("k_split"):
            kname = "split step: k_split_h + %s + %s" % ("k_split_e_sig" if args.thermal else "k_split_e",
                                                         "k_joule_sig + k_thermal_nodal + k_sigma_nodal" if getattr(args, "thermal_nodal", False)
                                                         else "k_joule_thermal" if args.thermal else "k_split_joule")
        else:
            kname = "coupled step: k_diffuse + k_sweep_tma<TH> (sweep alone %.3f ms)" % (kms / max(klaunch, 1))
    roofline = {"bound": "hbm", "kernel": kname, "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak if achieved else None, "traffic": ncu_traffic(kname, kcells),
                "peak_source": peak_src, "algorithmic_bytes_per_launch": bmin * kcells,
                "avg_launch_ms": avg_ms, "launches_timed": klaunch,
                "step_effective_GBps": bmin * value / world / 1e9, "step_frac_of_peak": bmin * value / world / 1e9 / peak,
                "frac_of_8TBps_nominal": (achieved / 8000.0) if achieved else None,
                "algorithmic_bytes_per_cell_update": bmin}
    if form == P.EM_FORM_EONLY:      # the same cell-updates/s expressed in the leapfrog's B_min: may exceed 1, not clipped
        roofline["frac_in_leapfrog_bytes"] = B_MIN[precision] * kcells / (avg_ms * 1e-3) / 1e9 / peak
    cpu = None
    if not args.no_cpu_baseline:
        rate, threads, sample, ms_cpu, _ = cpu_oracle_rate(args, args.cpu_seconds)
        cpu = {"value": rate, "unit": "cell-updates/s", "cores": threads, "kind": "oracle", "sample": sample,
               "single_thread_value": getattr(cpu_oracle_rate, "single_thread", None),
               "ms_per_step_on_sample": ms_cpu}
    line = {
        "metric": "EM cell-updates/sec", "value": value, "unit": "cell-updates/s", "n_gpus": world,
        "steps": K, "warmup": Wm, "ms_per_step": ms / K, "higher_is_better": True,
        "scaling": "strong" if slab is not None else "weak",
        "vs_baseline": None, "dtype": "f32" if precision == 32 else "f64", "data": "synthetic",
        "config": {"workload": "config %d: %s %dx%dx%d cells (%d), %d ports, %s loss, Joule map every %s steps"
                               % (args.config, p_global.name, p_global.nx, p_global.ny, p_global.nz, cells, p_global.n_ports,
                                  "EXP" if p.loss_mode else "CD", je or "-")
                               + (", walls -x+x-y+y-z+z = %s (1 = PMC)" % "".join(str(int(b)) for b in p.bc) if any(p.bc) else "")
                               + (", E-only three-level recurrence of eq. (2)" if form == P.EM_FORM_EONLY else "")
                               + (", %d Joule-map output(s) inside each timed repetition of %d steps (one output = %.2f ms, "
                                  "i.e. +%.3f ms/step at the config's cadence)" % (outputs[0], K, out_ms, out_ms / je) if je else "")
                               + (", two-way thermal coupling (%s)" % ("theta on the mesh nodes, split kernels" if getattr(args, "thermal_nodal", False) else
                                                                      "split kernels" if args.kernel == "split" else "coupled TMA sweep + conduction kernel") if args.thermal else ""),
                   "kernel_strategy": args.kernel, "l2": "state %.1f GB >> 126 MB L2 (no flush needed)" % (em.workspace_bytes / 1e9)
                   if em.workspace_bytes > 1e9 else "state fits L2: %.0f MB" % (em.workspace_bytes / 1e6),
                   "parallelism": ("z-slabs x%d, halo per step: %s" % (world, "Ex, Ey wall planes stored by the sweep into the "
                                   "neighbour's memory (peer mapping) + one 4-byte all-reduce" if slab.mode == "peer" else
                                   "pack kernel, NCCL send/recv, unpack kernel") if slab is not None else
                                   "replicas x%d" % world) if world > 1 else "single GPU"},
        "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": launches,
        "joule_total_J": q_total,
        "timing": {"reps": len(rep_ms), "ms_per_rep": rep_ms, "reported": "median", "reset_before_each_rep": True},
        "clocks": sampler.summary(),
    }
    print(json.dumps(line))
    em.close()
    if dist is not None:
        dist.destroy_process_group()


def main():
    args = parse()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_b200(args)


if __name__ == "__main__":
    main()
