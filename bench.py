#!/usr/bin/env python
"""bench.py -- atom-steps/s of the GMNN energy+force hot path on B200 (BASELINE.json `metric`).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload config5] [--mlp 3xf16]
    python bench.py --impl reference ...          # the fp64 CPU oracle on the host cores

One "step" is one NVE velocity-Verlet step of the workload through gmnn_md_verlet_steps: kick,
drift, skin test, neighbour rebuild when an atom moved more than skin/2, gather, pair forward,
contraction, MLP forward + backward, contraction backward, pair backward with the force reduction,
kick -- every row of SURVEY.md section 8(a) except the ensemble statistics (config 4, a parity
case).  `value` = atoms x steps / device time (CUDA events on the launching stream, inputs resident
in HBM).  `e2e` = the same metric through gmnn_energy_forces_host: every step copies the positions
from pinned host memory, evaluates energy and forces and copies forces and energy back.
N > 1 (torchrun): the path does not shard (replicas only) -- every rank runs an
independent replica on its own GPU, no data-path collective; `value` sums the replicas over the
slowest rank's time.

Only the `cpu_baseline` leg and `--impl reference` execute oracle/ (test infrastructure).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "atom-steps/s (GMNN energy+forces)"
UNIT = "atom-steps/s"
N_FEATURES = 360
MLP_NAMES = {"fp32": 0, "3xtf32": 1, "tf32": 2, "3xf16": 3}


def load_peaks():
    """MEASURED_PEAKS.json (driver-written) or the fallback B200_PROFILING.md states."""
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return {"hbm_gbs": float(d["hbm_gbs"]), "bf16_burst": float(d["bf16_tflops"]),
                "bf16_sustained": float(d.get("bf16_tflops_sustained", d["bf16_tflops"])),
                "sm_max_mhz": float(d.get("sm_max_mhz", 1965.0)), "source": "measured"}
    return {"hbm_gbs": 6650.0, "bf16_burst": 1590.0, "bf16_sustained": 1400.0, "sm_max_mhz": 1965.0,
            "source": "fallback"}


def stage_model(w, nl_mean, nc_mean, n_hidden_macs, mlp, forces="pairbuf"):
    """Algorithmic HBM bytes and flops per atom of each stage, keyed by the
    stage names gmnn_stage_times reports.  bound: which roof binds the stage by count."""
    F = N_FEATURES
    mlp_flops = 2.0 * n_hidden_macs  # one direction
    tensor = mlp != "fp32"
    return {
        "gather": dict(bytes=36.0, flops=0.0, bound="hbm"),
        "pair_forward": dict(bytes=4.0 * nl_mean + 420.0, flops=12.0 * nl_mean + 340.0 * nc_mean, bound="alu"),
        "contract_forward": dict(bytes=400.0 + 4.0 * F, flops=2.0 * 5000.0, bound="hbm"),
        "mlp_forward": dict(bytes=4.0 * F + 4.0, flops=mlp_flops, bound="tensor" if tensor else "alu"),
        # one head: fused into the last GEMM epilogue, what is left adds 4 partial sums per atom
        "mlp_heads": (dict(bytes=16.0 + 16.0 + 8.0, flops=8.0, bound="hbm") if w.model.n_heads == 1 and mlp != "fp32"
                      else dict(bytes=2048.0 + 8.0, flops=1024.0 * w.model.n_heads, bound="hbm")),
        "mlp_backward": dict(bytes=4.0 * F, flops=mlp_flops, bound="tensor" if tensor else "alu"),
        "contract_backward": dict(bytes=4.0 * F + 800.0, flops=2.0 * 15000.0, bound="hbm"),
        # gather form: both directions per entry; pair buffer: one direction, g_ij written to and read
        # back from the [N][cap] float4 buffer through the uint16 reverse-pair index
        "pair_backward": (dict(bytes=4.0 * nl_mean + 432.0, flops=12.0 * nl_mean + 1400.0 * nc_mean, bound="alu")
                          if forces == "gather" else
                          dict(bytes=(4.0 + 2.0 + 16.0 + 16.0) * nl_mean + 432.0, flops=12.0 * nl_mean + 700.0 * nc_mean,
                               bound="alu")),
        "outputs": dict(bytes=48.0, flops=0.0, bound="hbm"),
        "kick_drift": dict(bytes=76.0, flops=30.0, bound="hbm"),
        "kick_ke": dict(bytes=56.0, flops=20.0, bound="hbm"),
        "rebuild_if_moved": dict(bytes=0.0, flops=0.0, bound="hbm"),
    }


class ClockSampler:
    """nvidia-smi clocks and throttle reasons, sampled every 200 ms while the timed region runs."""

    Q = ("timestamp,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, device_index: int):
        self.proc = None
        self.path = "/tmp/gmnn_bench_clocks_%d.csv" % os.getpid()
        sel = []
        try:
            import torch

            uuid = str(torch.cuda.get_device_properties(device_index).uuid)
            sel = ["-i", uuid if uuid.startswith("GPU-") else "GPU-" + uuid]
        except Exception:
            sel = ["-i", str(device_index)]
        self.cmd = ["nvidia-smi", *sel, "--query-gpu=" + self.Q, "--format=csv,noheader,nounits", "-lms", "200"]

    def start(self):
        try:
            self.out = open(self.path, "w")
            self.proc = subprocess.Popen(self.cmd, stdout=self.out, stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self, t_begin=None, t_end=None):
        """Summary of the samples taken between the wall-clock times t_begin and t_end (time.time(); None: all).  The
        sampler is started BEFORE the warm-up steps, so that its start-up (a fork and ~100 ms of nvidia-smi initialisation)
        does not leave the GPU idle, and clocked down, right before the timed region."""
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        self.out.close()
        import datetime

        sm, smax, power, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        with open(self.path) as f:
            for line in f:
                c = [x.strip() for x in line.split(",")]
                if len(c) < 9:
                    continue
                if t_begin is not None and t_end is not None:
                    try:  # "2026/11/05 02:38:11.123": local time of the box, like time.time() through fromtimestamp
                        ts = datetime.datetime.strptime(c[0], "%Y/%m/%d %H:%M:%S.%f").timestamp()
                        if ts < t_begin - 0.25 or ts > t_end + 0.25:
                            continue
                    except ValueError:
                        pass
                c = c[1:]
                try:
                    sm.append(float(c[0]))
                    smax.append(float(c[1]))
                    power.append(float(c[2]))
                except ValueError:
                    continue
                for nm, v in zip(names, c[4:8]):
                    if v.lower().startswith("active"):
                        reasons.add(nm)
        try:
            os.remove(self.path)
        except OSError:
            pass
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        busy = [s for s, p in zip(sm, power) if p >= 0.5 * max(power)] or sm
        return {"sm_mhz": float(np.median(busy)), "sm_max_mhz": float(max(smax)), "power_w_max": float(max(power)),
                "samples": len(sm), "reasons": sorted(reasons)}


def make_bench_workload(name: str, weight_sets: str = "shared"):
    import workloads as wl

    if weight_sets == "species":  # one NN per species (north_star's variant of Eq. 4): 3 sets on the Li3PO4 boxes
        n_species = {"config1": 2, "config2": 5}.get(name, 3)
        return wl.make_workload(name, n_weight_sets=n_species)
    return wl.make_workload(name)


# ------------------------------------------------------------------------------------------------
# the oracle legs (cpu_baseline of our arm, and the whole reference arm)
# ------------------------------------------------------------------------------------------------
def oracle_sample_workload(workload_name: str, n_sample: int):
    """A box of the benchmarked workload's own family (composition, density, cutoff, skin, model)
    cut down to n_sample atoms so that the fp64 oracle finishes in seconds."""
    import workloads as wl

    if workload_name == "config2":
        return wl.ionic_liquid_box(n_pairs=max(8, n_sample // 24))
    if workload_name == "config1":
        return wl.tiny_box()
    skin = 1.0 if workload_name == "config5" else 0.0
    cfg = 5 if workload_name == "config5" else 3
    heads = 32 if workload_name == "config4" else 1
    return wl.li3po4_box(n_sample, skin=skin, config=cfg, n_heads=heads)


def oracle_prepare(w):
    from oracle import gmnn_oracle as orc

    r_list = float(np.float32(w.model.r_cut) + np.float32(w.skin))
    pairs = orc.auto_neighbors(w.positions, w.cell, w.pbc, r_list)
    return orc, orc.Model(w.model), pairs


def oracle_step(orc, model, w, pairs):
    t0 = time.perf_counter()
    if w.model.n_heads > 1:  # config 4: the step is the full ensemble evaluation (one forward, one backward per head)
        orc.ensemble(model, w.positions, w.species, w.cell, pairs)
    else:
        orc.energy_forces(model, w.positions, w.species, w.cell, pairs)
    return time.perf_counter() - t0


def cpu_baseline(workload_name: str, n_sample: int = 16384):
    if workload_name == "config4":
        n_sample = 2048  # 32 backward passes per evaluation
    w = oracle_sample_workload(workload_name, n_sample)
    orc, model, pairs = oracle_prepare(w)
    dt = oracle_step(orc, model, w, pairs)
    return {"value": w.n_atoms / dt, "unit": UNIT, "cores": orc.num_threads(), "kind": "oracle",
            "sample": "one fp64 %s evaluation (oracle/gmnn_oracle.c, OpenMP) of a %d-atom box of the "
                      "same family as %s (same density, species ratio, r_cut, skin, model), neighbour list prebuilt; "
                      "%.2f s" % ("shallow-ensemble (32 heads)" if w.model.n_heads > 1 else "energy+forces", w.n_atoms,
                                  workload_name, dt)}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    budget_s = 150.0
    probe = oracle_sample_workload(args.workload, 1024)
    orc, model, pairs = oracle_prepare(probe)
    oracle_step(orc, model, probe, pairs)
    rate = probe.n_atoms / oracle_step(orc, model, probe, pairs)  # atom-steps/s on this host
    n_sample = 1024
    for cand in (2048, 4096, 8192, 16384, 32768):
        if cand / rate * (args.steps + args.warmup) <= budget_s:
            n_sample = cand
    w = probe if n_sample == 1024 else oracle_sample_workload(args.workload, n_sample)
    if w is not probe:
        orc, model, pairs = oracle_prepare(w)
    for _ in range(args.warmup):
        oracle_step(orc, model, w, pairs)
    total = 0.0
    for _ in range(args.steps):
        total += oracle_step(orc, model, w, pairs)
    value = w.n_atoms * args.steps / total
    sample = ("each step = one fp64 energy+forces evaluation (oracle, OpenMP) of a %d-atom box of the family of %s, "
              "neighbour list prebuilt" % (w.n_atoms, args.workload))
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": args.workload, "sample_atoms": w.n_atoms},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": orc.num_threads(), "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


def max_over_ranks(x: float, world: int, device) -> float:
    """The slowest rank's time: replicas are independent, the job is as slow as its slowest member."""
    if world <= 1:
        return float(x)
    import torch
    import torch.distributed as dist

    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(n_atoms: int, steps: int, world: int, ms_max: float) -> float:
    """atom-steps/s of the whole job: every replica advances n_atoms atoms by `steps` steps."""
    return world * n_atoms * steps / (ms_max * 1e-3)


# ------------------------------------------------------------------------------------------------
# our arm
# ------------------------------------------------------------------------------------------------
SWITCHING_MD_STEPS = 200


def run_switching(args):
    """--workload config4_switching: the paper's switching-mode claim ("prediction times are
    nearly independent of the number of ensemble members") on the config-4 box under MD: ms per step of
    gmnn_md_ensemble_steps at several sampling rates against the same MD on a single-head model.  A side
    measurement (one GPU, graph-replayed MD loop), not the round's headline line."""
    import torch

    import paper_2505_22168_b200 as gm
    import workloads as wl

    torch.cuda.set_device(0)
    n = SWITCHING_MD_STEPS
    prec, fmode = MLP_NAMES[args.mlp], {"gather": 0, "pairbuf": 1}[args.forces]

    def timed(n_heads, rate):
        w = wl.li3po4_box(8192, n_heads=n_heads, skin=0.5)
        sysm = gm.System(gm.Model(w.model, mlp_precision=prec, force_mode=fmode), w.species)
        pos = torch.from_numpy(w.positions).cuda()
        vel = torch.from_numpy(w.velocities).cuda()
        mass = torch.from_numpy(w.masses).cuda()
        sysm.build_neighbors(pos, w.cell9, w.pbc, w.model.r_cut, w.skin)
        sysm.md_ensemble_steps(pos, vel, mass, w.dt_fs, max(args.warmup, 3) * 4, 4)  # warm-up, both modes
        torch.cuda.synchronize()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record()
        out = sysm.md_ensemble_steps(pos, vel, mass, w.dt_fs, n, rate)
        ev1.record()
        torch.cuda.synchronize()
        assert out["n_steps_done"] == n
        return ev0.elapsed_time(ev1) / n, len(out["sigma_e"]), out["n_rebuilds"]

    rows = {}
    for label, heads, rate in (("single_head", 1, 10 ** 9), ("m32_never", 32, 10 ** 9), ("m32_every_100", 32, 100),
                               ("m32_every_10", 32, 10), ("m32_every_1", 32, 1)):
        ms, ns, nreb = timed(heads, rate)
        rows[label] = {"ms_per_step": round(ms, 4), "samples": ns, "rebuilds": nreb}
    ms = rows["m32_every_100"]["ms_per_step"]
    print(json.dumps({
        "metric": "atom-steps/s (switching-mode shallow-ensemble MD)", "value": 8192 / (ms * 1e-3),
        "unit": "atom-steps/s", "n_gpus": 1, "steps": n, "warmup": max(args.warmup, 3) * 4, "ms_per_step": ms,
        "higher_is_better": True, "vs_baseline": None, "data": "synthetic", "dtype": "f32 (MLP mode: %s)" % args.mlp,
        "config": {"workload": "config4_switching", "n_atoms": 8192, "n_heads": 32, "skin": 0.5, "sampling_rate": 100,
                   "what": "li3po4_8192 with 32 heads, NVE on the mean energy, per-head pass every sampling_rate steps",
                   "mlp": args.mlp, "forces": args.forces},
        "rates": rows, "gpu_launches": int(gm.launch_count())}))
    return 0


def measure_run_peaks(dev, mlp):
    """Roofline denominators measured in THIS run ("measure them in the same run"): the fp32 FMA rate
    from the library's register-only FMA kernel, and dense fp16 / tf32 matmul rates (8192^3, cuBLAS through torch, the
    method of MEASURED_PEAKS.json) as the tensor roofs of the two split modes."""
    import torch

    import paper_2505_22168_b200 as gm

    # best of several calls (each: best of three 10-ms kernels): right after a long step the clock is still recovering
    out = {"fp32_fma_tflops": max(gm.measure_fp32_peak() for _ in range(4))}
    n = 8192

    def mm_rate(dtype, allow_tf32):
        torch.backends.cuda.matmul.allow_tf32 = allow_tf32
        a = torch.randn(n, n, device=dev, dtype=dtype)
        b = torch.randn(n, n, device=dev, dtype=dtype)
        torch.matmul(a, b)
        torch.cuda.synchronize()
        best = 0.0
        for _ in range(5):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            torch.matmul(a, b)
            e1.record()
            torch.cuda.synchronize()
            best = max(best, 2.0 * n ** 3 / (e0.elapsed_time(e1) * 1e-3) / 1e12)
        # sustained: back to back for about a second (the power cap pulls the clock down)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        reps = max(4, int(1.0 * best * 1e12 / (2.0 * n ** 3)))
        e0.record()
        for _ in range(reps):
            torch.matmul(a, b)
        e1.record()
        torch.cuda.synchronize()
        return best, 2.0 * n ** 3 * reps / (e0.elapsed_time(e1) * 1e-3) / 1e12

    if mlp in ("3xf16", "3xtf32", "tf32"):
        out["fp16_matmul_tflops_burst"], out["fp16_matmul_tflops_sustained"] = mm_rate(torch.float16, False)
    if mlp in ("3xtf32", "tf32"):
        out["tf32_matmul_tflops_burst"], out["tf32_matmul_tflops_sustained"] = mm_rate(torch.float32, True)
        torch.backends.cuda.matmul.allow_tf32 = False
    return out


def recorded_traffic(workload, mlp):
    """dram__bytes_read.sum + dram__bytes_write.sum per GEMM launch from the committed ncu capture of this workload and MLP
    mode (profiles/ncu_r2_gemm_traffic.json.txt, written from `ncu --set full`, command inside), or None: never a constant
    pasted into this file."""
    path = os.path.join(ROOT, "profiles", "ncu_r2_gemm_traffic.json.txt")
    if not os.path.exists(path):
        return None, None
    with open(path) as f:
        rec = json.load(f)
    ent = rec.get("%s/%s" % (workload, mlp))
    if not ent:
        return None, None
    return ent["dram_bytes_per_launch"], "profiles/ncu_r2_gemm_traffic.json.txt (ncu --set full of commit %s)" % rec.get("commit", "?")


def run_ours(args):
    import torch
    import torch.distributed as dist

    import paper_2505_22168_b200 as gm

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the GMNN path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    peaks = load_peaks()

    # what one "step" is: an MD step (default: every row of SURVEY 8(a) but a12), one gmnn_energy_forces call (--ef:
    # BASELINE.json config 3, "energy+forces throughput per N"), or one gmnn_ensemble_energy_forces call (config 4)
    mode = "ensemble" if args.workload == "config4" else ("ef" if args.ef else "md")
    w = make_bench_workload(args.workload, args.weight_sets)
    N = w.n_atoms
    mlp = MLP_NAMES[args.mlp]
    model = gm.Model(w.model, mlp_precision=mlp, force_mode={"gather": 0, "pairbuf": 1}[args.forces])
    sysm = gm.System(model, w.species)
    pos0 = torch.from_numpy(w.positions).to(dev)
    pos = pos0.clone()
    vel = torch.from_numpy(w.velocities).to(dev)
    masses = torch.from_numpy(w.masses).to(dev)
    if args.workload != "config5" and mode == "md":
        # long runs of the small boxes densify locally under the random-weight model: leave head room
        # (the list has a static capacity, like the paper's `extra_capacity`)
        vol = float(np.prod(w.cell.astype(np.float64)))
        sysm.set_int("capacity", int(2.0 * N / vol * 4.19 * (w.model.r_cut + w.skin) ** 3) + 64)
    sysm.build_neighbors(pos, w.cell9, w.pbc, w.model.r_cut, w.skin)
    if args.nvt > 0:
        sysm.set_nose_hoover(args.nvt, 100.0 * w.dt_fs, 3, 2, 3)
    counts = sysm.debug_read("count").astype(np.float64)
    nl_mean = float(counts.mean())
    r_list = w.model.r_cut + w.skin
    nc_mean = nl_mean * (w.model.r_cut / r_list) ** 3
    dims = [N_FEATURES, *w.model.hidden, w.model.n_heads]
    hidden_macs = sum(dims[l] * dims[l + 1] for l in range(len(dims) - 1))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    e_out = torch.empty(1, dtype=torch.float64, device=dev)
    ea_out = torch.empty(N, dtype=torch.float32, device=dev)
    f_out = torch.empty(N, 3, dtype=torch.float32, device=dev)

    def run_steps(n, series):
        """n steps of the timed kind; returns (epot + ekin series or None, rebuilds)."""
        if mode == "md":
            ep, ek, nr = sysm.md_verlet_steps(pos, vel, masses, w.dt_fs, n, want_series=series)
            return ((ep + ek) if series else None), nr
        for _ in range(n):
            if mode == "ef":
                sysm.energy_forces(pos, e_out, ea_out, f_out)
            else:
                sysm.ensemble_energy_forces(pos)
        return None, 0

    # ---- device-resident steps ----------------------------------------------------------------
    sysm.set_int("md_continue", 1)
    stream = torch.cuda.current_stream()
    total_rebuilds = 0
    sampler = ClockSampler(local)
    sampler.start()
    stages_on = not args.no_stages and mode != "ensemble"
    sysm.set_int("profile", 1 if stages_on else 0)  # the warm-up steps run the code path that is timed (events included)
    if args.warmup > 0:
        total_rebuilds += run_steps(args.warmup, True)[1]
    sysm.set_int("profile", 1 if stages_on else 0)  # drops the warm-up's stage events
    barrier()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    launches0 = gm.launch_count()
    t_begin = time.time()
    ev0.record(stream)
    etot_series, nreb = run_steps(args.steps, True)
    ev1.record(stream)
    barrier()
    t_end = time.time()
    launches = gm.launch_count() - launches0
    clocks = sampler.stop(t_begin, t_end)
    total_rebuilds += nreb
    ms = ev0.elapsed_time(ev1)
    stages = sysm.stage_times() if stages_on else []
    sysm.set_int("profile", 0)
    ms_max = max_over_ranks(ms, world, dev)
    value = whole_job_value(N, args.steps, world, ms_max)
    drift = None
    if etot_series is not None:
        etot = etot_series.cpu().numpy()
        drift = float(np.abs(etot - etot[0]).max() / N)

    # ---- end to end through the host-buffer entry ----------------------------------------------
    e2e_steps = max(3, min(args.steps, 10))
    hpos = torch.from_numpy(w.positions).pin_memory()
    hfrc = torch.empty(N, 3, dtype=torch.float32).pin_memory()
    sysm.build_neighbors(pos0, w.cell9, w.pbc, w.model.r_cut, w.skin)
    hp_np, hf_np = hpos.numpy(), hfrc.numpy()
    if mode == "ensemble":
        # the ensemble call has no host-buffer entry: positions from pinned memory in, the four statistics out, every call
        dpos = torch.empty_like(pos0)
        houts = [torch.empty(N, dtype=torch.float32).pin_memory(), torch.empty(N, dtype=torch.float32).pin_memory(),
                 torch.empty(N, 3, dtype=torch.float32).pin_memory(), torch.empty(N, 3, dtype=torch.float32).pin_memory()]

        def e2e_call():
            dpos.copy_(hpos, non_blocking=True)
            outs = sysm.ensemble_energy_forces(dpos)
            for h, o in zip(houts, outs):
                h.copy_(o, non_blocking=True)
            torch.cuda.synchronize()

        d2h = 32 * N
    else:
        def e2e_call():
            sysm.energy_forces_host(hp_np, hf_np)

        d2h = 12 * N + 8
    for _ in range(2):
        e2e_call()
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        e2e_call()
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    e2e = {"value": world * N * e2e_steps / max_over_ranks(e2e_s, world, dev), "unit": UNIT, "h2d_bytes_per_step": 12 * N,
           "d2h_bytes_per_step": d2h, "steps": e2e_steps,
           "what": ("gmnn_ensemble_energy_forces: pinned positions in, e_mean, e_var, f_mean, f_var out, every call" if mode == "ensemble"
                    else "gmnn_energy_forces_host: pinned positions in, forces and total energy out, every step")}
    # ---- roofs measured in this run, after BOTH timed regions (seconds of dense matmul at the power cap leave the part at
    # 1.36 GHz for a while: measured before the end-to-end loop they cost it 30 - 45 % on the small workloads) ------------
    run_peaks = measure_run_peaks(dev, args.mlp)

    # ---- per-stage roofline (live CUDA events of the timed region) ------------------------------
    sm = stage_model(w, nl_mean, nc_mean, hidden_macs, args.mlp, args.forces)
    # roofs: HBM and the fp16/bf16 tensor rate from MEASURED_PEAKS.json (driver-measured on this pool; sustained: the
    # kernels are timed inside a long step); fp32 FMA and tf32 measured in this run
    fp32_peak_tflops = run_peaks.get("fp32_fma_tflops") or float("nan")
    if args.mlp == "3xf16":
        tensor_peak, tensor_src = peaks["bf16_sustained"], "bf16_tflops_sustained of MEASURED_PEAKS.json (%s); fp16 runs at the bf16 rate: %.0f TFLOP/s sustained in this run" % (
            peaks["source"], run_peaks.get("fp16_matmul_tflops_sustained", float("nan")))
    else:
        tensor_peak = run_peaks.get("tf32_matmul_tflops_sustained", 0.5 * peaks["bf16_sustained"])
        tensor_src = "tf32 8192^3 matmul, sustained, measured in this run"
    stage_out = {}
    per_step_ms = {}
    for name, mean_ms, cnt in stages:
        per_step = mean_ms * cnt / args.steps
        per_step_ms[name] = per_step
        info = sm.get(name, dict(bytes=0.0, flops=0.0, bound="hbm"))
        sec = mean_ms * 1e-3
        ent = {"ms": round(mean_ms, 4), "per_step_ms": round(per_step, 4), "ns_per_atom": round(mean_ms * 1e6 / N, 3),
               "bound": info["bound"]}
        if sec > 0 and info["bytes"] > 0:
            ent["hbm_gbs"] = round(info["bytes"] * N / sec / 1e9, 1)
            ent["hbm_frac"] = round(ent["hbm_gbs"] / peaks["hbm_gbs"], 4)
        if sec > 0 and info["flops"] > 0:
            tf = info["flops"] * N / sec / 1e12
            ent["tflops"] = round(tf, 2)
            ent["flop_frac"] = round(tf / (tensor_peak if info["bound"] == "tensor" else fp32_peak_tflops), 4)
        stage_out[name] = ent
    # the dominant stage among those with an algorithmic byte / flop count (the in-loop list rebuild has none: it is
    # bookkeeping around a sort, and dominates only where the workload rebuilds at every step, i.e. config 3's skin 0)
    modelled = {k: v for k, v in per_step_ms.items() if sm.get(k, {}).get("bytes", 0.0) > 0 or sm.get(k, {}).get("flops", 0.0) > 0}
    dom = max(modelled, key=modelled.get) if modelled else None
    if dom is not None and args.mlp != "fp32" and "mlp_forward" in per_step_ms and "mlp_backward" in per_step_ms:
        # the GEMM launches of mlp_forward and mlp_backward are one kernel (k_gemm_tc[_pair]): it is the
        # dominant kernel if together they outweigh every other stage
        if per_step_ms["mlp_forward"] + per_step_ms["mlp_backward"] >= per_step_ms[dom]:
            dom = "mlp_forward"
    roofline = None
    if dom is not None:
        info = sm.get(dom, dict(bytes=0.0, flops=0.0, bound="hbm"))
        mean_ms = [m for n_, m, _ in stages if n_ == dom][0]
        sec = mean_ms * 1e-3
        if info["bound"] == "hbm":
            ach, peak, unit = info["bytes"] * N / sec / 1e9, peaks["hbm_gbs"], "GB/s"
        elif info["bound"] == "tensor":
            ach, peak, unit = info["flops"] * N / sec / 1e12, tensor_peak, "TFLOP/s"
        else:
            ach, peak, unit = info["flops"] * N / sec / 1e12, fp32_peak_tflops, "TFLOP/s"
        roofline = {"kernel": dom, "bound": info["bound"], "achieved": round(ach, 3), "peak": round(peak, 3),
                    "unit": unit, "frac": round(ach / peak, 4), "traffic": None,
                    "peak_source": {"hbm": "MEASURED_PEAKS.json hbm_gbs (%s)" % peaks["source"], "tensor": tensor_src,
                                    "alu": "fp32 FMA rate measured in this run (gmnn_measure_fp32_peak)"}[info["bound"]],
                    "share_of_step": round(per_step_ms[dom] / (ms_max / args.steps), 4),
                    "algorithmic_per_atom": {"bytes": info["bytes"], "flops": info["flops"]}}
        if info["bound"] == "tensor":
            # the four GEMM launches of a step (mlp_forward + mlp_backward) are one kernel family:
            # report them together, per launch
            t_f = [m for n_, m, _ in stages if n_ == "mlp_forward"][0]
            t_b = [m for n_, m, _ in stages if n_ == "mlp_backward"][0]
            n_launch = 2 * len(w.model.hidden) * w.model.n_weight_sets
            ach = 2.0 * info["flops"] * N / ((t_f + t_b) * 1e-3) / 1e12
            traffic, traffic_src = recorded_traffic(args.workload, args.mlp)
            roofline.update({"kernel": {"3xf16": "k_gemm_tc_pair<F16>", "3xtf32": "k_gemm_tc_pair"}.get(args.mlp, "k_gemm_tc"),
                             "launches_per_step": n_launch, "achieved": round(ach, 3), "frac": round(ach / peak, 4),
                             "avg_launch_ms": round((t_f + t_b) / n_launch, 4),
                             "share_of_step": round((per_step_ms["mlp_forward"] + per_step_ms["mlp_backward"])
                                                    / (ms_max / args.steps), 4),
                             # algorithmic = the fused count of SURVEY 8(d): G in, dG out, E_i out; what the unfused
                             # layers actually move through HBM (H, D, dZ written and re-read as fp32) is listed beside it
                             "algorithmic_per_atom": {"bytes": 4.0 * (2 * N_FEATURES + 1), "flops": 2.0 * info["flops"]},
                             "unfused_hbm_bytes_per_atom": 4.0 * (2 * N_FEATURES + (8 if w.model.n_heads == 1 else 9) * w.model.hidden[0]),
                             "traffic": traffic, "traffic_source": traffic_src})
        if info["bound"] == "tensor" and args.mlp in ("3xtf32", "3xf16"):
            roofline["note"] = ("achieved counts the ALGORITHMIC flops (one product per multiply-add); the %s split "
                                "executes 3 tensor-core MMAs per product, so tensor-pipe flops are 3x achieved"
                                % {"3xtf32": "3xTF32", "3xf16": "3xFP16"}[args.mlp])
            roofline["executed_tflops"] = round(3 * ach, 3)
            roofline["executed_frac"] = round(3 * ach / peak, 4)

    sysm.check()

    if rank == 0:
        what = {"md": w.name + ", %s velocity Verlet, dt %.2f fs, skin %.1f" % (
                    "NVT (Nose-Hoover chain 3/2/3, %g K)" % args.nvt if args.nvt > 0 else "NVE", w.dt_fs, w.skin),
                "ef": w.name + ", one gmnn_energy_forces call per step on a prebuilt list (skin %.1f)" % w.skin,
                "ensemble": w.name + ", one gmnn_ensemble_energy_forces call per step (%d heads: e_mean, e_var, f_mean, f_var)" % w.model.n_heads}[mode]
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_max / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": {"fp32": "f32", "3xtf32": "f32 (MLP: 3xTF32 split on tcgen05, fp32 accumulate)",
                      "3xf16": "f32 (MLP: 3xFP16 split on tcgen05, fp32 accumulate)",
                      "tf32": "tf32 MLP, f32 elsewhere"}[args.mlp],
            "data": "synthetic",
            "config": {"workload": args.workload, "step": mode, "n_atoms": N, "what": what, "mlp": args.mlp, "forces": args.forces,
                       "hidden": list(w.model.hidden), "n_heads": w.model.n_heads, "weight_sets": w.model.n_weight_sets,
                       "neighbors_in_list_mean": round(nl_mean, 2), "rebuilds_in_timed_region": nreb,
                       "l2": "inputs_exceed_l2" if N >= 65536 else "working set of this small case is L2-resident",
                       "replicas": world},
            "gpu_launches": launches, "clocks": clocks, "e2e": e2e, "roofline": roofline, "stages": stage_out,
            "peaks_measured_in_this_run": {k: round(v, 2) for k, v in run_peaks.items()},
            "energy_drift_ev_per_atom": drift, "ns_per_atom_step": ms_max * 1e6 / args.steps / N,
        }
        if world == 1 and not args.no_cpu_baseline:
            line["cpu_baseline"] = cpu_baseline(args.workload)
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="config5",
                    help="config5 (default, 1,048,576 atoms), config2, config3_<N>; config4: one gmnn_ensemble_energy_forces call per "
                         "step (32 heads); config4_switching: side measurement of the switching-mode ensemble MD (its own JSON line)")
    ap.add_argument("--ef", action="store_true",
                    help="a step is one gmnn_energy_forces call on a prebuilt list instead of one MD step (BASELINE.json config 3: "
                         "energy+forces throughput per N)")
    ap.add_argument("--mlp", default="3xf16", choices=sorted(MLP_NAMES),
                    help="3xf16 (default) / 3xtf32: tcgen05 tensor cores, fp32-accurate three-product split on fp16 / tf32 "
                         "operands; fp32: SIMT FMA; tf32: single pass")
    ap.add_argument("--forces", default="pairbuf", choices=["gather", "pairbuf"],
                    help="force reduction: gather form, or pair buffer with a reverse-pair index (both deterministic)")
    ap.add_argument("--weight-sets", default="shared", choices=["shared", "species"],
                    help="shared: one NN for all species (Eq. 4, the headline); species: one NN per species, the rows of the "
                         "MLP stage grouped by species (a side measurement)")
    ap.add_argument("--no-stages", action="store_true",
                    help="no per-stage CUDA events: the MD loop then replays its step as a CUDA graph (no roofline entry)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--nvt", type=float, default=0.0,
                    help="temperature in K: run the steps NVT with the paper's Nose-Hoover chain (3/2/3, tau = 100 dt; "
                         "PAPER.md:365-375) instead of NVE; recorded in config")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.workload == "config4_switching":
        return run_switching(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
