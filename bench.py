#!/usr/bin/env python
"""bench.py -- one JSON line: mesh points/s of the grid-integration hot path (gint_vlocal followed by gint_rho,
fp64) on the synthetic workloads of BASELINE.json, with the roofline fraction of the dominant kernel and the CPU
oracle timed beside it.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--cfg 4] [--impl ours|reference]

A "step" is one pass of the whole hot path over the whole mesh: gint_vlocal (Eq. 2) then gint_rho
(Eq. 3).  `value` = mesh points / step time (device-resident inputs, CUDA events on the launching
stream).  `e2e` = the same through the host-buffer C-ABI calls (H2D + kernels + D2H every step).
The path does not shard (BASELINE.json north_star: one GPU, no collectives): with --gpus N every rank runs an
independent replica ("replicas only") and value = N * points / max-over-ranks time.
--impl reference times the CPU oracle (oracle/), as it stands, on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

FP64_PEAK_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12     # 37.2: 148 SMs x 64 FP64 FMA/clk x 2 flop x 1.965 GHz
EVAL_FLOP_PER_INCIDENCE = 120.0                      # orbital evaluation per (point, atom)
METRIC = "mesh points/s for gint_vlocal and gint_rho (fp64); % of FP64/HBM roofline"


def alg_flops(st: dict) -> float:
    """Algorithmic flops of ONE call (vlocal or rho): unique orbital pairs + V*dV scaling + orbital evaluation."""
    return float(st["alg_sum_n2"] + st["alg_sum_n"]) + float(st["alg_sum_n"]) + EVAL_FLOP_PER_INCIDENCE * st["alg_incidence"]


TRAFFIC_CSV = os.path.join("profiles", "r3_traffic.csv")
FORCE_GRAD_FLOP_PER_INCIDENCE = 360.0                # value + gradient of the orbitals of one atom at one point (3x the value alone)


def force_alg_flops(st: dict) -> float:
    """Algorithmic flops of ONE gint_force_stress call: Psi needs every ORDERED pair of orbitals non-zero at a point
    (2 n_g^2; the mirror halving of Eq. 2 / Eq. 3 does not apply), then three gradient components times Psi (6 n_g), plus the
    evaluation of values and gradients."""
    return 2.0 * st["alg_sum_n2"] + 6.0 * st["alg_sum_n"] + FORCE_GRAD_FLOP_PER_INCIDENCE * st["alg_incidence"]


def csrc_digest() -> str:
    """sha256 over the sources of the timed gint_vlocal / gint_rho path (everything in csrc/ but the force kernels): the committed
    ncu capture names the digest it was taken on."""
    import hashlib
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_2409_09399_b200", "csrc")
    for name in sorted(os.listdir(d)):
        if name == "gint_force.cu":
            continue
        with open(os.path.join(d, name), "rb") as f:
            h.update(name.encode()); h.update(f.read())
    return h.hexdigest()[:16]


def ncu_traffic(cfg: int, batch, call: str):
    """DRAM bytes (dram__bytes_read.sum + dram__bytes_write.sum, summed over the kernels of one `call` = "vlocal_main" or
    "rho_main", all waves) from the committed ncu capture profiles/r3_traffic.csv, with a note.  A row is keyed by the config AND
    the grid-batch shape it was captured with (the launch the tuner chose may differ from run to run), and names the digest of the
    kernel sources: no row for this shape, or sources changed since, and the figure is not reported."""
    path = os.path.join(ROOT, TRAFFIC_CSV)
    shape = "x".join(str(int(b)) for b in batch)
    try:
        with open(path) as f:
            lines = [ln for ln in f.read().splitlines() if ln and not ln.startswith("#")]
        for ln in lines[1:]:
            c, b, k, rd, wr, digest = [x.strip() for x in ln.split(",")[:6]]
            if int(c) == cfg and b == shape and k == call:
                if digest != csrc_digest():
                    print(f"bench.py: {TRAFFIC_CSV} was captured on csrc digest {digest}, the tree is at {csrc_digest()}: "
                          "roofline.traffic not reported (re-capture with ncu)", file=sys.stderr)
                    return None, f"stale capture (csrc digest {digest} != {csrc_digest()})"
                return int(rd) + int(wr), f"{TRAFFIC_CSV}, batch {shape}, csrc digest {digest}"
    except (OSError, ValueError):
        pass
    return None, f"no capture for cfg {cfg} with batch {shape}"


def cpu_model() -> str:
    try:
        with open("/proc/cpuinfo") as f:
            for ln in f:
                if ln.startswith("model name"):
                    return ln.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def max_over_ranks(values, device, world: int):
    """Element-wise maximum over all ranks (torch.distributed all-reduce; identity for one rank)."""
    if world <= 1:
        return [float(v) for v in values]
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t.tolist()]


def job_value(npts: int, t_step: float, world: int) -> float:
    """Whole-job mesh points/s: the path does not shard, every rank runs a replica of the full mesh."""
    return world * npts / t_step


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for ln in self.proc.stdout:
            self.lines.append(ln.strip())

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def oracle_sample(w, V, D, plist, budget_s: float = 20.0):
    """Time the oracle (as it stands, OpenMP on all host cores) on a bounded sample: a contiguous run of pair keys
    for vlocal and a contiguous run of mesh points (whole a1-planes) for rho, sized from a short probe so that the
    two legs take about `budget_s` seconds together.  Returns (points/s equivalent of one vlocal+rho step, dict)."""
    from oracle import oracle as O
    npairs, npts = len(plist[0]), w.n_points
    plane = int(w.mesh[1]) * int(w.mesh[2])
    # probe
    n0p = min(npairs, 64)
    t0 = time.perf_counter(); O.vlocal(w, V, plist, sel=np.arange(n0p, dtype=np.int64)); tp = (time.perf_counter() - t0) / n0p
    mid = (int(w.mesh[0]) // 2) * plane
    n0g = min(npts, 4096)
    sel0 = np.arange(mid, mid + n0g, dtype=np.int64) % npts
    t0 = time.perf_counter(); O.rho(w, D, plist, sel=sel0); tg = (time.perf_counter() - t0) / n0g
    np_s = int(min(npairs, max(n0p, 0.5 * budget_s / tp)))
    ng_s = int(min(npts, max(n0g, 0.5 * budget_s / tg)))
    if ng_s < npts:
        ng_s = max(plane, ng_s // plane * plane) if ng_s >= plane else ng_s
    # sample in the middle of the list / mesh (atoms and planes are homogeneous in all five configs)
    p0 = (npairs - np_s) // 2
    g0 = ((int(w.mesh[0]) - max(1, ng_s // plane)) // 2) * plane if ng_s >= plane else mid
    t0 = time.perf_counter(); O.vlocal(w, V, plist, sel=np.arange(p0, p0 + np_s, dtype=np.int64)); t_v = time.perf_counter() - t0
    t0 = time.perf_counter(); O.rho(w, D, plist, sel=(np.arange(g0, g0 + ng_s, dtype=np.int64) % npts)); t_r = time.perf_counter() - t0
    t_step = t_v * npairs / np_s + t_r * npts / ng_s          # extrapolated full-mesh step
    info = {"kind": "oracle", "cores": O.threads(), "cpu": cpu_model(), "extrapolated": bool(np_s < npairs or ng_s < npts),
            "sample_fraction": {"vlocal_pair_keys": np_s / npairs, "rho_mesh_points": ng_s / npts},
            "sample": f"vlocal: {np_s} of {npairs} pair keys in {t_v:.2f} s; rho: {ng_s} of {npts} mesh points in {t_r:.2f} s; "
                      f"scaled to the full mesh (vlocal {t_v * npairs / np_s:.1f} s + rho {t_r * npts / ng_s:.1f} s per step)"}
    return npts / t_step, info


def run_reference(args):
    """--impl reference: the CPU oracle on a bounded sample per step (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return 0
    from oracle import oracle as O
    from paper_2409_09399_b200 import workloads as W
    w = W.make_workload(args.cfg)
    V = W.make_potential(w)
    plist = O.pairs(w)
    D = W.make_density_blocks(w, *plist)
    budget = max(4.0, min(20.0, 150.0 / max(1, args.steps + args.warmup)))
    vals, info = [], None
    for s in range(args.warmup + args.steps):
        v, info = oracle_sample(w, V, D, plist, budget_s=budget)
        if s >= args.warmup:
            vals.append(v)
    value = float(np.median(vals))
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": "mesh points/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * w.n_points / value,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name, "cfg": args.cfg, "mesh": [int(m) for m in w.mesh], "atoms": int(w.n_atoms),
                       "note": "CPU oracle, each step a bounded sample scaled to the full mesh"},
            "cpu_baseline": {"value": value, "unit": "mesh points/s", **info},
            "e2e": {"value": value, "unit": "mesh points/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--cfg", type=int, default=4, help="BASELINE.json configs[i]; 4 = TBG 10,444 atoms (headline); 5 = mixed-species bilayer (SURVEY 8f NEXT-4)")
    ap.add_argument("--impl", default="ours", choices=("ours", "reference"))
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-force", action="store_true", help="skip the (separately reported) gint_force_stress timing")
    ap.add_argument("--batch", default="", help="override grid-batch shape, e.g. 8,8,8")
    ap.add_argument("--csrc-digest", action="store_true", help="print the digest of the kernel sources (for profiles/r3_traffic.csv) and exit")
    args = ap.parse_args()
    if args.csrc_digest:
        print(csrc_digest())
        return 0
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import torch.distributed as dist
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the hot path has no CPU fallback")
    rank, world, local = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)

    from paper_2409_09399_b200 import workloads as W
    from paper_2409_09399_b200.gint import FLAG_TUNE, Gint, batch_flag, fp64_peak

    # same-run FP64 peak: DMMA / DFMA micro-benchmark of the library, in this process, before the timed region
    peak_measured = fp64_peak(local)

    t0 = time.perf_counter()
    w = W.make_workload(args.cfg)
    V = W.make_potential(w)
    # default: the library's init-time batch-shape tuner; --batch fixes the shape instead
    flags = batch_flag(*(int(x) for x in args.batch.split(","))) if args.batch else FLAG_TUNE
    t1 = time.perf_counter()
    g = Gint.from_workload(w, device=local, flags=flags)
    torch.cuda.synchronize()
    t_init = time.perf_counter() - t1
    plist = g.pairs()                      # integer pair list from the library (bit-checked against the oracle in tests/)
    D = W.make_density_blocks(w, *plist)
    st = g.stats()
    F_alg = alg_flops(st)
    npts = w.n_points

    V_d = torch.from_numpy(V).to(dev)
    D_d = torch.from_numpy(D).to(dev)
    H_d = torch.empty(g.n_values, dtype=torch.float64, device=dev)
    rho_d = torch.empty(npts, dtype=torch.float64, device=dev)
    stream = torch.cuda.current_stream()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing: inputs (V 8*npts B, D 8*n_values B) are larger than L2 for cfg >= 3; for the small
    # configs an L2 flush (write of a 256 MiB buffer) runs between steps, outside the per-call events.
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev) if 8 * (npts + g.n_values) < (200 << 20) else None
    for _ in range(args.warmup):
        g.vlocal(V_d, out=H_d); g.rho(D_d, out=rho_d)
    barrier()
    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(args.steps)]
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    barrier()
    wall0 = time.perf_counter()
    for s in range(args.steps):
        if flush is not None:
            flush.zero_()
        ev[s][0].record(stream)
        g.vlocal(V_d, out=H_d)
        ev[s][1].record(stream)
        g.rho(D_d, out=rho_d)
        ev[s][2].record(stream)
    barrier()
    wall = time.perf_counter() - wall0
    clocks = sampler.stop() if rank == 0 else None
    t_v = np.array([ev[s][0].elapsed_time(ev[s][1]) for s in range(args.steps)]) * 1e-3
    t_r = np.array([ev[s][1].elapsed_time(ev[s][2]) for s in range(args.steps)]) * 1e-3
    t_step = float(np.median(t_v + t_r))          # median over the steps
    # identity P4: sum_g V rho dV == <D, H> -- a full-size consistency check of the two kernels
    dV = abs(np.linalg.det(w.cell)) / npts
    lhs = float((V_d * rho_d).sum().item() * dV); rhs = float((D_d * H_d).sum().item())
    p4 = abs(lhs - rhs) / max(abs(lhs), 1e-300)

    # ---- per-kernel durations of the dominant kernels (CUDA events inside the library around the main kernel)
    kt = g.kernel_times()                     # seconds, last call of each: {"vlocal_main": .., "rho_main": ..}

    # ---- Pulay force + stress (Eq. 4 / Eq. 5): reported beside the step, not part of `value`
    force = None
    if not args.no_force:
        g.force_stress(V_d, D_d); torch.cuda.synchronize()
        fs = ClockSampler(local)
        if rank == 0:
            fs.start()
        tf = []
        for _ in range(2):
            g.force_stress(V_d, D_d); torch.cuda.synchronize(); tf.append(g.force_time())
        t_f = float(np.median(tf))
        F_force = force_alg_flops(st)
        force = {"ms": 1e3 * t_f, "points_per_s": npts / t_f,
                 "what": "gint_force_stress: forces of all atoms and the 3x3 stress in one call (k_sym_full + k_force_batch)",
                 "roofline": {"bound": "alu", "achieved": F_force / t_f / 1e12, "peak": FP64_PEAK_TFLOPS, "unit": "TFLOP/s",
                              "frac": F_force / t_f / 1e12 / FP64_PEAK_TFLOPS, "alg_flop_per_call": F_force,
                              "flops": "2 sum n_g^2 (Psi, every ordered orbital pair) + 6 sum n_g (grad . Psi) + 360 per (point, atom) incidence"},
                 "clocks": fs.stop() if rank == 0 else None}

    # ---- end to end through the host-buffer entry points (pinned host memory, H2D + D2H every step)
    e2e = None
    if not args.no_e2e:
        V_h = torch.from_numpy(V).pin_memory(); D_h = torch.from_numpy(D).pin_memory()
        H_h = torch.empty(g.n_values, dtype=torch.float64).pin_memory(); rho_h = torch.empty(npts, dtype=torch.float64).pin_memory()
        g.vlocal_host(V_h, H_h); g.rho_host(D_h, rho_h)
        barrier()
        n_e2e = max(1, args.steps)
        es = ClockSampler(local)
        if rank == 0:
            es.start()
        te0 = time.perf_counter()
        for _ in range(n_e2e):
            g.vlocal_host(V_h, H_h); g.rho_host(D_h, rho_h)      # each call synchronises its stream before returning
        barrier()
        t_e2e = (time.perf_counter() - te0) / n_e2e
        e2e = {"t": t_e2e, "h2d": 8 * (npts + g.n_values), "d2h": 8 * (g.n_values + npts), "steps": n_e2e,
               "clocks": es.stop() if rank == 0 else None}
        del V_h, D_h, H_h, rho_h

    t_step, t_e2e_max = max_over_ranks([t_step, e2e["t"] if e2e else 0.0], dev, world)
    if e2e:
        e2e["t"] = t_e2e_max

    if rank == 0:
        cpu = None
        if not args.no_cpu_baseline and world == 1:
            val, info = oracle_sample(w, V, D, plist, budget_s=20.0)
            cpu = {"value": val, "unit": "mesh points/s", **info}
        dom = "vlocal_main" if kt["vlocal_main"] >= kt["rho_main"] else "rho_main"
        achieved = F_alg / kt[dom] / 1e12
        traffic, traffic_note = ncu_traffic(args.cfg, (st["batch_bx"], st["batch_by"], st["batch_bz"]), dom)
        # context: the same kernel against the HBM roofline (measured copy bandwidth of this pool's B200s, MEASURED_PEAKS.json;
        # 6650 GB/s is the profiling guide's fallback).  Algorithmic bytes: V + canonical H (vlocal) / canonical D + rho (rho).
        try:
            with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
                hbm_peak, hbm_src = float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
        except (OSError, KeyError, ValueError):
            hbm_peak, hbm_src = 6650.0, "fallback (B200_PROFILING.md)"
        alg_bytes = 8.0 * (npts + st["n_canon"] * (g.n_values / max(1, g.n_pairs)))
        hbm_achieved = alg_bytes / kt[dom] / 1e9
        line = {
            "metric": METRIC, "value": job_value(npts, t_step, world), "unit": "mesh points/s", "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t_step, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name, "cfg": args.cfg, "mesh": [int(m) for m in w.mesh], "atoms": int(w.n_atoms),
                       "orbitals": int(g.n_orb), "pair_blocks": int(g.n_pairs),
                       "batch": [st["batch_bx"], st["batch_by"], st["batch_bz"]],
                       "batch_tuner": {"seconds": st["tune_us"] / 1e6, "tried_ns_per_point": {f"{a}x{b}x{c}": t for a, b, c, t in g.tune_report()}},
                       "l2": "inputs larger than L2" if flush is None else "L2 flushed between steps",
                       "parallelism": "replicas only" if world > 1 else "single GPU"},
            "vlocal_points_per_s": npts / float(np.median(t_v)), "rho_points_per_s": npts / float(np.median(t_r)),
            "ms_vlocal": 1e3 * float(np.median(t_v)), "ms_rho": 1e3 * float(np.median(t_r)), "init_s": t_init,
            "alg_flop_per_call": F_alg, "alg_tflops_vlocal": F_alg / float(np.median(t_v)) / 1e12,
            "alg_tflops_rho": F_alg / float(np.median(t_r)) / 1e12,
            "roofline_frac_vlocal": F_alg / kt["vlocal_main"] / 1e12 / FP64_PEAK_TFLOPS,
            "roofline_frac_rho": F_alg / kt["rho_main"] / 1e12 / FP64_PEAK_TFLOPS,
            "identity_P4_rel": p4,
            "roofline": {"bound": "alu", "kernel": dom, "achieved": achieved, "peak": FP64_PEAK_TFLOPS, "unit": "TFLOP/s",
                         "frac": achieved / FP64_PEAK_TFLOPS, "traffic": traffic,
                         "traffic_unit": "bytes per call: dram__bytes_read.sum + dram__bytes_write.sum over the call's kernels (k_eval_phi + k_tiles, all waves)",
                         "traffic_source": traffic_note,
                         "kernels": "k_eval_phi + k_tiles<%s> over all waves of one call (CUDA events inside the library)" % ("vlocal" if dom == "vlocal_main" else "rho"),
                         "peak_source": "stated: 148 SMs x 64 FP64 FMA/clk x 2 x 1.965 GHz (DESIGN.md 6); peak_measured = gint_fp64_peak in this process",
                         "peak_measured": peak_measured,
                         "kernel_ms": {k: 1e3 * v for k, v in kt.items()},
                         "hbm_context": {"achieved": hbm_achieved, "peak": hbm_peak, "unit": "GB/s", "frac": hbm_achieved / hbm_peak,
                                         "peak_source": hbm_src, "algorithmic_bytes": alg_bytes}},
            "clocks": clocks,
            "gpu_launches": args.steps * (st["launches_vlocal"] + st["launches_rho"]),
            "wall_s_timed_region": wall, "setup_s": t1 - t0,
        }
        if e2e:
            line["e2e"] = {"value": world * npts / e2e["t"], "unit": "mesh points/s", "h2d_bytes_per_step": e2e["h2d"],
                           "d2h_bytes_per_step": e2e["d2h"], "ms_per_step": 1e3 * e2e["t"], "steps": e2e["steps"],
                           "clocks": e2e["clocks"]}
        if force:
            line["force_stress"] = force
        if cpu:
            line["cpu_baseline"] = cpu
        print(json.dumps(line))
    g.close()
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
