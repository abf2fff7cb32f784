"""bench.py — forward and gradient env-steps/s of the dmx hot path on B200 (BASELINE.json metric).

A "step" is one pass of the whole hot path over one batch of synthetic environments: dmx_rollout (adaptive RK
forward with tape, S1-S9) followed by dmx_rollout_backward (reverse sweep with the CFD straight-through VJP,
S10-S12).  Workload at N=1: BASELINE config 2 (planar push, 4096 envs, fp64, Tsit5 rtol 1e-6, 250 control knots),
seeded synthetic inputs from paper_2506_14186_b200/workloads.py.  N>1: one process per GPU, envs sharded, no
data-path collective (weak scaling: every rank runs a full 4096-env batch with its own seed).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C2] [--nenv n] [--impl reference]

Prints ONE JSON line.  `--impl reference` times the CPU oracle (test infrastructure, as it stands) instead.
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

from paper_2506_14186_b200 import workloads as W  # noqa: E402

METRIC = "env-steps/s forward and gradient env-steps/s"
UNIT = "accepted env-steps/s (forward + reverse sweep)"
# Algorithmic FP64 work per unit: flops per attempted forward step
# (6 F evaluations + stage combinations + error norm) and per F evaluation, FMA = 2.
FLOPS_PER_ATTEMPT = dict(C1=7e2, C2=5e4, C3=1.2e5, C4=4.7e5, C5=3.9e5)
FLOPS_PER_FEVAL = dict(C1=1e2, C2=8e3, C3=2e4, C4=8e4, C5=6e4)


# dram__bytes_read.sum + dram__bytes_write.sum per launch from the ncu --set full captures of the default workload
# (profiles/r1_rollout_kernel.md, profiles/r1_backward_kernel.md); other workloads were not captured.
NCU_TRAFFIC_C2_F64_4096 = {"rollout_kernel": 0.571e9, "backward_kernel": 0.716e9}


def grad_flops_per_accepted(cfg, cfd):
    """gradient per accepted step = 6 F (recompute) + 6 VJP (2.5 F each) + 6 F~ solves when CFD is on."""
    return (6 + 15 + (6 if cfd else 0)) * FLOPS_PER_FEVAL[cfg]


class ClockSampler:
    """nvidia-smi clocks and throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self.proc:
            self.proc.terminate()
        sm, mx, reasons = [], 0.0, set()
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx = max(mx, float(r[1]))
            except (ValueError, IndexError):
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return dict(sm_mhz=float(np.median(sm)) if sm else None, sm_max_mhz=mx or None, reasons=sorted(reasons), samples=len(sm))


def make_workload(cfg, nenv, rank):
    kw = {}
    if nenv:
        kw["nenv"] = nenv
    if rank:
        kw["seed"] = 250614186 + int(cfg[1]) + 1000 * rank
    return W.make(cfg, **kw)


def oracle_sample(w, cfg, n_sample, cfd, threads):
    """Times the oracle (forward with tape + reverse sweep) on the first n_sample envs; returns env-steps/s."""
    from oracle import oracle as O
    orc = O.Oracle(w["model"])
    x0 = w["x0"][:n_sample]
    ctrl = None if w["ctrl"] is None else w["ctrl"][:n_sample]
    t0 = time.perf_counter()
    of = orc.rollout(x0, ctrl, w["nknot"], w["knot_dt"], None, w["horizon"], w["opts"], threads=threads)
    t_f = time.perf_counter() - t0
    _, g = w["loss_grad"](of["xT"], x0)
    t0 = time.perf_counter()
    orc.rollout_grad(x0, ctrl, w["nknot"], w["knot_dt"], None, w["horizon"], w["opts"], dLdxT=g, cfd_on=cfd, threads=threads,
                     want_params=False)
    t_g = time.perf_counter() - t0            # rollout_grad = forward with tape + reverse sweep
    acc = float(of["stats"]["n_accept"].sum())
    return dict(grad=acc / t_g, fwd=acc / t_f, accepted=acc, t_fwd=t_f, t_grad=t_g)


def run_reference(args, rank, world):
    """The tier's reference arm: the CPU oracle on the box's host cores, each step a bounded sample of the workload."""
    if rank != 0:
        return
    cfg = args.config
    w = make_workload(cfg, args.nenv, 0)
    cores = os.cpu_count() or 1
    n_sample = min(w["nenv"], args.ref_sample)
    vals = []
    for i in range(args.warmup + args.steps):
        r = oracle_sample(w, cfg, n_sample, w["cfd"], cores)
        if i >= args.warmup:
            vals.append(r)
    t = float(np.mean([r["t_grad"] for r in vals]))
    v = float(np.mean([r["accepted"] for r in vals])) / t
    sample = "first %d of %d envs of %s, forward with tape + reverse sweep%s" % (n_sample, w["nenv"], w["name"], " (CFD)" if w["cfd"] else "")
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": 1e3 * t, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": w["name"], "nenv": n_sample, "horizon_s": w["horizon"], "rtol": w["opts"]["rtol"]},
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "forward_env_steps_per_s": float(np.mean([r["fwd"] for r in vals])),
    }), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="dmx", choices=["dmx", "reference"])
    ap.add_argument("--config", default="C2", choices=list(W.CONFIGS))
    ap.add_argument("--nenv", type=int, default=0, help="0 = the BASELINE size of the config")
    ap.add_argument("--precision", type=int, default=64, choices=[64, 32])
    ap.add_argument("--ref-sample", type=int, default=256, help="envs per step of the reference arm / cpu_baseline")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-cfd", action="store_true")
    args = ap.parse_args()
    rank, world, local = int(os.environ.get("RANK", 0)), int(os.environ.get("WORLD_SIZE", 1)), int(os.environ.get("LOCAL_RANK", 0))
    if args.impl == "reference":
        return run_reference(args, rank, world)
    args.warmup = max(args.warmup, 3)

    import torch
    import torch.distributed as dist
    from paper_2506_14186_b200 import binding as B
    from paper_2506_14186_b200.sharding import max_over_ranks, sum_over_ranks
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the dmx path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    cfg = args.config
    w = make_workload(cfg, args.nenv, rank)
    nenv, cfd = w["nenv"], (w["cfd"] and not args.no_cfd)
    m = B.Model(w["model"], precision=args.precision, device=dev)
    np_dt = np.float64 if args.precision == 64 else np.float32
    x0_h = torch.from_numpy(np.ascontiguousarray(w["x0"], dtype=np_dt)).pin_memory()
    ctrl_h = None if w["ctrl"] is None else torch.from_numpy(np.ascontiguousarray(w["ctrl"], dtype=np_dt)).pin_memory()
    x0 = x0_h.to(dev); ctrl = None if ctrl_h is None else ctrl_h.to(dev)
    stats = m.alloc_stats(nenv)
    want_p = "mu" in w["grad_targets"] or "mass" in w["grad_targets"]

    # caller-side loss gradient dL/dx_T (not part of the method) with torch ops on the device, per config
    goal2 = torch.tensor([0.6, 0.0], dtype=m.dtype, device=dev); goal3 = torch.tensor([0.5, 0.0, 0.04], dtype=m.dtype, device=dev)

    def dLdxT_of(xT):
        g = torch.zeros_like(xT)
        if cfg in ("C1", "C3"): g[:, 0] = 1.0
        elif cfg == "C2": g[:, 2:4] = 2 * (xT[:, 2:4] - goal2)
        elif cfg == "C4": g[:, 7:10] = 2 * (xT[:, 7:10] - goal3)
        else: g[:, 0] = -1.0
        return g

    # size the tape from one untaped forward pass
    xT = m.rollout(x0, ctrl, w["nknot"], w["knot_dt"], None, w["horizon"], w["opts"], stats=stats)
    torch.cuda.synchronize()
    cap = int(stats["n_accept"].max().item() * 1.25) + 16
    tape = m.alloc_tape(nenv, cap)
    out = dict(dLdx0=torch.empty((nenv, 2 * m.nv), dtype=m.dtype, device=dev),
               dLdctrl=None if ctrl is None else torch.empty_like(ctrl),
               dLdparams=torch.empty((nenv, m.np_), dtype=m.dtype, device=dev) if want_p else None)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)      # > 126 MB L2
    stream = torch.cuda.current_stream(dev)

    def step(ev=None):
        """one pass of the hot path; ev = [e0, e1, e2] CUDA events recorded around forward and backward on the launch stream"""
        if ev: ev[0].record(stream)
        xT_ = m.rollout(x0, ctrl, w["nknot"], w["knot_dt"], None, w["horizon"], w["opts"], xT=xT, stats=stats, tape=tape)
        if ev: ev[1].record(stream)
        g = dLdxT_of(xT_)
        m.rollout_backward(ctrl, w["nknot"], None, w["opts"], xT_, g, cfd, tape, want_params=want_p, out=out)
        if ev: ev[2].record(stream)

    for _ in range(args.warmup):
        flush.fill_(1); step()
    torch.cuda.synchronize()
    peak64, _ = B.fma_peak(64, 1 << 15)
    peak32, _ = B.fma_peak(32, 1 << 15)
    if world > 1: dist.barrier()
    torch.cuda.synchronize()
    clocks = ClockSampler(local); clocks.start()
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(args.steps)]
    t_wall0 = time.perf_counter()
    for k in range(args.steps):
        flush.fill_(k)              # L2 flush between timed iterations (outside the event brackets)
        step(evs[k])
    torch.cuda.synchronize()
    if world > 1: dist.barrier()
    t_wall = time.perf_counter() - t_wall0
    clk = clocks.stop()
    t_f = sum(e[0].elapsed_time(e[1]) for e in evs) * 1e-3 / args.steps
    t_b = sum(e[1].elapsed_time(e[2]) for e in evs) * 1e-3 / args.steps
    t_step = sum(e[0].elapsed_time(e[2]) for e in evs) * 1e-3 / args.steps
    acc = float(stats["n_accept"].sum().item()); rej = float(stats["n_reject"].sum().item())
    fev = float(stats["n_feval"].sum().item())
    bad = int((stats["status"] != 0).sum().item())

    # end to end: pinned host inputs -> device, hot path, results -> host, every step
    res_h = [torch.empty(xT.shape, dtype=m.dtype).pin_memory(), torch.empty(out["dLdx0"].shape, dtype=m.dtype).pin_memory()]
    if ctrl is not None: res_h.append(torch.empty(ctrl.shape, dtype=m.dtype).pin_memory())
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    h2d = x0_h.numel() * x0_h.element_size() + (0 if ctrl_h is None else ctrl_h.numel() * ctrl_h.element_size())
    d2h = sum(t.numel() * t.element_size() for t in res_h)
    t_e2e = 0.0
    for k in range(args.steps):
        flush.fill_(k)
        e0.record(stream)
        x0.copy_(x0_h, non_blocking=True)
        if ctrl is not None: ctrl.copy_(ctrl_h, non_blocking=True)
        step()
        res_h[0].copy_(xT, non_blocking=True); res_h[1].copy_(out["dLdx0"], non_blocking=True)
        if ctrl is not None: res_h[2].copy_(out["dLdctrl"], non_blocking=True)
        e1.record(stream); e1.synchronize()
        t_e2e += e0.elapsed_time(e1) * 1e-3
    t_e2e /= args.steps

    t_step_max = max_over_ranks(t_step, dev); t_e2e_max = max_over_ranks(t_e2e, dev)
    acc_all = sum_over_ranks(acc, dev)
    if rank != 0:
        if world > 1: dist.destroy_process_group()
        return
    # roofline of the dominant kernel (bound by plain FP64 ALU arithmetic)
    peak = peak64 if args.precision == 64 else peak32
    fl_f = FLOPS_PER_ATTEMPT[cfg] * (acc + rej)
    fl_b = grad_flops_per_accepted(cfg, cfd) * acc
    dom = "backward_kernel" if t_b >= t_f else "rollout_kernel"
    fl_d, t_d = (fl_b, t_b) if t_b >= t_f else (fl_f, t_f)
    line = {
        "metric": METRIC, "value": acc_all / t_step_max, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": 1e3 * t_step_max, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64" if args.precision == 64 else "f32", "data": "synthetic",
        "config": {"workload": w["name"], "nenv_per_gpu": nenv, "horizon_s": w["horizon"], "rtol": w["opts"]["rtol"], "cfd_backward": bool(cfd),
                   "lanes_per_env": m.lanes, "l2": "flushed between timed iterations (256 MiB write)", "tape_steps": cap, "tape_record": "checkpoint + 6 stage rates",
                   "param_grads": bool(want_p)},
        "forward_env_steps_per_s": acc / t_f, "forward_attempted_steps_per_s": (acc + rej) / t_f, "backward_env_steps_per_s": acc / t_b,
        "ms_forward": 1e3 * t_f, "ms_backward": 1e3 * t_b, "accepted_steps": acc, "rejected_steps": rej, "f_evals": fev, "failed_envs": bad,
        "wall_s_timed_region": t_wall,
        "e2e": {"value": acc_all / t_e2e_max, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h},
        "gpu_launches": 2 * args.steps,
        "clocks": clk,
        "roofline": {"bound": "alu", "kernel": dom, "achieved": fl_d / t_d / 1e12, "peak": peak / 1e12, "unit": "TFLOP/s", "frac": fl_d / t_d / peak,
                     "traffic": NCU_TRAFFIC_C2_F64_4096[dom] if (cfg == "C2" and nenv == 4096 and args.precision == 64 and cfd) else None, "peak_source": "measured FMA-chain (dmx_fma_peak) in this run; nominal 37.2 (fp64) / 74.4 (fp32)",
                     "forward": {"achieved": fl_f / t_f / 1e12, "frac": fl_f / t_f / peak},
                     "backward": {"achieved": fl_b / t_b / 1e12, "frac": fl_b / t_b / peak},
                     "tape_gbs_write": acc * (m.nq + m.nv + 2 + 6 * m.nv) * (8 if args.precision == 64 else 4) / t_f / 1e9},
    }
    if not args.no_cpu_baseline:
        cores = os.cpu_count() or 1
        n_sample = min(nenv, args.ref_sample)
        r = oracle_sample(w, cfg, n_sample, cfd, cores)
        line["cpu_baseline"] = {"value": r["grad"], "unit": UNIT, "cores": cores, "kind": "oracle",
                                "sample": "first %d of %d envs, forward with tape + reverse sweep, %.1f s" % (n_sample, nenv, r["t_grad"] + r["t_fwd"]),
                                "forward_env_steps_per_s": r["fwd"]}
    print(json.dumps(line), flush=True)
    if world > 1: dist.destroy_process_group()


if __name__ == "__main__":
    main()
