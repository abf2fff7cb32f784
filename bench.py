"""bench.py — forward and gradient env-steps/s of the dmx hot path on B200 (BASELINE.json metric).

A "step" is one pass of the whole hot path over one batch of synthetic environments: dmx_rollout (adaptive RK
forward with tape, S1-S9) followed by dmx_rollout_backward (reverse sweep with the CFD straight-through VJP,
S10-S12), in the launch configuration a user of the library would use: one sizing pass (untaped forward) ->
dmx_tape_plan (longest environment first, per-environment tape slots) -> timed passes.

Headline line (`value`, `ms_per_step`, `e2e`, `--steps/--warmup`): BASELINE config 2 (planar push, 4096 envs, fp64,
Tsit5 rtol 1e-6, 250 control knots).  The largest single-GPU configuration, C4 (16 384 envs, 2 s horizon), costs
seconds per pass and cannot be repeated steps+warmup+e2e times inside the driver's limit, so it is measured in the
`per_config` block with its own (stated) repeat count, together with the other BASELINE configs (C1-C5, C3 also in
fp32) and the saturating-batch companions of C1 and C2.  N>1: one process per GPU; `--scaling weak`
(default) runs a full batch per rank with its own seed, `--scaling strong` shards ONE BASELINE batch over the ranks
with sharding.shard_range; no data-path collective either way.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C2] [--nenv n] [--impl reference]
                    [--no-per-config] [--per-config C1,C3] [--scaling weak|strong]

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

# Executed-FP64 fractions of the measured FMA peak (2*DFMA + DADD + DMUL per second / 33.8 TFLOP/s) and DRAM bytes per launch
# from the committed ncu --set full captures (profiles/r2_{rollout,backward}_kernel_{C2,C3,C5}.md).  They are constants of
# those captures, NOT measured in the run that prints them (a profiler cannot run inside a timed region); the JSON line
# labels them as such, next to the live algorithmic fraction.  Key: config_dtype_nenv of the capture.
NCU_EXECUTED = {
    "C2_f64_4096": {"rollout_kernel_executed_frac": 0.0339, "backward_kernel_executed_frac": 0.0349,
                    "rollout_kernel_dram_bytes": 5.701e+08, "backward_kernel_dram_bytes": 7.149e+08},
    "C3_f64_2048": {"rollout_kernel_executed_frac": 0.0108, "backward_kernel_executed_frac": 0.0097,
                    "rollout_kernel_dram_bytes": 3.224e+08, "backward_kernel_dram_bytes": 3.821e+08},
    "C5_f64_512": {"rollout_kernel_executed_frac": 0.0110, "backward_kernel_executed_frac": 0.0130,
                    "rollout_kernel_dram_bytes": 1.66e+09, "backward_kernel_dram_bytes": 1.713e+09},
}

# per_config rows: (key, config, nenv (0 = BASELINE size), precision, timed passes, oracle sample envs, checkpoint stride)
PER_CONFIG = [("C1", "C1", 0, 64, 3, 1024, 1), ("C2", "C2", 0, 64, 3, 256, 1), ("C3", "C3", 0, 64, 2, 256, 1), ("C3_fp32", "C3", 0, 32, 2, 0, 1),
              ("C4", "C4", 0, 64, 1, 16, 1), ("C5", "C5", 0, 64, 2, 16, 1),
              ("C1_saturating_65536", "C1", 65536, 64, 2, 0, 1), ("C2_saturating_32768", "C2", 32768, 64, 2, 0, 1),
              # the checkpoint-count knob: a checkpoint every 16 accepted steps, segments recomputed in the sweep
              ("C3_checkpoint_stride16", "C3", 0, 64, 1, 0, 16), ("C4_checkpoint_stride16", "C4", 0, 64, 1, 0, 16),
              # C3 with the step budget of PAPER.md:377, 493 (max_steps; 9x the median count): the one environment whose 4-iteration
              # Newton solves stop converging ends with status 1 instead of owning the launch
              ("C3_step_budget_4096", "C3", 0, 64, 2, 0, 1, {"max_steps": 4096})]


# ---- algorithmic FP64 work: analytic flop counts of the operations the method defines, FMA = 2, times
# the units the launch actually processed (F evaluations, Newton iterations, rows: counted by the kernels) ------------
def flop_model(model):
    nb, nv, nu = int(model["nbody"]), int(model["nv"]), int(model["nu"])
    parent = list(model["body_parent"]); jt = list(model["jnt_type"]); jb = list(model["jnt_body"])
    body_j = {b: t for b, t in zip(jb, jt)}
    ndof_of = lambda b: 0 if b not in body_j else (6 if body_j[b] == W.JNT_FREE else 1)
    anc_dofs, sub = [0] * nb, [1] * nb
    for b in range(1, nb):
        anc_dofs[b] = anc_dofs[parent[b]] + ndof_of(b)
    for b in range(nb - 1, 0, -1):
        if parent[b] > 0:
            sub[parent[b]] += sub[b]
    ntw = sum(anc_dofs[1:])
    kin = sum({W.JNT_HINGE: 440, W.JNT_SLIDE: 300, W.JNT_FREE: 65}.get(body_j.get(b), 120) for b in range(1, nb))
    dyn = 190 * (nb - 1) + 12 * ntw + 9 * sum(sub[1:])
    m_entries = 0
    for b in range(1, nb):          # M(i,j) with the deeper dof on body b: sum over its subtree of a 7-flop term
        m_entries += sub[b] * 7 * ndof_of(b) * (anc_dofs[b] - (ndof_of(b) - 1) / 2.0)
    dyn += m_entries + sum(sub[b] * 12 * ndof_of(b) for b in range(1, nb)) + 8 * nv + 4 * nu
    chol = nv ** 3 / 3.0 + nv ** 2
    solve = 2.0 * nv ** 2 + nv
    gt = list(model["geom_type"]); g2 = list(model["pair_geom2"]); g1 = list(model["pair_geom1"])
    nc = sum({W.GEOM_SPHERE: 1, W.GEOM_CAPSULE: 2, W.GEOM_BOX: 8}[gt[b]] for b in g2)
    collide = 35.0 * nc + 45.0 * sum(1 for a in g1 if gt[a] != W.GEOM_PLANE)
    avg_path = ntw / max(nb - 1, 1)
    return dict(nv=nv, base=kin + dyn + chol + solve + collide,          # S1-S4 + factor of M + a0, per F evaluation
                per_row=10.0 + 35.0 * avg_path / 4.0 + 2.0 * nv + 2,         # S5: scalars, Jacobian entries (per row), a_ref
                per_iter=chol + solve + 2.0 * nv ** 2 + 2.0 * nv,             # S6 per Newton iteration: g (M part), factor, solve, update
                per_rowiter=3.0 * nv * (nv + 1) / 2.0 + 7.0 * nv + 1,         # S6 per row and iteration: s, g (row part), H, J dl
                vjp=2.5 * (kin + dyn + collide) + chol + 2 * solve)           # S11 per stage without its solve (2-3 F)


def flops_forward(fm, fev, work3):
    it, rowit, rows = work3
    return fev * fm["base"] + rows * fm["per_row"] + it * fm["per_iter"] + rowit * fm["per_rowiter"]


def flops_backward(fm, accepted, work3, tape_stages=True):
    """6 VJPs per accepted step, their row terms, the solves the sweep actually ran (F~ with CFD; none without CFD in the
    stage-rate tape mode), and 6 recomputed F only in checkpoint-only mode."""
    it, rowit, rows = work3
    fl = 6 * accepted * fm["vjp"] + rows * (fm["per_row"] + 3.0 * fm["nv"]) + it * fm["per_iter"] + rowit * fm["per_rowiter"]
    if not tape_stages:
        fl += 6 * accepted * fm["base"]
    return fl


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


def make_workload(cfg, nenv, rank, world=1, strong=False):
    kw = {}
    if nenv:
        kw["nenv"] = nenv
    if rank and not strong:
        kw["seed"] = 250614186 + int(cfg[1]) + 1000 * rank
    w = W.make(cfg, **kw)
    if strong and world > 1:                      # one BASELINE batch, contiguous env ranges per rank
        from paper_2506_14186_b200.sharding import shard_range
        lo, hi = shard_range(w["nenv"], rank, world)
        w = dict(w); w["x0"] = np.ascontiguousarray(w["x0"][lo:hi]); w["nenv"] = hi - lo
        if w["ctrl"] is not None:
            w["ctrl"] = np.ascontiguousarray(w["ctrl"][lo:hi])
    return w


def oracle_sample(w, n_sample, cfd, threads):
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


def cpu_baseline_entry(w, n_sample, cfd):
    cores = os.cpu_count() or 1
    n_sample = min(w["nenv"], n_sample)
    r = oracle_sample(w, n_sample, cfd, cores)
    return {"value": r["grad"], "unit": UNIT, "cores": min(cores, n_sample), "kind": "oracle (forward-mode-dual VJP, as it stands: not an optimised baseline)",
            "sample": "first %d of %d envs, forward with tape + reverse sweep, %.1f s" % (n_sample, w["nenv"], r["t_grad"] + r["t_fwd"]),
            "forward_env_steps_per_s": r["fwd"]}


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
        r = oracle_sample(w, n_sample, w["cfd"], cores)
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


class Runner:
    """One workload on one device: sizing pass, plan, tape, and the timed pass."""

    def __init__(self, torch, B, dev, cfg, w, precision, cfd, stride=1):
        self.torch, self.cfg, self.w, self.cfd, self.dev, self.stride = torch, cfg, w, cfd, dev, stride
        self.m = m = B.Model(w["model"], precision=precision, device=dev)
        if stride > 1:
            m.set_checkpoint_stride(stride)
        self.nenv = w["nenv"]
        np_dt = np.float64 if precision == 64 else np.float32
        self.x0_h = torch.from_numpy(np.ascontiguousarray(w["x0"], dtype=np_dt)).pin_memory()
        self.ctrl_h = None if w["ctrl"] is None else torch.from_numpy(np.ascontiguousarray(w["ctrl"], dtype=np_dt)).pin_memory()
        self.x0 = self.x0_h.to(dev); self.ctrl = None if self.ctrl_h is None else self.ctrl_h.to(dev)
        self.stats = m.alloc_stats(self.nenv)
        self.want_p = "mu" in w["grad_targets"] or "mass" in w["grad_targets"]
        self.goal2 = torch.tensor([0.6, 0.0], dtype=m.dtype, device=dev); self.goal3 = torch.tensor([0.5, 0.0, 0.04], dtype=m.dtype, device=dev)
        self.stream = torch.cuda.current_stream(dev)
        # sizing pass: accepted steps per environment -> launch plan (order + tape slots, 25 % + 16 records of margin)
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
        ev[0].record(self.stream)
        self.xT = m.rollout(self.x0, self.ctrl, w["nknot"], w["knot_dt"], None, w["horizon"], w["opts"], stats=self.stats)
        ev[1].record(self.stream); torch.cuda.synchronize()
        self.ms_sizing = ev[0].elapsed_time(ev[1])
        self.plan, self.tape = m.plan(self.stats["n_accept"], margin_pct=25, pad=16)
        self.tape_uniform_bytes = m.tape_bytes(self.nenv, int(self.stats["n_accept"].max().item() * 1.25) + 16)
        self.out = dict(dLdx0=torch.empty((self.nenv, 2 * m.nv), dtype=m.dtype, device=dev),
                        dLdctrl=None if self.ctrl is None else torch.empty_like(self.ctrl),
                        dLdparams=torch.empty((self.nenv, m.np_), dtype=m.dtype, device=dev) if self.want_p else None)

    def dLdxT(self, xT):
        """caller-side loss gradient dL/dx_T (not part of the method), torch ops on the device"""
        g = self.torch.zeros_like(xT)
        cfg = self.cfg
        if cfg in ("C1", "C3"): g[:, 0] = 1.0
        elif cfg == "C2": g[:, 2:4] = 2 * (xT[:, 2:4] - self.goal2)
        elif cfg == "C4": g[:, 7:10] = 2 * (xT[:, 7:10] - self.goal3)
        else: g[:, 0] = -1.0
        return g

    def step(self, ev=None):
        """one pass of the hot path; ev = [e0, e1, e2] CUDA events recorded around forward and backward on the launch stream"""
        w, m = self.w, self.m
        if ev: ev[0].record(self.stream)
        xT_ = m.rollout(self.x0, self.ctrl, w["nknot"], w["knot_dt"], None, w["horizon"], w["opts"], xT=self.xT, stats=self.stats,
                        tape=self.tape, plan=self.plan)
        if ev: ev[1].record(self.stream)
        g = self.dLdxT(xT_)
        m.rollout_backward(self.ctrl, w["nknot"], None, w["opts"], xT_, g, self.cfd, self.tape, want_params=self.want_p, out=self.out,
                           plan=self.plan, stats=self.stats)
        if ev: ev[2].record(self.stream)

    def timed(self, flush, warm, reps):
        torch = self.torch
        for _ in range(warm):
            flush.fill_(1); self.step()
        torch.cuda.synchronize()
        evs = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(reps)]
        for k in range(reps):
            flush.fill_(k)              # L2 flush between timed iterations (outside the event brackets)
            self.step(evs[k])
        torch.cuda.synchronize()
        t_f = sum(e[0].elapsed_time(e[1]) for e in evs) * 1e-3 / reps
        t_b = sum(e[1].elapsed_time(e[2]) for e in evs) * 1e-3 / reps
        t_s = sum(e[0].elapsed_time(e[2]) for e in evs) * 1e-3 / reps
        return t_f, t_b, t_s

    def summary(self, t_f, t_b, t_s, peak):
        st, m, w = self.stats, self.m, self.w
        acc = float(st["n_accept"].sum().item()); rej = float(st["n_reject"].sum().item()); fev = float(st["n_feval"].sum().item())
        work = st["work"].sum(dim=0).double().cpu().numpy()
        fm = flop_model(w["model"])
        fl_f, fl_b = flops_forward(fm, fev, work[0:3]), flops_backward(fm, acc, work[3:6])
        sim = float(st["t_end"].sum().item())
        na = st["n_accept"]
        return {
            "workload": w["name"], "nenv": self.nenv, "dtype": "f64" if m.precision == 64 else "f32", "lanes_per_env": m.lanes,
            "checkpoint_stride": self.stride,
            "cfd_backward": bool(self.cfd), "param_grads": bool(self.want_p),
            "ms_forward": 1e3 * t_f, "ms_backward": 1e3 * t_b, "ms_step": 1e3 * t_s,
            "forward_env_steps_per_s": acc / t_f, "forward_attempted_steps_per_s": (acc + rej) / t_f, "backward_env_steps_per_s": acc / t_b,
            "gradient_env_steps_per_s": acc / t_s, "simulated_seconds_envs_per_s_forward": sim / t_f, "simulated_seconds_envs_per_s_gradient": sim / t_s,
            "accepted_steps": acc, "rejected_steps": rej, "f_evals": fev, "accepted_per_env_median": float(na.float().median().item()),
            "accepted_per_env_max": int(na.max().item()), "failed_envs": int((st["status"] != 0).sum().item()),
            "newton_unconverged_forward": int(st["n_newton_unconverged"].sum().item()),
            "newton_unconverged_backward": int(st["n_newton_unconverged_bwd"].sum().item()),
            "newton_iterations_forward": float(work[0]), "newton_iterations_backward": float(work[3]),
            "tape_bytes": int(self.tape.numel()), "tape_bytes_uniform_slots": int(self.tape_uniform_bytes),
            "tape_gbs_write": float(self.tape.numel()) / 1.25 / t_f / 1e9, "ms_sizing_pass": self.ms_sizing,
            "roofline": {"bound": "alu", "unit": "TFLOP/s", "peak": peak / 1e12,
                         "forward": {"achieved": fl_f / t_f / 1e12, "frac": fl_f / t_f / peak, "algorithmic_flops": fl_f},
                         "backward": {"achieved": fl_b / t_b / 1e12, "frac": fl_b / t_b / peak, "algorithmic_flops": fl_b}},
        }


def mpc_row(torch, B, dev):
    """one plan step of the gradient-based MPC of PAPER.md:167 (32 Adam iterations with clipping and keep-best,
    paper_2506_14186_b200/apps.py) on the C2 batch: wall time between two device synchronisations, after a warm-up plan step
    of 2 iterations."""
    try:
        from paper_2506_14186_b200 import apps
        w = make_workload("C2", 0, 0)
        m = B.Model(w["model"], precision=64, device=dev)
        goal = torch.tensor([0.6, 0.0], dtype=m.dtype, device=dev)

        def cost(xT):
            e = xT[:, 2:4] - goal
            g = torch.zeros_like(xT); g[:, 2:4] = 2 * e
            return (e * e).sum(1), g
        nenv = w["nenv"]
        mpc = apps.MPC(m, nenv, w["nknot"], w["knot_dt"], w["opts"], cost, cfd=True, iters=2, lr=0.01, clip=1.0, execute=16)
        x0, u0 = m.dev(w["x0"]), m.dev(w["ctrl"])
        mpc.plan_step(x0, u0)                                    # warm-up (sizes the tape)
        mpc.iters = 32
        torch.cuda.synchronize(); t0 = time.perf_counter()
        _, best, hist = mpc.plan_step(x0, u0)
        torch.cuda.synchronize(); dt = time.perf_counter() - t0
        steps = int(mpc.roll.stats["n_accept"].sum().item())
        return {"workload": w["name"], "nenv": nenv, "iterations": 32, "horizon_knots": w["nknot"], "s_per_plan_step": dt,
                "gradient_env_steps_per_s": 32 * steps / dt, "accepted_steps_last_rollout": steps,
                "mean_cost_first_iterate": float(hist[0].mean().item()), "mean_cost_best_iterate": float(best.mean().item()),
                "timing": "host wall clock around 32 x (dmx_rollout with tape, cost on the device, dmx_rollout_backward, dmx_adam_step), one status read-back per iteration"}
    except Exception as ex:            # noqa: BLE001
        return {"error": "%s: %s" % (type(ex).__name__, ex)}


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
    ap.add_argument("--no-per-config", action="store_true")
    ap.add_argument("--per-config", default="", help="comma-separated subset of per_config keys")
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"])
    ap.add_argument("--checkpoint-stride", type=int, default=1, help="tape keeps every k-th accepted step; segments recomputed in the sweep")
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
    strong = args.scaling == "strong"
    w = make_workload(cfg, args.nenv, rank, world, strong)
    cfd = w["cfd"] and not args.no_cfd
    run = Runner(torch, B, dev, cfg, w, args.precision, cfd, args.checkpoint_stride)
    m, nenv = run.m, run.nenv
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)      # > 126 MB L2
    stream = run.stream

    for _ in range(args.warmup):
        flush.fill_(1); run.step()
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
        run.step(evs[k])
    torch.cuda.synchronize()
    if world > 1: dist.barrier()
    t_wall = time.perf_counter() - t_wall0
    clk = clocks.stop()
    t_f = sum(e[0].elapsed_time(e[1]) for e in evs) * 1e-3 / args.steps
    t_b = sum(e[1].elapsed_time(e[2]) for e in evs) * 1e-3 / args.steps
    t_step = sum(e[0].elapsed_time(e[2]) for e in evs) * 1e-3 / args.steps
    peak = peak64 if args.precision == 64 else peak32
    head = run.summary(t_f, t_b, t_step, peak)
    acc = head["accepted_steps"]

    # end to end: pinned host inputs -> device, hot path, results -> host, every step
    xT, out, ctrl = run.xT, run.out, run.ctrl
    res_h = [torch.empty(xT.shape, dtype=m.dtype).pin_memory(), torch.empty(out["dLdx0"].shape, dtype=m.dtype).pin_memory()]
    if ctrl is not None: res_h.append(torch.empty(ctrl.shape, dtype=m.dtype).pin_memory())
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    h2d = run.x0_h.numel() * run.x0_h.element_size() + (0 if run.ctrl_h is None else run.ctrl_h.numel() * run.ctrl_h.element_size())
    d2h = sum(t.numel() * t.element_size() for t in res_h)
    t_e2e = 0.0
    for k in range(args.steps):
        flush.fill_(k)
        e0.record(stream)
        run.x0.copy_(run.x0_h, non_blocking=True)
        if ctrl is not None: ctrl.copy_(run.ctrl_h, non_blocking=True)
        run.step()
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
    dom = "backward_kernel" if t_b >= t_f else "rollout_kernel"
    rd = head["roofline"]["backward" if t_b >= t_f else "forward"]
    key = "%s_%s_%d" % (cfg, "f64" if args.precision == 64 else "f32", nenv)
    ncu = NCU_EXECUTED.get(key, {})
    line = {
        "metric": METRIC, "value": acc_all / t_step_max, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": 1e3 * t_step_max, "higher_is_better": True, "scaling": args.scaling, "vs_baseline": None,
        "dtype": "f64" if args.precision == 64 else "f32", "data": "synthetic",
        "config": {"workload": w["name"], "nenv_per_gpu": nenv, "horizon_s": w["horizon"], "rtol": w["opts"]["rtol"], "cfd_backward": bool(cfd),
                   "lanes_per_env": m.lanes, "l2": "flushed between timed iterations (256 MiB write)",
                   "tape": "planned slots (dmx_tape_plan from a sizing pass, 25 %% + 16 records margin), %d B" % run.tape.numel(),
                   "tape_record": "checkpoint + 6 stage rates" if args.checkpoint_stride == 1 else "checkpoint + first-stage rate every %d steps, 8-byte step schedule" % args.checkpoint_stride,
                   "param_grads": bool(run.want_p),
                   "headline": "C2 is the timed headline; the largest single-GPU config C4 (16384 envs) takes seconds per pass and is measured in "
                               "per_config with its own repeat count (1 warm-up + the stated timed passes)"},
        "forward_env_steps_per_s": head["forward_env_steps_per_s"], "forward_attempted_steps_per_s": head["forward_attempted_steps_per_s"],
        "backward_env_steps_per_s": head["backward_env_steps_per_s"],
        "simulated_seconds_envs_per_s_gradient": head["simulated_seconds_envs_per_s_gradient"],
        "ms_forward": 1e3 * t_f, "ms_backward": 1e3 * t_b, "accepted_steps": acc, "rejected_steps": head["rejected_steps"], "f_evals": head["f_evals"],
        "failed_envs": head["failed_envs"], "newton_unconverged_forward": head["newton_unconverged_forward"],
        "newton_unconverged_backward": head["newton_unconverged_backward"],
        "wall_s_timed_region": t_wall,
        "e2e": {"value": acc_all / t_e2e_max, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h},
        "gpu_launches": 3 * args.steps,       # rollout_kernel + backward_kernel + the caller-side loss-gradient fill per step
        "clocks": clk,
        "roofline": {"bound": "alu", "kernel": dom, "achieved": rd["achieved"], "peak": peak / 1e12, "unit": "TFLOP/s", "frac": rd["frac"],
                     "traffic": ncu.get(dom + "_dram_bytes"), "traffic_source": "ncu --set full capture in profiles/ (not this run)" if ncu else None,
                     "executed_frac_ncu": ncu.get(dom + "_executed_frac"),
                     "numerator": "analytic flops per unit (bench.py flop_model) x units counted by the kernels (F evaluations, rows, Newton iterations)",
                     "peak_source": "measured FMA-chain (dmx_fma_peak) in this run; nominal 37.2 (fp64) / 74.4 (fp32)",
                     "forward": head["roofline"]["forward"], "backward": head["roofline"]["backward"],
                     "tape_gbs_write": head["tape_gbs_write"]},
    }
    if not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline_entry(w, args.ref_sample, cfd)

    # ---- the other BASELINE configs and the saturating-batch companions, each with its own repeat count ----------------
    if not args.no_per_config and world == 1:
        want = [k for k in args.per_config.split(",") if k]
        per = {}
        del run
        torch.cuda.empty_cache()
        for row_ in PER_CONFIG:
            key_, c, n, prec, reps, n_orc, stride_ = row_[:7]
            if want and key_ not in want:
                continue
            try:
                wc = make_workload(c, n, 0)
                if len(row_) > 7:
                    wc["opts"] = dict(wc["opts"], **row_[7])
                rc = Runner(torch, B, dev, c, wc, prec, wc["cfd"], stride_)
                warm = 0 if c == "C4" else 1             # C4: the sizing pass is the only warm-up (a pass takes a minute)
                tf_, tb_, ts_ = rc.timed(flush, warm, reps)
                ent = rc.summary(tf_, tb_, ts_, peak64 if prec == 64 else peak32)
                ent["timed_passes"] = reps; ent["warmup_passes"] = warm
                if len(row_) > 7:
                    ent["opts_override"] = row_[7]
                k2 = "%s_%s_%d" % (c, "f64" if prec == 64 else "f32", wc["nenv"])
                if k2 in NCU_EXECUTED:
                    ent["roofline"]["executed_frac_ncu"] = {kk: vv for kk, vv in NCU_EXECUTED[k2].items() if kk.endswith("executed_frac")}
                if n_orc and not args.no_cpu_baseline:
                    ent["cpu_baseline"] = cpu_baseline_entry(wc, n_orc, wc["cfd"])
                per[key_] = ent
                del rc
            except Exception as ex:            # noqa: BLE001 - a failing companion row must not lose the headline
                per[key_] = {"error": "%s: %s" % (type(ex).__name__, ex)}
            torch.cuda.empty_cache()
        if not want or "C2_mpc_plan_step" in want:
            per["C2_mpc_plan_step"] = mpc_row(torch, B, dev)
        line["per_config"] = per
    print(json.dumps(line), flush=True)
    if world > 1: dist.destroy_process_group()


if __name__ == "__main__":
    main()
