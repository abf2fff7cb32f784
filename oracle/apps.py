"""ORACLE - test infrastructure only (see oracle/README.md).  Not part of the product path.

Plain NumPy restatement of the paper's optimisation loops around the simulator:
  adam_step   Adam with bias correction (Kingma & Ba 2015; "Adam optimizer with a learning rate of 0.01";
              PAPER.md:515 "b1 = 0.5, b2 = 0.9, eps = 1e-6") preceded by per-row gradient clipping (PAPER.md:167
              "gradient clipping, which is important as the scale of gradients changes massively in the presence of contacts")
  mpc_plan_step   one planning step of the gradient-based MPC of PAPER.md:167: `iters` Adam iterations on the control knots,
              keeping the best of the evaluated iterates ("we store the rollout cost of all gradient iterations and select
              the one with minimal cost"); rollouts and gradients come from oracle.Oracle.
Readings G22-G24: moments reset per plan step; iterates 0 .. iters-1 are the evaluated ones.
Pins: tests/test_apps.py (first step = lr * sign(g); constant gradient -> exactly linear path; clipped norm)."""
import numpy as np


def adam_step(x, g, m, v, t, lr, b1=0.9, b2=0.999, eps=1e-8, clip=0.0, active=None):
    """in place on x, m, v (all [nrow, len] float64); t = 1, 2, ...; rows with active[r] == 0 untouched"""
    for r in range(x.shape[0]):
        if active is not None and not active[r]:
            continue
        gr = g[r].astype(np.float64).copy()
        if clip > 0:
            nrm = np.sqrt(np.sum(gr * gr))
            if nrm > clip:
                gr = gr * (clip / nrm)
        m[r] = b1 * m[r] + (1.0 - b1) * gr
        v[r] = b2 * v[r] + (1.0 - b2) * gr * gr
        mhat = m[r] / (1.0 - b1 ** t)
        vhat = v[r] / (1.0 - b2 ** t)
        x[r] = x[r] - lr * mhat / (np.sqrt(vhat) + eps)


def mpc_plan_step(orc, x, plan, nknot, knot_dt, opts, cost, cfd=True, iters=32, lr=0.01, clip=1.0, betas=(0.9, 0.999), eps=1e-8,
                  params=None, threads=1):
    """-> (best plan, best cost [nenv], costs [iters, nenv], iterates [iters + 1, nenv, nknot, nu]).
    cost(xT) -> (cost [nenv], dcost/dxT [nenv, nq+nv]) in NumPy."""
    nenv = x.shape[0]
    u = plan.astype(np.float64).copy()
    m = np.zeros((nenv, u[0].size)); v = np.zeros_like(m)
    best_u = u.copy(); best_c = np.full(nenv, np.inf); hist = []; iterates = [u.copy()]
    horizon = nknot * knot_dt
    for it in range(iters):
        fwd = orc.rollout(x, u, nknot, knot_dt, params, horizon, opts, threads=threads)
        ok = fwd["stats"]["status"] == 0
        c, g = cost(fwd["xT"])
        c = np.where(ok, c, np.inf)
        better = c < best_c
        best_c = np.where(better, c, best_c)
        best_u[better] = u[better]
        hist.append(c)
        gr = orc.rollout_grad(x, u, nknot, knot_dt, params, horizon, opts, dLdxT=g, cfd_on=cfd, want_params=False, threads=threads)
        uf = u.reshape(nenv, -1)
        adam_step(uf, gr["dLdctrl"].reshape(nenv, -1), m, v, it + 1, lr, betas[0], betas[1], eps, clip, active=ok)
        u = uf.reshape(u.shape)
        iterates.append(u.copy())
    return best_u, best_c, np.stack(hist), np.stack(iterates)
