"""The paper's two applications as callers of the C-ABI: gradient-based model-predictive control
(section 5.2) and parameter identification from trajectory segments (PAPER.md:157 section 5.1, :515 E.2).

Everything that simulates or differentiates runs in libdmx (dmx_rollout, dmx_rollout_backward) and the optimiser update is
dmx_adam_step; this module only sequences those calls.  The task cost is the caller's: a callable on device tensors that
returns the cost per environment and its gradient with respect to the final state.  Readings (G22-G24):
the Adam moments are reset at every plan step; the plan returned by a plan step is the best of the iterates whose rollout
cost was computed (iterates 0 .. iters-1; the last update is never evaluated, as in "we store the rollout cost of all
gradient iterations and select the one with minimal cost"); a segment's loss is taken on its last state."""
import math

from . import binding as B

TAPE_FULL = 4      # dmx_stats.status of an environment whose tape slot overflowed (include/dmx.h)


class _TapedRollout:
    """forward with tape + reverse sweep for a fixed batch shape; grows the (uniform-slot) tape when an environment fills it"""

    def __init__(self, model, nenv, tape_steps):
        self.m, self.nenv, self.tape_steps = model, nenv, int(tape_steps)
        self.tape = model.alloc_tape(nenv, self.tape_steps)
        self.stats = model.alloc_stats(nenv)

    def forward(self, x, ctrl, nknot, knot_dt, params, horizon, opts):
        for _ in range(8):                                    # at most 256x the initial tape
            xT = self.m.rollout(x, ctrl, nknot, knot_dt, params, horizon, opts, stats=self.stats, tape=self.tape)
            st = self.stats["status"]
            if not bool((st == TAPE_FULL).any().item()):
                return xT, st
            self.tape_steps *= 2
            self.tape = None                                  # release before the larger one is allocated
            self.tape = self.m.alloc_tape(self.nenv, self.tape_steps)
        raise RuntimeError("tape of %d steps per environment still too small: set max_steps in the solver options" % self.tape_steps)

    def backward(self, ctrl, nknot, params, opts, xT, dLdxT, cfd, want_params):
        return self.m.rollout_backward(ctrl, nknot, params, opts, xT, dLdxT, cfd, self.tape, want_params=want_params,
                                       status=self.stats["status"])


class MPC:
    """Gradient-based MPC: at every plan step the control knots of the horizon are refined by `iters` Adam
    iterations (lr 0.01) on the rollout cost, with the gradient of every environment clipped to norm `clip` and the best
    evaluated iterate kept; the plan is executed for `execute` knots and shifted (warm start).  A batch of independent
    environments is planned at once.  cost(xT) -> (cost[nenv], dcost/dxT[nenv, nq+nv]) on device tensors."""

    def __init__(self, model, nenv, nknot, knot_dt, opts, cost, cfd=True, iters=32, lr=0.01, clip=1.0, execute=16,
                 betas=(0.9, 0.999), eps=1e-8, params=None, tape_steps=None):
        self.m, self.nenv, self.nknot, self.knot_dt, self.opts, self.cost = model, nenv, int(nknot), float(knot_dt), opts, cost
        self.cfd, self.iters, self.lr, self.clip, self.execute, self.betas, self.eps, self.params = cfd, iters, lr, clip, int(execute), betas, eps, params
        self.horizon = self.nknot * self.knot_dt
        self.roll = _TapedRollout(model, nenv, tape_steps or 4 * self.nknot + 64)
        T = model.torch
        self.mom1 = T.zeros((nenv, self.nknot, model.nu), dtype=model.dtype, device=model.device)
        self.mom2 = T.zeros_like(self.mom1)

    def plan_step(self, x, plan):
        """-> (best plan, its cost [nenv], costs of the evaluated iterates [iters, nenv]); `plan` is not modified"""
        T = self.m.torch
        u = plan.clone()
        self.mom1.zero_(); self.mom2.zero_()
        best_u, best_c, hist = plan.clone(), None, []
        for it in range(self.iters):
            xT, st = self.roll.forward(x, u, self.nknot, self.knot_dt, self.params, self.horizon, self.opts)
            c, g = self.cost(xT)
            c = T.where(st == 0, c, T.full_like(c, math.inf))               # a failed rollout is never the best
            better = c < best_c if best_c is not None else T.ones_like(c, dtype=T.bool)
            best_c = c.clone() if best_c is None else T.where(better, c, best_c)
            best_u = T.where(better[:, None, None], u, best_u)
            hist.append(c)
            gr = self.roll.backward(u, self.nknot, self.params, self.opts, xT, g.contiguous(), self.cfd, want_params=False)
            B.adam_step(u, gr["dLdctrl"], self.mom1, self.mom2, it + 1, self.lr, self.betas[0], self.betas[1], self.eps, self.clip,
                        active=(st == 0).to(T.uint8))
        return best_u, best_c, T.stack(hist)

    def execute_plan(self, x, plan):
        """simulate the first `execute` knots of the plan (no tape) -> next state"""
        return self.m.rollout(x, plan, self.nknot, self.knot_dt, self.params, self.execute * self.knot_dt, self.opts)

    def shift(self, plan):
        """warm start of the next plan step: drop the executed knots, hold the last one"""
        T = self.m.torch
        return T.cat([plan[:, self.execute:], plan[:, -1:].expand(-1, self.execute, -1)], dim=1).contiguous()

    def run(self, x0, plan0, n_plan_steps):
        """the MPC loop -> dict(x [nenv, nq+nv] final state, plan, cost [n_plan_steps, nenv] of the executed states)"""
        T = self.m.torch
        x, plan, costs = x0, plan0, []
        for _ in range(n_plan_steps):
            plan, _, _ = self.plan_step(x, plan)
            x = self.execute_plan(x, plan)
            costs.append(self.cost(x)[0])
            plan = self.shift(plan)
        return dict(x=x, plan=plan, cost=T.stack(costs))


def quat_to_mat(q):
    """rotation matrices [n, 9] of unit quaternions (w, x, y, z) [n, 4]; torch ops (differentiable), caller side"""
    w, x, y, z = q[:, 0], q[:, 1], q[:, 2], q[:, 3]
    rows = [1 - 2 * (y * y + z * z), 2 * (x * y - w * z), 2 * (x * z + w * y),
            2 * (x * y + w * z), 1 - 2 * (x * x + z * z), 2 * (y * z - w * x),
            2 * (x * z - w * y), 2 * (y * z + w * x), 1 - 2 * (x * x + y * y)]
    import torch
    return torch.stack(rows, dim=1)


class SysID:
    """Identification of simulation parameters from trajectory segments.  Environment e holds one
    segment: start state x_start[e] and the recorded state x_end[e] `horizon` seconds later.  One parameter vector is
    shared by all segments; its entries listed in `free` are optimised through p = softplus(theta) (PAPER.md E.2.1:
    "constrained using ... a softplus function"), the others stay at p0.  Loss: mean over segments of the squared error
    of position, rotation matrix (quaternions are converted first), and w_vel times that of the velocities.
    Optimiser: Adam with b1 = 0.5, b2 = 0.9, eps = 1e-6 through dmx_adam_step."""

    def __init__(self, model, x_start, x_end, horizon, opts, p0, free, free_quat_adr=3, lr=0.02, cfd=False, w_vel=0.01,
                 betas=(0.5, 0.9), eps=1e-6, tape_steps=4096):
        T = model.torch
        self.m, self.x0, self.x1, self.horizon, self.opts, self.cfd, self.lr, self.w_vel = model, x_start, x_end, float(horizon), opts, cfd, lr, w_vel
        self.betas, self.eps, self.qa = betas, eps, free_quat_adr
        self.nenv = x_start.shape[0]
        self.free = T.as_tensor(list(free), dtype=T.long, device=model.device)
        self.p0 = p0.to(model.device, model.dtype).clone()
        pf = self.p0[self.free]
        self.theta = T.where(pf > 20, pf, T.log(T.expm1(pf))).reshape(1, -1).contiguous()       # softplus^-1
        self.mom1, self.mom2, self.t = T.zeros_like(self.theta), T.zeros_like(self.theta), 0
        self.roll = _TapedRollout(model, self.nenv, tape_steps)

    def params(self):
        T = self.m.torch
        p = self.p0.clone()
        p[self.free] = T.nn.functional.softplus(self.theta[0])
        return p

    def loss_and_grad(self, xT):
        """-> (loss scalar, dloss/dxT [nenv, nq+nv]); torch autograd over the nenv x (nq+nv) end states only"""
        T = self.m.torch
        nq, qa = self.m.nq, self.qa
        x = xT.detach().clone().requires_grad_(True)
        e_pos = x[:, :qa] - self.x1[:, :qa]
        e_rot = quat_to_mat(x[:, qa:qa + 4]) - quat_to_mat(self.x1[:, qa:qa + 4])
        e_vel = x[:, nq:] - self.x1[:, nq:]
        loss = ((e_pos ** 2).sum(1) + (e_rot ** 2).sum(1) + self.w_vel * (e_vel ** 2).sum(1)).mean()
        (g,) = T.autograd.grad(loss, x)
        return loss.detach(), g

    def step(self):
        """one optimisation step -> loss before the update"""
        T = self.m.torch
        p = self.params()
        pe = p.reshape(1, -1).expand(self.nenv, -1).contiguous()
        xT, st = self.roll.forward(self.x0, None, 0, 0.0, pe, self.horizon, self.opts)
        if bool((st != 0).any().item()):
            raise RuntimeError("SysID: %d segment rollouts failed" % int((st != 0).sum().item()))
        loss, g = self.loss_and_grad(xT)
        gr = self.roll.backward(None, 0, pe, self.opts, xT, g.contiguous(), self.cfd, want_params=True)
        gp = gr["dLdparams"].sum(0)[self.free]                                          # shared parameters: sum over segments
        gth = (gp * T.sigmoid(self.theta[0])).reshape(1, -1).contiguous()               # d softplus / d theta
        self.t += 1
        B.adam_step(self.theta, gth, self.mom1, self.mom2, self.t, self.lr, self.betas[0], self.betas[1], self.eps, 0.0)
        return float(loss.item())

    def fit(self, n_steps):
        return [self.step() for _ in range(n_steps)]
