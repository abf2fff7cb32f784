"""Thin Python binding of the C-ABI in include/dmx.h (argument marshalling only).

PyTorch is used for device memory and the CUDA stream; every step of the path runs in the CUDA
kernels of libdmx.so.  There is no CPU fallback: importing works without a GPU (so that the symbol
table can be checked), but any call that computes raises if the library or a device is missing.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("DMX_LIB", os.path.join(_HERE, "libdmx.so"))

SYMBOLS = ["dmx_model_create", "dmx_model_destroy", "dmx_model_set_tape_stages", "dmx_model_set_checkpoint_stride", "dmx_model_np", "dmx_model_nc", "dmx_model_default_params",
           "dmx_model_lanes", "dmx_tape_bytes", "dmx_tape_bytes_records", "dmx_plan_bytes", "dmx_tape_plan",
           "dmx_rollout", "dmx_rollout_grad", "dmx_rollout_backward", "dmx_rollout_backward_adjoint", "dmx_rollout_grad_adjoint",
           "dmx_rollout_backward_noalloc", "dmx_noalloc_scratch_bytes",
           "dmx_vector_field", "dmx_vjp_field", "dmx_adam_step", "dmx_fma_peak", "dmx_debug_counters", "dmx_last_error"]

_pd, _pi = C.POINTER(C.c_double), C.POINTER(C.c_int)
_INT_FIELDS = ["nbody", "njnt", "nq", "nv", "nu", "ngeom", "npair"]
_PTR_FIELDS = [
    ("body_parent", "i"), ("body_pos", "d"), ("body_quat", "d"), ("body_mass", "d"), ("body_ipos", "d"),
    ("body_iquat", "d"), ("body_inertia_unit", "d"),
    ("jnt_type", "i"), ("jnt_body", "i"), ("jnt_qadr", "i"), ("jnt_vadr", "i"),
    ("jnt_axis", "d"), ("jnt_pos", "d"), ("jnt_damping", "d"), ("jnt_armature", "d"),
    ("geom_type", "i"), ("geom_body", "i"), ("geom_size", "d"), ("geom_pos", "d"), ("geom_quat", "d"),
    ("pair_geom1", "i"), ("pair_geom2", "i"), ("pair_condim", "i"),
    ("pair_friction", "d"), ("pair_solref", "d"), ("pair_solimp", "d"), ("pair_solimp_cfd", "d"), ("pair_cfd_beta", "d"),
    ("act_type", "i"), ("act_jnt", "i"), ("act_gear", "d"), ("act_kp", "d"), ("act_kd", "d"),
]


class ModelDesc(C.Structure):
    _fields_ = ([(n, C.c_int) for n in _INT_FIELDS] + [(n, _pi if t == "i" else _pd) for n, t in _PTR_FIELDS] +
                [("gravity", C.c_double * 3), ("newton_iters", C.c_int), ("ls_iters", C.c_int), ("qpos0", _pd)])


class SolverOpts(C.Structure):
    _fields_ = [("tableau", C.c_int), ("rtol", C.c_double), ("atol", C.c_double), ("h0", C.c_double),
                ("pcoeff", C.c_double), ("icoeff", C.c_double), ("safety", C.c_double), ("fac_min", C.c_double),
                ("fac_max", C.c_double), ("max_steps", C.c_int)]


class Stats(C.Structure):
    _fields_ = [("n_accept", C.c_void_p), ("n_reject", C.c_void_p), ("n_feval", C.c_void_p),
                ("n_newton_unconverged", C.c_void_p), ("status", C.c_void_p),
                ("h_min", C.c_void_p), ("h_max", C.c_void_p), ("t_end", C.c_void_p), ("n_newton_unconverged_bwd", C.c_void_p), ("work", C.c_void_p)]


_lib = None


def load():
    """dlopen libdmx.so (built in-tree by build.py); raises if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError("libdmx.so not built: run `python -m paper_2506_14186_b200.build` (no CPU fallback exists)")
        L = C.CDLL(LIB_PATH)
        L.dmx_last_error.restype = C.c_char_p
        L.dmx_tape_bytes.restype = C.c_size_t
        L.dmx_tape_bytes.argtypes = [C.c_void_p, C.c_int, C.c_int]
        L.dmx_tape_bytes_records.restype = C.c_size_t
        L.dmx_tape_bytes_records.argtypes = [C.c_void_p, C.c_int, C.c_longlong]
        L.dmx_plan_bytes.restype = C.c_size_t
        L.dmx_plan_bytes.argtypes = [C.c_int]
        L.dmx_tape_plan.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_size_t, C.c_void_p]
        L.dmx_model_create.argtypes = [C.POINTER(ModelDesc), C.c_int, C.POINTER(C.c_void_p)]
        L.dmx_model_destroy.argtypes = [C.c_void_p]
        for f in ("dmx_model_np", "dmx_model_nc", "dmx_model_lanes"):
            getattr(L, f).argtypes = [C.c_void_p]
        L.dmx_model_default_params.argtypes = [C.c_void_p, C.c_void_p]
        L.dmx_model_set_tape_stages.argtypes = [C.c_void_p, C.c_int]
        L.dmx_model_set_checkpoint_stride.argtypes = [C.c_void_p, C.c_int]
        vp, i, d, sz = C.c_void_p, C.c_int, C.c_double, C.c_size_t
        L.dmx_rollout.argtypes = [vp, i, vp, vp, i, d, vp, d, C.POINTER(SolverOpts), vp, i, vp, C.POINTER(Stats), vp, sz, vp, vp]
        L.dmx_rollout_grad.argtypes = [vp, i, vp, vp, i, d, vp, d, C.POINTER(SolverOpts), vp, i, vp, i, vp, vp, vp, vp,
                                       C.POINTER(Stats), vp, sz, vp, vp]
        L.dmx_rollout_backward.argtypes = [vp, i, vp, i, vp, C.POINTER(SolverOpts), vp, vp, i, vp, vp, vp, C.POINTER(Stats), vp, sz, vp, vp]
        L.dmx_rollout_backward_noalloc.argtypes = [vp, i, vp, i, vp, C.POINTER(SolverOpts), vp, vp, i, vp, vp, vp, C.POINTER(Stats), vp, sz, vp, vp]
        L.dmx_noalloc_scratch_bytes.restype = C.c_size_t
        L.dmx_noalloc_scratch_bytes.argtypes = []
        L.dmx_rollout_backward_adjoint.argtypes = [vp, i, vp, i, vp, C.POINTER(SolverOpts), C.POINTER(SolverOpts), vp, vp, i, vp, vp, vp,
                                                   C.POINTER(Stats), vp, vp, i, vp, sz, vp, vp]
        L.dmx_rollout_grad_adjoint.argtypes = [vp, i, vp, vp, i, d, vp, d, C.POINTER(SolverOpts), C.POINTER(SolverOpts), vp, i, vp, i, vp, vp, vp, vp,
                                               C.POINTER(Stats), vp, vp, i, vp, sz, vp, vp]
        L.dmx_vector_field.argtypes = [vp, i, vp, vp, vp, i, vp, vp, vp]
        L.dmx_vjp_field.argtypes = [vp, i, vp, vp, vp, vp, i, vp, vp, vp, vp, vp]
        L.dmx_adam_step.argtypes = [i, i, i, vp, vp, vp, vp, vp, i, d, d, d, d, d, vp]
        L.dmx_fma_peak.argtypes = [i, i, _pd, _pd]
        L.dmx_debug_counters.argtypes = [vp, vp]
        _lib = L
    return _lib


def _err():
    return load().dmx_last_error().decode()


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("dmx needs a CUDA device (no CPU fallback)")
    return torch


def _ptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


def _opts(o):
    return SolverOpts(int(o["tableau"]), o["rtol"], o["atol"], o["h0"], o["pcoeff"], o["icoeff"], o["safety"],
                      o["fac_min"], o["fac_max"], int(o["max_steps"]))


def fma_peak(precision=64, iters=1 << 16):
    """Measured FMA-chain peak (FLOP/s) of the CUDA cores; roofline denominator."""
    _torch()
    f, ms = C.c_double(0), C.c_double(0)
    if load().dmx_fma_peak(int(precision), int(iters), C.byref(f), C.byref(ms)) != 0:
        raise RuntimeError("dmx_fma_peak: " + _err())
    return f.value, ms.value


def adam_step(x, g, mom1, mom2, t, lr, b1=0.9, b2=0.999, eps=1e-8, clip=0.0, active=None, stream=None):
    """dmx_adam_step: one clipped Adam update of every (active) row of x[nrow, ...] in place; t = 1, 2, ...."""
    T = _torch()
    nrow = x.shape[0]
    ln = x.numel() // nrow
    for a in (g, mom1, mom2):
        if a.dtype != x.dtype or a.numel() != x.numel() or not a.is_contiguous():
            raise ValueError("adam_step: g / mom1 / mom2 must be contiguous tensors of x's type and size")
    if not x.is_contiguous() or x.dtype not in (T.float64, T.float32):
        raise ValueError("adam_step: x must be a contiguous float64 / float32 tensor")
    if active is not None and (active.dtype != T.uint8 or active.numel() != nrow):
        raise ValueError("adam_step: active must be a uint8 tensor with one entry per row")
    sp = stream.cuda_stream if stream is not None else T.cuda.current_stream(x.device).cuda_stream
    rc = load().dmx_adam_step(64 if x.dtype == T.float64 else 32, int(nrow), int(ln), _ptr(x), _ptr(g), _ptr(mom1), _ptr(mom2), _ptr(active),
                              int(t), float(lr), float(b1), float(b2), float(eps), float(clip), C.c_void_p(sp))
    if rc != 0:
        raise RuntimeError("dmx_adam_step: " + _err())


class Model:
    """dmx_model handle.  `model` is the dict of flat arrays built by workloads.ModelBuilder."""

    def __init__(self, model, precision=64, device="cuda:0"):
        self.torch = _torch()
        self.device = self.torch.device(device)
        self.torch.cuda.set_device(self.device)
        L = load()
        d = ModelDesc()
        keep = []
        for n in _INT_FIELDS:
            setattr(d, n, int(model[n]))
        for n, t in _PTR_FIELDS:
            a = np.ascontiguousarray(model[n], dtype=np.int32 if t == "i" else np.float64)
            keep.append(a)
            setattr(d, n, a.ctypes.data_as(_pi if t == "i" else _pd))
        for k in range(3):
            d.gravity[k] = float(model["gravity"][k])
        d.newton_iters, d.ls_iters = int(model["newton_iters"]), int(model["ls_iters"])
        q0 = np.ascontiguousarray(model["qpos0"], dtype=np.float64)
        d.qpos0 = q0.ctypes.data_as(_pd)
        h = C.c_void_p()
        if L.dmx_model_create(C.byref(d), int(precision), C.byref(h)) != 0:
            raise RuntimeError("dmx_model_create: " + _err())
        self.h = h
        self.precision = int(precision)
        self.dtype = self.torch.float64 if precision == 64 else self.torch.float32
        self.nq, self.nv, self.nu = int(model["nq"]), int(model["nv"]), int(model["nu"])
        self.np_ = L.dmx_model_np(h)
        self.nc = L.dmx_model_nc(h)
        self.lanes = L.dmx_model_lanes(h)

    def __del__(self):
        if getattr(self, "h", None) and load is not None:      # at interpreter exit the module globals may be gone already
            load().dmx_model_destroy(self.h)
            self.h = None

    def set_tape_stages(self, on):
        """1 (default): tape also holds the stage rates, no recomputation in the reverse sweep; 0: checkpoints only."""
        if load().dmx_model_set_tape_stages(self.h, int(bool(on))) != 0:
            raise RuntimeError("dmx_model_set_tape_stages: " + _err())

    def set_checkpoint_stride(self, k):
        """1 (default): a tape record per accepted step; k > 1: a checkpoint every k steps + the step schedule, segments
        recomputed in the reverse sweep (dmx.h)."""
        if load().dmx_model_set_checkpoint_stride(self.h, int(k)) != 0:
            raise RuntimeError("dmx_model_set_checkpoint_stride: " + _err())

    def default_params(self):
        p = np.zeros(self.np_)
        load().dmx_model_default_params(self.h, p.ctypes.data_as(C.c_void_p))
        return p

    def debug_counters(self):
        a = np.zeros(32, dtype=np.uint64)
        if load().dmx_debug_counters(self.h, a.ctypes.data_as(C.c_void_p)) != 0:
            raise RuntimeError("dmx_debug_counters: " + _err())
        return a

    def tape_bytes(self, nenv, tape_steps):
        return int(load().dmx_tape_bytes(self.h, int(nenv), int(tape_steps)))

    # ---- helpers -------------------------------------------------------------------------------
    def dev(self, a, dtype=None):
        """numpy / tensor -> contiguous device tensor of the model's real type (None passes through)."""
        if a is None:
            return None
        t = self.torch.as_tensor(a)
        return t.to(device=self.device, dtype=dtype or self.dtype).contiguous()

    def alloc_stats(self, nenv):
        T = self.torch
        s = dict(n_accept=T.zeros(nenv, dtype=T.int32, device=self.device), n_reject=T.zeros(nenv, dtype=T.int32, device=self.device),
                 n_feval=T.zeros(nenv, dtype=T.int32, device=self.device),
                 n_newton_unconverged=T.zeros(nenv, dtype=T.int32, device=self.device),
                 status=T.zeros(nenv, dtype=T.int32, device=self.device),
                 h_min=T.zeros(nenv, dtype=T.float64, device=self.device), h_max=T.zeros(nenv, dtype=T.float64, device=self.device),
                 t_end=T.zeros(nenv, dtype=T.float64, device=self.device),
                 n_newton_unconverged_bwd=T.zeros(nenv, dtype=T.int32, device=self.device),
                 work=T.zeros((nenv, 6), dtype=T.int64, device=self.device))
        return s

    @staticmethod
    def _stats_struct(s):
        if s is None:
            return None
        return Stats(*[(s[k].data_ptr() if s.get(k) is not None else None) for k in
                       ("n_accept", "n_reject", "n_feval", "n_newton_unconverged", "status", "h_min", "h_max", "t_end", "n_newton_unconverged_bwd", "work")])

    def alloc_tape(self, nenv, tape_steps):
        return self.torch.empty(self.tape_bytes(nenv, tape_steps), dtype=self.torch.uint8, device=self.device)

    def plan(self, n_accept, margin_pct=25, pad=16, stream=None):
        """dmx_tape_plan on the accepted-step counts of a previous pass (device int32 [nenv]).  Returns (plan, tape):
        the plan buffer and a tape sized for it - sum_e (n + n*margin_pct//100 + pad) records, the formula of dmx.h."""
        T = self.torch
        nenv = n_accept.shape[0]
        n_accept = n_accept.to(device=self.device, dtype=T.int32).contiguous()
        plan = T.empty(int(load().dmx_plan_bytes(nenv)), dtype=T.uint8, device=self.device)
        if load().dmx_tape_plan(self.h, nenv, _ptr(n_accept), int(margin_pct), int(pad), _ptr(plan), plan.numel(), self._stream(stream)) != 0:
            raise RuntimeError("dmx_tape_plan: " + _err())
        n64 = n_accept.to(T.int64)
        total = int((n64 + n64 * int(margin_pct) // 100 + int(pad)).sum().item())
        tape = T.empty(int(load().dmx_tape_bytes_records(self.h, nenv, total)), dtype=T.uint8, device=self.device)
        return plan, tape

    def _stream(self, stream):
        s = stream if stream is not None else self.torch.cuda.current_stream(self.device)
        return C.c_void_p(s.cuda_stream)

    # ---- the C-ABI calls (device tensors in, device tensors out) ---------------------------------
    def rollout(self, x0, ctrl, nknot, knot_dt, params, horizon, opts, h_replay=None, xT=None, stats=None, tape=None, stream=None, plan=None):
        nenv = x0.shape[0]
        xT = self.torch.empty_like(x0) if xT is None else xT
        st = self._stats_struct(stats)
        o = _opts(opts)
        nrep = 0 if h_replay is None else h_replay.shape[1]
        rc = load().dmx_rollout(self.h, nenv, _ptr(x0), _ptr(ctrl), int(nknot), float(knot_dt), _ptr(params), float(horizon), C.byref(o),
                                _ptr(h_replay), nrep, _ptr(xT), C.byref(st) if st else None, _ptr(tape),
                                0 if tape is None else tape.numel(), _ptr(plan), self._stream(stream))
        if rc != 0:
            raise RuntimeError("dmx_rollout: " + _err())
        return xT

    def rollout_backward(self, ctrl, nknot, params, opts, xT, dLdxT, cfd_on, tape, want_params=True, status=None, stream=None,
                         out=None, plan=None, stats=None):
        """status: device int32 [nenv] marking environments to skip; stats: dict whose n_newton_unconverged_bwd is written."""
        T = self.torch
        nenv = xT.shape[0]
        if out is None:
            out = dict(dLdx0=T.empty((nenv, 2 * self.nv), dtype=self.dtype, device=self.device),
                       dLdctrl=T.empty((nenv, nknot, self.nu), dtype=self.dtype, device=self.device) if (ctrl is not None and nknot > 0) else None,
                       dLdparams=T.empty((nenv, self.np_), dtype=self.dtype, device=self.device) if want_params else None)
        o = _opts(opts)
        st = Stats()
        if status is not None:
            st.status = status.data_ptr()
        if stats is not None and stats.get("n_newton_unconverged_bwd") is not None:
            st.n_newton_unconverged_bwd = stats["n_newton_unconverged_bwd"].data_ptr()
        if stats is not None and stats.get("work") is not None:
            st.work = stats["work"].data_ptr()
        rc = load().dmx_rollout_backward(self.h, nenv, _ptr(ctrl), int(nknot), _ptr(params), C.byref(o), _ptr(xT), _ptr(dLdxT), int(cfd_on),
                                         _ptr(out["dLdx0"]), _ptr(out["dLdctrl"]), _ptr(out["dLdparams"]), C.byref(st), _ptr(tape),
                                         tape.numel(), _ptr(plan), self._stream(stream))
        if rc != 0:
            raise RuntimeError("dmx_rollout_backward: " + _err())
        return out

    def rollout_grad(self, x0, ctrl, nknot, knot_dt, params, horizon, opts, dLdxT, cfd_on, tape, h_replay=None, want_params=True,
                     stats=None, stream=None, out=None, plan=None):
        T = self.torch
        nenv = x0.shape[0]
        if out is None:
            out = dict(xT=T.empty_like(x0), dLdx0=T.empty((nenv, 2 * self.nv), dtype=self.dtype, device=self.device),
                       dLdctrl=T.empty((nenv, nknot, self.nu), dtype=self.dtype, device=self.device) if (ctrl is not None and nknot > 0) else None,
                       dLdparams=T.empty((nenv, self.np_), dtype=self.dtype, device=self.device) if want_params else None)
        st = self._stats_struct(stats)
        o = _opts(opts)
        nrep = 0 if h_replay is None else h_replay.shape[1]
        rc = load().dmx_rollout_grad(self.h, nenv, _ptr(x0), _ptr(ctrl), int(nknot), float(knot_dt), _ptr(params), float(horizon), C.byref(o),
                                     _ptr(h_replay), nrep, _ptr(dLdxT), int(cfd_on), _ptr(out["xT"]), _ptr(out["dLdx0"]), _ptr(out["dLdctrl"]),
                                     _ptr(out["dLdparams"]), C.byref(st) if st else None, _ptr(tape), tape.numel(), _ptr(plan), self._stream(stream))
        if rc != 0:
            raise RuntimeError("dmx_rollout_grad: " + _err())
        return out

    def rollout_backward_noalloc(self, ctrl, nknot, params, opts, xT, dLdxT, cfd_on, tape, out, status=None, stream=None, plan=None, stats=None):
        """dmx_rollout_backward_noalloc: the reverse sweep with its scratch in the library's static device array.  `out` must
        hold preallocated dLdx0 / dLdctrl / dLdparams tensors (this wrapper allocates nothing either)."""
        o = _opts(opts)
        st = Stats()
        if status is not None:
            st.status = status.data_ptr()
        if stats is not None and stats.get("n_newton_unconverged_bwd") is not None:
            st.n_newton_unconverged_bwd = stats["n_newton_unconverged_bwd"].data_ptr()
        if stats is not None and stats.get("work") is not None:
            st.work = stats["work"].data_ptr()
        rc = load().dmx_rollout_backward_noalloc(self.h, xT.shape[0], _ptr(ctrl), int(nknot), _ptr(params), C.byref(o), _ptr(xT), _ptr(dLdxT),
                                                 int(cfd_on), _ptr(out["dLdx0"]), _ptr(out.get("dLdctrl")), _ptr(out.get("dLdparams")), C.byref(st),
                                                 _ptr(tape), tape.numel(), _ptr(plan), self._stream(stream))
        if rc != 0:
            raise RuntimeError("dmx_rollout_backward_noalloc: " + _err())
        return out

    def _adj_out(self, nenv, ctrl, nknot, want_params, with_xT, like):
        T = self.torch
        out = dict(dLdx0=T.empty((nenv, 2 * self.nv), dtype=self.dtype, device=self.device),
                   dLdctrl=T.empty((nenv, nknot, self.nu), dtype=self.dtype, device=self.device) if (ctrl is not None and nknot > 0) else None,
                   dLdparams=T.empty((nenv, self.np_), dtype=self.dtype, device=self.device) if want_params else None,
                   adj_info=T.zeros((nenv, 3), dtype=T.int32, device=self.device))
        if with_xT:
            out["xT"] = T.empty_like(like)
        return out

    def rollout_grad_adjoint(self, x0, ctrl, nknot, knot_dt, params, horizon, opts, adj_opts, dLdxT, cfd_on, tape, h_replay=None,
                             want_params=True, stats=None, stream=None, plan=None, adj_replay=None):
        """dmx_rollout_grad_adjoint: forward with tape, then the continuous adjoint solved backwards under adj_opts.
        Returns the dict of rollout_grad plus adj_info (int32 [nenv, 3]: accepted / rejected sub-steps, status)."""
        nenv = x0.shape[0]
        out = self._adj_out(nenv, ctrl, nknot, want_params, True, x0)
        st = self._stats_struct(stats)
        o, oa = _opts(opts), _opts(adj_opts)
        nrep = 0 if h_replay is None else h_replay.shape[1]
        rc = load().dmx_rollout_grad_adjoint(self.h, nenv, _ptr(x0), _ptr(ctrl), int(nknot), float(knot_dt), _ptr(params), float(horizon),
                                             C.byref(o), C.byref(oa), _ptr(h_replay), nrep, _ptr(dLdxT), int(cfd_on), _ptr(out["xT"]),
                                             _ptr(out["dLdx0"]), _ptr(out["dLdctrl"]), _ptr(out["dLdparams"]), C.byref(st) if st else None,
                                             _ptr(out["adj_info"]), _ptr(adj_replay), 0 if adj_replay is None else adj_replay.shape[1],
                                             _ptr(tape), tape.numel(), _ptr(plan), self._stream(stream))
        if rc != 0:
            raise RuntimeError("dmx_rollout_grad_adjoint: " + _err())
        return out

    def rollout_backward_adjoint(self, ctrl, nknot, params, opts, adj_opts, xT, dLdxT, cfd_on, tape, want_params=True, stream=None, plan=None,
                                 stats=None, adj_replay=None):
        nenv = xT.shape[0]
        out = self._adj_out(nenv, ctrl, nknot, want_params, False, xT)
        o, oa = _opts(opts), _opts(adj_opts)
        st = Stats()
        if stats is not None and stats.get("n_newton_unconverged_bwd") is not None:
            st.n_newton_unconverged_bwd = stats["n_newton_unconverged_bwd"].data_ptr()
        if stats is not None and stats.get("work") is not None:
            st.work = stats["work"].data_ptr()
        rc = load().dmx_rollout_backward_adjoint(self.h, nenv, _ptr(ctrl), int(nknot), _ptr(params), C.byref(o), C.byref(oa), _ptr(xT), _ptr(dLdxT),
                                                 int(cfd_on), _ptr(out["dLdx0"]), _ptr(out["dLdctrl"]), _ptr(out["dLdparams"]), C.byref(st),
                                                 _ptr(out["adj_info"]), _ptr(adj_replay), 0 if adj_replay is None else adj_replay.shape[1],
                                                 _ptr(tape), tape.numel(), _ptr(plan), self._stream(stream))
        if rc != 0:
            raise RuntimeError("dmx_rollout_backward_adjoint: " + _err())
        return out

    def vector_field(self, x, u=None, params=None, cfd=False, stream=None):
        T = self.torch
        n = x.shape[0]
        acc = T.empty((n, self.nv), dtype=self.dtype, device=self.device)
        nrow = T.zeros(n, dtype=T.int32, device=self.device)
        rc = load().dmx_vector_field(self.h, n, _ptr(x), _ptr(u), _ptr(params), int(cfd), _ptr(acc), _ptr(nrow), self._stream(stream))
        if rc != 0:
            raise RuntimeError("dmx_vector_field: " + _err())
        return acc, nrow

    def vjp_field(self, x, u, params, kappa, cfd=False, want_params=True, stream=None):
        T = self.torch
        n = x.shape[0]
        mk = lambda k: T.empty((n, max(k, 1)), dtype=self.dtype, device=self.device)
        qb, vb, ub = mk(self.nv), mk(self.nv), mk(self.nu)
        pb = mk(self.np_) if want_params else None
        rc = load().dmx_vjp_field(self.h, n, _ptr(x), _ptr(u), _ptr(params), _ptr(kappa), int(cfd), _ptr(qb), _ptr(vb), _ptr(ub), _ptr(pb),
                                  self._stream(stream))
        if rc != 0:
            raise RuntimeError("dmx_vjp_field: " + _err())
        return qb, vb, ub[:, :self.nu], pb
