"""ORACLE — test infrastructure only.  ctypes marshalling for oracle/liboracle.so.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It imports nothing from the product package; model descriptions and
inputs arrive as plain dicts / numpy arrays (built by paper_2506_14186_b200/workloads.py,
which holds no method arithmetic).
"""
import ctypes as C
import os
import subprocess
import threading
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB = os.path.join(_HERE, "liboracle.so")
_SRC = ["capi.cpp", "adjoint.hpp", "rk.hpp", "field.hpp", "solve.hpp", "contact.hpp", "kin.hpp", "model.hpp", "dual.hpp"]


def build(force=False):
    """g++ -O2, no fast-math, no FMA contraction (D4), generic x86-64."""
    src_m = max(os.path.getmtime(os.path.join(_HERE, s)) for s in _SRC)
    if not force and os.path.exists(_LIB) and os.path.getmtime(_LIB) >= src_m:
        return _LIB
    cmd = ["g++", "-std=c++17", "-O2", "-fPIC", "-shared", "-ffp-contract=off", "-o", _LIB, os.path.join(_HERE, "capi.cpp")]
    subprocess.check_call(cmd)
    return _LIB


_F8 = np.ctypeslib.ndpointer(dtype=np.float64, flags="C_CONTIGUOUS")
_I4 = np.ctypeslib.ndpointer(dtype=np.int32, flags="C_CONTIGUOUS")
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


class _Desc(C.Structure):
    _fields_ = ([(n, C.c_int) for n in _INT_FIELDS] + [(n, _pi if t == "i" else _pd) for n, t in _PTR_FIELDS] +
                [("gravity", C.c_double * 3), ("newton_iters", C.c_int), ("ls_iters", C.c_int), ("qpos0", _pd)])


class _Opts(C.Structure):
    _fields_ = [("tableau", C.c_int), ("rtol", C.c_double), ("atol", C.c_double), ("h0", C.c_double),
                ("pcoeff", C.c_double), ("icoeff", C.c_double), ("safety", C.c_double), ("fac_min", C.c_double),
                ("fac_max", C.c_double), ("max_steps", C.c_int)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(_LIB)
        _lib.orc_model_create.restype = C.c_void_p
        _lib.orc_last_error.restype = C.c_char_p
        _lib.orc_impedance.restype = C.c_double
        _lib.orc_impedance_cfd.restype = C.c_double
        _lib.orc_softplus.restype = C.c_double
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _f8(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64)


class Oracle:
    """CPU fp64 oracle of the hot path for one model description (dict of arrays)."""

    def __init__(self, model):
        L = lib()
        d = _Desc()
        self._keep = []
        for n in _INT_FIELDS:
            setattr(d, n, int(model[n]))
        for n, t in _PTR_FIELDS:
            a = np.ascontiguousarray(model[n], dtype=np.int32 if t == "i" else np.float64)
            self._keep.append(a)
            setattr(d, n, a.ctypes.data_as(_pi if t == "i" else _pd))
        for k in range(3):
            d.gravity[k] = float(model["gravity"][k])
        d.newton_iters, d.ls_iters = int(model["newton_iters"]), int(model["ls_iters"])
        q0 = np.ascontiguousarray(model["qpos0"], dtype=np.float64); self._keep.append(q0)
        d.qpos0 = q0.ctypes.data_as(_pd)
        self.h = L.orc_model_create(C.byref(d))
        if not self.h:
            raise ValueError("oracle model_create: " + L.orc_last_error().decode())
        self.h = C.c_void_p(self.h)
        self.nq, self.nv, self.nu, self.nbody, self.npair = (int(model[k]) for k in ("nq", "nv", "nu", "nbody", "npair"))
        self.np_ = L.orc_np(self.h)
        self.nc = L.orc_nc(self.h)

    def __del__(self):
        if getattr(self, "h", None) and lib is not None:        # module globals may be gone at interpreter exit
            lib().orc_model_destroy(self.h)
            self.h = None

    # ---- pieces (pins) ----
    def default_params(self):
        p = np.zeros(self.np_); lib().orc_default_params(self.h, _p(p)); return p

    def invweight(self):
        bw, pw = np.zeros(self.nbody), np.zeros(self.npair)
        lib().orc_invweight(self.h, _p(bw), _p(pw)); return bw, pw

    def mass_matrix(self, q, p=None):
        M = np.zeros((self.nv, self.nv)); lib().orc_mass_matrix(self.h, _p(_f8(q)), _p(_f8(p)), _p(M)); return M

    def inverse_dynamics(self, q, v, a, p=None):
        o = np.zeros(self.nv); lib().orc_inverse_dynamics(self.h, _p(_f8(q)), _p(_f8(v)), _p(_f8(a)), _p(_f8(p)), _p(o)); return o

    def kinematics(self, q, v):
        nb = self.nbody
        pos, mat, com, w, cv = np.zeros((nb, 3)), np.zeros((nb, 3, 3)), np.zeros((nb, 3)), np.zeros((nb, 3)), np.zeros((nb, 3))
        lib().orc_kinematics(self.h, _p(_f8(q)), _p(_f8(v)), _p(pos), _p(mat), _p(com), _p(w), _p(cv))
        return dict(pos=pos, mat=mat, com=com, angvel=w, comvel=cv)

    def world_inertia(self, q, p=None):
        I = np.zeros((self.nbody, 3, 3)); lib().orc_world_inertia(self.h, _p(_f8(q)), _p(_f8(p)), _p(I)); return I

    def collide(self, q):
        nc = self.nc
        r, n, pos, t1, t2 = np.zeros(nc), np.zeros((nc, 3)), np.zeros((nc, 3)), np.zeros((nc, 3)), np.zeros((nc, 3))
        lib().orc_collide(self.h, _p(_f8(q)), _p(r), _p(n), _p(pos), _p(t1), _p(t2))
        return dict(r=r, n=n, pos=pos, t1=t1, t2=t2)

    def rows(self, q, v, p=None, cfd=False):
        nmax = 4 * self.nc
        J, aref, D, r = np.zeros((nmax, self.nv)), np.zeros(nmax), np.zeros(nmax), np.zeros(nmax)
        nr = lib().orc_rows(self.h, _p(_f8(q)), _p(_f8(v)), _p(_f8(p)), int(cfd), _p(J), _p(aref), _p(D), _p(r))
        return dict(J=J[:nr].copy(), aref=aref[:nr].copy(), D=D[:nr].copy(), r=r[:nr].copy())

    def vector_field(self, q, v, u=None, p=None, cfd=False):
        acc = np.zeros(self.nv); conv = C.c_int(0)
        u = np.zeros(max(self.nu, 1)) if u is None else _f8(u)
        nr = lib().orc_vector_field(self.h, _p(_f8(q)), _p(_f8(v)), _p(u), _p(_f8(p)), int(cfd), _p(acc), C.byref(conv))
        return acc, nr, bool(conv.value)

    def vjp_field(self, q, v, u, p, kappa, cfd=False, want_p=True):
        qb, vb, ub = np.zeros(self.nv), np.zeros(self.nv), np.zeros(max(self.nu, 1))
        pb = np.zeros(self.np_) if want_p else None
        u = np.zeros(max(self.nu, 1)) if u is None else _f8(u)
        rc = lib().orc_vjp_field(self.h, _p(_f8(q)), _p(_f8(v)), _p(u), _p(_f8(p)), _p(_f8(kappa)), int(cfd), _p(qb), _p(vb), _p(ub), _p(pb))
        if rc != 0:
            raise RuntimeError("oracle vjp_field failed")
        return qb, vb, ub[: self.nu], pb

    def retract(self, q, delta):
        o = np.zeros(self.nq); lib().orc_retract(self.h, _p(_f8(q)), _p(_f8(delta)), _p(o)); return o

    def ambient_to_tangent(self, x, g):
        lam = np.zeros(2 * self.nv); lib().orc_ambient_to_tangent(self.h, _p(_f8(x)), _p(_f8(g)), _p(lam)); return lam

    # ---- rollouts ----
    @staticmethod
    def _opts(o):
        return _Opts(int(o["tableau"]), o["rtol"], o["atol"], o["h0"], o["pcoeff"], o["icoeff"], o["safety"],
                     o["fac_min"], o["fac_max"], int(o["max_steps"]))

    def _run(self, fn, nenv, threads):
        """Shard envs over plain threads (ctypes releases the GIL); each env is single-threaded code."""
        threads = max(1, min(threads, nenv))
        if threads == 1:
            fn(0, nenv); return
        bounds = np.linspace(0, nenv, threads + 1).astype(int)
        ts = [threading.Thread(target=fn, args=(int(bounds[i]), int(bounds[i + 1]))) for i in range(threads)]
        [t.start() for t in ts]; [t.join() for t in ts]

    def rollout(self, x0, ctrl, nknot, knot_dt, params, horizon, opts, h_replay=None, n_hout=0, threads=1):
        x0 = _f8(x0); nenv = x0.shape[0]
        ctrl, params, h_replay = _f8(ctrl), _f8(params), _f8(h_replay)
        xT = np.zeros_like(x0); ist = np.zeros((nenv, 5), dtype=np.int32); dst = np.zeros((nenv, 3))
        hout = np.zeros((nenv, n_hout)) if n_hout > 0 else None
        o = self._opts(opts); nrep = 0 if h_replay is None else h_replay.shape[1]
        L = lib()

        def fn(e0, e1):
            L.orc_rollout(self.h, e0, e1, _p(x0), _p(ctrl), int(nknot), C.c_double(knot_dt), _p(params), C.c_double(horizon),
                          C.byref(o), _p(h_replay), nrep, _p(xT), _p(ist), _p(dst), _p(hout), int(n_hout))
        self._run(fn, nenv, threads)
        return dict(xT=xT, stats=_stats(ist, dst), h=hout)

    def rollout_grad(self, x0, ctrl, nknot, knot_dt, params, horizon, opts, dLdxT=None, loss_grad=None, cfd_on=False,
                     h_replay=None, want_params=True, threads=1):
        """dLdxT may be given, or computed by the caller-side loss_grad(xT, x0) after an oracle forward pass."""
        x0 = _f8(x0); nenv = x0.shape[0]
        ctrl, params, h_replay = _f8(ctrl), _f8(params), _f8(h_replay)
        if dLdxT is None:
            fwd = self.rollout(x0, ctrl, nknot, knot_dt, params, horizon, opts, h_replay=h_replay, threads=threads)
            dLdxT = loss_grad(fwd["xT"], x0)[1]
        dLdxT = _f8(dLdxT)
        xT = np.zeros_like(x0); ist = np.zeros((nenv, 5), dtype=np.int32); dst = np.zeros((nenv, 3))
        g0 = np.zeros((nenv, 2 * self.nv))
        gc = np.zeros((nenv, nknot, self.nu)) if (ctrl is not None and nknot > 0) else None
        gp = np.zeros((nenv, self.np_)) if want_params else None
        o = self._opts(opts); nrep = 0 if h_replay is None else h_replay.shape[1]
        L = lib()

        def fn(e0, e1):
            L.orc_rollout_grad(self.h, e0, e1, _p(x0), _p(ctrl), int(nknot), C.c_double(knot_dt), _p(params), C.c_double(horizon),
                               C.byref(o), _p(h_replay), nrep, _p(dLdxT), int(cfd_on), _p(xT), _p(ist), _p(dst), _p(g0), _p(gc), _p(gp))
        self._run(fn, nenv, threads)
        return dict(xT=xT, stats=_stats(ist, dst), dLdx0=g0, dLdctrl=gc, dLdparams=gp)


def _adjoint(self, x0, ctrl, nknot, knot_dt, params, horizon, opts, adj_opts, dLdxT, cfd_on=False, h_replay=None, want_params=True, threads=1,
             adj_replay=None, n_adj_hout=0):
    """Optimize-then-discretize gradient (adjoint.hpp): forward with tape, then the continuous adjoint solved backwards
    with its own error-controlled steps under adj_opts.  Returns the fields of rollout_grad plus adj_accept / adj_reject /
    adj_status per environment."""
    x0 = _f8(x0); nenv = x0.shape[0]
    ctrl, params, h_replay, dLdxT = _f8(ctrl), _f8(params), _f8(h_replay), _f8(dLdxT)
    xT = np.zeros_like(x0); ist = np.zeros((nenv, 5), dtype=np.int32); dst = np.zeros((nenv, 3)); asub = np.zeros((nenv, 3), dtype=np.int32)
    g0 = np.zeros((nenv, 2 * self.nv))
    gc = np.zeros((nenv, nknot, self.nu)) if (ctrl is not None and nknot > 0) else None
    gp = np.zeros((nenv, self.np_)) if want_params else None
    o, oa = self._opts(opts), self._opts(adj_opts); nrep = 0 if h_replay is None else h_replay.shape[1]
    adj_replay = _f8(adj_replay); narep = 0 if adj_replay is None else adj_replay.shape[1]
    hout = np.zeros((nenv, n_adj_hout)) if n_adj_hout > 0 else None
    L = lib()

    def fn(e0, e1):
        L.orc_rollout_grad_adjoint(self.h, e0, e1, _p(x0), _p(ctrl), int(nknot), C.c_double(knot_dt), _p(params), C.c_double(horizon),
                                   C.byref(o), C.byref(oa), _p(h_replay), nrep, _p(dLdxT), int(cfd_on), _p(xT), _p(ist), _p(dst), _p(asub),
                                   _p(g0), _p(gc), _p(gp), _p(adj_replay), narep, _p(hout), int(n_adj_hout))
    self._run(fn, nenv, threads)
    return dict(xT=xT, stats=_stats(ist, dst), dLdx0=g0, dLdctrl=gc, dLdparams=gp, adj_accept=asub[:, 0].copy(), adj_reject=asub[:, 1].copy(),
                adj_status=asub[:, 2].copy(), adj_h=hout)


Oracle.rollout_grad_adjoint = _adjoint


def _stats(ist, dst):
    return dict(n_accept=ist[:, 0].copy(), n_reject=ist[:, 1].copy(), n_feval=ist[:, 2].copy(),
                n_newton_unconverged=ist[:, 3].copy(), status=ist[:, 4].copy(),
                h_min=dst[:, 0].copy(), h_max=dst[:, 1].copy(), t_end=dst[:, 2].copy())


def contact_solve(M, a0, J, aref, D, n_it=4, n_ls=16):
    nv, nr = len(a0), len(aref)
    x, f, act = np.zeros(nv), np.zeros(max(nr, 1)), np.zeros(max(nr, 1), dtype=np.int32)
    it = lib().orc_contact_solve(nv, nr, _p(_f8(M)), _p(_f8(a0)), _p(_f8(J).reshape(-1) if nr else np.zeros(1)), _p(_f8(aref) if nr else np.zeros(1)),
                                 _p(_f8(D) if nr else np.zeros(1)), n_it, n_ls, _p(x), _p(f), _p(act))
    return dict(x=x, f=f[:nr], active=act[:nr].astype(bool), converged=it > 0, iters=abs(it))


def tableau(which):
    c, a, b, e = np.zeros(7), np.zeros((7, 7)), np.zeros(7), np.zeros(7)
    lib().orc_tableau(int(which), _p(c), _p(a), _p(b), _p(e)); return c, a, b, e


def impedance(solimp, r):
    return lib().orc_impedance(_p(_f8(solimp)), C.c_double(r))


def impedance_cfd(solimp_cfd, r):
    return lib().orc_impedance_cfd(_p(_f8(solimp_cfd)), C.c_double(r))


def softplus(z, beta):
    return lib().orc_softplus(C.c_double(z), C.c_double(beta))
