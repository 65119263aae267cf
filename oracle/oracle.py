"""ctypes front end of the CPU oracle (oracle/dd4dvar_oracle.c).

TEST INFRASTRUCTURE: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this.  Argument marshalling only; all arithmetic is in the C
file, each function citing the PAPER.md passage it follows.
"""
from __future__ import annotations

import ctypes as C
import numpy as np

from . import build as _build

_lib = None
_EVALFN = C.CFUNCTYPE(None, C.c_void_p, C.POINTER(C.c_double), C.c_int,
                      C.POINTER(C.c_double), C.POINTER(C.c_double))


def _load():
    global _lib
    if _lib is not None:
        return _lib
    lib = C.CDLL(_build.build())
    dp = C.POINTER(C.c_double)
    ip = C.POINTER(C.c_int)
    lib.orc_create.restype = C.c_void_p
    lib.orc_create.argtypes = [C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, C.c_double,
                               C.c_double, C.c_int, C.c_int, C.c_int, C.c_int, C.c_double,
                               C.c_double, C.c_double, C.c_int, C.c_int, C.c_int, C.c_int,
                               C.c_double, ip]
    lib.orc_destroy.argtypes = [C.c_void_p]
    lib.orc_nsub.argtypes = [C.c_void_p]
    lib.orc_sub_info.argtypes = [C.c_void_p, C.c_int, ip]
    lib.orc_row_tables.argtypes = [C.c_void_p, dp, dp]
    lib.orc_sub_weight.argtypes = [C.c_void_p, C.c_int, C.c_int, dp]
    lib.orc_step.argtypes = [C.c_void_p, dp, dp]
    lib.orc_step_tlm.argtypes = [C.c_void_p, dp, dp, dp]
    lib.orc_step_adj.argtypes = [C.c_void_p, dp, dp, dp]
    lib.orc_forecast.argtypes = [C.c_void_p, dp, C.c_int, ip, dp]
    lib.orc_set_background.argtypes = [C.c_void_p, dp, dp]
    lib.orc_set_observations.argtypes = [C.c_void_p, C.c_int, ip, C.POINTER(C.c_longlong), ip, dp, dp]
    lib.orc_eval_global.argtypes = [C.c_void_p, dp, dp, dp, dp]
    lib.orc_eval_local_one.argtypes = [C.c_void_p, C.c_int, dp, dp, dp, dp]
    lib.orc_get_control.argtypes = [C.c_void_p, C.c_int, dp]
    lib.orc_get_trajectory.argtypes = [C.c_void_p, C.c_int, dp]
    lib.orc_run.argtypes = [C.c_void_p, C.c_int, dp, dp]
    lib.orc_global_4dvar.argtypes = [C.c_void_p, C.c_int, dp, dp]
    lib.orc_run_gn.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, dp, dp]
    lib.orc_gn_hessvec.argtypes = [C.c_void_p, C.c_int, dp, dp, dp]
    lib.orc_gn_local.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, dp, dp]
    lib.orc_lbfgs.restype = C.c_double
    lib.orc_lbfgs.argtypes = [C.c_long, C.c_int, C.c_int, C.c_int, C.c_double, _EVALFN, C.c_void_p, dp]
    lib.orc_sweep_range.restype = C.c_double
    lib.orc_sweep_range.argtypes = [C.c_void_p, C.c_int, C.c_int, dp]
    _lib = lib
    return lib


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _c(a):
    return np.ascontiguousarray(a, dtype=np.float64)


SUB_FIELDS = ("a", "b", "jw", "oi0", "oi1", "oj0", "oj1", "ei0", "ej0", "ex", "ey",
              "gx", "gys", "gyn", "s", "e")


class Oracle:
    """One DD-4DVar problem instance on the CPU oracle (host arrays everywhere)."""

    def __init__(self, nlon, nlat, dt, nsteps, p_lon=1, p_lat=1, q_time=1, overlap=0,
                 mu=1.0, lam=1.0, radius=6.371e6, omega=7.292e-5, gravity=9.806,
                 cos_clamp=float(np.cos(np.deg2rad(50.0))), diffusion=0.02,
                 lbfgs_m=5, n_inner=5, max_backtrack=20, armijo_c1=1e-4, bg_later=0.0):
        lib = _load()
        st = C.c_int(0)
        self._h = lib.orc_create(nlon, nlat, radius, omega, gravity, cos_clamp, diffusion,
                                 p_lon, p_lat, q_time, overlap, mu, lam, dt, nsteps,
                                 lbfgs_m, n_inner, max_backtrack, armijo_c1, C.byref(st))
        if not self._h:
            raise ValueError(f"orc_create failed with status {st.value}")
        self.lib = lib
        self.nlon, self.nlat, self.nsteps = nlon, nlat, nsteps
        self.shape = (3, nlat, nlon)
        self.nsub = lib.orc_nsub(self._h)
        self.subs = [self.sub_info(k) for k in range(self.nsub)]
        self.set_bg_weight(bg_later)

    @classmethod
    def from_workload(cls, w, **kw):
        args = dict(nlon=w.nlon, nlat=w.nlat, dt=w.dt, nsteps=w.nsteps, p_lon=w.p_lon,
                    p_lat=w.p_lat, q_time=w.q_time, overlap=w.overlap, mu=w.mu, lam=w.lam,
                    lbfgs_m=w.lbfgs_m, n_inner=w.n_inner, max_backtrack=w.max_backtrack,
                    armijo_c1=w.armijo_c1, bg_later=getattr(w, "bg_later", 0.0))
        args.update(kw)
        return cls(**args)

    def close(self):
        if getattr(self, "_h", None):
            self.lib.orc_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_bg_weight(self, w):
        """weight of (25a) in windows j > 0 (R7): 0 = only at t_0 (default), 1 = as printed"""
        self.lib.orc_set_bg_weight.argtypes = [C.c_void_p, C.c_double]
        self.lib.orc_set_bg_weight.restype = None
        self.lib.orc_set_bg_weight(self._h, float(w))

    # ---- geometry
    def set_overlap_levels(self, on):
        """(25c) case 1 on every level of the window (eq (21), read literally) instead of the control level only."""
        self.lib.orc_set_overlap_levels.argtypes = [C.c_void_p, C.c_int]
        self.lib.orc_set_overlap_levels.restype = None
        self.lib.orc_set_overlap_levels(self._h, int(bool(on)))

    def sub_info(self, k):
        out = (C.c_int * 16)()
        self.lib.orc_sub_info(self._h, k, out)
        return dict(zip(SUB_FIELDS, list(out)))

    def sub_shape(self, k):
        s = self.subs[k]
        return (3, s["ey"], s["ex"])

    def row_tables(self):
        out = np.zeros((6, self.nlat))
        cm = C.c_double(0)
        self.lib.orc_row_tables(self._h, _dp(out), C.byref(cm))
        return dict(f=out[0], t=out[1], cz=out[2], rp=out[3], rm=out[4], mc=out[5], cm=cm.value)

    def sub_weight(self, k, level):
        s = self.subs[k]
        out = np.zeros((s["ey"], s["ex"]))
        self.lib.orc_sub_weight(self._h, k, level, _dp(out))
        return out

    # ---- model
    def step(self, Z):
        Z = _c(Z); out = np.empty(self.shape)
        self.lib.orc_step(self._h, _dp(Z), _dp(out))
        return out

    def step_tlm(self, Z, dZ):
        Z = _c(Z); dZ = _c(dZ); out = np.empty(self.shape)
        self.lib.orc_step_tlm(self._h, _dp(Z), _dp(dZ), _dp(out))
        return out

    def step_adj(self, Z, L1):
        Z = _c(Z); L1 = _c(L1); out = np.empty(self.shape)
        self.lib.orc_step_adj(self._h, _dp(Z), _dp(L1), _dp(out))
        return out

    def forecast(self, x0, levels):
        x0 = _c(x0)
        lv = np.ascontiguousarray(levels, dtype=np.int32)
        out = np.empty((lv.size,) + self.shape)
        self.lib.orc_forecast(self._h, _dp(x0), lv.size, lv.ctypes.data_as(C.POINTER(C.c_int)), _dp(out))
        return out

    # ---- problem data
    def set_background(self, xb, sigma_b):
        xb = _c(xb); sb = _c(sigma_b)
        rc = self.lib.orc_set_background(self._h, _dp(xb), _dp(sb))
        if rc:
            raise RuntimeError(f"orc_set_background -> {rc}")

    def set_observations(self, obs):
        lv = np.ascontiguousarray(obs.levels, dtype=np.int32)
        off = np.ascontiguousarray(obs.offsets, dtype=np.int64)
        idx = np.ascontiguousarray(obs.index, dtype=np.int32)
        val = _c(obs.value); so = _c(obs.sigma_o)
        rc = self.lib.orc_set_observations(
            self._h, lv.size, lv.ctypes.data_as(C.POINTER(C.c_int)),
            off.ctypes.data_as(C.POINTER(C.c_longlong)), idx.ctypes.data_as(C.POINTER(C.c_int)),
            _dp(val), _dp(so))
        if rc:
            raise RuntimeError(f"orc_set_observations -> {rc}")

    # ---- functionals
    def eval_global(self, x0, want_grad=True):
        x0 = _c(x0)
        J = C.c_double(0); parts = np.zeros(2)
        g = np.empty(self.shape) if want_grad else None
        rc = self.lib.orc_eval_global(self._h, _dp(x0), C.byref(J), _dp(g) if want_grad else None, _dp(parts))
        if rc:
            raise RuntimeError(f"orc_eval_global -> {rc}")
        return J.value, g, parts

    def eval_local(self, k, x, want_grad=True, want_traj=False):
        """J_ji, its parts (total,bg,obs,ov_space,ov_pred,ov_succ), dJ/dx, local trajectory."""
        x = _c(x); s = self.subs[k]
        parts = np.zeros(6)
        g = np.empty(self.sub_shape(k)) if want_grad else None
        tr = np.empty((s["e"] - s["s"] + 1,) + self.sub_shape(k)) if want_traj else None
        rc = self.lib.orc_eval_local_one(self._h, k, _dp(x), _dp(parts), _dp(g) if want_grad else None,
                                         _dp(tr) if want_traj else None)
        if rc:
            raise RuntimeError(f"orc_eval_local_one -> {rc}")
        return parts, g, tr

    def get_control(self, k):
        out = np.empty(self.sub_shape(k))
        self.lib.orc_get_control(self._h, k, _dp(out))
        return out

    def get_trajectory(self, level):
        out = np.empty(self.shape)
        self.lib.orc_get_trajectory(self._h, level, _dp(out))
        return out

    def run(self, outer_iters):
        an = np.empty(self.shape); hist = np.zeros((outer_iters + 1, 3))
        rc = self.lib.orc_run(self._h, outer_iters, _dp(an), _dp(hist))
        if rc:
            raise RuntimeError(f"orc_run -> {rc}")
        return an, hist

    def run_gn(self, outer_iters, n_gn=2, n_cg=5):
        """Algorithm 1 with the paper's own local minimiser: incremental Gauss-Newton (Alg 5-6),
        normal equations solved by n_cg CG iterations in w-space (eq (42)-(46))."""
        an = np.empty(self.shape); hist = np.zeros((outer_iters + 1, 3))
        rc = self.lib.orc_run_gn(self._h, outer_iters, n_gn, n_cg, _dp(an), _dp(hist))
        if rc:
            raise RuntimeError(f"orc_run_gn -> {rc}")
        return an, hist

    def gn_hessvec(self, k, x, p):
        """H_GN p of subdomain k about the control x (p and the result in w-space)."""
        x = _c(x); p = _c(p); out = np.empty_like(p)
        rc = self.lib.orc_gn_hessvec(self._h, k, _dp(x), _dp(p), _dp(out))
        if rc:
            raise RuntimeError(f"orc_gn_hessvec -> {rc}")
        return out

    def gn_local(self, k, x, n_gn, n_cg):
        """n_gn Gauss-Newton iterations on subdomain k from the control x; returns (x_new, J_first, J_last)."""
        x = np.array(_c(x), copy=True); jj = np.zeros(2)
        rc = self.lib.orc_gn_local(self._h, k, n_gn, n_cg, _dp(x), _dp(jj))
        if rc:
            raise RuntimeError(f"orc_gn_local -> {rc}")
        return x, jj[0], jj[1]

    def global_4dvar(self, rounds):
        an = np.empty(self.shape); hist = np.zeros(rounds + 1)
        rc = self.lib.orc_global_4dvar(self._h, rounds, _dp(an), _dp(hist))
        if rc:
            raise RuntimeError(f"orc_global_4dvar -> {rc}")
        return an, hist

    def sweep_range(self, k0, k1):
        cs = C.c_double(0)
        pts = self.lib.orc_sweep_range(self._h, k0, k1, C.byref(cs))
        return pts, cs.value


def lbfgs_minimize(fun, w0, m=5, n_iter=50, max_backtrack=20, c1=1e-4):
    """The oracle's L-BFGS on a Python function fun(w) -> (J, g); for the dense-solve pin."""
    lib = _load()
    w = _c(w0).copy(); n = w.size

    def cb(ctx, wp, want_grad, Jp, gp):
        wv = np.ctypeslib.as_array(wp, shape=(n,))
        J, g = fun(wv.copy())
        Jp[0] = J
        if want_grad:
            np.ctypeslib.as_array(gp, shape=(n,))[:] = g

    J = lib.orc_lbfgs(n, m, n_iter, max_backtrack, c1, _EVALFN(cb), None, _dp(w))
    return w, J
