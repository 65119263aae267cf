"""Thin ctypes binding of include/dd4dvar.h: argument marshalling only.

Every step of the hot path runs in the CUDA kernels of libdd4dvar.so.  PyTorch supplies device
memory (workspaces, inputs, outputs) and the stream.  There is no CPU fallback: without the
built library or without a CUDA device the constructor raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIBPATH = os.path.join(HERE, "libdd4dvar.so")

SUB_FIELDS = ("a", "b", "jw", "oi0", "oi1", "oj0", "oj1", "ei0", "ej0", "ex", "ey",
              "gx", "gys", "gyn", "s", "e")


class Grid(C.Structure):
    _fields_ = [("nlon", C.c_int), ("nlat", C.c_int), ("radius", C.c_double), ("omega", C.c_double),
                ("gravity", C.c_double), ("cos_clamp", C.c_double), ("diffusion", C.c_double)]


class Decomp(C.Structure):
    _fields_ = [("p_lon", C.c_int), ("p_lat", C.c_int), ("q_time", C.c_int), ("overlap", C.c_int),
                ("mu", C.c_double), ("lam", C.c_double)]


class Window(C.Structure):
    _fields_ = [("dt", C.c_double), ("nsteps", C.c_int)]


class Opts(C.Structure):
    _fields_ = [("lbfgs_m", C.c_int), ("n_inner", C.c_int), ("max_backtrack", C.c_int),
                ("armijo_c1", C.c_double), ("path", C.c_int)]


class DD4DVarError(RuntimeError):
    def __init__(self, fn, code, text=""):
        super().__init__(f"{fn} -> {code}: {text}")
        self.code = code


_lib = None

EXPORTS = [
    "dd4dvar_create", "dd4dvar_workspace_bytes", "dd4dvar_set_workspace", "dd4dvar_set_background",
    "dd4dvar_obs_workspace_bytes", "dd4dvar_set_observations", "dd4dvar_run", "dd4dvar_eval_global",
    "dd4dvar_eval_local", "dd4dvar_eval_local_host", "dd4dvar_sweep_async", "dd4dvar_get_controls", "dd4dvar_get_trajectory",
    "dd4dvar_get_local_trajectory", "dd4dvar_forecast", "dd4dvar_forecast_static", "dd4dvar_num_subdomains",
    "dd4dvar_subdomain_info", "dd4dvar_control_offset", "dd4dvar_active_path", "dd4dvar_launch_count",
    "dd4dvar_measure_peaks", "dd4dvar_set_bg_weight", "dd4dvar_run_gn", "dd4dvar_gn_hessvec", "dd4dvar_set_history_global", "dd4dvar_set_overlap_levels", "dd4dvar_set_owned_windows", "dd4dvar_exchange_buffer",
    "dd4dvar_get_local_stats", "dd4dvar_gather_analysis", "dd4dvar_set_phase_timing", "dd4dvar_get_phase_ms",
    "dd4dvar_last_error", "dd4dvar_destroy",
]


def load_library():
    """Load libdd4dvar.so (built in-tree by paper_2205_06649_b200/build.py) and declare the ABI."""
    global _lib
    if _lib is not None:
        return _lib
    path = os.environ.get("DD4DVAR_LIB", LIBPATH)     # override: an alternative build of the same ABI
    if not os.path.exists(path):
        raise DD4DVarError("load_library", -4, f"{LIBPATH} is missing: run `python -m paper_2205_06649_b200.build`")
    lib = C.CDLL(path)
    vp, dp, ip = C.c_void_p, C.c_void_p, C.POINTER(C.c_int)   # device pointers travel as integers
    hd = C.POINTER(C.c_double)
    lib.dd4dvar_create.argtypes = [C.POINTER(Grid), C.POINTER(Decomp), C.POINTER(Window), C.POINTER(Opts), vp, C.POINTER(vp)]
    lib.dd4dvar_workspace_bytes.restype = C.c_size_t
    lib.dd4dvar_workspace_bytes.argtypes = [vp]
    lib.dd4dvar_set_workspace.argtypes = [vp, dp, C.c_size_t]
    lib.dd4dvar_set_background.argtypes = [vp, dp, hd]
    lib.dd4dvar_obs_workspace_bytes.restype = C.c_size_t
    lib.dd4dvar_obs_workspace_bytes.argtypes = [vp, C.c_longlong]
    lib.dd4dvar_set_observations.argtypes = [vp, C.c_int, ip, C.POINTER(C.c_longlong), dp, dp, hd, dp, C.c_size_t]
    lib.dd4dvar_run.argtypes = [vp, C.c_int, dp, hd]
    lib.dd4dvar_run_gn.argtypes = [vp, C.c_int, C.c_int, C.c_int, dp, hd]
    lib.dd4dvar_gn_hessvec.argtypes = [vp, dp, dp, dp]
    lib.dd4dvar_eval_global.argtypes = [vp, dp, hd, dp]
    lib.dd4dvar_eval_local.argtypes = [vp, dp, hd, hd, dp]
    lib.dd4dvar_eval_local_host.argtypes = [vp, C.c_void_p, hd, C.c_void_p]
    lib.dd4dvar_sweep_async.argtypes = [vp, C.c_int]
    lib.dd4dvar_get_controls.argtypes = [vp, dp]
    lib.dd4dvar_get_trajectory.argtypes = [vp, C.c_int, dp]
    lib.dd4dvar_get_local_trajectory.argtypes = [vp, C.c_int, dp]
    lib.dd4dvar_forecast.argtypes = [vp, dp, C.c_int, ip, dp]
    lib.dd4dvar_forecast_static.argtypes = [C.POINTER(Grid), C.POINTER(Window), dp, C.c_int, ip, dp, vp, C.c_char_p, C.c_size_t]
    lib.dd4dvar_num_subdomains.argtypes = [vp]
    lib.dd4dvar_subdomain_info.argtypes = [vp, C.c_int, ip]
    lib.dd4dvar_control_offset.restype = C.c_longlong
    lib.dd4dvar_control_offset.argtypes = [vp, C.c_int]
    lib.dd4dvar_active_path.argtypes = [vp]
    lib.dd4dvar_launch_count.restype = C.c_longlong
    lib.dd4dvar_launch_count.argtypes = [vp]
    lib.dd4dvar_measure_peaks.argtypes = [vp, hd]
    lib.dd4dvar_set_bg_weight.argtypes = [vp, C.c_double]
    lib.dd4dvar_set_history_global.argtypes = [vp, C.c_int]
    lib.dd4dvar_set_overlap_levels.argtypes = [vp, C.c_int]
    lib.dd4dvar_set_owned_windows.argtypes = [vp, C.c_int, C.c_int]
    lib.dd4dvar_exchange_buffer.argtypes = [vp, C.c_int, C.POINTER(C.c_void_p), C.POINTER(C.c_longlong)]
    lib.dd4dvar_get_local_stats.argtypes = [vp, hd, hd]
    lib.dd4dvar_gather_analysis.argtypes = [vp, dp]
    lib.dd4dvar_set_phase_timing.argtypes = [vp, C.c_int]
    lib.dd4dvar_get_phase_ms.argtypes = [vp, hd]
    lib.dd4dvar_last_error.restype = C.c_char_p
    lib.dd4dvar_last_error.argtypes = [vp]
    lib.dd4dvar_destroy.restype = None
    lib.dd4dvar_destroy.argtypes = [vp]
    _lib = lib
    return lib


def _hd(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def measure_peaks(device="cuda:0"):
    """dd4dvar_measure_peaks: fp64 FMA / ADD rates, LDS.64 bandwidth, 64-bit shuffle rate of the device."""
    import numpy as np
    import torch
    lib = load_library()
    dev = torch.device(device)
    out = np.zeros(6)
    with torch.cuda.device(dev):
        st = torch.cuda.current_stream(dev)
        rc = lib.dd4dvar_measure_peaks(C.c_void_p(st.cuda_stream), _hd(out))
    if rc:
        raise DD4DVarError("dd4dvar_measure_peaks", rc)
    nsm, mhz = out[4], out[5]
    return {"fp64_fma_tflops": out[0], "fp64_add_tinstr_s": out[1], "lds64_bytes_per_s": out[2],
            "lds64_bytes_per_clk_per_sm": out[2] / (nsm * mhz * 1e6), "shfl64_per_s": out[3],
            "shfl64_bytes_per_clk_per_sm": 8.0 * out[3] / (nsm * mhz * 1e6), "sm_count": int(nsm), "sm_clock_mhz": mhz}


STATIC_SCRATCH_BYTES = 16 << 20     # DD4DVAR_STATIC_SCRATCH_BYTES of include/dd4dvar.h


def forecast_static(x0, levels, out, dt, nsteps, radius=6.371e6, omega=7.292e-5, gravity=9.806,
                    cos_clamp=float(np.cos(np.deg2rad(50.0))), diffusion=0.02, stream=None):
    """dd4dvar_forecast_static: the model forecast for a caller that cannot allocate device memory for the library
    (the device is owned by another pool, or is full, or the caller must not stall it with cudaMalloc).  No handle,
    no workspace: the library steps the model inside a 16 MiB array that is part of its image, so the grid is limited
    to about 349 000 cells (DD4DVarError with code -6 beyond that).  Nothing is allocated here either: `x0`
    ([3][nlat][nlon]) and `out` ([len(levels)][3][nlat][nlon]) are the caller's fp64 CUDA tensors; `out` is filled and
    returned.  Calls share the library's array: do not let two of them overlap on one GPU.  Make the first call on a
    device during set-up, outside stream capture."""
    import torch
    lib = load_library()
    if not (x0.is_cuda and out.is_cuda and x0.dtype == torch.float64 and out.dtype == torch.float64
            and x0.is_contiguous() and out.is_contiguous() and x0.dim() == 3 and x0.shape[0] == 3):
        raise DD4DVarError("dd4dvar_forecast_static", -1, "x0 and out must be contiguous fp64 CUDA tensors, x0 [3][nlat][nlon]")
    lv = np.ascontiguousarray(levels, dtype=np.int32)
    if tuple(out.shape) != (lv.size,) + tuple(x0.shape) or out.device != x0.device:
        raise DD4DVarError("dd4dvar_forecast_static", -1, "out must be [len(levels)][3][nlat][nlon] on x0's device")
    g = Grid(int(x0.shape[2]), int(x0.shape[1]), radius, omega, gravity, cos_clamp, diffusion)
    w = Window(dt, nsteps)
    err = C.create_string_buffer(512)
    with torch.cuda.device(x0.device):
        st = stream if stream is not None else torch.cuda.current_stream(x0.device)
        rc = lib.dd4dvar_forecast_static(C.byref(g), C.byref(w), x0.data_ptr(), lv.size,
                                         lv.ctypes.data_as(C.POINTER(C.c_int)), out.data_ptr(),
                                         C.c_void_p(st.cuda_stream), err, len(err))
    if rc:
        raise DD4DVarError("dd4dvar_forecast_static", rc, err.value.decode())
    return out


class DD4DVar:
    """One DD-4DVar problem on one GPU.  Tensors in and out are torch CUDA fp64 tensors."""

    def __init__(self, nlon, nlat, dt, nsteps, p_lon=1, p_lat=1, q_time=1, overlap=0, mu=1.0, lam=1.0,
                 radius=6.371e6, omega=7.292e-5, gravity=9.806,
                 cos_clamp=float(np.cos(np.deg2rad(50.0))), diffusion=0.02, lbfgs_m=5, n_inner=5,
                 max_backtrack=20, armijo_c1=1e-4, path=0, device="cuda:0", stream=None, bg_later=0.0):
        import torch
        self.torch = torch
        self.lib = load_library()
        if not torch.cuda.is_available():
            raise DD4DVarError("DD4DVar", -4, "no CUDA device: the library has no CPU fallback")
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        g = Grid(nlon, nlat, radius, omega, gravity, cos_clamp, diffusion)
        d = Decomp(p_lon, p_lat, q_time, overlap, mu, lam)
        w = Window(dt, nsteps)
        o = Opts(lbfgs_m, n_inner, max_backtrack, armijo_c1, path)
        h = C.c_void_p()
        rc = self.lib.dd4dvar_create(C.byref(g), C.byref(d), C.byref(w), C.byref(o),
                                     C.c_void_p(self.stream.cuda_stream), C.byref(h))
        if rc:
            raise DD4DVarError("dd4dvar_create", rc)
        self._h = h
        rc = self.lib.dd4dvar_set_bg_weight(h, float(bg_later))
        if rc:
            raise DD4DVarError("dd4dvar_set_bg_weight", rc)
        self.nlon, self.nlat, self.nsteps = nlon, nlat, nsteps
        self.shape = (3, nlat, nlon)
        self.nsub = self.lib.dd4dvar_num_subdomains(h)
        self.subs = [self.sub_info(k) for k in range(self.nsub)]
        self.offsets = [self.lib.dd4dvar_control_offset(h, k) for k in range(self.nsub + 1)]
        self.ctot = self.offsets[-1]
        nbytes = self.lib.dd4dvar_workspace_bytes(h)
        self.workspace_bytes = nbytes
        self._ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        base = (self._ws.data_ptr() + 255) & ~255
        self._check("dd4dvar_set_workspace", self.lib.dd4dvar_set_workspace(h, base, nbytes))
        self._obs_ws = None

    @classmethod
    def from_workload(cls, w, **kw):
        args = dict(nlon=w.nlon, nlat=w.nlat, dt=w.dt, nsteps=w.nsteps, p_lon=w.p_lon, p_lat=w.p_lat,
                    q_time=w.q_time, overlap=w.overlap, mu=w.mu, lam=w.lam, lbfgs_m=w.lbfgs_m,
                    n_inner=w.n_inner, max_backtrack=w.max_backtrack, armijo_c1=w.armijo_c1,
                    bg_later=getattr(w, "bg_later", 0.0))
        args.update(kw)
        return cls(**args)

    # ---- plumbing
    def _check(self, fn, rc):
        if rc:
            raise DD4DVarError(fn, rc, self.lib.dd4dvar_last_error(self._h).decode())

    def _dev(self, a):
        t = self.torch.as_tensor(a, dtype=self.torch.float64, device=self.device).contiguous()
        return t

    def close(self):
        if getattr(self, "_h", None):
            self.torch.cuda.synchronize(self.device)
            self.lib.dd4dvar_destroy(self._h)
            self._h = None
            self._ws = None
            self._obs_ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- geometry
    def sub_info(self, k):
        out = (C.c_int * 16)()
        self._check("dd4dvar_subdomain_info", self.lib.dd4dvar_subdomain_info(self._h, k, out))
        return dict(zip(SUB_FIELDS, list(out)))

    def sub_shape(self, k):
        s = self.subs[k]
        return (3, s["ey"], s["ex"])

    def split(self, flat):
        """View an "all subdomains" tensor as a list of [3][ey][ex] tensors."""
        out = []
        for k in range(self.nsub):
            n = int(np.prod(self.sub_shape(k)))
            out.append(flat[self.offsets[k]:self.offsets[k] + n].view(self.sub_shape(k)))
        return out

    def pack(self, arrays):
        """Concatenate per-subdomain arrays (numpy or torch) into an "all subdomains" device tensor."""
        flat = self.torch.zeros(self.ctot, dtype=self.torch.float64, device=self.device)
        for k, a in enumerate(arrays):
            t = self._dev(a).reshape(-1)
            flat[self.offsets[k]:self.offsets[k] + t.numel()] = t
        return flat

    @property
    def active_path(self):
        return self.lib.dd4dvar_active_path(self._h)

    @property
    def launch_count(self):
        return self.lib.dd4dvar_launch_count(self._h)

    # ---- problem data
    def set_background(self, xb, sigma_b):
        xb = self._dev(xb)
        sb = np.ascontiguousarray(sigma_b, dtype=np.float64)
        self._check("dd4dvar_set_background", self.lib.dd4dvar_set_background(self._h, xb.data_ptr(), _hd(sb)))

    def set_observations(self, obs):
        torch = self.torch
        lv = np.ascontiguousarray(obs.levels, dtype=np.int32)
        off = np.ascontiguousarray(obs.offsets, dtype=np.int64)
        so = np.ascontiguousarray(obs.sigma_o, dtype=np.float64)
        idx = torch.as_tensor(np.ascontiguousarray(obs.index, dtype=np.int32), device=self.device)
        val = self._dev(obs.value)
        total = int(off[-1]) if lv.size else 0
        nbytes = self.lib.dd4dvar_obs_workspace_bytes(self._h, total)
        self._obs_ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        base = (self._obs_ws.data_ptr() + 255) & ~255
        rc = self.lib.dd4dvar_set_observations(
            self._h, lv.size, lv.ctypes.data_as(C.POINTER(C.c_int)), off.ctypes.data_as(C.POINTER(C.c_longlong)),
            idx.data_ptr(), val.data_ptr(), _hd(so), base, nbytes)
        self._check("dd4dvar_set_observations", rc)

    # ---- the hot path and the driver
    def eval_local(self, controls, want_grad=True):
        """controls: "all subdomains" device tensor.  Returns (costs[nsub], parts[nsub][5], grads)."""
        torch = self.torch
        controls = self._dev(controls)
        costs = np.zeros(self.nsub); parts = np.zeros((self.nsub, 5))
        grads = torch.empty(self.ctot, dtype=torch.float64, device=self.device) if want_grad else None
        rc = self.lib.dd4dvar_eval_local(self._h, controls.data_ptr(), _hd(costs), _hd(parts),
                                         grads.data_ptr() if want_grad else None)
        self._check("dd4dvar_eval_local", rc)
        return costs, parts, grads

    def eval_local_host(self, h_controls, h_costs, h_grads=None):
        """End to end with host buffers (pinned torch CPU tensors or numpy arrays), copies inside."""
        def ptr(a):
            return a.data_ptr() if hasattr(a, "data_ptr") else a.ctypes.data
        rc = self.lib.dd4dvar_eval_local_host(self._h, ptr(h_controls), h_costs.ctypes.data_as(C.POINTER(C.c_double)),
                                              ptr(h_grads) if h_grads is not None else None)
        self._check("dd4dvar_eval_local_host", rc)

    def eval_global(self, x0, want_grad=True):
        torch = self.torch
        x0 = self._dev(x0)
        J = np.zeros(1)
        g = torch.empty(self.shape, dtype=torch.float64, device=self.device) if want_grad else None
        rc = self.lib.dd4dvar_eval_global(self._h, x0.data_ptr(), _hd(J), g.data_ptr() if want_grad else None)
        self._check("dd4dvar_eval_global", rc)
        return float(J[0]), g

    def sweep_async(self, mode=1):
        """0: forward + costs, 1: forward + costs + adjoint (the gradient sweep), 2: adjoint only."""
        self._check("dd4dvar_sweep_async", self.lib.dd4dvar_sweep_async(self._h, int(mode)))

    def run(self, outer_iters):
        torch = self.torch
        an = torch.empty(self.shape, dtype=torch.float64, device=self.device)
        hist = np.zeros((outer_iters + 1, 3))
        self._check("dd4dvar_run", self.lib.dd4dvar_run(self._h, outer_iters, an.data_ptr(), _hd(hist)))
        return an, hist

    def run_gn(self, outer_iters, n_gn=2, n_cg=5):
        """Algorithm 1 with the Gauss-Newton + CG local minimiser (Alg 5-7)."""
        torch = self.torch
        an = torch.empty(self.shape, dtype=torch.float64, device=self.device)
        hist = np.zeros((outer_iters + 1, 3))
        self._check("dd4dvar_run_gn", self.lib.dd4dvar_run_gn(self._h, outer_iters, int(n_gn), int(n_cg),
                                                              an.data_ptr(), _hd(hist)))
        return an, hist

    def gn_hessvec(self, controls, p):
        """H_GN p of every subdomain about `controls` (flat control layout; p and the result in w-space)."""
        torch = self.torch
        controls = self._dev(controls); p = self._dev(p)
        out = torch.empty(self.ctot, dtype=torch.float64, device=self.device)
        self._check("dd4dvar_gn_hessvec", self.lib.dd4dvar_gn_hessvec(self._h, controls.data_ptr(), p.data_ptr(),
                                                                      out.data_ptr()))
        return out

    # ---- sharded runs (one process per GPU owns a block of time windows; see parallel.py)
    def set_owned_windows(self, j0, j1):
        self._check("dd4dvar_set_owned_windows", self.lib.dd4dvar_set_owned_windows(self._h, int(j0), int(j1)))

    def exchange_view(self, which):
        """fp64 view (no copy) of an exchange buffer inside the workspace: 0 frozen controls, 1 predecessor end states."""
        ptr = C.c_void_p(); cnt = C.c_longlong()
        self._check("dd4dvar_exchange_buffer", self.lib.dd4dvar_exchange_buffer(self._h, int(which), C.byref(ptr), C.byref(cnt)))
        off = ptr.value - self._ws.data_ptr()
        assert off >= 0 and off % 8 == 0 and off + 8 * cnt.value <= self._ws.numel()
        return self._ws[off:off + 8 * cnt.value].view(self.torch.float64)

    def local_stats(self):
        J = np.zeros(self.nsub); dm = np.zeros(self.nsub)
        self._check("dd4dvar_get_local_stats", self.lib.dd4dvar_get_local_stats(self._h, _hd(J), _hd(dm)))
        return J, dm

    def gather_analysis(self):
        an = self.torch.empty(self.shape, dtype=self.torch.float64, device=self.device)
        self._check("dd4dvar_gather_analysis", self.lib.dd4dvar_gather_analysis(self._h, an.data_ptr()))
        return an

    def set_overlap_levels(self, on):
        """(25c) case 1 on every level of the window (generic kernels only; before set_background)."""
        self._check("dd4dvar_set_overlap_levels", self.lib.dd4dvar_set_overlap_levels(self._h, int(bool(on))))

    def set_phase_timing(self, on):
        """Record CUDA-event marks inside run(): phase_ms() then gives the device time of the last run per phase."""
        self._check("dd4dvar_set_phase_timing", self.lib.dd4dvar_set_phase_timing(self._h, int(bool(on))))

    def phase_ms(self):
        out = np.zeros(5)
        self._check("dd4dvar_get_phase_ms", self.lib.dd4dvar_get_phase_ms(self._h, _hd(out)))
        return dict(zip(("sweeps", "lbfgs", "exchange", "jglobal", "gather"), out.tolist()))

    def set_history_global(self, on):
        self._check("dd4dvar_set_history_global", self.lib.dd4dvar_set_history_global(self._h, int(bool(on))))

    def get_controls(self):
        torch = self.torch
        out = torch.empty(self.ctot, dtype=torch.float64, device=self.device)
        self._check("dd4dvar_get_controls", self.lib.dd4dvar_get_controls(self._h, out.data_ptr()))
        return out

    def get_trajectory(self, level):
        torch = self.torch
        out = torch.empty(self.shape, dtype=torch.float64, device=self.device)
        self._check("dd4dvar_get_trajectory", self.lib.dd4dvar_get_trajectory(self._h, level, out.data_ptr()))
        return out

    def get_local_trajectory(self, k):
        torch = self.torch
        s = self.subs[k]
        out = torch.empty((s["e"] - s["s"] + 1,) + self.sub_shape(k), dtype=torch.float64, device=self.device)
        self._check("dd4dvar_get_local_trajectory",
                    self.lib.dd4dvar_get_local_trajectory(self._h, k, out.data_ptr()))
        return out

    def forecast(self, x0, levels):
        """Model only: states at the given ascending levels, returned as a numpy array."""
        torch = self.torch
        x0 = self._dev(x0)
        lv = np.ascontiguousarray(levels, dtype=np.int32)
        out = torch.empty((lv.size,) + self.shape, dtype=torch.float64, device=self.device)
        rc = self.lib.dd4dvar_forecast(self._h, x0.data_ptr(), lv.size, lv.ctypes.data_as(C.POINTER(C.c_int)),
                                       out.data_ptr())
        self._check("dd4dvar_forecast", rc)
        return out.cpu().numpy()
