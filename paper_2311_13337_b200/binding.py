"""Thin Python binding of the C ABI in include/tvbx.h (argument marshalling only).

Every step of the hot path runs in the CUDA kernels of libtvbx.so; PyTorch is used only for device
buffers and streams.  There is no CPU fallback: importing works without a GPU (so the symbol table
can be checked), but any compute call fails with TvbxError(TVBX_ECUDA) when no device is present, and
loading fails loudly when the library has not been built.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_ROOT = os.path.dirname(_HERE)
LIB_PATH = os.path.join(_HERE, "libtvbx.so")
SRC_DIR = os.path.join(_HERE, "csrc")
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared"]

TVBX_OK, TVBX_EINVAL, TVBX_ENOMEM, TVBX_ECUDA, TVBX_ESTATE = 0, -1, -2, -3, -4
TVBX_F32, TVBX_F64 = 0, 1
TVBX_FC_AUTO, TVBX_FC_FP32, TVBX_FC_TF32 = 0, 1, 2   # tvbx_sweep_opts.fc_mode

# parameter ids (include/tvbx.h enum tvbx_param_id)
PARAM_IDS = dict(
    G=0, b_e=1, a_e=2, tau_w_e=3, v=4, wNoise=5, E_L_e=6, E_L_i=7, T=8, c_Fee=9, c_Fei=10, c_Fie=11,
    c_Fii=12, b_i=13, a_i=14, tau_w_i=15, g_L=16, C_m=17, Q_e=18, tau_e=19, E_e=20, Q_i=21, tau_i=22,
    E_i=23, N_tot=24, p_conn=25, g_inh=26, tau_OU=27, mu_OU=28, sigma_OU=29, muV0=30, dmuV0=31, sV0=32,
    dsV0=33, tauVN0=34, dtauVN0=35, eps_nu=36, muV_local=37, kappa=38)
P_POLY_E, P_POLY_I, N_PARAMS, N_SWEEPABLE = 39, 49, 59, 13


class TvbxError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"tvbx error {code}: {msg}")
        self.code = code


class ModelParams(C.Structure):
    _fields_ = [("p", C.c_double * N_PARAMS)]


class Axis(C.Structure):
    _fields_ = [("param_id", C.c_int32), ("n", C.c_int32), ("lo", C.c_double), ("hi", C.c_double),
                ("values", C.POINTER(C.c_double))]


class SweepOpts(C.Structure):
    _fields_ = [("precision", C.c_int32), ("sims_per_cta", C.c_int32), ("n_sims", C.c_int64),
                ("sim_ids", C.POINTER(C.c_int64)), ("chunk_samples", C.c_int64),
                ("threads_per_cta", C.c_int32), ("ctas_per_group", C.c_int32),
                ("fc_mode", C.c_int32), ("rate_stats_inhibitory", C.c_int32), ("rate_threshold_khz", C.c_double),
                ("latency_form", C.c_int32), ("reserved0", C.c_int32), ("updown_threshold_khz", C.c_double)]


class RunOpts(C.Structure):
    _fields_ = [("noise_on", C.c_int32), ("ds", C.c_int32), ("discard_steps", C.c_int64),
                ("traj", C.c_void_p), ("traj_steps", C.c_int64), ("traj_on_device", C.c_int32),
                ("reserved", C.c_int32), ("cuda_stream", C.c_void_p)]


EXPORTS = [
    "tvbx_default_params", "tvbx_create_connectome", "tvbx_destroy_connectome", "tvbx_sweep_create",
    "tvbx_sweep_destroy", "tvbx_sweep_set_initial", "tvbx_run", "tvbx_fc_readout", "tvbx_fc_scores", "tvbx_rate_stats",
    "tvbx_state_durations", "tvbx_top_k", "tvbx_sweep_size",
    "tvbx_sweep_param", "tvbx_sweep_ext_id", "tvbx_delay_index", "tvbx_ring_len", "tvbx_steps_done",
    "tvbx_samples_kept", "tvbx_sweep_state", "tvbx_launch_info", "tvbx_launch_count", "tvbx_kernel_name", "tvbx_fc_kernel_name", "tvbx_last_error",
    "tvbx_version", "tvbx_trim_memory", "tvbx_sweep_reset", "tvbx_profile_enable", "tvbx_profile_read", "tvbx_bytes_copied", "tvbx_diag_tf_closed2",
    "tvbx_top_k_noalloc",
]
NOALLOC_MAX_SCORES = 1 << 20        # include/tvbx_noalloc.h TVBX_NOALLOC_MAX_SCORES


def build(force: bool = False, verbose: bool = False, jobs: int = 0) -> str:
    """Compile csrc/*.cu for sm_100a into libtvbx.so (in-tree).  nvcc cross-compiles without a GPU.  Every .cu is its own
    translation unit (the integrator instances are spread over tvbx_k_*.cu), compiled in parallel into build/obj/*.o and
    linked; an object is rebuilt when its source or any header (csrc/*.h, *.cuh, include/*.h) is newer."""
    from concurrent.futures import ThreadPoolExecutor
    cus = sorted(f for f in os.listdir(SRC_DIR) if f.endswith(".cu"))
    hdrs = [os.path.join(SRC_DIR, f) for f in os.listdir(SRC_DIR) if f.endswith((".h", ".cuh"))]
    inc = os.path.join(_ROOT, "include")
    hdrs += [os.path.join(inc, f) for f in os.listdir(inc) if f.endswith(".h")]
    newest_hdr = max(os.path.getmtime(f) for f in hdrs)
    obj_dir = os.path.join(_ROOT, "build", "obj")
    os.makedirs(obj_dir, exist_ok=True)
    flags = [f for f in NVCC_FLAGS if f != "-shared"]
    todo, objs = [], []
    for f in cus:
        src, obj = os.path.join(SRC_DIR, f), os.path.join(obj_dir, f[:-3] + ".o")
        objs.append(obj)
        if force or not os.path.exists(obj) or os.path.getmtime(obj) < max(os.path.getmtime(src), newest_hdr):
            cmd = ["nvcc", *flags, "-c", "-o", obj, src]
            if verbose:
                cmd.insert(1, "-Xptxas=-v")
            todo.append(cmd)
    if todo:
        with ThreadPoolExecutor(max_workers=jobs or min(len(todo), os.cpu_count() or 4)) as ex:
            for r in ex.map(lambda c: subprocess.run(c, capture_output=True, text=True), todo):
                if verbose and r.stderr:
                    print(r.stderr)
                if r.returncode != 0:
                    raise RuntimeError("nvcc failed: " + " ".join(r.args) + "\n" + r.stdout + r.stderr)
    stale = [o for o in os.listdir(obj_dir) if os.path.join(obj_dir, o) not in objs]
    for o in stale:
        os.remove(os.path.join(obj_dir, o))
    if todo or stale or not os.path.exists(LIB_PATH) or os.path.getmtime(LIB_PATH) < max(os.path.getmtime(o) for o in objs):
        subprocess.check_call(["nvcc", "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB_PATH, *objs])
    return LIB_PATH


_lib = None


def lib():
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: run `python -c 'import __graft_entry__ as g; g.build()'` "
                              "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        vp, i32, i64, dbl = C.c_void_p, C.c_int32, C.c_int64, C.c_double
        dp, fp = C.POINTER(C.c_double), C.POINTER(C.c_float)
        sig = {
            "tvbx_default_params": [C.POINTER(ModelParams)],
            "tvbx_create_connectome": [i32, dp, dp, C.POINTER(vp)],
            "tvbx_destroy_connectome": [vp],
            "tvbx_sweep_create": [vp, C.POINTER(ModelParams), i32, C.POINTER(Axis), C.c_uint64,
                                  C.POINTER(SweepOpts), C.POINTER(vp)],
            "tvbx_sweep_destroy": [vp],
            "tvbx_sweep_set_initial": [vp, dp],
            "tvbx_run": [vp, i64, dbl, C.POINTER(RunOpts)],
            "tvbx_fc_readout": [vp, vp, vp, vp, i32, vp],
            "tvbx_fc_scores": [vp, vp, vp, vp, vp, i32, vp],
            "tvbx_rate_stats": [vp, vp, vp, vp, vp, vp, vp, i32, vp],
            "tvbx_state_durations": [vp, vp, vp, vp, vp, i32, vp],
            "tvbx_top_k": [vp, i32, vp, i32, C.POINTER(i64), fp, C.POINTER(i32), vp],
            "tvbx_sweep_size": [vp, C.POINTER(i64), C.POINTER(i64), C.POINTER(i32)],
            "tvbx_sweep_param": [vp, i64, i32, dp],
            "tvbx_sweep_ext_id": [vp, i64, C.POINTER(i64)],
            "tvbx_delay_index": [vp, i64, i32, i32, dbl, C.POINTER(i32)],
            "tvbx_ring_len": [vp, i64, dbl, C.POINTER(i32), C.POINTER(i32)],
            "tvbx_steps_done": [vp, C.POINTER(i64)],
            "tvbx_samples_kept": [vp, C.POINTER(i64)],
            "tvbx_sweep_state": [vp, dp, dp],
            "tvbx_launch_info": [vp, C.POINTER(i32)],
            "tvbx_launch_count": [vp, C.POINTER(i64)],
            "tvbx_kernel_name": [vp, C.c_char_p, i32],
            "tvbx_fc_kernel_name": [vp, C.c_char_p, i32],
            "tvbx_sweep_reset": [vp, vp],
            "tvbx_trim_memory": [C.POINTER(i64)],
            "tvbx_profile_enable": [vp, i32],
            "tvbx_profile_read": [vp, dp, C.POINTER(i64)],
            "tvbx_bytes_copied": [vp, C.POINTER(i64), C.POINTER(i64)],
            "tvbx_diag_tf_closed2": [C.POINTER(ModelParams), i32, dp, dp, dp, dp, dp],
            "tvbx_top_k_noalloc": [vp, i32, i32, vp, vp, vp],
        }
        for name, argtypes in sig.items():
            fn = getattr(L, name)
            fn.argtypes = argtypes
            fn.restype = i32
        L.tvbx_last_error.restype = C.c_char_p
        L.tvbx_version.restype = i32
        _lib = L
    return _lib


def _chk(rc):
    if rc != 0:
        raise TvbxError(rc, lib().tvbx_last_error().decode())


def _dptr(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def default_params() -> np.ndarray:
    m = ModelParams()
    _chk(lib().tvbx_default_params(C.byref(m)))
    return np.array(m.p[:], dtype=np.float64)


class Connectome:
    """tvbx_create_connectome / tvbx_destroy_connectome.  W[k, j] = weight of source j into target k."""

    def __init__(self, W, L_mm):
        W = np.ascontiguousarray(W, dtype=np.float64)
        L = np.ascontiguousarray(L_mm, dtype=np.float64)
        assert W.ndim == 2 and W.shape[0] == W.shape[1] and W.shape == L.shape
        self.n = W.shape[0]
        self._h = C.c_void_p()
        _chk(lib().tvbx_create_connectome(self.n, _dptr(W), _dptr(L), C.byref(self._h)))

    def close(self):
        if getattr(self, "_h", None):
            lib().tvbx_destroy_connectome(self._h)
            self._h = None

    __del__ = close


class Sweep:
    """tvbx_sweep_create ... tvbx_sweep_destroy.

    axes: list of dicts {name | param_id, lo, hi, n, values (optional list)} (workloads.config axes).
    params: optional full default vector (N_PARAMS float64, include/tvbx.h order) or dict of overrides.
    """

    def __init__(self, conn: Connectome, axes, seed=0, params=None, precision=TVBX_F32, sims_per_cta=0,
                 sim_ids=None, chunk_samples=0, threads_per_cta=0, init=None, ctas_per_group=0, fc_mode=0, rate_threshold_khz=0.0,
                 rate_stats_inhibitory=False, latency_form=0, updown_threshold_khz=0.0):
        L = lib()
        self.conn = conn
        m = ModelParams()
        _chk(L.tvbx_default_params(C.byref(m)))
        if params is not None:
            if isinstance(params, dict):
                for k, v in params.items():
                    if k == "poly_e":
                        m.p[P_POLY_E:P_POLY_E + 10] = list(map(float, v))
                    elif k == "poly_i":
                        m.p[P_POLY_I:P_POLY_I + 10] = list(map(float, v))
                    else:
                        m.p[PARAM_IDS[k]] = float(v)
            else:
                vec = np.asarray(params, dtype=np.float64)
                assert vec.shape == (N_PARAMS,)
                for i in range(N_PARAMS):
                    m.p[i] = float(vec[i])
        ax = (Axis * max(1, len(axes)))()
        keep = []
        for i, a in enumerate(axes):
            ax[i].param_id = a["param_id"] if "param_id" in a else PARAM_IDS[a["name"]]
            ax[i].n = int(a["n"]); ax[i].lo = float(a["lo"]); ax[i].hi = float(a["hi"])
            if a.get("values") is not None:
                arr = np.ascontiguousarray(a["values"], dtype=np.float64)
                keep.append(arr)
                ax[i].values = _dptr(arr)
        o = SweepOpts()
        o.precision = precision; o.sims_per_cta = sims_per_cta; o.chunk_samples = chunk_samples
        o.threads_per_cta = threads_per_cta; o.ctas_per_group = ctas_per_group; o.fc_mode = fc_mode; o.rate_threshold_khz = rate_threshold_khz; o.rate_stats_inhibitory = int(bool(rate_stats_inhibitory)); o.latency_form = int(latency_form)
        o.updown_threshold_khz = float(updown_threshold_khz)
        self.rate_stats_inhibitory = bool(rate_stats_inhibitory)
        if sim_ids is not None:
            ids = np.ascontiguousarray(sim_ids, dtype=np.int64)
            keep.append(ids)
            o.n_sims = ids.size
            o.sim_ids = ids.ctypes.data_as(C.POINTER(C.c_int64))
        self._h = C.c_void_p()
        _chk(L.tvbx_sweep_create(conn._h, C.byref(m), len(axes), ax, seed, C.byref(o), C.byref(self._h)))
        ns, gs, nr = C.c_int64(), C.c_int64(), C.c_int32()
        _chk(L.tvbx_sweep_size(self._h, C.byref(ns), C.byref(gs), C.byref(nr)))
        self.n_sims, self.grid_size, self.n_regions = ns.value, gs.value, nr.value
        self.precision = precision
        if init is not None:
            a = np.ascontiguousarray(init, dtype=np.float64)
            _chk(L.tvbx_sweep_set_initial(self._h, _dptr(a)))

    def close(self):
        if getattr(self, "_h", None):
            lib().tvbx_sweep_destroy(self._h)
            self._h = None

    __del__ = close

    # ---- tvbx_run --------------------------------------------------------------------------------
    def run(self, steps, dt=0.1, noise_on=False, ds=10, discard_steps=0, traj_steps=0, traj_device=False,
            stream=None):
        """Advance all sims.  Returns the trajectory of the first traj_steps steps of this call,
        [n_sims][traj_steps][7][N] (numpy on host, or a torch CUDA tensor if traj_device), else None."""
        o = RunOpts()
        o.noise_on = int(bool(noise_on)); o.ds = int(ds); o.discard_steps = int(discard_steps)
        o.cuda_stream = _stream_ptr(stream)
        traj = None
        if traj_steps > 0:
            traj_steps = min(int(traj_steps), int(steps))
            shape = (self.n_sims, traj_steps, 7, self.n_regions)
            if traj_device:
                import torch
                traj = torch.zeros(shape, device="cuda",
                                   dtype=torch.float64 if self.precision == TVBX_F64 else torch.float32)
                o.traj = traj.data_ptr(); o.traj_on_device = 1
            else:
                traj = np.zeros(shape, dtype=np.float64 if self.precision == TVBX_F64 else np.float32)
                o.traj = traj.ctypes.data
            o.traj_steps = traj_steps
        _chk(lib().tvbx_run(self._h, int(steps), float(dt), C.byref(o)))
        return traj

    # ---- tvbx_fc_readout -------------------------------------------------------------------------
    def fc_readout(self, device=False, stream=None, out=None):
        """-> (fc [S][N][N], mean_e [S][N], mean_i [S][N]) float32; numpy (host) or torch CUDA tensors.
        `out`: optional preallocated triple of the right kind."""
        S, N = self.n_sims, self.n_regions
        if device:
            import torch
            fc, me, mi = out if out is not None else (
                torch.empty((S, N, N), device="cuda", dtype=torch.float32),
                torch.empty((S, N), device="cuda", dtype=torch.float32),
                torch.empty((S, N), device="cuda", dtype=torch.float32))
            _chk(lib().tvbx_fc_readout(self._h, fc.data_ptr(), me.data_ptr(), mi.data_ptr(), 1, _stream_ptr(stream)))
        else:
            fc, me, mi = out if out is not None else (
                np.empty((S, N, N), np.float32), np.empty((S, N), np.float32), np.empty((S, N), np.float32))
            _chk(lib().tvbx_fc_readout(self._h, fc.ctypes.data, me.ctypes.data, mi.ctypes.data, 0, _stream_ptr(stream)))
        return fc, me, mi

    # ---- accessors ---------------------------------------------------------------------------------
    def param(self, sim, name_or_id):
        pid = name_or_id if isinstance(name_or_id, int) else PARAM_IDS[name_or_id]
        out = C.c_double()
        _chk(lib().tvbx_sweep_param(self._h, sim, pid, C.byref(out)))
        return out.value

    def ext_id(self, sim):
        out = C.c_int64()
        _chk(lib().tvbx_sweep_ext_id(self._h, sim, C.byref(out)))
        return out.value

    def delay_index(self, sim, k, j, dt=0.0):
        out = C.c_int32()
        _chk(lib().tvbx_delay_index(self._h, sim, k, j, dt, C.byref(out)))
        return out.value

    def ring_len(self, sim, dt=0.0):
        h, hp = C.c_int32(), C.c_int32()
        _chk(lib().tvbx_ring_len(self._h, sim, dt, C.byref(h), C.byref(hp)))
        return h.value, hp.value

    def steps_done(self):
        out = C.c_int64()
        _chk(lib().tvbx_steps_done(self._h, C.byref(out)))
        return out.value

    def samples_kept(self):
        out = C.c_int64()
        _chk(lib().tvbx_samples_kept(self._h, C.byref(out)))
        return out.value

    def state(self):
        """-> (y [S][7][N], ou [S][N]) float64 on host (synchronises)."""
        y = np.zeros((self.n_sims, 7, self.n_regions)); ou = np.zeros((self.n_sims, self.n_regions))
        _chk(lib().tvbx_sweep_state(self._h, _dptr(y), _dptr(ou)))
        return y, ou

    def launch_info(self):
        a = (C.c_int32 * 10)()
        _chk(lib().tvbx_launch_info(self._h, a))
        keys = ("ctas", "threads", "sims_per_cta", "regs", "smem", "passes", "chunk_samples", "local_bytes", "ctas_per_group", "latency_form")
        return dict(zip(keys, a[:]))

    def reset(self, stream=None):
        _chk(lib().tvbx_sweep_reset(self._h, _stream_ptr(stream)))

    def profile_enable(self, on=True):
        _chk(lib().tvbx_profile_enable(self._h, int(bool(on))))

    def profile_read(self):
        """-> {kernel class: (summed ms, launches)} since the last read (synchronises the events)."""
        ms = (C.c_double * 4)(); n = (C.c_int64 * 4)()
        _chk(lib().tvbx_profile_read(self._h, ms, n))
        return {k: (ms[i], n[i]) for i, k in enumerate(("integrate", "fc", "readout", "reset"))}

    def bytes_copied(self):
        a, b = C.c_int64(), C.c_int64()
        _chk(lib().tvbx_bytes_copied(self._h, C.byref(a), C.byref(b)))
        return a.value, b.value

    def fc_scores(self, ref_fc=None, device=False, stream=None):
        """tvbx_fc_scores -> dict(fcsc [S], mean_fc [S], fitness [S] if ref_fc is given) float32; numpy or torch CUDA."""
        S = self.n_sims
        ref = None if ref_fc is None else np.ascontiguousarray(ref_fc, dtype=np.float64)
        if ref is not None:
            assert ref.shape == (self.n_regions, self.n_regions)
        names = ["fcsc", "fitness", "mean_fc"] if ref is not None else ["fcsc", "mean_fc"]
        if device:
            import torch
            out = {k: torch.empty((S,), device="cuda", dtype=torch.float32) for k in names}
            ptr = {k: v.data_ptr() for k, v in out.items()}
        else:
            out = {k: np.empty((S,), np.float32) for k in names}
            ptr = {k: v.ctypes.data for k, v in out.items()}
        _chk(lib().tvbx_fc_scores(self._h, None if ref is None else ref.ctypes.data, ptr["fcsc"], ptr.get("fitness"),
                                  ptr["mean_fc"], 1 if device else 0, _stream_ptr(stream)))
        return out

    def rate_stats(self, device=False, stream=None):
        """tvbx_rate_stats -> (var_e, max_e float32 [S][N], n_above_e int32 [S][N]), followed by (var_i, max_i,
        n_above_i) if the sweep was created with rate_stats_inhibitory; numpy or torch CUDA."""
        S, N = self.n_sims, self.n_regions
        pops = 2 if self.rate_stats_inhibitory else 1
        if device:
            import torch
            out = []
            for _ in range(pops):
                out += [torch.empty((S, N), device="cuda", dtype=torch.float32), torch.empty((S, N), device="cuda", dtype=torch.float32),
                        torch.empty((S, N), device="cuda", dtype=torch.int32)]
            ptr = [t.data_ptr() for t in out]
        else:
            out = []
            for _ in range(pops):
                out += [np.empty((S, N), np.float32), np.empty((S, N), np.float32), np.empty((S, N), np.int32)]
            ptr = [a.ctypes.data for a in out]
        ptr += [None] * (6 - len(ptr))
        _chk(lib().tvbx_rate_stats(self._h, *ptr, 1 if device else 0, _stream_ptr(stream)))
        return tuple(out)

    def state_durations(self, device=False, stream=None):
        """tvbx_state_durations -> (n_up int32, mean_up_ms float32, n_down int32, mean_down_ms float32), each [S][N]."""
        S, N = self.n_sims, self.n_regions
        if device:
            import torch
            out = [torch.empty((S, N), device="cuda", dtype=d) for d in (torch.int32, torch.float32, torch.int32, torch.float32)]
            ptr = [t.data_ptr() for t in out]
        else:
            out = [np.empty((S, N), d) for d in (np.int32, np.float32, np.int32, np.float32)]
            ptr = [a.ctypes.data for a in out]
        _chk(lib().tvbx_state_durations(self._h, *ptr, 1 if device else 0, _stream_ptr(stream)))
        return tuple(out)

    def top_k(self, k, which="fcsc", ref_fc=None, stream=None):
        """tvbx_top_k -> (external sim ids int64 [n], scores float32 [n]), best first; which in fcsc / fitness / mean_fc."""
        ref = None if ref_fc is None else np.ascontiguousarray(ref_fc, dtype=np.float64)
        ids = np.zeros(k, np.int64); sc = np.zeros(k, np.float32); n = C.c_int32()
        _chk(lib().tvbx_top_k(self._h, {"fcsc": 0, "fitness": 1, "mean_fc": 2}[which], None if ref is None else ref.ctypes.data, int(k),
                              ids.ctypes.data_as(C.POINTER(C.c_int64)), sc.ctypes.data_as(C.POINTER(C.c_float)), C.byref(n), _stream_ptr(stream)))
        return ids[:n.value], sc[:n.value]

    def kernel_name(self):
        buf = C.create_string_buffer(64)
        _chk(lib().tvbx_kernel_name(self._h, buf, 64))
        return buf.value.decode()

    def fc_kernel_name(self):
        buf = C.create_string_buffer(64)
        _chk(lib().tvbx_fc_kernel_name(self._h, buf, 64))
        return buf.value.decode()

    def launch_count(self):
        out = C.c_int64()
        _chk(lib().tvbx_launch_count(self._h, C.byref(out)))
        return out.value


def _stream_ptr(stream):
    if stream is None:
        return None
    if isinstance(stream, int):
        return stream
    return stream.cuda_stream      # torch.cuda.Stream


def diag_tf_closed2(fe, fi, w_e, w_i, params=None):
    """tvbx_diag_tf_closed2: the product kernel's packed transfer function evaluated on the device (FP32) ->
    [n][2][7] float64: per point and population (e, i): F, F_e, F_i, F_ee, F_ei, F_ii (unscaled by kappa), mu_V."""
    fe, fi, w_e, w_i = (np.ascontiguousarray(x, dtype=np.float64) for x in (fe, fi, w_e, w_i))
    n = fe.size
    assert fi.size == n and w_e.size == n and w_i.size == n
    m = None
    if params is not None:
        m = ModelParams()
        _chk(lib().tvbx_default_params(C.byref(m)))
        for k, v in params.items():
            m.p[PARAM_IDS[k]] = float(v)
    out = np.zeros((n, 2, 7))
    _chk(lib().tvbx_diag_tf_closed2(C.byref(m) if m is not None else None, n, _dptr(fe), _dptr(fi), _dptr(w_e), _dptr(w_i), _dptr(out)))
    return out


def top_k_noalloc(scores, k, out_idx, out_val, stream=None):
    """tvbx_top_k_noalloc (include/tvbx_noalloc.h): the k largest of the float32 CUDA tensor `scores` [n], best first, ties to
    the lower index, written to the caller's CUDA tensors out_idx (int32) and out_val (float32), both of >= min(k, n)
    entries.  Allocates nothing and does not synchronise: one kernel on `stream`, scratch in a static device array of the
    library (n <= NOALLOC_MAX_SCORES; calls that overlap on the GPU race on it).  Returns min(k, n)."""
    import torch
    n = int(scores.numel())
    m = min(int(k), n)
    assert scores.is_cuda and scores.dtype == torch.float32 and scores.is_contiguous()
    assert out_idx.is_cuda and out_idx.dtype == torch.int32 and out_idx.is_contiguous() and out_idx.numel() >= m
    assert out_val.is_cuda and out_val.dtype == torch.float32 and out_val.is_contiguous() and out_val.numel() >= m
    _chk(lib().tvbx_top_k_noalloc(scores.data_ptr(), n, int(k), out_idx.data_ptr(), out_val.data_ptr(), _stream_ptr(stream)))
    return m


def trim_memory() -> int:
    """tvbx_trim_memory: return the library's cached device buffers to the driver; bytes freed."""
    out = C.c_int64()
    _chk(lib().tvbx_trim_memory(C.byref(out)))
    return out.value


def sweep_from_config(cfg: dict, W, L_mm, **kw):
    """Convenience: (Connectome, Sweep) for a workloads.config() dict."""
    conn = Connectome(W, L_mm)
    params = dict(cfg.get("fixed", {}))
    params.update(kw.pop("params", {}) or {})
    sw = Sweep(conn, cfg["axes"], seed=kw.pop("seed", cfg["seed"]), params=params, **kw)
    return conn, sw
