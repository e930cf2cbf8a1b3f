"""ctypes wrapper around oracle/tvb_adex_oracle.cpp  --  TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs import this.
It never imports the CUDA package and the CUDA package never imports it.  Marshalling only; all
arithmetic is in the C++ file.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "tvb_adex_oracle.cpp")
_LIB = os.path.join(_HERE, "liboracle.so")

# -ffp-contract=off: no FMA contraction, so the FP64 arithmetic is the plain IEEE sequence written
# in the source; -O2, no fast-math.
_CXXFLAGS = ["-O2", "-std=c++17", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off"]


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["g++", *_CXXFLAGS, "-o", _LIB, _SRC])
    return _LIB


_dp = C.POINTER(C.c_double)


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.orc_num_params.restype = C.c_int
        L.orc_axis_value.restype = C.c_double
        L.orc_axis_value.argtypes = [C.c_double, C.c_double, C.c_int, C.c_int]
        L.orc_grid_digits.argtypes = [C.c_int, C.POINTER(C.c_int), C.c_longlong, C.POINTER(C.c_int)]
        L.orc_delay_index.restype = C.c_int
        L.orc_delay_index.argtypes = [C.c_double, C.c_double, C.c_double]
        L.orc_philox4x32_10.argtypes = [C.POINTER(C.c_uint), C.POINTER(C.c_uint), C.POINTER(C.c_uint)]
        L.orc_uniform23.restype = C.c_double
        L.orc_uniform23.argtypes = [C.c_uint]
        L.orc_normal.restype = C.c_double
        L.orc_normal.argtypes = [C.c_ulonglong, C.c_longlong, C.c_int, C.c_longlong]
        L.orc_tf.argtypes = [_dp, C.c_int, C.c_double, C.c_double, C.c_double, _dp, _dp]
        L.orc_create.restype = C.c_void_p
        L.orc_create.argtypes = [C.c_int, _dp, _dp, C.c_longlong, _dp, C.POINTER(C.c_longlong),
                                 C.c_ulonglong]
        L.orc_destroy.argtypes = [C.c_void_p]
        L.orc_set_initial.argtypes = [C.c_void_p, _dp]
        L.orc_set_unwrapped_history.argtypes = [C.c_void_p, C.c_int]
        L.orc_run.argtypes = [C.c_void_p, C.c_longlong, C.c_double, C.c_int, C.c_int, C.c_longlong,
                              _dp, C.c_longlong, C.c_int]
        L.orc_num_samples.restype = C.c_longlong
        L.orc_num_samples.argtypes = [C.c_void_p]
        L.orc_samples.argtypes = [C.c_void_p, C.c_longlong, _dp, _dp]
        L.orc_state.argtypes = [C.c_void_p, C.c_longlong, _dp, _dp]
        L.orc_ring_len.restype = C.c_int
        L.orc_ring_len.argtypes = [C.c_void_p, C.c_longlong]
        L.orc_steps_done.restype = C.c_longlong
        L.orc_steps_done.argtypes = [C.c_void_p]
        L.orc_fc_readout.argtypes = [C.c_void_p, _dp, _dp, _dp]
        L.orc_max_threads.restype = C.c_int
        _lib = L
    return _lib


def _p(a):
    return a.ctypes.data_as(_dp) if a is not None else None


# ------------------------------------------------------------------ scalar helpers
def axis_value(lo, hi, n, i):
    return lib().orc_axis_value(lo, hi, n, i)


def grid_digits(n_per_axis, s):
    n = len(n_per_axis)
    a = (C.c_int * n)(*n_per_axis)
    d = (C.c_int * n)()
    lib().orc_grid_digits(n, a, s, d)
    return list(d)


def delay_index(L_mm, v, dt):
    return lib().orc_delay_index(L_mm, v, dt)


def philox4x32_10(ctr, key):
    c = (C.c_uint * 4)(*ctr)
    k = (C.c_uint * 2)(*key)
    o = (C.c_uint * 4)()
    lib().orc_philox4x32_10(c, k, o)
    return tuple(int(x) for x in o)


def uniform23(x):
    return lib().orc_uniform23(x)


def normal(seed, sim, region, step):
    return lib().orc_normal(seed, sim, region, step)


def tf(params, pop, x_e, x_i, W):
    """-> (array of 6: F, F_e, F_i, F_ee, F_ei, F_ii ; mu_V)"""
    params = np.ascontiguousarray(params, dtype=np.float64)
    out = np.zeros(6)
    mu = C.c_double()
    lib().orc_tf(_p(params), pop, x_e, x_i, W, _p(out), C.byref(mu))
    return out, mu.value


# ------------------------------------------------------------------ the sweep object
class OracleSweep:
    """S independent simulations on one connectome.  params: [S][NP] float64 (workloads order)."""

    def __init__(self, W, L_mm, params, seed=0, ext_ids=None, init=None, unwrapped=False):
        L = lib()
        self.W = np.ascontiguousarray(W, dtype=np.float64)
        self.L = np.ascontiguousarray(L_mm, dtype=np.float64)
        self.params = np.ascontiguousarray(np.atleast_2d(params), dtype=np.float64)
        assert self.params.shape[1] == L.orc_num_params()
        self.N = self.W.shape[0]
        self.S = self.params.shape[0]
        ids = None
        if ext_ids is not None:
            ids = np.ascontiguousarray(ext_ids, dtype=np.int64)
            assert ids.shape == (self.S,)
        self._h = L.orc_create(self.N, _p(self.W), _p(self.L), self.S, _p(self.params),
                               ids.ctypes.data_as(C.POINTER(C.c_longlong)) if ids is not None else None,
                               seed)
        if not self._h:
            raise MemoryError("orc_create failed")
        if init is not None:
            a = np.ascontiguousarray(init, dtype=np.float64)
            assert L.orc_set_initial(self._h, _p(a)) == 0
        if unwrapped:
            assert L.orc_set_unwrapped_history(self._h, 1) == 0

    def close(self):
        if self._h:
            lib().orc_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def run(self, steps, dt=0.1, noise_on=False, ds=10, discard_steps=0, traj_steps=0, n_threads=0):
        """Advance all sims; returns the trajectory [S][traj_steps][7][N] (float64) or None."""
        traj = None
        if traj_steps > 0:
            traj_steps = min(traj_steps, steps)
            traj = np.zeros((self.S, traj_steps, 7, self.N))
        rc = lib().orc_run(self._h, steps, dt, int(bool(noise_on)), ds, discard_steps, _p(traj),
                           traj_steps, n_threads)
        if rc != 0:
            raise ValueError(f"orc_run rc={rc}")
        return traj

    def samples(self, s):
        ns = lib().orc_num_samples(self._h)
        xe = np.zeros((ns, self.N)); xi = np.zeros((ns, self.N))
        lib().orc_samples(self._h, s, _p(xe), _p(xi))
        return xe, xi

    def state(self, s):
        y = np.zeros((7, self.N)); ou = np.zeros(self.N)
        lib().orc_state(self._h, s, _p(y), _p(ou))
        return y, ou

    def ring_len(self, s):
        return lib().orc_ring_len(self._h, s)

    def steps_done(self):
        return lib().orc_steps_done(self._h)

    def fc_readout(self):
        fc = np.zeros((self.S, self.N, self.N)); me = np.zeros((self.S, self.N)); mi = np.zeros((self.S, self.N))
        rc = lib().orc_fc_readout(self._h, _p(fc), _p(me), _p(mi))
        if rc != 0:
            raise RuntimeError(f"orc_fc_readout rc={rc}")
        return fc, me, mi


def max_threads():
    return lib().orc_max_threads()
