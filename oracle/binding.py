"""ctypes binding of oracle/oracle.cpp (TEST INFRASTRUCTURE, not the product).

``build_oracle()`` compiles ``liboracle.so`` next to the source with g++;
``Oracle`` wraps one chain with numpy host arrays.  See oracle.cpp for the
citations of every step.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "oracle.cpp"
_LIB = _HERE / "liboracle.so"
_CXXFLAGS = ["-O3", "-mavx2", "-mfma", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-std=c++17"]

_lib = None


def build_oracle(force: bool = False) -> Path:
    """Compile the oracle if the shared object is missing or older than its source."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        tmp = _LIB.with_suffix(f".so.tmp{os.getpid()}")
        subprocess.run(["g++", *_CXXFLAGS, "-o", str(tmp), str(_SRC)], check=True)
        os.replace(tmp, _LIB)
    return _LIB


class _Stats(C.Structure):
    _fields_ = [("accepted", C.c_uint64), ("veto_overlap", C.c_uint64), ("veto_wall", C.c_uint64),
                ("near_ties", C.c_uint64), ("E_running", C.c_double)]


def load_oracle():
    global _lib
    if _lib is not None:
        return _lib
    build_oracle()
    try:
        lib = C.CDLL(str(_LIB))
    except OSError:
        build_oracle(force=True)
        lib = C.CDLL(str(_LIB))
    dp, u8p, u32p, u64p, vp = (C.POINTER(C.c_double), C.POINTER(C.c_uint8), C.POINTER(C.c_uint32),
                               C.POINTER(C.c_uint64), C.c_void_p)
    lib.oracle_philox4x32_10.argtypes = [u32p, u32p, u32p]
    lib.oracle_philox4x32_10.restype = None
    lib.oracle_uniform_open01.argtypes = [C.c_uint32, C.c_uint32]
    lib.oracle_uniform_open01.restype = C.c_double
    lib.oracle_init.argtypes = [C.POINTER(vp), C.c_int64, dp, dp, dp, C.c_double, C.c_double,
                                C.c_double, C.c_uint64, C.c_int]
    lib.oracle_free.argtypes = [vp]
    lib.oracle_free.restype = None
    lib.oracle_set_threads.argtypes = [vp, C.c_int]
    lib.oracle_sweep.argtypes = [vp, C.c_int64]
    lib.oracle_partial_sweep.argtypes = [vp, C.c_int64, C.c_int64]
    lib.oracle_set_position_bits.argtypes = [vp, C.c_int]
    lib.oracle_energy.argtypes = [vp, dp]
    lib.oracle_pair_hist.argtypes = [vp, C.c_double, C.c_int, C.c_double, u64p, u64p]
    lib.oracle_get_positions.argtypes = [vp, dp]
    lib.oracle_set_positions.argtypes = [vp, dp]
    lib.oracle_get_sweep_index.argtypes = [vp, u64p]
    lib.oracle_set_sweep_index.argtypes = [vp, C.c_uint64]
    lib.oracle_get_stats.argtypes = [vp, C.POINTER(_Stats)]
    lib.oracle_get_trial_log.argtypes = [vp, dp, u8p, dp, dp, dp]
    _lib = lib
    return lib


def _dp(a: np.ndarray):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def philox4x32_10(ctr, key):
    lib = load_oracle()
    c = (C.c_uint32 * 4)(*[int(v) & 0xFFFFFFFF for v in ctr])
    k = (C.c_uint32 * 2)(*[int(v) & 0xFFFFFFFF for v in key])
    o = (C.c_uint32 * 4)()
    lib.oracle_philox4x32_10(c, k, o)
    return tuple(int(v) for v in o)


def uniform_open01(lo: int, hi: int) -> float:
    return float(load_oracle().oracle_uniform_open01(lo & 0xFFFFFFFF, hi & 0xFFFFFFFF))


class OracleError(RuntimeError):
    def __init__(self, code):
        super().__init__({-1: "EINVAL", -2: "EOVERLAP", -3: "EOUTSIDE"}.get(code, str(code)))
        self.code = code


class Oracle:
    """One serial Metropolis chain on the host. ``pos`` is [3, N] float64."""

    def __init__(self, pos, charges, diameters, cavity_R, bjerrum_length, max_disp, seed,
                 validate=True, threads=1):
        self._lib = load_oracle()
        pos = np.ascontiguousarray(pos, dtype=np.float64)
        q = np.ascontiguousarray(charges, dtype=np.float64)
        d = np.ascontiguousarray(diameters, dtype=np.float64)
        assert pos.ndim == 2 and pos.shape[0] == 3
        self.N = pos.shape[1]
        assert q.shape == (self.N,) and d.shape == (self.N,)
        self._h = C.c_void_p()
        rc = self._lib.oracle_init(C.byref(self._h), self.N, _dp(pos), _dp(q), _dp(d), cavity_R,
                                   bjerrum_length, max_disp, seed, 1 if validate else 0)
        if rc != 0:
            self._h = None
            raise OracleError(rc)
        if threads != 1:
            self.set_threads(threads)

    def __del__(self):
        if getattr(self, "_h", None):
            self._lib.oracle_free(self._h)
            self._h = None

    def _ck(self, rc):
        if rc != 0:
            raise OracleError(rc)

    def set_threads(self, n):
        self._ck(self._lib.oracle_set_threads(self._h, int(n)))

    def set_position_bits(self, bits):
        """32: positions are held as FP32 values, arithmetic stays FP64; 64: the default."""
        self._ck(self._lib.oracle_set_position_bits(self._h, int(bits)))

    def sweep(self, n=1):
        self._ck(self._lib.oracle_sweep(self._h, int(n)))

    def partial_sweep(self, first, count):
        self._ck(self._lib.oracle_partial_sweep(self._h, int(first), int(count)))

    def energy(self) -> float:
        e = C.c_double()
        self._ck(self._lib.oracle_energy(self._h, C.byref(e)))
        return e.value

    def pair_hist(self, bin_width, nbins, centre_rmax, hist=None, n_centres=None):
        if hist is None:
            hist = np.zeros((2, 2, nbins), dtype=np.uint64)
        if n_centres is None:
            n_centres = np.zeros(2, dtype=np.uint64)
        self._ck(self._lib.oracle_pair_hist(self._h, bin_width, nbins, centre_rmax,
                                            hist.ctypes.data_as(C.POINTER(C.c_uint64)),
                                            n_centres.ctypes.data_as(C.POINTER(C.c_uint64))))
        return hist, n_centres

    @property
    def positions(self) -> np.ndarray:
        out = np.empty((3, self.N), dtype=np.float64)
        self._ck(self._lib.oracle_get_positions(self._h, _dp(out)))
        return out

    @positions.setter
    def positions(self, pos):
        pos = np.ascontiguousarray(pos, dtype=np.float64)
        assert pos.shape == (3, self.N)
        self._ck(self._lib.oracle_set_positions(self._h, _dp(pos)))

    @property
    def sweep_index(self) -> int:
        s = C.c_uint64()
        self._ck(self._lib.oracle_get_sweep_index(self._h, C.byref(s)))
        return s.value

    @sweep_index.setter
    def sweep_index(self, s):
        self._ck(self._lib.oracle_set_sweep_index(self._h, int(s)))

    def stats(self) -> dict:
        st = _Stats()
        self._ck(self._lib.oracle_get_stats(self._h, C.byref(st)))
        return {"accepted": st.accepted, "veto_overlap": st.veto_overlap, "veto_wall": st.veto_wall,
                "near_ties": st.near_ties, "E_running": st.E_running}

    def trial_log(self) -> dict:
        N = self.N
        dE = np.empty(N); scale = np.empty(N); t = np.empty(N); trial = np.empty((3, N))
        flags = np.empty(N, dtype=np.uint8)
        self._ck(self._lib.oracle_get_trial_log(self._h, _dp(dE), flags.ctypes.data_as(C.POINTER(C.c_uint8)),
                                                _dp(scale), _dp(t), _dp(trial)))
        return {"dE": dE, "flags": flags, "scale": scale, "t": t, "trial": trial}
