"""Thin Python binding of libmcb200.so (include/mcb200.h): argument marshalling only.

PyTorch is used for device memory and streams; every step of the hot path runs in the CUDA
kernels of csrc/.  There is no CPU fallback: if the shared library is missing or the device is
not a B200-class GPU, the calls raise.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

import numpy as np
import torch

_PKG = Path(__file__).resolve().parent
_LIBPATH = _PKG / "libmcb200.so"

MC_OK, MC_EINVAL, MC_EOVERLAP, MC_EOUTSIDE, MC_ENOSPACE, MC_ECUDA, MC_ESTALL = 0, -1, -2, -3, -4, -5, -6
_CODES = {-1: "MC_EINVAL", -2: "MC_EOVERLAP", -3: "MC_EOUTSIDE", -4: "MC_ENOSPACE", -5: "MC_ECUDA", -6: "MC_ESTALL"}

EXPORTS = (
    "mc_workspace_bytes", "mc_init", "mc_sweep", "mc_energy", "mc_energy_dev", "mc_energy_noalloc", "mc_pair_hist", "mc_sweep_host",
    "mc_sweep_timed", "mc_sweep_reduction",
    "mc_get_positions", "mc_set_positions", "mc_set_state", "mc_get_sweep_index", "mc_set_sweep_index", "mc_get_stats",
    "mc_get_trial_log", "mc_free", "mc_last_error", "mc_measure_fp64_peak", "mc_set_option", "mc_get_option",
    "mc_debug_counters", "mc_debug_peek", "mc_plan_check",
    "mc_get_launch_count",
)


class MCError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"{_CODES.get(code, code)}: {msg}")
        self.code = code


class mc_stats(C.Structure):
    _fields_ = [("accepted", C.c_uint64), ("veto_overlap", C.c_uint64), ("veto_wall", C.c_uint64),
                ("near_ties", C.c_uint64), ("E_running", C.c_double)]


_lib = None


def load_library() -> C.CDLL:
    """dlopen libmcb200.so (built by paper_1602_05716_b200.build); raises if it is not there."""
    global _lib
    if _lib is not None:
        return _lib
    if not _LIBPATH.exists():
        raise ImportError(f"{_LIBPATH} is missing: build it with `python -m paper_1602_05716_b200.build` "
                          "(there is no CPU fallback)")
    lib = C.CDLL(str(_LIBPATH))
    vp, i64, u64, dbl = C.c_void_p, C.c_int64, C.c_uint64, C.c_double
    lib.mc_workspace_bytes.argtypes = [i64]; lib.mc_workspace_bytes.restype = C.c_size_t
    lib.mc_init.argtypes = [C.POINTER(vp), i64, vp, vp, vp, dbl, dbl, dbl, u64, vp, C.c_size_t, vp, C.c_int]
    lib.mc_sweep.argtypes = [vp, i64]
    lib.mc_sweep_reduction.argtypes = [vp, i64]
    lib.mc_energy.argtypes = [vp, C.POINTER(dbl)]
    lib.mc_energy_dev.argtypes = [vp, vp]
    lib.mc_energy_noalloc.argtypes = [i64, vp, vp, dbl, vp, vp]
    lib.mc_sweep_timed.argtypes = [vp, i64, C.POINTER(dbl)]
    lib.mc_pair_hist.argtypes = [vp, dbl, C.c_int, dbl, vp, vp]
    lib.mc_sweep_host.argtypes = [vp, i64, vp, C.POINTER(dbl), vp, C.POINTER(mc_stats)]
    lib.mc_get_positions.argtypes = [vp, vp]
    lib.mc_set_positions.argtypes = [vp, vp]
    lib.mc_set_state.argtypes = [vp, vp, u64, dbl]
    lib.mc_get_sweep_index.argtypes = [vp, C.POINTER(u64)]
    lib.mc_set_sweep_index.argtypes = [vp, u64]
    lib.mc_get_stats.argtypes = [vp, C.POINTER(mc_stats)]
    lib.mc_get_trial_log.argtypes = [vp, vp, vp]
    lib.mc_free.argtypes = [vp]
    lib.mc_last_error.argtypes = []; lib.mc_last_error.restype = C.c_char_p
    lib.mc_measure_fp64_peak.argtypes = [vp, dbl, C.POINTER(dbl)]
    lib.mc_set_option.argtypes = [vp, C.c_char_p, i64]
    lib.mc_get_option.argtypes = [vp, C.c_char_p, C.POINTER(i64)]
    lib.mc_get_launch_count.argtypes = [vp, C.POINTER(u64)]
    lib.mc_debug_counters.argtypes = [vp, C.POINTER(C.c_int64)]
    lib.mc_debug_peek.argtypes = [vp, C.POINTER(C.c_int32), C.c_int]
    lib.mc_plan_check.argtypes = [i64, C.c_int, C.c_int, C.c_int, C.POINTER(C.c_int64)]
    for name in EXPORTS:
        if name not in ("mc_workspace_bytes", "mc_last_error"):
            getattr(lib, name).restype = C.c_int
    _lib = lib
    return lib


def _check(rc: int):
    if rc != MC_OK:
        raise MCError(rc, (load_library().mc_last_error() or b"").decode())


def _dev_f64(t, shape, device):
    t = torch.as_tensor(t, dtype=torch.float64)
    t = t.to(device).contiguous()
    assert tuple(t.shape) == tuple(shape), (tuple(t.shape), tuple(shape))
    return t


# ---- functions with the C ABI's names ----------------------------------------------------------
def mc_workspace_bytes(N: int) -> int:
    return int(load_library().mc_workspace_bytes(int(N)))


def mc_plan_check(N: int, rows_per_thread: int, far_cols: int, far_workers: int) -> dict:
    """Host-only check that the persistent kernel's items cover every column exactly once per chunk."""
    out = (C.c_int64 * 4)()
    _check(load_library().mc_plan_check(int(N), int(rows_per_thread), int(far_cols), int(far_workers), out))
    return {"items": out[0], "violations": out[1], "max_item_cols": out[2], "urgent": out[3]}


def mc_measure_fp64_peak(millis: float = 50.0) -> float:
    """Thread-level FP64 FMA instructions per second sustained by a register-resident loop."""
    out = C.c_double()
    _check(load_library().mc_measure_fp64_peak(C.c_void_p(torch.cuda.current_stream().cuda_stream), millis,
                                               C.byref(out)))
    return out.value


def mc_energy_noalloc(pos: torch.Tensor, charges: torch.Tensor, bjerrum_length: float, out: torch.Tensor) -> torch.Tensor:
    """From-scratch energy of the configuration ``pos`` ([3][N], CUDA float64) with ``charges`` ([N]) into ``out``
    (CUDA float64, one element) on the current stream; allocates nothing (include/mcb200.h: mc_energy_noalloc)."""
    for t in (pos, charges, out):
        assert t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()
    N = charges.numel()
    assert tuple(pos.shape) == (3, N) and out.numel() >= 1
    with torch.cuda.device(pos.device):
        _check(load_library().mc_energy_noalloc(int(N), pos.data_ptr(), charges.data_ptr(), float(bjerrum_length),
                                                out.data_ptr(), C.c_void_p(torch.cuda.current_stream().cuda_stream)))
    return out


class MCSystem:
    """One Markov chain on the current CUDA device (wraps an ``mc_handle``)."""

    def __init__(self, pos, charges, diameters, cavity_R, bjerrum_length, max_disp, seed, validate=True,
                 device=None):
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1602_05716_b200 needs a CUDA device (B200); there is no CPU fallback")
        self._lib = load_library()
        self.device = torch.device(device if device is not None else f"cuda:{torch.cuda.current_device()}")
        pos_np_shape = tuple(pos.shape)
        assert len(pos_np_shape) == 2 and pos_np_shape[0] == 3, "pos must be [3, N]"
        self.N = int(pos_np_shape[1])
        with torch.cuda.device(self.device):
            p = _dev_f64(pos, (3, self.N), self.device)
            q = _dev_f64(charges, (self.N,), self.device)
            d = _dev_f64(diameters, (self.N,), self.device)
            nbytes = mc_workspace_bytes(self.N)
            self._ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            base = self._ws.data_ptr()
            self._ws_ptr = (base + 255) // 256 * 256
            self._stream = torch.cuda.current_stream(self.device)
            self._h = C.c_void_p()
            rc = self._lib.mc_init(C.byref(self._h), self.N, p.data_ptr(), q.data_ptr(), d.data_ptr(),
                                   float(cavity_R), float(bjerrum_length), float(max_disp), int(seed),
                                   self._ws_ptr, nbytes, C.c_void_p(self._stream.cuda_stream), 1 if validate else 0)
        if rc != MC_OK:
            self._h = None
            _check(rc)

    # -- lifetime --
    def close(self):
        if getattr(self, "_h", None):
            self._lib.mc_free(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- the hot path --
    def mc_sweep(self, n: int = 1):
        _check(self._lib.mc_sweep(self._h, int(n)))

    sweep = mc_sweep

    def mc_sweep_reduction(self, n: int = 1):
        """The paper's comparison code: the same chain, one kernel launch per trial."""
        _check(self._lib.mc_sweep_reduction(self._h, int(n)))

    def mc_energy(self) -> float:
        e = C.c_double()
        _check(self._lib.mc_energy(self._h, C.byref(e)))
        return e.value

    energy = mc_energy

    def mc_energy_dev(self, out=None) -> torch.Tensor:
        if out is None:
            out = torch.empty(1, dtype=torch.float64, device=self.device)
        assert out.is_cuda and out.dtype == torch.float64 and out.numel() >= 1
        _check(self._lib.mc_energy_dev(self._h, out.data_ptr()))
        return out

    def mc_sweep_timed(self, n: int = 1) -> float:
        """mc_sweep(n) as one launch of k_sweep with an event pair around it: its device time in ms."""
        ms = C.c_double()
        _check(self._lib.mc_sweep_timed(self._h, int(n), C.byref(ms)))
        return ms.value

    def mc_pair_hist(self, bin_width, nbins, centre_rmax, hist=None, n_centres=None):
        if hist is None:
            hist = torch.zeros((2, 2, nbins), dtype=torch.int64, device=self.device)
        if n_centres is None:
            n_centres = torch.zeros(2, dtype=torch.int64, device=self.device)
        assert hist.is_cuda and hist.is_contiguous() and hist.numel() == 4 * nbins and hist.element_size() == 8
        assert n_centres.is_cuda and n_centres.numel() == 2 and n_centres.element_size() == 8
        _check(self._lib.mc_pair_hist(self._h, float(bin_width), int(nbins), float(centre_rmax), hist.data_ptr(),
                                      n_centres.data_ptr()))
        return hist, n_centres

    pair_hist = mc_pair_hist

    def mc_sweep_host(self, n, pos_in=None, pos_out=None, E_running_in=None):
        """n sweeps through pinned host tensors; returns (pos_out, stats dict).  ``E_running_in``: the running
        energy that belongs to ``pos_in`` (taken on trust: no from-scratch pass), or None to recompute it."""
        st = mc_stats()
        if pos_in is not None:
            assert not pos_in.is_cuda and pos_in.dtype == torch.float64 and pos_in.is_contiguous()
            assert tuple(pos_in.shape) == (3, self.N)
        if pos_out is not None:
            assert not pos_out.is_cuda and pos_out.dtype == torch.float64 and pos_out.is_contiguous()
            assert tuple(pos_out.shape) == (3, self.N)
        e_in = C.byref(C.c_double(float(E_running_in))) if E_running_in is not None else None
        _check(self._lib.mc_sweep_host(self._h, int(n), pos_in.data_ptr() if pos_in is not None else None, e_in,
                                       pos_out.data_ptr() if pos_out is not None else None, C.byref(st)))
        return pos_out, _stats_dict(st)

    # -- accessors --
    def mc_get_positions(self) -> torch.Tensor:
        out = torch.empty((3, self.N), dtype=torch.float64, device=self.device)
        _check(self._lib.mc_get_positions(self._h, out.data_ptr()))
        return out

    def mc_set_positions(self, pos):
        p = _dev_f64(pos, (3, self.N), self.device)
        _check(self._lib.mc_set_positions(self._h, p.data_ptr()))
        self._keep = p  # keep alive until the stream has consumed it

    def mc_set_state(self, pos, sweep_index: int, E_running: float):
        p = _dev_f64(pos, (3, self.N), self.device)
        _check(self._lib.mc_set_state(self._h, p.data_ptr(), int(sweep_index), float(E_running)))
        self._keep = p

    @property
    def positions(self) -> np.ndarray:
        return self.mc_get_positions().cpu().numpy()

    @positions.setter
    def positions(self, pos):
        self.mc_set_positions(pos)

    @property
    def sweep_index(self) -> int:
        s = C.c_uint64()
        _check(self._lib.mc_get_sweep_index(self._h, C.byref(s)))
        return s.value

    @sweep_index.setter
    def sweep_index(self, s: int):
        _check(self._lib.mc_set_sweep_index(self._h, int(s)))

    def mc_get_stats(self) -> dict:
        st = mc_stats()
        _check(self._lib.mc_get_stats(self._h, C.byref(st)))
        return _stats_dict(st)

    stats = mc_get_stats

    def mc_get_trial_log(self) -> dict:
        dE = torch.empty(self.N, dtype=torch.float64, device=self.device)
        flags = torch.empty(self.N, dtype=torch.uint8, device=self.device)
        _check(self._lib.mc_get_trial_log(self._h, dE.data_ptr(), flags.data_ptr()))
        return {"dE": dE.cpu().numpy(), "flags": flags.cpu().numpy()}

    trial_log = mc_get_trial_log

    def mc_set_option(self, key: str, value: int):
        _check(self._lib.mc_set_option(self._h, key.encode(), int(value)))

    def mc_get_option(self, key: str) -> int:
        v = C.c_int64()
        _check(self._lib.mc_get_option(self._h, key.encode(), C.byref(v)))
        return v.value

    def mc_debug_counters(self) -> list:
        out = (C.c_int64 * 16)()
        _check(self._lib.mc_debug_counters(self._h, out))
        return list(out)

    def mc_debug_peek(self, n: int) -> list:
        out = (C.c_int32 * abs(n))()
        _check(self._lib.mc_debug_peek(self._h, out, n))
        return list(out)

    def mc_get_launch_count(self) -> int:
        n = C.c_uint64()
        _check(self._lib.mc_get_launch_count(self._h, C.byref(n)))
        return n.value

    def synchronize(self):
        self._stream.synchronize()


def _stats_dict(st: mc_stats) -> dict:
    return {"accepted": st.accepted, "veto_overlap": st.veto_overlap, "veto_wall": st.veto_wall,
            "near_ties": st.near_ties, "E_running": st.E_running}


def mc_init(pos, charges, diameters, cavity_R, bjerrum_length, max_disp, seed, validate=True) -> MCSystem:
    """north_star's mc_init(positions, charges, diameters, cavity_R, bjerrum_length, max_disp, seed)."""
    return MCSystem(pos, charges, diameters, cavity_R, bjerrum_length, max_disp, seed, validate=validate)
