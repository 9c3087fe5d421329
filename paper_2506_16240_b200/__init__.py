"""paper_2506_16240_b200 -- Python binding of libmicsa.so (include/micsa.h).

Argument marshalling only: every step of the MicSA path (sweep, daemon
refresh, reductions) runs in the CUDA kernels of ``csrc/``.  PyTorch is used
for device memory (the workspace tensor) and the CUDA stream, nothing else.
There is no CPU fallback: importing this package raises if ``libmicsa.so`` has
not been built (``python -m paper_2506_16240_b200.build``), and creating a
context raises without a CUDA device.

Method names mirror the C ABI: ``micsa_create`` -> ``MicSA(...)``,
``micsa_sweep`` -> ``.sweep(n)``, ``micsa_refresh_demons`` ->
``.refresh_demons(T, step)``, ``micsa_measure`` -> ``.measure()``,
``micsa_anneal`` -> ``.anneal(schedule)`` ...
"""
from __future__ import annotations

import ctypes
from pathlib import Path

import numpy as np

_PKG = Path(__file__).resolve().parent
LIB_PATH = _PKG / "libmicsa.so"

MICSA_OK, MICSA_ERR_INVALID, MICSA_ERR_NOMEM, MICSA_ERR_CUDA = 0, -1, -2, -3

EXPORTS = (
    "micsa_last_error", "micsa_create", "micsa_create_ex", "micsa_workspace_bytes",
    "micsa_destroy", "micsa_synchronize", "micsa_set_couplings", "micsa_set_spins",
    "micsa_set_daemons", "micsa_set_demons", "micsa_get_state", "micsa_sweep", "micsa_half_sweep",
    "micsa_refresh_demons", "micsa_debug_thresholds", "micsa_debug_philox", "micsa_measure_i64",
    "micsa_measure", "micsa_anneal", "micsa_counters", "micsa_layout_info",
    "micsa_set_tuning",
    "micsa_prefetch_refresh", "micsa_measure_begin", "micsa_measure_end", "micsa_sweep_measure",
    "micsa_measure_noalloc",
    "micsa_measure_c4", "micsa_xi", "micsa_effective_temperature", "micsa_metropolis_sweep", "micsa_metropolis_half_sweep", "micsa_debug_metropolis_thresholds",
    "micsa_set_gamma", "micsa_select_daemon_set",
    "micsa_wander", "micsa_set_walkers", "micsa_set_time", "micsa_get_time",
    "micsa_gauss_create", "micsa_gauss_destroy", "micsa_gauss_set_couplings", "micsa_gauss_set_state",
    "micsa_gauss_get_state", "micsa_gauss_refresh", "micsa_gauss_sweep", "micsa_gauss_half_sweep",
    "micsa_gauss_wander", "micsa_gauss_set_walkers", "micsa_gauss_measure", "micsa_gauss_counters",
    "micsa_gauss_synchronize",
)


class MicsaError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"micsa error {code}: {msg}")
        self.code = code


class _Step(ctypes.Structure):
    _fields_ = [("T", ctypes.c_double), ("n_sweeps", ctypes.c_int32),
                ("measure_every", ctypes.c_int32)]


class _Trace(ctypes.Structure):
    _fields_ = [("capacity", ctypes.c_int64), ("n_rows", ctypes.c_int64),
                ("sweep", ctypes.c_void_p), ("T", ctypes.c_void_p),
                ("E", ctypes.c_void_p), ("E_daemon", ctypes.c_void_p),
                ("Q", ctypes.c_void_p)]


def _load() -> ctypes.CDLL:
    try:
        return _bind()
    except AttributeError:
        # a stale binary from an older header: rebuild once, then fail loudly
        from .build import build as _build
        _build(force=True)
        return _bind()


def _bind() -> ctypes.CDLL:
    if not LIB_PATH.exists():
        # a fresh checkout has no binary: compile it now (nvcc, sm_100a); there is
        # nothing to fall back to if that fails
        from .build import build as _build
        try:
            _build()
        except Exception as exc:
            raise ImportError(
                f"{LIB_PATH} is missing and `python -m paper_2506_16240_b200.build` failed "
                f"({exc}). This package has no CPU fallback.") from exc
    lib = ctypes.CDLL(str(LIB_PATH))
    vp, i32, u32, u64, f64 = (ctypes.c_void_p, ctypes.c_int, ctypes.c_uint32,
                              ctypes.c_uint64, ctypes.c_double)
    lib.micsa_last_error.restype = ctypes.c_char_p
    lib.micsa_last_error.argtypes = []
    lib.micsa_create.restype = vp
    lib.micsa_create.argtypes = [i32, i32, i32, u64]
    lib.micsa_create_ex.restype = vp
    lib.micsa_create_ex.argtypes = [i32, i32, i32, u64, i32, vp, ctypes.c_size_t, vp]
    lib.micsa_gauss_create.restype = vp
    lib.micsa_gauss_create.argtypes = [i32, i32, i32, u64, i32, vp]
    lib.micsa_workspace_bytes.restype = ctypes.c_size_t
    lib.micsa_workspace_bytes.argtypes = [i32, i32, i32]
    for name, args in (
            ("micsa_destroy", [vp]), ("micsa_synchronize", [vp]),
            ("micsa_set_couplings", [vp, vp]), ("micsa_set_spins", [vp, vp]),
            ("micsa_set_daemons", [vp, vp]), ("micsa_set_demons", [vp, vp]), ("micsa_get_state", [vp, vp, vp, vp]),
            ("micsa_sweep", [vp, i32]), ("micsa_sweep_measure", [vp, i32]),
            ("micsa_metropolis_sweep", [vp, f64, u32, i32]), ("micsa_metropolis_half_sweep", [vp, f64, u32, i32]),
            ("micsa_debug_metropolis_thresholds", [f64, vp]),
            ("micsa_set_gamma", [vp, i32]), ("micsa_select_daemon_set", [vp, i32]),
            ("micsa_wander", [vp, i32, i32, i32]), ("micsa_set_walkers", [vp, i32]),
            ("micsa_set_time", [vp, ctypes.c_int64]), ("micsa_get_time", [vp, vp]), ("micsa_half_sweep", [vp, i32]),
            ("micsa_refresh_demons", [vp, f64, u32]),
            ("micsa_prefetch_refresh", [vp, f64, u32]),
            ("micsa_debug_thresholds", [f64, vp]), ("micsa_debug_philox", [u64, vp, i32, vp]), ("micsa_effective_temperature", [f64, vp]),
            ("micsa_measure_i64", [vp, vp, vp, vp]),
            ("micsa_measure_noalloc", [vp, vp]),
            ("micsa_measure_c4", [vp, vp]), ("micsa_xi", [vp, i32, f64, vp, vp, vp]), ("micsa_measure_begin", [vp]), ("micsa_measure_end", [vp, vp, vp, vp]), ("micsa_measure", [vp, vp, vp, vp]),
            ("micsa_anneal", [vp, vp, i32, u32, vp, vp]),
            ("micsa_counters", [vp, vp, vp, vp]), ("micsa_layout_info", [vp, vp]),
            ("micsa_set_tuning", [vp, i32, i32]),
            ("micsa_gauss_destroy", [vp]), ("micsa_gauss_set_couplings", [vp, vp]),
            ("micsa_gauss_set_state", [vp, vp, vp]), ("micsa_gauss_get_state", [vp, vp, vp, vp]),
            ("micsa_gauss_refresh", [vp, f64, u32]), ("micsa_gauss_sweep", [vp, i32]),
            ("micsa_gauss_half_sweep", [vp, i32]), ("micsa_gauss_wander", [vp, i32, i32, i32]),
            ("micsa_gauss_set_walkers", [vp, i32, ctypes.c_int64]), ("micsa_gauss_measure", [vp, vp, vp, vp]),
            ("micsa_gauss_counters", [vp, vp, vp]), ("micsa_gauss_synchronize", [vp])):
        fn = getattr(lib, name)
        fn.restype = i32
        fn.argtypes = args
    return lib


_lib = _load()


def last_error() -> str:
    return _lib.micsa_last_error().decode()


def _check(rc):
    if rc != MICSA_OK:
        raise MicsaError(rc, last_error())


def _ptr(a):
    return None if a is None else ctypes.c_void_p(a.ctypes.data)


def debug_thresholds(T: float) -> np.ndarray:
    """micsa_debug_thresholds: the integer thresholds of Eq. (11) (R7)."""
    thr = np.zeros(3, dtype=np.uint64)
    _check(_lib.micsa_debug_thresholds(float(T), _ptr(thr)))
    return thr


def debug_philox(seed: int, counters) -> np.ndarray:
    """micsa_debug_philox: the library's device Philox4x32-10 on counters [n][4] (test hook, pin P6)."""
    c = np.ascontiguousarray(counters, dtype=np.uint32).reshape(-1, 4)
    out = np.empty_like(c)
    _check(_lib.micsa_debug_philox(int(seed), _ptr(c), c.shape[0], _ptr(out)))
    return out


def xi(C4, c_min=0.0):
    """micsa_xi: (I_1, I_2, I_3, xi_12, xi_23 / xi_12) of Eq. (17)-(18) from C4(r), r = 0 .. len - 1."""
    C4 = np.ascontiguousarray(C4, dtype=np.float64)
    I = np.zeros(3, np.float64)
    a, b = ctypes.c_double(0.0), ctypes.c_double(0.0)
    _check(_lib.micsa_xi(_ptr(C4), C4.size, float(c_min), _ptr(I), ctypes.byref(a), ctypes.byref(b)))
    return float(I[0]), float(I[1]), float(I[2]), float(a.value), float(b.value)


def effective_temperature(e_daemon_per_variable: float) -> float:
    """Invert Eq. (12): the temperature of daemons holding this energy per auxiliary variable."""
    T = ctypes.c_double(0.0)
    _check(_lib.micsa_effective_temperature(float(e_daemon_per_variable), ctypes.byref(T)))
    return float(T.value)


def debug_metropolis_thresholds(T: float) -> np.ndarray:
    thr = np.zeros(3, dtype=np.uint64)
    _check(_lib.micsa_debug_metropolis_thresholds(float(T), _ptr(thr)))
    return thr


def workspace_bytes(L, n_samples, n_replicas) -> int:
    return int(_lib.micsa_workspace_bytes(L, n_samples, n_replicas))


class MicSA:
    """One MicSA context (micsa_create_ex).  Device memory and stream come from
    torch when ``use_torch`` (default), else the library allocates itself."""

    def __init__(self, L, n_samples, n_replicas, seed, sample_offset=0, device=0,
                 use_torch=True, stream=None):
        self.L, self.n_samples, self.n_replicas = int(L), int(n_samples), int(n_replicas)
        self.N = self.L ** 3
        self.n_sys = self.n_samples * self.n_replicas
        self.n_pairs = self.n_samples * (self.n_replicas * (self.n_replicas - 1) // 2)
        self.seed = int(seed)
        self._h = None
        self._ws = None
        self._stream = None
        ws_ptr, ws_bytes, stream_ptr = None, 0, None
        if use_torch:
            import torch
            if not torch.cuda.is_available():
                raise MicsaError(MICSA_ERR_CUDA, "no CUDA device (this library has no CPU fallback)")
            torch.cuda.set_device(device)
            nbytes = workspace_bytes(self.L, self.n_samples, self.n_replicas)
            if nbytes == 0:
                raise MicsaError(MICSA_ERR_INVALID, last_error())
            self._ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=f"cuda:{device}")
            base = self._ws.data_ptr()
            ws_ptr = (base + 255) // 256 * 256
            ws_bytes = nbytes
            self._stream = stream if stream is not None else torch.cuda.current_stream()
            stream_ptr = self._stream.cuda_stream
        h = _lib.micsa_create_ex(self.L, self.n_samples, self.n_replicas, self.seed,
                                 int(sample_offset), ws_ptr, ws_bytes, stream_ptr)
        if not h:
            raise MicsaError(MICSA_ERR_INVALID, last_error())
        self._h = ctypes.c_void_p(h)

    # -- life cycle
    def destroy(self):
        if self._h is not None:
            _lib.micsa_destroy(self._h)
            self._h = None
            self._ws = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.destroy()

    def synchronize(self):
        _check(_lib.micsa_synchronize(self._h))

    # -- state in / out (canonical layouts of micsa.h)
    def set_couplings(self, J):
        J = np.ascontiguousarray(J, dtype=np.int8)
        assert J.shape == (self.n_samples, 3, self.N), J.shape
        _check(_lib.micsa_set_couplings(self._h, _ptr(J)))

    def set_spins(self, s):
        s = np.ascontiguousarray(s, dtype=np.int8)
        assert s.shape == (self.n_samples, self.n_replicas, self.N), s.shape
        _check(_lib.micsa_set_spins(self._h, _ptr(s)))

    def set_daemons(self, m):
        m = np.ascontiguousarray(m, dtype=np.uint8)
        assert m.shape == (self.n_samples, self.n_replicas, self.N), m.shape
        _check(_lib.micsa_set_daemons(self._h, _ptr(m)))

    def get_state(self, spins=True, daemons=True, couplings=True):
        s = np.empty((self.n_samples, self.n_replicas, self.N), np.int8) if spins else None
        m = np.empty((self.n_samples, self.n_replicas, self.N), np.uint8) if daemons else None
        J = np.empty((self.n_samples, 3, self.N), np.int8) if couplings else None
        _check(_lib.micsa_get_state(self._h, _ptr(s), _ptr(m), _ptr(J)))
        return s, m, J

    # -- hot path
    def sweep(self, n=1):
        _check(_lib.micsa_sweep(self._h, int(n)))

    def sweep_measure(self, n=1):
        """n sweeps, then the measurement queued (fetch it with measure_end)."""
        _check(_lib.micsa_sweep_measure(self._h, int(n)))

    def metropolis_sweep(self, T, tau0, n=1):
        _check(_lib.micsa_metropolis_sweep(self._h, float(T), int(tau0), int(n)))

    def metropolis_half_sweep(self, T, tau, parity):
        _check(_lib.micsa_metropolis_half_sweep(self._h, float(T), int(tau), int(parity)))

    def set_gamma(self, gamma):
        _check(_lib.micsa_set_gamma(self._h, int(gamma)))

    def select_daemon_set(self, alpha):
        _check(_lib.micsa_select_daemon_set(self._h, int(alpha)))

    def wander(self, axis=0, sign=+1, parity=0):
        _check(_lib.micsa_wander(self._h, int(axis), int(sign), int(parity)))

    def set_walkers(self, mode):
        _check(_lib.micsa_set_walkers(self._h, int(mode)))

    def set_time(self, t):
        _check(_lib.micsa_set_time(self._h, int(t)))

    def get_time(self) -> int:
        t = ctypes.c_int64(0)
        _check(_lib.micsa_get_time(self._h, ctypes.byref(t)))
        return int(t.value)

    def half_sweep(self, parity):
        _check(_lib.micsa_half_sweep(self._h, int(parity)))

    def refresh_demons(self, T, step):
        _check(_lib.micsa_refresh_demons(self._h, float(T), int(step)))

    def prefetch_refresh(self, T, step):
        _check(_lib.micsa_prefetch_refresh(self._h, float(T), int(step)))

    def measure_i64(self):
        E = np.empty(self.n_sys, np.int64)
        Ed = np.empty(self.n_sys, np.int64)
        Q = np.empty(self.n_pairs, np.int64) if self.n_replicas >= 2 else None
        _check(_lib.micsa_measure_i64(self._h, _ptr(E), _ptr(Ed), _ptr(Q)))
        return E, Ed, (Q if Q is not None else np.empty(0, np.int64))

    @property
    def row_len(self) -> int:
        """int64 elements of a measurement row: E[n_sys] | E_daemon[n_sys] | Q[n_pairs]."""
        return 2 * self.n_sys + self.n_pairs

    def measure_noalloc(self, row):
        """micsa_measure_noalloc: queue the measurement into `row`, a caller-owned contiguous torch.int64 CUDA tensor
        of at least row_len elements (or an integer device address).  Nothing is allocated, copied or synchronised;
        the sums are in row[:n_sys], row[n_sys:2 n_sys], row[2 n_sys:row_len] once the stream gets there."""
        if isinstance(row, int):
            ptr = row
        else:
            if str(row.dtype) != "torch.int64" or not row.is_cuda or not row.is_contiguous() or row.numel() < self.row_len:
                raise MicsaError(MICSA_ERR_INVALID, "row must be a contiguous torch.int64 CUDA tensor of >= row_len elements")
            ptr = row.data_ptr()
        _check(_lib.micsa_measure_noalloc(self._h, ctypes.c_void_p(ptr)))

    def measure_c4(self):
        """S[pair, axis, r] = sum_x q_x q_{x + r e_axis} (exact int64), r = 0..L/2, for every replica pair a < b of
        every sample, pairs ordered like Q of measure()."""
        S = np.empty((self.n_pairs, 3, self.L // 2 + 1), np.int64)
        _check(_lib.micsa_measure_c4(self._h, _ptr(S)))
        return S

    def measure_begin(self):
        _check(_lib.micsa_measure_begin(self._h))

    def measure_end(self):
        E = np.empty(self.n_sys, np.int64)
        Ed = np.empty(self.n_sys, np.int64)
        Q = np.empty(self.n_pairs, np.int64) if self.n_replicas >= 2 else None
        _check(_lib.micsa_measure_end(self._h, _ptr(E), _ptr(Ed), _ptr(Q)))
        return E, Ed, (Q if Q is not None else np.empty(0, np.int64))

    def measure(self):
        e = np.empty(self.n_sys, np.float64)
        ed = np.empty(self.n_sys, np.float64)
        q = np.empty(self.n_pairs, np.float64) if self.n_replicas >= 2 else None
        _check(_lib.micsa_measure(self._h, _ptr(e), _ptr(ed), _ptr(q)))
        return e, ed, (q if q is not None else np.empty(0, np.float64))

    def anneal(self, schedule, step0=0, trace=True):
        """schedule: iterable of (T, n_sweeps, measure_every).  Returns a dict
        with the measurement rows (exact int64 sums) and min_energy (E/N)."""
        sched = list(schedule)
        arr = (_Step * max(len(sched), 1))()
        rows = 0
        for k, (T, n, every) in enumerate(sched):
            arr[k].T, arr[k].n_sweeps, arr[k].measure_every = float(T), int(n), int(every)
            if every > 0:
                rows += int(n) // int(every)
        min_e = np.empty(self.n_sys, np.float64)
        out = {}
        tr = None
        if trace:
            cap = max(rows, 1)
            out = {"sweep": np.zeros(cap, np.int64), "T": np.zeros(cap, np.float64),
                   "E": np.zeros((cap, self.n_sys), np.int64),
                   "Edem": np.zeros((cap, self.n_sys), np.int64),
                   "Q": np.zeros((cap, self.n_pairs), np.int64)}
            tr = _Trace(cap, 0, out["sweep"].ctypes.data, out["T"].ctypes.data,
                        out["E"].ctypes.data, out["Edem"].ctypes.data,
                        out["Q"].ctypes.data if self.n_pairs else None)
        _check(_lib.micsa_anneal(self._h, arr, len(sched), int(step0), _ptr(min_e),
                                 ctypes.byref(tr) if tr is not None else None))
        if trace:
            out = {k: v[:rows] for k, v in out.items()}
            assert tr.n_rows == rows
        out["min_energy"] = min_e
        return out

    # -- accounting
    def counters(self):
        a, r, p = ctypes.c_uint64(), ctypes.c_uint64(), ctypes.c_uint64()
        _check(_lib.micsa_counters(self._h, ctypes.byref(a), ctypes.byref(r), ctypes.byref(p)))
        return {"attempts": a.value, "rns_drawn": r.value, "philox_calls": p.value}

    def set_tuning(self, key, value):
        """micsa_set_tuning: 'sweep_kernel' (1 row-marching, 2 pipelined row-marching),
        'pipe_rows' (4, 8), 'pdl' (0, 1), 'pipe_planes' (1, 4), 'fuse_measure' (0, 1), 'fuse_walk' (0, 1),
        'l2_groups' (0, 1), 'small_path' (0, 1), 'small_items' (0 default, 1..1024)."""
        k = {"sweep_kernel": 0, "pipe_rows": 2, "pdl": 3, "pipe_planes": 4, "fuse_measure": 5, "fuse_walk": 6, "l2_groups": 7, "small_path": 8, "small_items": 9}[key]
        _check(_lib.micsa_set_tuning(self._h, k, int(value)))

    def layout_info(self):
        info = np.zeros(5, np.uint64)
        _check(_lib.micsa_layout_info(self._h, _ptr(info)))
        return {"state_bytes": int(info[0]), "compulsory_bytes_per_sweep": int(info[1]),
                "words_per_site": int(info[2]), "bond_bits": int(info[3]),
                "launches": int(info[4])}


class GaussMicSA:
    """Continuous daemons / walkers with real couplings (micsa_gauss_*; Sec. 2.4 Eq. 9, Appendix C).
    Argument marshalling only; the library allocates its own device memory, `stream` is a torch stream or None."""

    def __init__(self, L, n_samples, n_replicas, seed, sample_offset=0, stream=None):
        self.L, self.n_samples, self.n_replicas = int(L), int(n_samples), int(n_replicas)
        self.N = self.L ** 3
        self.n_sys = self.n_samples * self.n_replicas
        self.n_pairs = self.n_samples * (self.n_replicas * (self.n_replicas - 1) // 2)
        self._stream = stream
        h = _lib.micsa_gauss_create(self.L, self.n_samples, self.n_replicas, int(seed), int(sample_offset),
                                    stream.cuda_stream if stream is not None else None)
        if not h:
            raise MicsaError(MICSA_ERR_INVALID, last_error())
        self._h = ctypes.c_void_p(h)

    def destroy(self):
        if self._h is not None:
            _lib.micsa_gauss_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.destroy()

    def set_couplings(self, J):
        J = np.ascontiguousarray(J, dtype=np.float64)
        assert J.shape == (self.n_samples, 3, self.N), J.shape
        _check(_lib.micsa_gauss_set_couplings(self._h, _ptr(J)))

    def set_state(self, s=None, n=None):
        if s is not None:
            s = np.ascontiguousarray(s, dtype=np.int8)
            assert s.shape == (self.n_samples, self.n_replicas, self.N)
        if n is not None:
            n = np.ascontiguousarray(n, dtype=np.float64)
            assert n.shape == (self.n_samples, self.n_replicas, self.N)
        _check(_lib.micsa_gauss_set_state(self._h, _ptr(s), _ptr(n)))

    def get_state(self, spins=True, daemons=True, couplings=True):
        s = np.empty((self.n_samples, self.n_replicas, self.N), np.int8) if spins else None
        n = np.empty((self.n_samples, self.n_replicas, self.N), np.float64) if daemons else None
        J = np.empty((self.n_samples, 3, self.N), np.float64) if couplings else None
        _check(_lib.micsa_gauss_get_state(self._h, _ptr(s), _ptr(n), _ptr(J)))
        return s, n, J

    def refresh(self, T, step):
        _check(_lib.micsa_gauss_refresh(self._h, float(T), int(step)))

    def sweep(self, n=1):
        _check(_lib.micsa_gauss_sweep(self._h, int(n)))

    def half_sweep(self, parity):
        _check(_lib.micsa_gauss_half_sweep(self._h, int(parity)))

    def wander(self, axis=0, sign=+1, parity=0):
        _check(_lib.micsa_gauss_wander(self._h, int(axis), int(sign), int(parity)))

    def set_walkers(self, mode, t=0):
        _check(_lib.micsa_gauss_set_walkers(self._h, int(mode), int(t)))

    def measure(self):
        E = np.empty(self.n_sys, np.float64)
        Ed = np.empty(self.n_sys, np.float64)
        Q = np.empty(self.n_pairs, np.int64) if self.n_replicas >= 2 else None
        _check(_lib.micsa_gauss_measure(self._h, _ptr(E), _ptr(Ed), _ptr(Q)))
        return E, Ed, (Q if Q is not None else np.empty(0, np.int64))

    def counters(self):
        a, r = ctypes.c_uint64(), ctypes.c_uint64()
        _check(_lib.micsa_gauss_counters(self._h, ctypes.byref(a), ctypes.byref(r)))
        return {"attempts": a.value, "rns_drawn": r.value}

    def synchronize(self):
        _check(_lib.micsa_gauss_synchronize(self._h))
