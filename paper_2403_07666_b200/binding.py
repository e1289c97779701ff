"""Thin ctypes binding of libqs.so (include/qs.h): argument marshalling only.

PyTorch is used for exactly two things: it owns the device workspace (one uint8 tensor handed to
``qs_init_device``) and the CUDA stream the library enqueues on.  Every step of the path runs in the
library's own kernels; there is no Python or CPU fallback — without the built library or without a
CUDA device the constructor raises.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import numpy as np

from .build import build as _build_lib

c_double_p = C.POINTER(C.c_double)
c_int32_p = C.POINTER(C.c_int32)


class QsGeometry(C.Structure):
    _fields_ = [("n_rings", C.c_int32), ("r", c_double_p), ("z", c_double_p), ("area", c_double_p),
                ("turn_id", c_int32_p), ("n_turns", C.c_int32), ("lattice", C.c_int32),
                ("layers", C.c_int32), ("turns_per_layer", C.c_int32), ("cells_per_side", C.c_int32),
                ("wire_size", C.c_double), ("r_inner", C.c_double), ("softening", C.c_double),
                ("h_conv", C.c_double * 4), ("T_bath", C.c_double),
                ("Bext0", C.c_double), ("Bext_rate", C.c_double), ("Bext_max", C.c_double),
                ("flags", C.c_int32), ("turn_share", c_double_p)]


class QsMaterial(C.Structure):
    _fields_ = [("Ec", C.c_double), ("n_exp", C.c_double), ("Jc0", C.c_double), ("Tc", C.c_double),
                ("B0", C.c_double), ("eps_coef", C.c_double), ("eps_exp", C.c_double), ("Y", C.c_double),
                ("rho_n", C.c_double), ("jc0_scale", c_double_p), ("C3", C.c_double), ("C1", C.c_double),
                ("k_in", C.c_double), ("k_between", C.c_double), ("theta", C.c_double),
                ("cg_tol", C.c_double), ("cg_maxit", C.c_int32),
                ("T_fluxjump", C.c_double), ("dEdt_spike", C.c_double), ("heat_adi_substeps", C.c_int32)]


class QsStats(C.Structure):
    _fields_ = [("cg_iters", C.c_int32), ("heat_substeps", C.c_int32), ("event_word", C.c_int32),
                ("sweeps", C.c_int32), ("cg_relres", C.c_double), ("U_terminal", C.c_double),
                ("Tmax", C.c_double), ("joule_power", C.c_double), ("t", C.c_double), ("I", C.c_double),
                ("launches", C.c_int64), ("pair_evals", C.c_int64), ("dJ_max", C.c_double)]


class QsProfile(C.Structure):
    _fields_ = [("ms", C.c_double * 8), ("launches", C.c_int64 * 8)]


PROFILE_CLASSES = ["sweep_M", "sweep_field", "material", "heat", "events", "cg_vector"]

# every symbol include/qs.h declares: (name, restype, argtypes)
_VP = C.c_void_p
SYMBOLS = [
    ("qs_init", C.c_int, [C.POINTER(QsGeometry), C.POINTER(QsMaterial), C.POINTER(_VP)]),
    ("qs_step", C.c_int, [_VP, C.c_double, C.c_double]),
    ("qs_step_rk", C.c_int, [_VP, C.c_double, C.c_double, C.c_double, C.c_double, c_double_p, c_double_p, c_double_p]),
    ("qs_read", C.c_int, [_VP, c_double_p, c_double_p, c_double_p, c_double_p]),
    ("qs_workspace_bytes", C.c_size_t, [C.POINTER(QsGeometry)]),
    ("qs_init_device", C.c_int, [C.POINTER(QsGeometry), C.POINTER(QsMaterial), _VP, C.c_size_t, _VP, C.POINTER(_VP)]),
    ("qs_write", C.c_int, [_VP, c_double_p, c_double_p, C.c_double, C.c_double]),
    ("qs_read_rate", C.c_int, [_VP, c_double_p]),
    ("qs_write_rate", C.c_int, [_VP, c_double_p]),
    ("qs_debug_inject_failure", C.c_int, [_VP, C.c_int32]),
    ("qs_matvec", C.c_int, [_VP, c_double_p, c_double_p]),
    ("qs_matvec_device", C.c_int, [_VP, _VP, _VP]),
    ("qs_matvec_noalloc", C.c_int, [C.c_int32, _VP, _VP, C.c_double, _VP, _VP, _VP]),
    ("qs_field", C.c_int, [_VP, c_double_p, c_double_p]),
    ("qs_solve", C.c_int, [_VP, c_double_p, c_double_p, C.c_int32, c_int32_p, c_double_p]),
    ("qs_solve_device", C.c_int, [_VP, _VP, _VP, C.c_int32, c_int32_p, c_double_p]),
    ("qs_material_eval", C.c_int, [_VP, C.c_double]),
    ("qs_set_aux", C.c_int, [_VP, C.c_int32]),
    ("qs_heat", C.c_int, [_VP, C.c_double]),
    ("qs_heat_adi", C.c_int, [_VP, C.c_double, C.c_int32]),
    ("qs_set_fields", C.c_int, [_VP, c_double_p, c_double_p]),
    ("qs_read_aux", C.c_int, [_VP, c_double_p, c_double_p, c_double_p, c_double_p]),
    ("qs_stats", C.c_int, [_VP, C.POINTER(QsStats)]),
    ("qs_profile_enable", C.c_int, [_VP, C.c_int32]),
    ("qs_profile_read", C.c_int, [_VP, C.POINTER(QsProfile)]),
    ("qs_fp64_peak", C.c_int, [c_double_p, c_double_p]),
    ("qs_issue_probe", C.c_int, [C.c_int32, c_double_p]),
    ("qs_pair_eval", C.c_int, [C.c_int32, c_double_p, c_double_p, C.c_int32, c_double_p, c_double_p, c_double_p, c_int32_p]),
    ("qs_events", C.c_int, [_VP, c_int32_p, c_double_p, c_int32_p]),
    ("qs_wire_stats", C.c_int, [_VP, c_double_p]),
    ("qs_sync", C.c_int, [_VP]),
    ("qs_last_error", C.c_char_p, []),
    ("qs_free", None, [_VP]),
]

_lib = None


def load_library(path: Optional[str] = None) -> C.CDLL:
    """dlopen libqs.so (building it in-tree with nvcc first if it is missing or stale)."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    if path is None:
        path = _build_lib()            # raises if nvcc fails; never falls back to anything else
    lib = C.CDLL(path)
    for name, res, args in SYMBOLS:
        fn = getattr(lib, name)          # AttributeError if the library does not export it
        fn.restype = res
        fn.argtypes = args
    _lib = lib
    return lib


class QsError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"libqs error {code}: {msg}")
        self.code = code


def _dp(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(c_double_p)


def _f64(a, n=None) -> np.ndarray:
    out = np.ascontiguousarray(a, dtype=np.float64)
    if n is not None and out.size != n:
        raise ValueError(f"expected {n} elements, got {out.size}")
    return out


NOALLOC_MAX_RINGS = 16384


def matvec_noalloc(r, z, softening: float, x, y, stream=None) -> None:
    """qs_matvec_noalloc: y = M x on free rings with all scratch in the library's static device array (no allocation,
    no handle).  r, z, x, y: float64 CUDA tensors of n elements on the current device; enqueued on `stream` (a
    torch.cuda.Stream, default: the current stream).  Calls that overlap on the GPU race on the shared array."""
    import torch
    lib = load_library()
    n = int(r.numel())
    st = torch.cuda.current_stream() if stream is None else stream
    rc = lib.qs_matvec_noalloc(n, _VP(r.data_ptr()), _VP(z.data_ptr()), float(softening), _VP(x.data_ptr()),
                               _VP(y.data_ptr()), _VP(st.cuda_stream))
    if rc < 0:
        raise QsError(rc, lib.qs_last_error().decode())


def fp64_peak():
    """(TFLOP/s, effective SM MHz) of the DFMA probe kernel on the current CUDA device."""
    lib = load_library()
    tf, mhz = C.c_double(0.0), C.c_double(0.0)
    rc = lib.qs_fp64_peak(C.byref(tf), C.byref(mhz))
    if rc < 0:
        raise QsError(rc, lib.qs_last_error().decode())
    return tf.value, mhz.value


def issue_probe() -> dict:
    """SM cycles per DFMA warp-instruction per sub-partition: 3 register operands / 2 + immediate / + integer ALU."""
    lib = load_library()
    out = {}
    for mode, name in ((1, "dfma_3reg"), (2, "dfma_2reg_imm"), (3, "dfma_2reg_imm_plus_1_alu")):
        v = C.c_double(0.0)
        rc = lib.qs_issue_probe(mode, C.byref(v))
        if rc < 0:
            raise QsError(rc, lib.qs_last_error().decode())
        out[name] = v.value
    return out


def pair_eval(A2, B2, cls: int = -1):
    """(M, K, E, class used) of the sweeps' per-pair arithmetic for given A2, B2 arrays (test hook)."""
    lib = load_library()
    a, b = _f64(A2), _f64(B2, None)
    n = a.size
    M, K, E = np.empty(n), np.empty(n), np.empty(n)
    used = np.empty(n, dtype=np.int32)
    rc = lib.qs_pair_eval(n, _dp(a), _dp(b), int(cls), _dp(M), _dp(K), _dp(E), used.ctypes.data_as(c_int32_p))
    if rc < 0:
        raise QsError(rc, lib.qs_last_error().decode())
    return M, K, E, used


class QS:
    """One simulation handle.  ``geometry`` / ``material`` are objects with the fields of
    ``qs_geometry`` / ``qs_material`` (e.g. ``workloads.Geometry`` / ``workloads.Material``)."""

    def __init__(self, geometry, material, device: int = 0, no_operator: bool = False, torch_memory: bool = True,
                 lattice_tables: bool = False, patch_precond: bool = True, heat_blocked: bool = False,
                 patch_subwire: bool = False):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2403_07666_b200 needs a CUDA device: there is no CPU path")
        self._lib = load_library()
        self._torch = torch
        self.N = int(geometry.r.shape[0])
        self.n_turns = int(geometry.n_turns)
        self._keep = []                              # host arrays referenced by the structs
        g = QsGeometry()
        g.n_rings = self.N
        for name in ("r", "z", "area"):
            arr = _f64(getattr(geometry, name), self.N)
            self._keep.append(arr)
            setattr(g, name, _dp(arr))
        if geometry.turn_id is not None and self.n_turns > 0:
            tid = np.ascontiguousarray(geometry.turn_id, dtype=np.int32)
            self._keep.append(tid)
            g.turn_id = tid.ctypes.data_as(c_int32_p)
        g.n_turns = self.n_turns
        g.lattice = int(geometry.lattice)
        g.layers, g.turns_per_layer, g.cells_per_side = int(geometry.layers), int(geometry.turns_per_layer), int(geometry.cells_per_side)
        g.wire_size, g.r_inner, g.softening = float(geometry.wire_size), float(geometry.r_inner), float(geometry.softening)
        g.h_conv = (C.c_double * 4)(*[float(v) for v in geometry.h_conv])
        g.T_bath = float(geometry.T_bath)
        g.Bext0, g.Bext_rate, g.Bext_max = float(geometry.Bext0), float(geometry.Bext_rate), float(geometry.Bext_max)
        g.flags = (1 if no_operator else 0) | (2 if lattice_tables else 0) | (0 if patch_precond else 4) | (8 if heat_blocked else 0) | \
                  (16 if patch_subwire else 0)
        share = getattr(geometry, "turn_share", None)
        if share is not None and self.n_turns > 0:
            sh = _f64(share, self.n_turns)
            self._keep.append(sh)
            g.turn_share = _dp(sh)
        m = QsMaterial()
        for name, _ in QsMaterial._fields_:
            if name == "jc0_scale":
                if material.jc0_scale is not None:
                    arr = _f64(material.jc0_scale, self.N)
                    self._keep.append(arr)
                    m.jc0_scale = _dp(arr)
            elif name == "cg_maxit":
                m.cg_maxit = int(material.cg_maxit)
            elif name == "heat_adi_substeps":
                m.heat_adi_substeps = int(getattr(material, "heat_adi_substeps", 0))
            else:
                setattr(m, name, float(getattr(material, name)))
        self._h = _VP()
        self.device = torch.device("cuda", device)
        with torch.cuda.device(self.device):
            if torch_memory:
                nbytes = self._lib.qs_workspace_bytes(C.byref(g))
                if nbytes == 0:
                    raise QsError(-1, self._lib.qs_last_error().decode())
                self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
                base = (self.workspace.data_ptr() + 255) // 256 * 256
                self.stream = torch.cuda.Stream(device=self.device)
                rc = self._lib.qs_init_device(C.byref(g), C.byref(m), _VP(base), nbytes, _VP(self.stream.cuda_stream),
                                              C.byref(self._h))
            else:
                self.workspace, self.stream = None, None
                rc = self._lib.qs_init(C.byref(g), C.byref(m), C.byref(self._h))
        self._check(rc)

    # ---- plumbing -------------------------------------------------------------------------------
    def _check(self, rc: int) -> int:
        if rc < 0:
            raise QsError(rc, self._lib.qs_last_error().decode())
        return rc

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            self._lib.qs_free(self._h)
            self._h = _VP()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    # ---- the three calls -------------------------------------------------------------------------
    def step(self, dt: float, I_ramp: float) -> int:
        return self._check(self._lib.qs_step(self._h, float(dt), float(I_ramp)))

    def step_rk(self, dt_try: float, I_ramp: float, rtol: float, dt_min: float):
        """Embedded Heun-Euler step with error control: returns (event word, dt taken, dt suggested next, err)."""
        taken, nxt, err = C.c_double(0.0), C.c_double(0.0), C.c_double(0.0)
        rc = self._check(self._lib.qs_step_rk(self._h, float(dt_try), float(I_ramp), float(rtol), float(dt_min),
                                               C.byref(taken), C.byref(nxt), C.byref(err)))
        return rc, taken.value, nxt.value, err.value

    def read(self, J=True, T=True, B=True, E=True, out=None):
        """Returns (J, T, B, E) as numpy arrays (B = [Br, Bz] concatenated); skipped entries are None.
        ``out`` may hold preallocated (e.g. pinned) float64 arrays of the right sizes."""
        N = self.N
        bufs = list(out) if out is not None else [np.empty(N) if J else None, np.empty(N) if T else None,
                                                   np.empty(2 * N) if B else None, np.empty(N) if E else None]
        self._check(self._lib.qs_read(self._h, *[_dp(b) for b in bufs]))
        return tuple(bufs)

    # ---- extras ----------------------------------------------------------------------------------
    def write(self, J=None, T=None, t: float = 0.0, I: float = 0.0):
        Ja = None if J is None else _f64(J, self.N)
        Ta = None if T is None else _f64(T, self.N)
        self._check(self._lib.qs_write(self._h, _dp(Ja), _dp(Ta), float(t), float(I)))

    def read_rate(self) -> np.ndarray:
        """I' = dI/dt per ring of the last step's solve (the next step's CG start)."""
        x = np.empty(self.N)
        self._check(self._lib.qs_read_rate(self._h, _dp(x)))
        return x

    def write_rate(self, Idot):
        self._check(self._lib.qs_write_rate(self._h, _dp(_f64(Idot, self.N))))

    def debug_inject_failure(self, where: int):
        self._check(self._lib.qs_debug_inject_failure(self._h, int(where)))

    def matvec(self, x) -> np.ndarray:
        xa = _f64(x, self.N)
        y = np.empty(self.N)
        self._check(self._lib.qs_matvec(self._h, _dp(xa), _dp(y)))
        return y

    def matvec_device(self, x, y):
        """x, y: float64 CUDA tensors of N elements on this handle's device; enqueued on self.stream."""
        self._check(self._lib.qs_matvec_device(self._h, _VP(x.data_ptr()), _VP(y.data_ptr())))

    def field(self, I) -> np.ndarray:
        Ia = _f64(I, self.N)
        B = np.empty(2 * self.N)
        self._check(self._lib.qs_field(self._h, _dp(Ia), _dp(B)))
        return B

    def solve(self, b, maxit: int = 0):
        ba = _f64(b, self.N)
        x = np.empty(self.N)
        it, rel = C.c_int32(0), C.c_double(0.0)
        rc = self._check(self._lib.qs_solve(self._h, _dp(ba), _dp(x), int(maxit), C.byref(it), C.byref(rel)))
        return x, it.value, rel.value, rc

    def solve_device(self, b, x, maxit: int = 0):
        it, rel = C.c_int32(0), C.c_double(0.0)
        rc = self._check(self._lib.qs_solve_device(self._h, _VP(b.data_ptr()), _VP(x.data_ptr()), int(maxit),
                                                   C.byref(it), C.byref(rel)))
        return it.value, rel.value, rc

    def material_eval(self, dt: float = 0.0, aux: bool = True):
        """S2 alone on the current (J, T, B); aux: also store dE/dJ for read_aux (the step never does)."""
        self._check(self._lib.qs_set_aux(self._h, 1 if aux else 0))
        self._check(self._lib.qs_material_eval(self._h, float(dt)))

    def heat(self, dt: float) -> int:
        return self._check(self._lib.qs_heat(self._h, float(dt)))

    def heat_adi(self, dt: float, m: int) -> int:
        return self._check(self._lib.qs_heat_adi(self._h, float(dt), int(m)))

    def set_fields(self, B=None, Q=None):
        Ba = None if B is None else _f64(B, 2 * self.N)
        Qa = None if Q is None else _f64(Q, self.N)
        self._check(self._lib.qs_set_fields(self._h, _dp(Ba), _dp(Qa)))

    def read_aux(self):
        N = self.N
        Q, d, Jc, rho = np.empty(N), np.empty(N), np.empty(N), np.empty(N)
        self._check(self._lib.qs_read_aux(self._h, _dp(Q), _dp(d), _dp(Jc), _dp(rho)))
        return dict(Q=Q, dEdJ=d, Jc=Jc, rho=rho)

    def stats(self) -> dict:
        s = QsStats()
        self._check(self._lib.qs_stats(self._h, C.byref(s)))
        return {name: getattr(s, name) for name, _ in QsStats._fields_}

    def profile_enable(self, on: bool = True):
        self._check(self._lib.qs_profile_enable(self._h, 1 if on else 0))

    def profile_read(self) -> dict:
        """{class name: (summed ms, launches)} since the last read; resets the totals."""
        p = QsProfile()
        self._check(self._lib.qs_profile_read(self._h, C.byref(p)))
        return {name: (p.ms[k], int(p.launches[k])) for k, name in enumerate(PROFILE_CLASSES)}

    def events(self):
        nt = max(self.n_turns, 0)
        fl, tf, cnt = np.zeros(nt, dtype=np.int32), np.zeros(nt), np.zeros(nt, dtype=np.int32)
        if nt:
            self._check(self._lib.qs_events(self._h, fl.ctypes.data_as(c_int32_p), _dp(tf), cnt.ctypes.data_as(c_int32_p)))
        return fl, tf, cnt

    WIRE_KEYS = ("E_joule", "Q_FJ", "P_max", "T_max", "t_q", "T_q", "P_q", "Q_q")

    def wire_stats(self) -> dict:
        """Per-wire statistics (see qs_wire_stats in include/qs.h): {name: array [n_turns]}."""
        nt = max(self.n_turns, 0)
        out = np.zeros(8 * nt)
        if nt:
            self._check(self._lib.qs_wire_stats(self._h, _dp(out)))
        return {k: out[j * nt:(j + 1) * nt].copy() for j, k in enumerate(self.WIRE_KEYS)}

    def sync(self):
        self._check(self._lib.qs_sync(self._h))
