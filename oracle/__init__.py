"""CPU oracle for the collide-and-stream path -- TEST INFRASTRUCTURE, not the product.

Thin ctypes wrapper over `oracle/lbm_oracle.cpp` (plain fp64 C++, two-lattice push written
from eq (2.6), (2.7), (2.11) of the paper).  Only `tests/`,
`__graft_entry__.smoke()` and `bench.py`'s `cpu_baseline` / `--impl reference` legs may import
this package.  It imports nothing from `paper_2607_05668_b200` and shares no code with it; the
only shared module is `workloads` (seeded inputs, no method arithmetic).
"""
from __future__ import annotations

import ctypes as C
from typing import Optional, Sequence

import numpy as np

from . import build as _build

MAXM = 32
SYSTEM_ID = {"advection2d": 0, "burgers2d": 1, "swe2d": 2, "euler2d": 3, "adr2d": 4, "nsf3d": 5, "mhd3d": 6, "urf2d": 7, "maxwell2d": 8, "allencahn2d": 9, "inse2d": 10, "elasticity2d": 11, "nsf2d": 12,
             "swe2d_bathy": 13, "hcnsf3d": 14, "mhd2d": 15}


class _Spec(C.Structure):
    _fields_ = [
        ("system", C.c_int32), ("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32),
        ("bc", C.c_int32), ("shifted", C.c_int32), ("mms_id", C.c_int32), ("n_threads", C.c_int32),
        ("ox", C.c_int32), ("oy", C.c_int32), ("oz", C.c_int32), ("pad_", C.c_int32),
        ("dx", C.c_double), ("lam", C.c_double), ("g_tau", C.c_double), ("t0", C.c_double),
        ("par", C.c_double * 16), ("mms_par", C.c_double * 16),
        ("tau_R", C.c_double * MAXM), ("omega", C.c_double * MAXM), ("U_ref", C.c_double * MAXM),
        ("collision", C.c_int32), ("pad2_", C.c_int32), ("trt_magic", C.c_double),
    ]


_lib = None


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        L.orc_create.restype = C.c_void_p
        L.orc_create.argtypes = [C.POINTER(_Spec)]
        L.orc_destroy.argtypes = [C.c_void_p]
        dp = C.POINTER(C.c_double)
        for name, args in {
            "orc_init_from_U": [C.c_void_p, dp], "orc_set_f": [C.c_void_p, dp],
            "orc_step": [C.c_void_p, C.c_int], "orc_read_f": [C.c_void_p, dp], "orc_read_U": [C.c_void_p, dp],
            "orc_time": [C.c_void_p, C.POINTER(C.c_int64), dp], "orc_omega": [C.c_void_p, dp], "orc_omega_plus": [C.c_void_p, dp],
            "orc_exact_U": [C.c_void_p, C.c_double, dp],
            "orc_flux_source": [C.c_void_p, dp, dp, dp, dp], "orc_set_aux": [C.c_void_p, dp],
            "orc_system_n_aux": [C.c_int], "orc_equilibrium": [C.c_void_p, dp, dp, dp],
            "orc_mms_source": [C.c_void_p, C.c_double, C.c_double, C.c_double, C.c_double, dp],
            "orc_exact_point": [C.c_void_p, C.c_double, C.c_double, C.c_double, C.c_double, dp],
            "orc_max_wave_speed": [C.c_void_p, dp],
            "orc_stream_index_map": [C.c_void_p, C.c_int, C.POINTER(C.c_int64)],
            "orc_system_info": [C.c_int] + [C.POINTER(C.c_int)] * 4,
            "orc_lattice": [C.c_int, C.POINTER(C.c_int), dp, dp],
        }.items():
            getattr(L, name).argtypes = args
            getattr(L, name).restype = C.c_int
        L.orc_threads.restype = C.c_int
        _lib = L
    return _lib


def _dp(a: np.ndarray):
    assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(C.POINTER(C.c_double))


def system_info(system: str):
    mc, mt, d, q = C.c_int(), C.c_int(), C.c_int(), C.c_int()
    assert lib().orc_system_info(SYSTEM_ID[system], mc, mt, d, q) == 0
    return mc.value, mt.value, d.value, q.value


def lattice(dim: int):
    """(c[Q][3] int, w[Q], c_s^2) of D2Q5 / D3Q7, Table SM1."""
    Q = 2 * dim + 1
    c = np.zeros((Q, 3), dtype=np.int32)
    w = np.zeros(Q)
    cs2 = C.c_double()
    assert lib().orc_lattice(dim, c.ctypes.data_as(C.POINTER(C.c_int)), _dp(w), C.byref(cs2)) == 0
    return c, w, cs2.value


def n_threads() -> int:
    return lib().orc_threads()


class OracleGrid:
    """One periodic (or Dirichlet-MMS) grid of the oracle."""

    def __init__(self, system: str, nx: int, ny: int, nz: int, dx: float, lam: float,
                 params: Sequence[float] = (), tau_R=0.0, g_tau: float = 0.0,
                 mms_id: int = 0, mms_params: Sequence[float] = (), bc: str = "periodic",
                 shifted: bool = False, U_ref: Optional[Sequence[float]] = None,
                 omega: Optional[Sequence[float]] = None, origin=(0, 0, 0), t0: float = 0.0,
                 n_threads: int = 0, collision: str = "bgk", trt_magic: float = 0.25):
        self.system = system
        self.m_conserved, self.m_total, self.dim, self.Q = system_info(system)
        self.nx, self.ny, self.nz = nx, ny, nz
        self.n_aux = lib().orc_system_n_aux(SYSTEM_ID[system])
        s = _Spec()
        s.system = SYSTEM_ID[system]
        s.nx, s.ny, s.nz = nx, ny, nz
        s.bc = {"periodic": 0, "dirichlet_mms": 1}[bc]
        s.shifted = int(bool(shifted))
        s.mms_id = mms_id
        s.n_threads = n_threads
        s.collision = {"bgk": 0, "trt": 1, "regularized": 2}[collision]
        s.trt_magic = trt_magic
        s.ox, s.oy, s.oz = origin
        s.dx, s.lam, s.g_tau, s.t0 = dx, lam, g_tau, t0
        for i, v in enumerate(params):
            s.par[i] = v
        for i, v in enumerate(mms_params):
            s.mms_par[i] = v
        tr = np.broadcast_to(np.asarray(tau_R, dtype=np.float64), (self.m_conserved,)) if np.ndim(tau_R) == 0 \
            else np.asarray(tau_R, dtype=np.float64)
        for k in range(self.m_conserved):
            s.tau_R[k] = float(tr[k])
        for k in range(MAXM):
            s.omega[k] = -1.0
        if omega is not None:
            om = np.broadcast_to(np.asarray(omega, dtype=np.float64), (self.m_total,))
            for k in range(self.m_total):
                s.omega[k] = float(om[k])
        if U_ref is not None:
            for k, v in enumerate(U_ref):
                s.U_ref[k] = v
        self._spec = s
        self._h = lib().orc_create(C.byref(s))
        if not self._h:
            raise ValueError("orc_create failed (bad system / dims)")

    @classmethod
    def from_workload(cls, w, **kw):
        args = dict(system=w.system, nx=w.nx, ny=w.ny, nz=w.nz, dx=w.dx, lam=w.lam, params=w.params,
                    tau_R=w.tau_R, g_tau=w.g_tau, mms_id=w.mms_id, mms_params=w.mms_params, U_ref=w.U_ref)
        args.update(kw)
        return cls(**args)

    def close(self):
        if self._h:
            lib().orc_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def shape_U(self):
        return (self.m_total, self.nz, self.ny, self.nx)

    @property
    def shape_f(self):
        return (self.m_total, self.Q, self.nz, self.ny, self.nx)

    def init_from_U(self, U: np.ndarray):
        U = np.ascontiguousarray(U, dtype=np.float64)
        assert U.shape == self.shape_U
        assert lib().orc_init_from_U(self._h, _dp(U)) == 0

    def set_aux(self, A: np.ndarray):
        """Prescribed coefficient fields A[n_aux][nz][ny][nx] (bed slope; porosity and solid velocity)."""
        A = np.ascontiguousarray(A, dtype=np.float64)
        assert A.shape == (self.n_aux, self.nz, self.ny, self.nx)
        assert lib().orc_set_aux(self._h, _dp(A)) == 0

    def set_f(self, f: np.ndarray):
        f = np.ascontiguousarray(f, dtype=np.float64)
        assert f.shape == self.shape_f
        assert lib().orc_set_f(self._h, _dp(f)) == 0

    def step(self, n: int = 1):
        rc = lib().orc_step(self._h, int(n))
        if rc != 0:
            raise RuntimeError(f"orc_step -> {rc}")

    def read_U(self) -> np.ndarray:
        U = np.empty(self.shape_U)
        assert lib().orc_read_U(self._h, _dp(U)) == 0
        return U

    def read_f(self) -> np.ndarray:
        f = np.empty(self.shape_f)
        assert lib().orc_read_f(self._h, _dp(f)) == 0
        return f

    def time(self):
        st, t = C.c_int64(), C.c_double()
        lib().orc_time(self._h, C.byref(st), C.byref(t))
        return st.value, t.value

    def omega(self) -> np.ndarray:
        o = np.empty(self.m_total)
        lib().orc_omega(self._h, _dp(o))
        return o

    def omega_plus(self) -> np.ndarray:
        o = np.empty(self.m_total)
        lib().orc_omega_plus(self._h, _dp(o))
        return o

    def exact_U(self, t: float) -> np.ndarray:
        U = np.empty(self.shape_U)
        if lib().orc_exact_U(self._h, float(t), _dp(U)) != 0:
            raise ValueError("no manufactured solution for this (system, mms_id)")
        return U

    def flux_source(self, U: Sequence[float], A: Optional[Sequence[float]] = None):
        U = np.ascontiguousarray(U, dtype=np.float64)
        F = np.zeros((self.m_total, 3))
        S = np.zeros(self.m_total)
        Aa = np.zeros(max(self.n_aux, 1)) if A is None else np.ascontiguousarray(A, dtype=np.float64)
        lib().orc_flux_source(self._h, _dp(U), _dp(Aa), _dp(F), _dp(S))
        return F, S

    def equilibrium(self, U, F) -> np.ndarray:
        U = np.ascontiguousarray(U, dtype=np.float64)
        F = np.ascontiguousarray(F, dtype=np.float64)
        feq = np.zeros((self.m_total, self.Q))
        lib().orc_equilibrium(self._h, _dp(U), _dp(F), _dp(feq))
        return feq

    def mms_source(self, t, x, y, z=0.0) -> np.ndarray:
        s = np.zeros(self.m_total)
        if lib().orc_mms_source(self._h, t, x, y, z, _dp(s)) != 0:
            raise ValueError("no manufactured solution")
        return s

    def exact_point(self, t, x, y, z=0.0) -> np.ndarray:
        q = np.zeros(self.m_total)
        if lib().orc_exact_point(self._h, t, x, y, z, _dp(q)) != 0:
            raise ValueError("no manufactured solution")
        return q

    def max_wave_speed(self):
        o = np.zeros(3)
        lib().orc_max_wave_speed(self._h, _dp(o))
        return float(o[0]), float(o[1]), float(o[2])

    def stream_index_map(self, direction: int) -> np.ndarray:
        out = np.empty((self.nz, self.ny, self.nx), dtype=np.int64)
        assert lib().orc_stream_index_map(self._h, direction, out.ctypes.data_as(C.POINTER(C.c_int64))) == 0
        return out


def run(w, steps: Optional[int] = None, U0: Optional[np.ndarray] = None, **kw) -> np.ndarray:
    """Initialise from the workload's U(x,0), step, read back U."""
    g = OracleGrid.from_workload(w, **kw)
    if g.n_aux:
        g.set_aux(w.aux_fields())
    g.init_from_U(w.initial_U() if U0 is None else U0)
    g.step(w.steps if steps is None else steps)
    U = g.read_U()
    g.close()
    return U
