"""paper_2607_05668_b200 -- Python binding of liblbmk.so (the C-ABI of include/lbmk.h).

Argument marshalling only: every step of the collide-and-stream path runs in the CUDA kernels behind the
C-ABI.  PyTorch supplies device memory (the workspace tensor) and the CUDA stream, nothing else.  There is
no CPU fallback: importing works without a GPU (so the symbol table can be checked), but every compute call
needs a CUDA device and raises `LbmkError` otherwise.  This package never imports `oracle/`.

Two layers:
  * module-level functions named exactly like the C entry points (`lbmk_system_create`, `lbmk_step`, ...),
    taking/returning plain Python values and ctypes handles;
  * `System` / `Grid`: small RAII holders that own the handles and the torch workspace, plus
    `Grid.from_workload(w)` for the seeded workloads of `workloads/`.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

import numpy as np

from . import _build

__all__ = ["LbmkError", "System", "Grid", "lib", "SYSTEM_ID", "STATUS"]

LBMK_OK = 0
STATUS = {0: "LBMK_OK", 1: "LBMK_EINVAL", 2: "LBMK_ENOMEM", 3: "LBMK_ECUDA", 4: "LBMK_ESUBCHAR", 5: "LBMK_ESTATE",
          6: "LBMK_EUNSUPPORTED"}
LBMK_D2Q5, LBMK_D3Q7 = 0, 1
LBMK_F64, LBMK_F32_SHIFTED, LBMK_F64_SHIFTED = 0, 1, 2
LBMK_PERIODIC, LBMK_DIRICHLET_MMS = 0, 1
LBMK_OPT_PATTERN, LBMK_OPT_KERNEL, LBMK_OPT_STEPPING = 0, 1, 2
LBMK_STEPPING_AUTO, LBMK_STEPPING_LAUNCH, LBMK_STEPPING_PERSISTENT, LBMK_STEPPING_CLUSTER, LBMK_STEPPING_RESIDENT = 0, 1, 2, 3, 4
LBMK_PATTERN_AUTO, LBMK_PATTERN_PULL2, LBMK_PATTERN_AA = 0, 1, 2
LBMK_KERNEL_AUTO, LBMK_KERNEL_NODE, LBMK_KERNEL_ROW, LBMK_KERNEL_TWOPASS = 0, 1, 2, 3
SYSTEM_ID = {"advection2d": 0, "burgers2d": 1, "swe2d": 2, "euler2d": 3, "adr2d": 4, "nsf3d": 5, "mhd3d": 6, "urf2d": 7, "maxwell2d": 8, "allencahn2d": 9, "inse2d": 10, "elasticity2d": 11, "nsf2d": 12,
             "swe2d_bathy": 13, "hcnsf3d": 14, "mhd2d": 15}
PRECISION = {"f64": LBMK_F64, "f32s": LBMK_F32_SHIFTED, "f64s": LBMK_F64_SHIFTED}
PATTERN = {"auto": 0, "pull2": 1, "aa": 2}
KERNEL = {"auto": 0, "node": 1, "row": 2, "twopass": 3}
STEPPING = {"auto": 0, "launch": 1, "persistent": 2, "cluster": 3, "resident": 4}

# every symbol include/lbmk.h declares: (restype, argtypes)
_dp = C.POINTER(C.c_double)
_vp = C.c_void_p
SYMBOLS = {
    "lbmk_system_create": (C.c_int, [C.c_int, C.c_int, _dp, C.c_int, C.POINTER(_vp)]),
    "lbmk_system_info": (C.c_int, [_vp] + [C.POINTER(C.c_int)] * 4),
    "lbmk_system_aux_count": (C.c_int, [_vp, C.POINTER(C.c_int)]),
    "lbmk_system_set_relaxation": (C.c_int, [_vp, _dp, C.c_int, C.c_double]),
    "lbmk_system_set_omega": (C.c_int, [_vp, _dp, C.c_int]),
    "lbmk_system_set_reference": (C.c_int, [_vp, _dp, C.c_int]),
    "lbmk_system_set_mms": (C.c_int, [_vp, C.c_int, _dp, C.c_int]),
    "lbmk_system_set_wave_speed_bound": (C.c_int, [_vp, C.c_double]),
    "lbmk_system_set_collision": (C.c_int, [_vp, C.c_int, C.c_double]),
    "lbmk_grid_omega_plus": (C.c_int, [_vp, _dp]),
    "lbmk_system_destroy": (None, [_vp]),
    "lbmk_grid_create": (C.c_int, [_vp, C.c_int, C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_int, _vp, C.POINTER(_vp)]),
    "lbmk_grid_set_option": (C.c_int, [_vp, C.c_int, C.c_longlong]),
    "lbmk_grid_get_option": (C.c_int, [_vp, C.c_int, C.POINTER(C.c_longlong)]),
    "lbmk_grid_workspace_bytes": (C.c_int, [_vp, C.POINTER(C.c_size_t)]),
    "lbmk_grid_bind_workspace": (C.c_int, [_vp, _vp, C.c_size_t]),
    "lbmk_grid_destroy": (None, [_vp]),
    "lbmk_init_from_U": (C.c_int, [_vp, _vp, C.c_int, C.c_double]),
    "lbmk_set_populations": (C.c_int, [_vp, _vp, C.c_int, C.c_double]),
    "lbmk_set_aux_fields": (C.c_int, [_vp, _vp, C.c_int]),
    "lbmk_step": (C.c_int, [_vp, C.c_int]),
    "lbmk_read_U": (C.c_int, [_vp, _vp, C.c_int]),
    "lbmk_read_populations": (C.c_int, [_vp, _vp, C.c_int]),
    "lbmk_time": (C.c_int, [_vp, C.POINTER(C.c_longlong), _dp]),
    "lbmk_check_subcharacteristic": (C.c_int, [_vp, _dp]),
    "lbmk_error_norms": (C.c_int, [_vp, _dp]),
    "lbmk_error_norms_noalloc": (C.c_int, [_vp, _vp]),
    "lbmk_grid_set_origin": (C.c_int, [_vp, C.c_int, C.c_int, C.c_int]),
    "lbmk_grid_set_slab": (C.c_int, [_vp, C.c_int]),
    "lbmk_halo_bytes": (C.c_int, [_vp, C.POINTER(C.c_size_t)]),
    "lbmk_halo_pack": (C.c_int, [_vp, _vp, _vp]),
    "lbmk_halo_unpack": (C.c_int, [_vp, _vp, _vp]),
    "lbmk_halo_pack_on": (C.c_int, [_vp, _vp, _vp, _vp]),
    "lbmk_halo_unpack_on": (C.c_int, [_vp, _vp, _vp, _vp]),
    "lbmk_step_slab": (C.c_int, [_vp]),
    "lbmk_stream_wait_boundary": (C.c_int, [_vp, _vp]),
    "lbmk_step_slab_peer": (C.c_int, [_vp]),
    "lbmk_grid_population_buffers": (C.c_int, [_vp, C.POINTER(_vp), C.POINTER(_vp), C.POINTER(C.c_longlong)]),
    "lbmk_grid_set_halo_peers": (C.c_int, [_vp, _vp, _vp, C.c_longlong, _vp, _vp]),
    "lbmk_grid_wait_stream": (C.c_int, [_vp, _vp]),
    "lbmk_stream_index_map": (C.c_int, [_vp, C.c_int, _vp, C.c_int]),
    "lbmk_generated_flux": (C.c_int, [C.c_int, _dp, _dp, _dp, C.c_int, C.c_double, C.c_double, C.c_double, _dp, _dp]),
    "lbmk_flux_selfcheck": (C.c_int, [_vp, _dp]),
    "lbmk_lattice_constants": (C.c_int, [C.c_int, C.POINTER(C.c_int), _dp, _dp]),
    "lbmk_grid_omega": (C.c_int, [_vp, _dp]),
    "lbmk_grid_launch_count": (C.c_int, [_vp, C.POINTER(C.c_longlong)]),
    "lbmk_last_step_ms": (C.c_int, [_vp, C.POINTER(C.c_float)]),
    "lbmk_last_error": (C.c_char_p, [_vp]),
    "lbmk_version": (C.c_char_p, []),
    "lbmk_copy_bandwidth": (C.c_int, [_vp, _vp, C.c_size_t, C.c_int, _vp, _dp]),
}


class LbmkError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"{STATUS.get(status, status)}: {message}")
        self.status = status


_lib = None


def lib() -> C.CDLL:
    """Load (building in-tree if needed) liblbmk.so.  Fails loudly if it cannot be built or loaded."""
    global _lib
    if _lib is None:
        path = _build.LIB if (os.path.exists(_build.LIB) and not _build.needs_build()) else _build.build()
        L = C.CDLL(path)
        for name, (res, args) in SYMBOLS.items():
            fn = getattr(L, name)           # AttributeError if a declared symbol is missing
            fn.restype = res
            fn.argtypes = args
        _lib = L
    return _lib


def _check(status: int, grid=None):
    if status != LBMK_OK:
        msg = lib().lbmk_last_error(grid)
        raise LbmkError(status, msg.decode() if msg else "")


def _darr(v: Sequence[float]):
    a = np.ascontiguousarray(np.atleast_1d(np.asarray(v, dtype=np.float64)))
    return a, a.ctypes.data_as(_dp)


# ---------------------------------------------------------------------------------- C-named thin wrappers
def lbmk_version() -> str:
    return lib().lbmk_version().decode()


def lbmk_last_error(grid_h=None) -> str:
    msg = lib().lbmk_last_error(grid_h)
    return msg.decode() if msg else ""


def lbmk_system_create(system_id: int, lattice: int, params: Sequence[float]):
    h = _vp()
    a, p = _darr(list(params) if len(params) else [0.0])
    _check(lib().lbmk_system_create(system_id, lattice, p, len(params), C.byref(h)))
    return h


def lbmk_system_info(sys_h):
    v = [C.c_int() for _ in range(4)]
    _check(lib().lbmk_system_info(sys_h, *[C.byref(x) for x in v]))
    return tuple(x.value for x in v)      # m_conserved, m_total, dim, Q


def lbmk_system_aux_count(sys_h) -> int:
    v = C.c_int()
    _check(lib().lbmk_system_aux_count(sys_h, C.byref(v)))
    return v.value


def lbmk_system_set_relaxation(sys_h, tau_R, g_tau: float):
    a, p = _darr(tau_R)
    _check(lib().lbmk_system_set_relaxation(sys_h, p, a.size, float(g_tau)))


def lbmk_system_set_omega(sys_h, omega):
    a, p = _darr(omega)
    _check(lib().lbmk_system_set_omega(sys_h, p, a.size))


def lbmk_system_set_reference(sys_h, U0):
    a, p = _darr(U0)
    _check(lib().lbmk_system_set_reference(sys_h, p, a.size))


def lbmk_system_set_mms(sys_h, mms_id: int, mms_params: Sequence[float]):
    a, p = _darr(list(mms_params) if len(mms_params) else [0.0])
    _check(lib().lbmk_system_set_mms(sys_h, int(mms_id), p, len(mms_params)))


def lbmk_system_set_collision(sys_h, collision: int, magic: float = 0.25):
    _check(lib().lbmk_system_set_collision(sys_h, int(collision), float(magic)))


def lbmk_grid_omega_plus(grid_h, m_total: int):
    o = np.zeros(m_total)
    _check(lib().lbmk_grid_omega_plus(grid_h, o.ctypes.data_as(_dp)), grid_h)
    return o


def lbmk_system_set_wave_speed_bound(sys_h, s_max: float):
    _check(lib().lbmk_system_set_wave_speed_bound(sys_h, float(s_max)))


def lbmk_system_destroy(sys_h):
    lib().lbmk_system_destroy(sys_h)


def lbmk_grid_create(sys_h, nx, ny, nz, bc, dx, lam, precision, cuda_stream: int):
    h = _vp()
    _check(lib().lbmk_grid_create(sys_h, nx, ny, nz, bc, float(dx), float(lam), precision, _vp(cuda_stream), C.byref(h)))
    return h


def lbmk_grid_set_option(grid_h, key: int, value: int):
    _check(lib().lbmk_grid_set_option(grid_h, key, value), grid_h)


def lbmk_grid_get_option(grid_h, key: int) -> int:
    v = C.c_longlong()
    _check(lib().lbmk_grid_get_option(grid_h, key, C.byref(v)), grid_h)
    return v.value


def lbmk_grid_workspace_bytes(grid_h) -> int:
    v = C.c_size_t()
    _check(lib().lbmk_grid_workspace_bytes(grid_h, C.byref(v)), grid_h)
    return v.value


def lbmk_grid_bind_workspace(grid_h, device_ptr: int, nbytes: int):
    _check(lib().lbmk_grid_bind_workspace(grid_h, _vp(device_ptr), nbytes), grid_h)


def lbmk_grid_destroy(grid_h):
    lib().lbmk_grid_destroy(grid_h)


def lbmk_init_from_U(grid_h, ptr: int, on_device: bool, t0: float = 0.0):
    _check(lib().lbmk_init_from_U(grid_h, _vp(ptr), int(on_device), float(t0)), grid_h)


def lbmk_set_populations(grid_h, ptr: int, on_device: bool, t0: float = 0.0):
    _check(lib().lbmk_set_populations(grid_h, _vp(ptr), int(on_device), float(t0)), grid_h)


def lbmk_set_aux_fields(grid_h, ptr: int, on_device: bool):
    _check(lib().lbmk_set_aux_fields(grid_h, _vp(ptr), int(on_device)), grid_h)


def lbmk_step(grid_h, n_steps: int):
    _check(lib().lbmk_step(grid_h, int(n_steps)), grid_h)


def lbmk_read_U(grid_h, ptr: int, on_device: bool):
    _check(lib().lbmk_read_U(grid_h, _vp(ptr), int(on_device)), grid_h)


def lbmk_read_populations(grid_h, ptr: int, on_device: bool):
    _check(lib().lbmk_read_populations(grid_h, _vp(ptr), int(on_device)), grid_h)


def lbmk_time(grid_h):
    s, t = C.c_longlong(), C.c_double()
    _check(lib().lbmk_time(grid_h, C.byref(s), C.byref(t)), grid_h)
    return s.value, t.value


def lbmk_check_subcharacteristic(grid_h, raise_on_violation: bool = True):
    out = np.zeros(3)
    st = lib().lbmk_check_subcharacteristic(grid_h, out.ctypes.data_as(_dp))
    if st != LBMK_OK and (raise_on_violation or st != 4):
        _check(st, grid_h)
    return (float(out[0]), float(out[1]), float(out[2])), st


def lbmk_grid_set_origin(grid_h, ox: int, oy: int, oz: int):
    _check(lib().lbmk_grid_set_origin(grid_h, ox, oy, oz), grid_h)


def lbmk_grid_set_slab(grid_h, enable: bool):
    _check(lib().lbmk_grid_set_slab(grid_h, int(enable)), grid_h)


def lbmk_halo_bytes(grid_h) -> int:
    n = C.c_size_t()
    _check(lib().lbmk_halo_bytes(grid_h, C.byref(n)), grid_h)
    return n.value


def lbmk_halo_pack(grid_h, send_lo: int, send_hi: int):
    _check(lib().lbmk_halo_pack(grid_h, _vp(send_lo), _vp(send_hi)), grid_h)


def lbmk_halo_unpack(grid_h, recv_lo: int, recv_hi: int):
    _check(lib().lbmk_halo_unpack(grid_h, _vp(recv_lo), _vp(recv_hi)), grid_h)


def lbmk_halo_pack_on(grid_h, send_lo: int, send_hi: int, cuda_stream: int):
    _check(lib().lbmk_halo_pack_on(grid_h, _vp(send_lo), _vp(send_hi), _vp(cuda_stream)), grid_h)


def lbmk_halo_unpack_on(grid_h, recv_lo: int, recv_hi: int, cuda_stream: int):
    _check(lib().lbmk_halo_unpack_on(grid_h, _vp(recv_lo), _vp(recv_hi), _vp(cuda_stream)), grid_h)


def lbmk_step_slab(grid_h):
    _check(lib().lbmk_step_slab(grid_h), grid_h)


def lbmk_step_slab_peer(grid_h):
    _check(lib().lbmk_step_slab_peer(grid_h), grid_h)


def lbmk_grid_population_buffers(grid_h):
    """(f0, f1, first node of the upper ghost plane): device pointers of the grid's two population buffers."""
    f0, f1, n0 = _vp(), _vp(), C.c_longlong()
    _check(lib().lbmk_grid_population_buffers(grid_h, C.byref(f0), C.byref(f1), C.byref(n0)), grid_h)
    return f0.value, f1.value, n0.value


def lbmk_grid_set_halo_peers(grid_h, lo_f0: int, lo_f1: int, lo_upper_ghost_first_node: int, hi_f0: int, hi_f1: int):
    _check(lib().lbmk_grid_set_halo_peers(grid_h, _vp(lo_f0), _vp(lo_f1), int(lo_upper_ghost_first_node), _vp(hi_f0), _vp(hi_f1)), grid_h)


def lbmk_stream_wait_boundary(grid_h, cuda_stream: int):
    _check(lib().lbmk_stream_wait_boundary(grid_h, _vp(cuda_stream)), grid_h)


def lbmk_grid_wait_stream(grid_h, cuda_stream: int):
    _check(lib().lbmk_grid_wait_stream(grid_h, _vp(cuda_stream)), grid_h)


def lbmk_error_norms(grid_h, m_total: int) -> np.ndarray:
    out = np.zeros((m_total, 6))
    _check(lib().lbmk_error_norms(grid_h, out.ctypes.data_as(_dp)), grid_h)
    return out


LBMK_NOALLOC_SCRATCH_BYTES = 4 * 1024 * 1024


def lbmk_error_norms_noalloc(grid_h, out_device_ptr: int):
    """[m_total][6] doubles into DEVICE memory at out_device_ptr; enqueued on the grid's stream, nothing allocated, not synchronised."""
    _check(lib().lbmk_error_norms_noalloc(grid_h, _vp(out_device_ptr)), grid_h)


def lbmk_stream_index_map(grid_h, direction: int, ptr: int, on_device: bool):
    _check(lib().lbmk_stream_index_map(grid_h, direction, _vp(ptr), int(on_device)), grid_h)


def lbmk_generated_flux(system_id: int, U, A, params, dx: float, lam: float, g_tau: float, m_total: int):
    Ua, Up = _darr(U)
    Aa, Ap = _darr(A if A is not None and len(A) else [0.0])
    Pa, Pp = _darr(list(params) if len(params) else [0.0])
    F, S = np.zeros((m_total, 3)), np.zeros(m_total)
    _check(lib().lbmk_generated_flux(system_id, Up, Ap, Pp, len(params), float(dx), float(lam), float(g_tau),
                                     F.ctypes.data_as(_dp), S.ctypes.data_as(_dp)))
    return F, S


def lbmk_flux_selfcheck(grid_h) -> float:
    v = C.c_double()
    _check(lib().lbmk_flux_selfcheck(grid_h, C.byref(v)), grid_h)
    return v.value


def lbmk_lattice_constants(lattice: int):
    Q = 5 if lattice == LBMK_D2Q5 else 7
    c = np.zeros((Q, 3), dtype=np.int32)
    w = np.zeros(Q)
    cs2 = C.c_double()
    _check(lib().lbmk_lattice_constants(lattice, c.ctypes.data_as(C.POINTER(C.c_int)), w.ctypes.data_as(_dp), C.byref(cs2)))
    return c, w, cs2.value


def lbmk_grid_omega(grid_h, m_total: int):
    o = np.zeros(m_total)
    _check(lib().lbmk_grid_omega(grid_h, o.ctypes.data_as(_dp)), grid_h)
    return o


def lbmk_grid_launch_count(grid_h) -> int:
    v = C.c_longlong()
    _check(lib().lbmk_grid_launch_count(grid_h, C.byref(v)), grid_h)
    return v.value


def lbmk_last_step_ms(grid_h) -> float:
    v = C.c_float()
    _check(lib().lbmk_last_step_ms(grid_h, C.byref(v)), grid_h)
    return v.value


def lbmk_copy_bandwidth(dst_ptr: int, src_ptr: int, nbytes: int, reps: int, cuda_stream: int) -> float:
    v = C.c_double()
    _check(lib().lbmk_copy_bandwidth(_vp(dst_ptr), _vp(src_ptr), nbytes, reps, _vp(cuda_stream), C.byref(v)))
    return v.value


# ---------------------------------------------------------------------------------- RAII holders
class System:
    """Declared system of conservation laws (handle owner)."""

    def __init__(self, name: str, params: Sequence[float] = (), tau_R=0.0, g_tau: float = 0.0,
                 U_ref: Optional[Sequence[float]] = None, mms_id: int = 0, mms_params: Sequence[float] = (),
                 omega=None, s_max: float = 0.0, collision: str = "bgk", trt_magic: float = 0.25):
        self.name = name
        sid = SYSTEM_ID[name]
        lattice = LBMK_D3Q7 if name in ("nsf3d", "mhd3d", "hcnsf3d") else LBMK_D2Q5
        self.h = lbmk_system_create(sid, lattice, list(params))
        self.m_conserved, self.m_total, self.dim, self.Q = lbmk_system_info(self.h)
        self.n_aux = lbmk_system_aux_count(self.h)
        lbmk_system_set_relaxation(self.h, tau_R, g_tau if self.m_total > self.m_conserved else 1.0)
        if U_ref is not None:
            lbmk_system_set_reference(self.h, list(U_ref))
        if mms_id:
            lbmk_system_set_mms(self.h, mms_id, list(mms_params))
        if omega is not None:
            lbmk_system_set_omega(self.h, omega)
        if s_max:
            lbmk_system_set_wave_speed_bound(self.h, s_max)
        if collision != "bgk":
            lbmk_system_set_collision(self.h, {"bgk": 0, "trt": 1, "regularized": 2}[collision], trt_magic)

    def close(self):
        if getattr(self, "h", None):
            lbmk_system_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class Grid:
    """A grid bound to a torch-owned device workspace on `device`, enqueuing on torch's current stream."""

    def __init__(self, system: System, nx: int, ny: int, nz: int, dx: float, lam: float, precision: str = "f64",
                 bc: str = "periodic", pattern: str = "auto", kernel: str = "auto", device: str = "cuda:0",
                 origin: Sequence[int] = (0, 0, 0), slab: bool = False, stepping: str = "auto"):
        import torch
        if not torch.cuda.is_available():
            raise LbmkError(3, "no CUDA device: the collide-and-stream path has no CPU fallback")
        self.torch = torch
        self.system = system
        self.nx, self.ny, self.nz = nx, ny, nz
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.stream = torch.cuda.current_stream(self.device)
        self.h = lbmk_grid_create(system.h, nx, ny, nz, {"periodic": 0, "dirichlet_mms": 1}[bc], dx, lam,
                                  PRECISION[precision], self.stream.cuda_stream)
        if tuple(origin) != (0, 0, 0):
            lbmk_grid_set_origin(self.h, *[int(o) for o in origin])
        self.slab = bool(slab)
        if pattern != "auto":
            lbmk_grid_set_option(self.h, LBMK_OPT_PATTERN, PATTERN[pattern])
        if kernel != "auto":
            lbmk_grid_set_option(self.h, LBMK_OPT_KERNEL, KERNEL[kernel])
        if stepping != "auto":
            lbmk_grid_set_option(self.h, LBMK_OPT_STEPPING, STEPPING[stepping])
        if slab:
            lbmk_grid_set_slab(self.h, True)
        self.workspace_bytes = lbmk_grid_workspace_bytes(self.h)
        self.workspace = torch.empty(self.workspace_bytes, dtype=torch.uint8, device=self.device)
        lbmk_grid_bind_workspace(self.h, self.workspace.data_ptr(), self.workspace_bytes)
        self.pattern = {1: "pull2", 2: "aa"}[lbmk_grid_get_option(self.h, LBMK_OPT_PATTERN)]
        self.kernel = {1: "node", 2: "row", 3: "twopass"}[lbmk_grid_get_option(self.h, LBMK_OPT_KERNEL)]
        self.stepping = {1: "launch", 2: "persistent", 3: "cluster", 4: "resident"}[lbmk_grid_get_option(self.h, LBMK_OPT_STEPPING)]

    @classmethod
    def from_workload(cls, w, precision: Optional[str] = None, omega=None, declare_bound: bool = True, collision: str = "bgk",
                      trt_magic: float = 0.25, **kw):
        s = System(w.system, params=w.params, tau_R=w.tau_R, g_tau=w.g_tau, U_ref=w.U_ref, mms_id=w.mms_id,
                   mms_params=w.mms_params if w.mms_id else (), omega=omega, s_max=w.s_max if declare_bound else 0.0,
                   collision=collision, trt_magic=trt_magic)
        kw.setdefault("origin", getattr(w, "origin", (0, 0, 0)))
        g = cls(s, w.nx, w.ny, w.nz, w.dx, w.lam, precision=precision or w.precision, **kw)
        if s.n_aux:
            g.set_aux_fields(w.aux_fields())        # prescribed coefficient fields are inputs of the workload, like U(x, 0)
        return g

    # shapes
    @property
    def shape_U(self):
        return (self.system.m_total, self.nz, self.ny, self.nx)

    @property
    def shape_f(self):
        return (self.system.m_total, self.system.Q, self.nz, self.ny, self.nx)

    @property
    def shape_aux(self):
        return (self.system.n_aux, self.nz, self.ny, self.nx)

    def _in(self, a, shape):
        """(pointer, on_device, keepalive) of a numpy array (host) or torch tensor (host or device)."""
        torch = self.torch
        if isinstance(a, np.ndarray):
            a = np.ascontiguousarray(a, dtype=np.float64)
            assert a.shape == tuple(shape), (a.shape, shape)
            return a.ctypes.data, False, a
        assert a.dtype == torch.float64 and a.is_contiguous() and tuple(a.shape) == tuple(shape)
        return a.data_ptr(), a.is_cuda, a

    def init_from_U(self, U, t0: float = 0.0):
        p, dev, keep = self._in(U, self.shape_U)
        lbmk_init_from_U(self.h, p, dev, t0)

    def set_aux_fields(self, A):
        p, dev, keep = self._in(A, self.shape_aux)
        lbmk_set_aux_fields(self.h, p, dev)

    def set_populations(self, f, t0: float = 0.0):
        p, dev, keep = self._in(f, self.shape_f)
        lbmk_set_populations(self.h, p, dev, t0)

    def step(self, n: int = 1):
        lbmk_step(self.h, n)

    def read_U(self, out=None):
        """fp64 U[m_total][nz][ny][nx]: into `out` (numpy / torch, host or device) or a new numpy array."""
        if out is None:
            out = np.empty(self.shape_U)
        p, dev, keep = self._in(out, self.shape_U)
        assert keep is out, "output must be C-contiguous fp64"
        lbmk_read_U(self.h, p, dev)
        return out

    def read_populations(self, out=None):
        if out is None:
            out = np.empty(self.shape_f)
        p, dev, keep = self._in(out, self.shape_f)
        assert keep is out
        lbmk_read_populations(self.h, p, dev)
        return out

    def stream_index_map(self, direction: int) -> np.ndarray:
        out = np.empty((self.nz, self.ny, self.nx), dtype=np.int64)
        lbmk_stream_index_map(self.h, direction, out.ctypes.data, False)
        return out

    def max_wave_speed(self):
        return lbmk_check_subcharacteristic(self.h, raise_on_violation=False)

    def error_norms(self):
        """Relative (L1, L2, Linf) errors per component against the manufactured solution at the current time."""
        o = lbmk_error_norms(self.h, self.system.m_total)
        with np.errstate(divide="ignore", invalid="ignore"):
            return np.stack([o[:, 0] / o[:, 3], np.sqrt(o[:, 1] / o[:, 4]), o[:, 2] / o[:, 5]], axis=1)

    def check_subcharacteristic(self):
        return lbmk_check_subcharacteristic(self.h, raise_on_violation=True)[0]

    def omega(self):
        return lbmk_grid_omega(self.h, self.system.m_total)

    def time(self):
        return lbmk_time(self.h)

    def launch_count(self) -> int:
        return lbmk_grid_launch_count(self.h)

    def last_step_ms(self) -> float:
        return lbmk_last_step_ms(self.h)

    def synchronize(self):
        self.stream.synchronize()

    def close(self):
        if getattr(self, "h", None):
            self.torch.cuda.synchronize(self.device)
            lbmk_grid_destroy(self.h)
            self.h = None
            self.workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def run(w, steps: Optional[int] = None, U0=None, **kw) -> np.ndarray:
    """Initialise from the workload's U(x,0), step, read back U (the GPU counterpart of a whole config run)."""
    g = Grid.from_workload(w, **kw)
    g.init_from_U(w.initial_U() if U0 is None else U0)
    g.step(w.steps if steps is None else steps)
    U = g.read_U()
    g.close()
    return U
