"""Thin Python binding of the C ABI in include/etics.h (argument marshalling only).

Every function has the name of the C entry point it calls; all arithmetic of the method runs in the CUDA
kernels behind that call.  PyTorch is used for device memory and streams only.  There is no CPU fallback: if
`libetics.so` is missing or cannot be loaded, `lib()` raises.
"""
from __future__ import annotations

import ctypes as C
import os

import torch

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libetics.so")

ETICS_OK = 0
ETICS_ERR_ARG, ETICS_ERR_LIMIT, ETICS_ERR_ALIGN, ETICS_ERR_WORKSPACE, ETICS_ERR_CUDA = -1, -2, -3, -4, -5
ETICS_ERR_STATIC_LIMIT = -6
ETICS_MAX_LMAX, ETICS_MAX_NMAX = 10, 32
ETICS_STATIC_MAX_TABLE = 1386
ETICS_WS_SCF_COEFFS, ETICS_WS_SCF_FORCE, ETICS_WS_MEX_FORCE, ETICS_WS_SCF_FORCE_F32 = 0, 1, 2, 3
ETICS_WHAT_BOTH, ETICS_WHAT_POTENTIAL, ETICS_WHAT_FORCE = 0, 1, 2

# every symbol include/etics.h declares (tests check that the library exports all of them)
EXPORTS = [
    "etics_status_string", "etics_init", "etics_workspace_bytes", "etics_scf_coeffs", "etics_scf_force",
    "etics_mex_force", "etics_scf_combine", "etics_scf_force_f32", "etics_scf_force_ex", "etics_mex_force_ex", "etics_mex_sort", "etics_host_scratch_bytes", "etics_scf_full_host",
    "etics_mex_full_host", "etics_mex_force_timed", "etics_probe_dfma", "etics_probe_copy",
    "etics_kernel_launches", "etics_step_host_scratch_bytes", "etics_step_host", "etics_stepper_workspace_bytes", "etics_stepper_create", "etics_stepper_step", "etics_stepper_set_coefficient_interval", "etics_stepper_destroy",
    "etics_scf_coeffs_static_max_table", "etics_scf_coeffs_static",
    "etics_mex_shard_rows", "etics_mex_shard_moments", "etics_mex_shard_bases", "etics_mex_shard_force",
]

_lib = None
_vp, _ll, _i, _sz = C.c_void_p, C.c_longlong, C.c_int, C.c_size_t


class EticsError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        super().__init__(f"{where}: {status_string(status)} ({status})")


def lib() -> C.CDLL:
    """Load libetics.so (built by paper_1406_4254_b200.build); fails loudly if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise FileNotFoundError(
            f"{LIB_PATH} not found: build it with `python -m paper_1406_4254_b200.build` "
            "(there is no CPU fallback for the ETICS hot path)")
    L = C.CDLL(LIB_PATH)
    L.etics_status_string.restype = C.c_char_p
    L.etics_status_string.argtypes = [_i]
    L.etics_init.restype = _i
    L.etics_init.argtypes = []
    L.etics_workspace_bytes.restype = _sz
    L.etics_workspace_bytes.argtypes = [_i, _ll, _i, _i]
    L.etics_scf_coeffs.restype = _i
    L.etics_scf_coeffs.argtypes = [_vp, _vp, _ll, _i, _i, _vp, _vp, _vp, _sz, _vp]
    L.etics_scf_coeffs_static_max_table.restype = _sz
    L.etics_scf_coeffs_static_max_table.argtypes = []
    L.etics_scf_coeffs_static.restype = _i
    L.etics_scf_coeffs_static.argtypes = [_vp, _vp, _ll, _i, _i, _vp, _vp, _vp]
    L.etics_scf_force.restype = _i
    L.etics_scf_force.argtypes = [_vp, _ll, _i, _i, _vp, _vp, _vp, _vp, _vp, _sz, _vp]
    L.etics_mex_force.restype = _i
    L.etics_mex_force.argtypes = [_vp, _vp, _ll, _i, _vp, _vp, _vp, _sz, _vp]
    L.etics_scf_force_f32.restype = _i
    L.etics_scf_force_f32.argtypes = [_vp, _ll, _i, _i, _vp, _vp, _i, _vp, _vp, _vp, _sz, _vp]
    L.etics_scf_combine.restype = _i
    L.etics_scf_combine.argtypes = [_vp, _i, _ll, _vp, _vp]
    L.etics_scf_force_ex.restype = _i
    L.etics_scf_force_ex.argtypes = [_vp, _ll, _i, _i, _vp, _vp, _i, _vp, _vp, _vp, _sz, _vp]
    L.etics_mex_force_ex.restype = _i
    L.etics_mex_force_ex.argtypes = [_vp, _vp, _ll, _i, _i, _vp, _vp, _vp, _sz, _vp]
    L.etics_mex_sort.restype = _i
    L.etics_mex_sort.argtypes = [_vp, _ll, _vp, _vp, _vp, _sz, _vp]
    L.etics_mex_shard_rows.restype = _i
    L.etics_mex_shard_rows.argtypes = [_i]
    L.etics_mex_shard_moments.restype = _i
    L.etics_mex_shard_moments.argtypes = [_vp, _vp, _ll, _i, _vp, _vp, _sz, _vp]
    L.etics_mex_shard_bases.restype = _i
    L.etics_mex_shard_bases.argtypes = [_vp, _i, _i, _i, _vp, _vp]
    L.etics_mex_shard_force.restype = _i
    L.etics_mex_shard_force.argtypes = [_ll, _i, _i, _vp, _vp, _vp, _vp, _sz, _vp]
    L.etics_host_scratch_bytes.restype = _sz
    L.etics_host_scratch_bytes.argtypes = [_i, _ll, _i, _i]
    L.etics_scf_full_host.restype = _i
    L.etics_scf_full_host.argtypes = [_vp, _vp, _ll, _i, _i, _vp, _vp, _vp, _vp, _vp, _sz, _vp]
    L.etics_mex_full_host.restype = _i
    L.etics_mex_full_host.argtypes = [_vp, _vp, _ll, _i, _vp, _vp, _vp, _sz, _vp]
    L.etics_mex_force_timed.restype = _i
    L.etics_mex_force_timed.argtypes = [_vp, _vp, _ll, _i, _vp, _vp, _vp, _sz, _vp, C.POINTER(C.c_float)]
    L.etics_kernel_launches.restype = _i
    L.etics_kernel_launches.argtypes = [_i, _ll]
    L.etics_step_host_scratch_bytes.restype = _sz
    L.etics_step_host_scratch_bytes.argtypes = [_ll, _i, _i, _i]
    L.etics_step_host.restype = _i
    L.etics_step_host.argtypes = [_vp, _vp, _ll, _i, _i, _i, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _sz, _vp, _vp]
    L.etics_stepper_workspace_bytes.restype = _sz
    L.etics_stepper_workspace_bytes.argtypes = [_i, _ll, _i, _i]
    L.etics_stepper_create.restype = _i
    L.etics_stepper_create.argtypes = [C.POINTER(_vp), _i, _vp, _vp, _vp, _ll, _i, _i, C.c_double, _vp, _vp, _vp, _sz, _i, _vp]
    L.etics_stepper_step.restype = _i
    L.etics_stepper_step.argtypes = [_vp, _i]
    L.etics_stepper_set_coefficient_interval.restype = _i
    L.etics_stepper_set_coefficient_interval.argtypes = [_vp, _i]
    L.etics_stepper_destroy.restype = _i
    L.etics_stepper_destroy.argtypes = [_vp]
    L.etics_probe_dfma.restype = _i
    L.etics_probe_dfma.argtypes = [_i, _vp, C.POINTER(C.c_double), _vp]
    L.etics_probe_copy.restype = _i
    L.etics_probe_copy.argtypes = [_vp, _vp, _sz, _vp]
    _lib = L
    return L


def status_string(status: int) -> str:
    return lib().etics_status_string(status).decode()


def num_lm(lmax: int) -> int:
    return (lmax + 1) * (lmax + 2) // 2


def _stream(stream) -> int:
    if stream is None:
        return torch.cuda.current_stream().cuda_stream
    return stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream)


def _dev(t: torch.Tensor, name: str, dtype=torch.float64) -> int:
    if not (t.is_cuda and t.dtype == dtype and t.is_contiguous()):
        raise TypeError(f"{name}: expected a contiguous CUDA tensor of dtype {dtype}")
    return t.data_ptr()


def _check(status: int, where: str) -> None:
    if status != ETICS_OK:
        raise EticsError(status, where)


def etics_init() -> None:
    _check(lib().etics_init(), "etics_init")


def etics_workspace_bytes(which: int, N: int, nmax: int, lmax: int) -> int:
    return lib().etics_workspace_bytes(which, N, nmax, lmax)


def _workspace(which: int, N: int, nmax: int, lmax: int, device, workspace):
    need = etics_workspace_bytes(which, N, nmax, lmax)
    if workspace is None:
        workspace = torch.empty(max(need, 256), dtype=torch.uint8, device=device)
    return workspace, workspace.numel() * workspace.element_size()


def etics_scf_coeffs(pos, mass, nmax: int, lmax: int, A=None, B=None, workspace=None, stream=None):
    """pos (3,N), mass (N,) CUDA fp64 -> A, B (T,) CUDA fp64.  See include/etics.h."""
    N = mass.shape[0]
    T = (nmax + 1) * num_lm(lmax)
    if A is None:
        A = torch.empty(T, dtype=torch.float64, device=pos.device)
    if B is None:
        B = torch.empty(T, dtype=torch.float64, device=pos.device)
    workspace, wsb = _workspace(ETICS_WS_SCF_COEFFS, N, nmax, lmax, pos.device, workspace)
    assert pos.shape == (3, N) and A.shape == (T,) and B.shape == (T,)
    s = lib().etics_scf_coeffs(_dev(pos, "pos"), _dev(mass, "mass"), N, nmax, lmax, _dev(A, "A"), _dev(B, "B"),
                               workspace.data_ptr(), wsb, _stream(stream))
    _check(s, "etics_scf_coeffs")
    return A, B


def etics_scf_coeffs_static_max_table() -> int:
    """Largest T = (nmax+1) * num_lm(lmax) etics_scf_coeffs_static accepts."""
    return int(lib().etics_scf_coeffs_static_max_table())


def etics_scf_coeffs_static(pos, mass, nmax: int, lmax: int, A, B, stream=None):
    """etics_scf_coeffs with the block partials in the library's own __device__ array: no workspace, nothing allocated
    (neither here: the caller passes A, B (T,) CUDA fp64).  T <= ETICS_STATIC_MAX_TABLE.  See include/etics.h."""
    N = mass.shape[0]
    T = (nmax + 1) * num_lm(lmax)
    assert pos.shape == (3, N) and A.shape == (T,) and B.shape == (T,)
    s = lib().etics_scf_coeffs_static(_dev(pos, "pos"), _dev(mass, "mass"), N, nmax, lmax, _dev(A, "A"), _dev(B, "B"),
                                      _stream(stream))
    _check(s, "etics_scf_coeffs_static")
    return A, B


def etics_scf_force(pos, nmax: int, lmax: int, A, B, acc=None, pot=None, stream=None):
    """pos (3,N), A, B (T,) CUDA fp64 -> acc (3,N), pot (N,)."""
    N = pos.shape[1]
    T = (nmax + 1) * num_lm(lmax)
    if acc is None:
        acc = torch.empty((3, N), dtype=torch.float64, device=pos.device)
    if pot is None:
        pot = torch.empty(N, dtype=torch.float64, device=pos.device)
    assert pos.shape == (3, N) and A.shape == (T,) and B.shape == (T,) and acc.shape == (3, N) and pot.shape == (N,)
    s = lib().etics_scf_force(_dev(pos, "pos"), N, nmax, lmax, _dev(A, "A"), _dev(B, "B"), _dev(acc, "acc"),
                              _dev(pot, "pot"), None, 0, _stream(stream))
    _check(s, "etics_scf_force")
    return acc, pot


def etics_mex_force(pos, mass, lmax: int, acc=None, pot=None, workspace=None, stream=None):
    """pos (3,N), mass (N,) CUDA fp64 -> acc (3,N), pot (N,) at the particles' original indices."""
    N = mass.shape[0]
    if acc is None:
        acc = torch.empty((3, N), dtype=torch.float64, device=pos.device)
    if pot is None:
        pot = torch.empty(N, dtype=torch.float64, device=pos.device)
    workspace, wsb = _workspace(ETICS_WS_MEX_FORCE, N, 0, lmax, pos.device, workspace)
    assert pos.shape == (3, N) and acc.shape == (3, N) and pot.shape == (N,)
    s = lib().etics_mex_force(_dev(pos, "pos"), _dev(mass, "mass"), N, lmax, _dev(acc, "acc"), _dev(pot, "pot"),
                              workspace.data_ptr(), wsb, _stream(stream))
    _check(s, "etics_mex_force")
    return acc, pot


def etics_scf_combine(parts, out=None, stream=None):
    """parts (R, len) CUDA fp64, the ranks' tables in rank order -> out (len,) = their sum in that order."""
    R, n = parts.shape
    if out is None:
        out = torch.empty(n, dtype=torch.float64, device=parts.device)
    _check(lib().etics_scf_combine(_dev(parts, "parts"), R, n, _dev(out, "out"), _stream(stream)), "etics_scf_combine")
    return out


def _opt(t, name):
    return None if t is None else _dev(t, name)


def etics_scf_force_ex(pos, nmax: int, lmax: int, A, B, what: int, acc=None, pot=None, stream=None):
    """etics_scf_force with a selector: ETICS_WHAT_POTENTIAL returns (None, pot), ETICS_WHAT_FORCE returns (acc, None)."""
    N = pos.shape[1]
    if acc is None and what != ETICS_WHAT_POTENTIAL:
        acc = torch.empty((3, N), dtype=torch.float64, device=pos.device)
    if pot is None and what != ETICS_WHAT_FORCE:
        pot = torch.empty(N, dtype=torch.float64, device=pos.device)
    s = lib().etics_scf_force_ex(_dev(pos, "pos"), N, nmax, lmax, _dev(A, "A"), _dev(B, "B"), what, _opt(acc, "acc"),
                                 _opt(pot, "pot"), None, 0, _stream(stream))
    _check(s, "etics_scf_force_ex")
    return (None if what == ETICS_WHAT_POTENTIAL else acc), (None if what == ETICS_WHAT_FORCE else pot)


def etics_scf_force_f32(pos, nmax: int, lmax: int, A, B, what: int = ETICS_WHAT_BOTH, acc=None, pot=None, workspace=None, stream=None):
    """Single-precision evaluation (fp64 arrays in and out); see include/etics.h."""
    N = pos.shape[1]
    if acc is None and what != ETICS_WHAT_POTENTIAL:
        acc = torch.empty((3, N), dtype=torch.float64, device=pos.device)
    if pot is None and what != ETICS_WHAT_FORCE:
        pot = torch.empty(N, dtype=torch.float64, device=pos.device)
    workspace, wsb = _workspace(ETICS_WS_SCF_FORCE_F32, N, nmax, lmax, pos.device, workspace)
    s = lib().etics_scf_force_f32(_dev(pos, "pos"), N, nmax, lmax, _dev(A, "A"), _dev(B, "B"), what, _opt(acc, "acc"),
                                  _opt(pot, "pot"), workspace.data_ptr(), wsb, _stream(stream))
    _check(s, "etics_scf_force_f32")
    return (None if what == ETICS_WHAT_POTENTIAL else acc), (None if what == ETICS_WHAT_FORCE else pot)


def etics_mex_force_ex(pos, mass, lmax: int, what: int, acc=None, pot=None, workspace=None, stream=None):
    """etics_mex_force with a selector (see etics_scf_force_ex)."""
    N = mass.shape[0]
    if acc is None and what != ETICS_WHAT_POTENTIAL:
        acc = torch.empty((3, N), dtype=torch.float64, device=pos.device)
    if pot is None and what != ETICS_WHAT_FORCE:
        pot = torch.empty(N, dtype=torch.float64, device=pos.device)
    workspace, wsb = _workspace(ETICS_WS_MEX_FORCE, N, 0, lmax, pos.device, workspace)
    s = lib().etics_mex_force_ex(_dev(pos, "pos"), _dev(mass, "mass"), N, lmax, what, _opt(acc, "acc"), _opt(pot, "pot"),
                                 workspace.data_ptr(), wsb, _stream(stream))
    _check(s, "etics_mex_force_ex")
    return (None if what == ETICS_WHAT_POTENTIAL else acc), (None if what == ETICS_WHAT_FORCE else pot)


MEX_STAGES = ("sort", "sort_fallback", "gather_totals", "unused", "tilescan", "evaluate")


def etics_mex_force_timed(pos, mass, lmax: int, acc, pot, workspace, stream=None):
    """etics_mex_force with CUDA events between the stages; synchronises; returns {stage: ms}."""
    N = mass.shape[0]
    ms = (C.c_float * 6)()
    s = lib().etics_mex_force_timed(_dev(pos, "pos"), _dev(mass, "mass"), N, lmax, _dev(acc, "acc"), _dev(pot, "pot"),
                                    workspace.data_ptr(), workspace.numel() * workspace.element_size(), _stream(stream), ms)
    _check(s, "etics_mex_force_timed")
    return dict(zip(MEX_STAGES, [float(v) for v in ms]))


def etics_mex_sort(pos, keys_sorted=None, perm=None, workspace=None, stream=None):
    """pos (3,N) CUDA fp64 -> keys_sorted (N,) int64 holding the uint64 bit patterns, perm (N,) int32 holding uint32."""
    N = pos.shape[1]
    if keys_sorted is None:
        keys_sorted = torch.empty(N, dtype=torch.int64, device=pos.device)
    if perm is None:
        perm = torch.empty(N, dtype=torch.int32, device=pos.device)
    workspace, wsb = _workspace(ETICS_WS_MEX_FORCE, N, 0, 0, pos.device, workspace)
    s = lib().etics_mex_sort(_dev(pos, "pos"), N, _dev(keys_sorted, "keys_sorted", torch.int64),
                             _dev(perm, "perm", torch.int32), workspace.data_ptr(), wsb, _stream(stream))
    _check(s, "etics_mex_sort")
    return keys_sorted, perm


def etics_mex_shard_rows(lmax: int) -> int:
    return lib().etics_mex_shard_rows(lmax)


def etics_mex_shard_moments(pos, mass, lmax: int, workspace, totals=None, stream=None):
    """Phase 1 of the radius-partitioned MEX for one shard: -> totals (R,), the shard's moment vector.  `workspace` (a CUDA
    byte tensor of etics_workspace_bytes(ETICS_WS_MEX_FORCE, N, 0, lmax)) carries the shard's state to etics_mex_shard_force."""
    N = mass.shape[0]
    if totals is None:
        totals = torch.empty(etics_mex_shard_rows(lmax), dtype=torch.float64, device=pos.device)
    assert pos.shape == (3, N)
    s = lib().etics_mex_shard_moments(_dev(pos, "pos"), _dev(mass, "mass"), N, lmax, _dev(totals, "totals"),
                                      workspace.data_ptr(), workspace.numel() * workspace.element_size(), _stream(stream))
    _check(s, "etics_mex_shard_moments")
    return totals


def etics_mex_shard_bases(parts, rank: int, lmax: int, base=None, stream=None):
    """parts (nparts, R) CUDA fp64, the shards' moment vectors in radius order -> base (R,) of shard `rank`."""
    nparts, R = parts.shape
    assert R == etics_mex_shard_rows(lmax)
    if base is None:
        base = torch.empty(R, dtype=torch.float64, device=parts.device)
    _check(lib().etics_mex_shard_bases(_dev(parts, "parts"), nparts, rank, lmax, _dev(base, "base"), _stream(stream)),
           "etics_mex_shard_bases")
    return base


def etics_mex_shard_force(N: int, lmax: int, what: int, base, workspace, acc=None, pot=None, stream=None):
    """Phase 2: scans from `base`, evaluation; acc (3,N), pot (N,) at the shard's local indices."""
    if acc is None and what != ETICS_WHAT_POTENTIAL:
        acc = torch.empty((3, N), dtype=torch.float64, device=base.device)
    if pot is None and what != ETICS_WHAT_FORCE:
        pot = torch.empty(N, dtype=torch.float64, device=base.device)
    s = lib().etics_mex_shard_force(N, lmax, what, _dev(base, "base"), _opt(acc, "acc"), _opt(pot, "pot"),
                                    workspace.data_ptr(), workspace.numel() * workspace.element_size(), _stream(stream))
    _check(s, "etics_mex_shard_force")
    return (None if what == ETICS_WHAT_POTENTIAL else acc), (None if what == ETICS_WHAT_FORCE else pot)


def etics_host_scratch_bytes(method: int, N: int, nmax: int, lmax: int) -> int:
    return lib().etics_host_scratch_bytes(method, N, nmax, lmax)


def _host(t: torch.Tensor, name: str) -> int:
    if t.is_cuda or t.dtype != torch.float64 or not t.is_contiguous():
        raise TypeError(f"{name}: expected a contiguous CPU float64 tensor")
    return t.data_ptr()


def etics_scf_full_host(pos_h, mass_h, nmax: int, lmax: int, acc_h, pot_h, scratch, A_h=None, B_h=None, stream=None):
    """Host buffers in/out (pinned recommended); `scratch` is a CUDA uint8 tensor of etics_host_scratch_bytes(0,...)."""
    N = mass_h.shape[0]
    s = lib().etics_scf_full_host(_host(pos_h, "pos_h"), _host(mass_h, "mass_h"), N, nmax, lmax,
                                  None if A_h is None else _host(A_h, "A_h"), None if B_h is None else _host(B_h, "B_h"),
                                  _host(acc_h, "acc_h"), _host(pot_h, "pot_h"),
                                  scratch.data_ptr(), scratch.numel() * scratch.element_size(), _stream(stream))
    _check(s, "etics_scf_full_host")


def etics_mex_full_host(pos_h, mass_h, lmax: int, acc_h, pot_h, scratch, stream=None):
    N = mass_h.shape[0]
    s = lib().etics_mex_full_host(_host(pos_h, "pos_h"), _host(mass_h, "mass_h"), N, lmax,
                                  _host(acc_h, "acc_h"), _host(pot_h, "pot_h"),
                                  scratch.data_ptr(), scratch.numel() * scratch.element_size(), _stream(stream))
    _check(s, "etics_mex_full_host")


def etics_kernel_launches(which: int, N: int) -> int:
    return lib().etics_kernel_launches(which, N)


def etics_step_host_scratch_bytes(N: int, nmax: int, lmax: int, mex_lmax: int) -> int:
    return lib().etics_step_host_scratch_bytes(N, nmax, lmax, mex_lmax)


def etics_step_host(pos_h, mass_h, nmax: int, lmax: int, mex_lmax: int, acc_scf_h, pot_scf_h, acc_mex_h, pot_mex_h, scratch,
                    A_h=None, B_h=None, stream=None, copy_stream=None):
    """One upload, SCF + MEX full force calculations, results to host buffers; copy_stream (a torch stream) overlaps the copies."""
    N = mass_h.shape[0]
    s = lib().etics_step_host(_host(pos_h, "pos_h"), _host(mass_h, "mass_h"), N, nmax, lmax, mex_lmax,
                              None if A_h is None else _host(A_h, "A_h"), None if B_h is None else _host(B_h, "B_h"),
                              _host(acc_scf_h, "acc_scf_h"), _host(pot_scf_h, "pot_scf_h"), _host(acc_mex_h, "acc_mex_h"),
                              _host(pot_mex_h, "pot_mex_h"), scratch.data_ptr(), scratch.numel() * scratch.element_size(),
                              _stream(stream), None if copy_stream is None else _stream(copy_stream))
    _check(s, "etics_step_host")


def etics_probe_dfma(iters: int, sink, stream=None) -> float:
    """Enqueue the fp64-FMA probe; returns the number of floating-point operations it performs."""
    flops = C.c_double(0.0)
    s = lib().etics_probe_dfma(iters, _dev(sink, "sink"), C.byref(flops), _stream(stream))
    _check(s, "etics_probe_dfma")
    return flops.value


def etics_probe_copy(dst, src, stream=None) -> int:
    nbytes = src.numel() * src.element_size()
    s = lib().etics_probe_copy(dst.data_ptr(), src.data_ptr(), nbytes, _stream(stream))
    _check(s, "etics_probe_copy")
    return 2 * nbytes


def etics_stepper_workspace_bytes(method: int, N: int, nmax: int, lmax: int) -> int:
    return lib().etics_stepper_workspace_bytes(method, N, nmax, lmax)


def etics_stepper_create(method: int, pos, vel, mass, nmax: int, lmax: int, dt: float, acc, pot, workspace, use_graph: bool = True,
                         stream=None):
    """Returns the opaque handle (a ctypes void pointer) of a stepper over the caller's CUDA tensors."""
    h = _vp()
    s = lib().etics_stepper_create(C.byref(h), method, _dev(pos, "pos"), _dev(vel, "vel"), _dev(mass, "mass"), mass.shape[0], nmax, lmax,
                                   float(dt), _dev(acc, "acc"), _dev(pot, "pot"), workspace.data_ptr(),
                                   workspace.numel() * workspace.element_size(), int(bool(use_graph)), _stream(stream))
    _check(s, "etics_stepper_create")
    return h


def etics_stepper_step(handle, nsteps: int = 1) -> None:
    _check(lib().etics_stepper_step(handle, nsteps), "etics_stepper_step")


def etics_stepper_set_coefficient_interval(handle, every: int) -> None:
    _check(lib().etics_stepper_set_coefficient_interval(handle, every), "etics_stepper_set_coefficient_interval")


def etics_stepper_destroy(handle) -> None:
    _check(lib().etics_stepper_destroy(handle), "etics_stepper_destroy")


class Stepper:
    """Keeps the tensors a stepper handle refers to alive (etics_stepper_* of include/etics.h): kick-drift-kick steps with
    the SCF (method 0) or MEX (method 1) force.  pos, vel are updated in place; acc, pot hold the acceleration / potential
    at the current positions."""

    def __init__(self, method: int, pos, vel, mass, dt: float, nmax: int = 0, lmax: int = 0, use_graph: bool = True, stream=None):
        N = mass.shape[0]
        self.pos, self.vel, self.mass = pos, vel, mass
        self.acc = torch.empty((3, N), dtype=torch.float64, device=pos.device)
        self.pot = torch.empty(N, dtype=torch.float64, device=pos.device)
        self.workspace = torch.empty(etics_stepper_workspace_bytes(method, N, nmax, lmax), dtype=torch.uint8, device=pos.device)
        self._h = etics_stepper_create(method, pos, vel, mass, nmax, lmax, dt, self.acc, self.pot, self.workspace, use_graph, stream)

    def set_coefficient_interval(self, every: int) -> None:
        etics_stepper_set_coefficient_interval(self._h, every)

    def step(self, nsteps: int = 1) -> None:
        etics_stepper_step(self._h, nsteps)

    def close(self) -> None:
        if self._h is not None:
            etics_stepper_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
