"""ctypes binding over libnbody_b200.so -- same names as the C ABI, argument marshalling only.

Every step of the path runs in the library's CUDA kernels; nothing here computes.  PyTorch
tensors are used for device memory and streams only (``tensor.data_ptr()``,
``torch.cuda.current_stream().cuda_stream``).  There is no CPU fallback: if the shared library
is missing or no sm_100 device is present, calls raise.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Tuple

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libnbody_b200.so")

NB_OK = 0
_lib = None


class NBError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        l = lib()
        msg = l.nb_status_string(status).decode()
        cuda = l.nb_last_cuda_error()
        super().__init__(f"{where}: status {status} ({msg}); last cudaError_t = {cuda}")


def lib() -> ctypes.CDLL:
    """Loads the in-tree shared library (raises if it has not been built: no fallback)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise FileNotFoundError(
                f"{LIB_PATH} is missing: build it with `python -m paper_astro_ph_0703100_b200.build` "
                "(or __graft_entry__.build()); there is no fallback path")
        l = ctypes.CDLL(LIB_PATH)
        i64, f32, p, ci = ctypes.c_int64, ctypes.c_float, ctypes.c_void_p, ctypes.c_int
        l.nb_force.argtypes = [i64, p, i64, p, p, f32, p, p, p]
        l.nb_force.restype = ci
        l.nb_force_noalloc.argtypes = [i64, p, i64, p, p, f32, p, p, p]
        l.nb_force_noalloc.restype = ci
        l.nb_force_host.argtypes = [i64, p, i64, p, p, f32, p, p]
        l.nb_force_host.restype = ci
        l.nb_leapfrog_kdk.argtypes = [i64, p, p, p, f32, f32, i64, p, p, p]
        l.nb_leapfrog_kdk.restype = ci
        l.nb_kick_drift.argtypes = [i64, p, p, p, f32, ci, f32, p]
        l.nb_kick_drift.restype = ci
        l.nb_kick.argtypes = [i64, p, p, f32, p]
        l.nb_kick.restype = ci
        l.nb_force_jerk.argtypes = [i64, p, p, i64, p, p, p, f32, p, p, p, p]
        l.nb_force_jerk.restype = ci
        for fn in (l.nb_cunbody_force, l.nb_cunbody_force_jerk_pot, l.nb_cunbody_lennard_jones):
            fn.argtypes = [p, p, p, i64, i64, p]
            fn.restype = ci
        l.nb_pack_j.argtypes = [i64, p, p, p, p]
        l.nb_pack_j.restype = ci
        l.nb_force_packed.argtypes = [i64, p, i64, p, f32, p, p, p]
        l.nb_force_packed.restype = ci
        l.nb_force_eps_i.argtypes = [i64, p, p, i64, p, p, p, p, p]
        l.nb_force_eps_i.restype = ci
        l.nb_force_batched.argtypes = [i64, p, p, i64, p, i64, p, p, f32, p, p, p]
        l.nb_force_batched.restype = ci
        l.nb_force_batched_packed.argtypes = [i64, p, p, i64, p, i64, p, f32, p, p, p]
        l.nb_force_batched_packed.restype = ci
        l.nb_force_batched_indexed.argtypes = [i64, p, p, i64, p, i64, p, i64, p, f32, p, p, p]
        l.nb_force_batched_indexed.restype = ci
        l.nb_force_jerk_host.argtypes = [i64, p, p, i64, p, p, p, f32, p, p, p]
        l.nb_force_jerk_host.restype = ci
        l.nb_plan_query_jerk.argtypes = [i64, i64, ci, ctypes.POINTER(i64)]
        l.nb_plan_query_jerk.restype = ci
        l.nb_hermite4.argtypes = [i64, p, p, p, f32, f32, i64, p, p, p, p]
        l.nb_hermite4.restype = ci
        l.nb_hermite4_block_step.argtypes = [i64, p, p, p, p, p, p, i64, p, ctypes.c_double, f32, p]
        l.nb_hermite4_block_step.restype = ci
        l.nb_block_schedule.argtypes = [i64, p, p, p, p, p, p]
        l.nb_block_schedule.restype = ci
        l.nb_block_step_size.argtypes = [i64, p, p, p, p, p, f32, p, p]
        l.nb_block_step_size.restype = ci
        l.nb_plan_query.argtypes = [i64, i64, ci, ctypes.POINTER(i64)]
        l.nb_plan_query.restype = ci
        l.nb_plan_query_small.argtypes = [i64, i64, ci, ctypes.POINTER(i64)]
        l.nb_plan_query_small.restype = ci
        l.nb_plan_query_small_jerk.argtypes = [i64, i64, ci, ctypes.POINTER(i64)]
        l.nb_plan_query_small_jerk.restype = ci
        l.nb_debug_set.argtypes = [ctypes.c_char_p, ctypes.c_char_p]
        l.nb_debug_set.restype = ci
        l.nb_debug_plan_exhaustive.argtypes = [i64, i64, ci, ci, ctypes.POINTER(i64)]
        l.nb_debug_plan_exhaustive.restype = ci
        l.nb_debug_plans_computed.restype = i64
        l.nb_release_stream.argtypes = [p]
        l.nb_release_stream.restype = ci
        l.nb_last_launch_count.restype = i64
        l.nb_release_workspace.restype = ci
        l.nb_profile_enable.argtypes = [ci]
        l.nb_profile_enable.restype = ci
        l.nb_profile_read.argtypes = [ctypes.POINTER(i64), ctypes.POINTER(ctypes.c_double)]
        l.nb_profile_read.restype = ci
        l.nb_status_string.argtypes = [ci]
        l.nb_status_string.restype = ctypes.c_char_p
        l.nb_last_cuda_error.restype = ci
        l.nb_version.restype = ci
        _lib = l
    return _lib


def _check(status: int, where: str) -> None:
    if status != NB_OK:
        raise NBError(status, where)


def _dev_f32(t, name: str, shape_tail: Tuple[int, ...]):
    import torch
    if not isinstance(t, torch.Tensor) or not t.is_cuda or t.dtype != torch.float32 or not t.is_contiguous():
        raise TypeError(f"{name} must be a contiguous float32 CUDA tensor")
    if tuple(t.shape[1:]) != shape_tail:
        raise ValueError(f"{name} must have shape [n{''.join(', %d' % s for s in shape_tail)}]")
    return t


def _stream_ptr(stream) -> int:
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return int(s.cuda_stream)


def force(x_i, x_j, m_j, eps2: float, acc_out=None, pot_out=None, want_pot: bool = True, stream=None):
    """nb_force on CUDA tensors.  Returns (acc [n_i,3], pot [n_i] or None); asynchronous on the stream."""
    import torch
    _dev_f32(x_i, "x_i", (3,)); _dev_f32(x_j, "x_j", (3,)); _dev_f32(m_j, "m_j", ())
    n_i, n_j = x_i.shape[0], x_j.shape[0]
    if m_j.shape[0] != n_j:
        raise ValueError("m_j length != n_j")
    if acc_out is None:
        acc_out = torch.empty((n_i, 3), dtype=torch.float32, device=x_i.device)
    if pot_out is None and want_pot:
        pot_out = torch.empty((n_i,), dtype=torch.float32, device=x_i.device)
    _dev_f32(acc_out, "acc_out", (3,))
    if pot_out is not None:
        _dev_f32(pot_out, "pot_out", ())
    with torch.cuda.device(x_i.device):
        st = lib().nb_force(n_i, x_i.data_ptr(), n_j, x_j.data_ptr(), m_j.data_ptr(), float(eps2),
                            acc_out.data_ptr(), None if pot_out is None else pot_out.data_ptr(), _stream_ptr(stream))
    _check(st, "nb_force")
    return acc_out, pot_out


NOALLOC_MAX_I = 4096            # NB_NOALLOC_MAX_I (include/nbody_b200.h)


def force_noalloc(x_i, x_j, m_j, eps2: float, acc_out, pot_out=None, stream=None):
    """nb_force_noalloc on CUDA tensors: nb_force without any device allocation (n_i <= NOALLOC_MAX_I; the scratch is a
    static array inside the library, shared by all calls on the device).  The caller passes the outputs, so that this
    wrapper allocates nothing either.  Returns (acc_out, pot_out); asynchronous on the stream."""
    import torch
    _dev_f32(x_i, "x_i", (3,)); _dev_f32(x_j, "x_j", (3,)); _dev_f32(m_j, "m_j", ())
    n_i, n_j = x_i.shape[0], x_j.shape[0]
    if m_j.shape[0] != n_j:
        raise ValueError("m_j length != n_j")
    _dev_f32(acc_out, "acc_out", (3,))
    if acc_out.shape[0] != n_i or (pot_out is not None and pot_out.shape[0] != n_i):
        raise ValueError("output length != n_i")
    if pot_out is not None:
        _dev_f32(pot_out, "pot_out", ())
    with torch.cuda.device(x_i.device):
        st = lib().nb_force_noalloc(n_i, x_i.data_ptr(), n_j, x_j.data_ptr(), m_j.data_ptr(), float(eps2),
                                    acc_out.data_ptr(), None if pot_out is None else pot_out.data_ptr(), _stream_ptr(stream))
    _check(st, "nb_force_noalloc")
    return acc_out, pot_out


def force_jerk(x_i, v_i, x_j, v_j, m_j, eps2: float, acc_out=None, jerk_out=None, pot_out=None, want_pot: bool = True,
               stream=None):
    """nb_force_jerk on CUDA tensors.  Returns (acc [n_i,3], jerk [n_i,3], pot [n_i] or None); asynchronous."""
    import torch
    for t, name in ((x_i, "x_i"), (v_i, "v_i"), (x_j, "x_j"), (v_j, "v_j")):
        _dev_f32(t, name, (3,))
    _dev_f32(m_j, "m_j", ())
    n_i, n_j = x_i.shape[0], x_j.shape[0]
    if v_i.shape[0] != n_i or v_j.shape[0] != n_j or m_j.shape[0] != n_j:
        raise ValueError("array lengths differ")
    if acc_out is None:
        acc_out = torch.empty((n_i, 3), dtype=torch.float32, device=x_i.device)
    if jerk_out is None:
        jerk_out = torch.empty((n_i, 3), dtype=torch.float32, device=x_i.device)
    if pot_out is None and want_pot:
        pot_out = torch.empty((n_i,), dtype=torch.float32, device=x_i.device)
    _dev_f32(acc_out, "acc_out", (3,)); _dev_f32(jerk_out, "jerk_out", (3,))
    if pot_out is not None:
        _dev_f32(pot_out, "pot_out", ())
    with torch.cuda.device(x_i.device):
        st = lib().nb_force_jerk(n_i, x_i.data_ptr(), v_i.data_ptr(), n_j, x_j.data_ptr(), v_j.data_ptr(), m_j.data_ptr(),
                                 float(eps2), acc_out.data_ptr(), jerk_out.data_ptr(),
                                 None if pot_out is None else pot_out.data_ptr(), _stream_ptr(stream))
    _check(st, "nb_force_jerk")
    return acc_out, jerk_out, pot_out


def _cunbody(fn_name: str, p_xj, p_xi, idim: int, jdim: int, fdim: int, p_fi, stream):
    import torch
    _dev_f32(p_xj, "p_xj", (jdim,)); _dev_f32(p_xi, "p_xi", (idim,))
    ni, nj = p_xi.shape[0], p_xj.shape[0]
    if p_fi is None:
        p_fi = torch.empty((ni, fdim), dtype=torch.float32, device=p_xi.device)
    _dev_f32(p_fi, "p_fi", (fdim,))
    with torch.cuda.device(p_xi.device):
        st = getattr(lib(), fn_name)(p_xj.data_ptr(), p_xi.data_ptr(), p_fi.data_ptr(), ni, nj, _stream_ptr(stream))
    _check(st, fn_name)
    return p_fi


def cunbody_force(p_xj, p_xi, p_fi=None, stream=None):
    """nb_cunbody_force: the paper's cunbody_api call for the Fig. A.3 pipeline.  p_xj [nj,4], p_xi [ni,4] -> p_fi [ni,3]."""
    return _cunbody("nb_cunbody_force", p_xj, p_xi, 4, 4, 3, p_fi, stream)


def cunbody_force_jerk_pot(p_xj, p_xi, p_fi=None, stream=None):
    """nb_cunbody_force_jerk_pot: the Fig. A.4 pipeline.  p_xj [nj,7], p_xi [ni,6] -> p_fi [ni,7]."""
    return _cunbody("nb_cunbody_force_jerk_pot", p_xj, p_xi, 6, 7, 7, p_fi, stream)


def cunbody_lennard_jones(p_xj, p_xi, p_fi=None, stream=None):
    """nb_cunbody_lennard_jones: 12-6 Lennard-Jones with Lorentz-Berthelot mixing.  p_xj [nj,5], p_xi [ni,5] =
    (x, y, z, sigma/2, sqrt(eps)) -> p_fi [ni,4] = (Fx, Fy, Fz, U)."""
    return _cunbody("nb_cunbody_lennard_jones", p_xj, p_xi, 5, 5, 4, p_fi, stream)


def pack_j(x_j, m_j, xm_out, stream=None):
    """nb_pack_j: writes (x, y, z, m) records of x_j / m_j into the first n_j rows of xm_out [>= n_j, 4]."""
    _dev_f32(x_j, "x_j", (3,)); _dev_f32(m_j, "m_j", ()); _dev_f32(xm_out, "xm_out", (4,))
    n_j = x_j.shape[0]
    if m_j.shape[0] != n_j or xm_out.shape[0] < n_j:
        raise ValueError("array lengths differ")
    import torch
    with torch.cuda.device(x_j.device):
        st = lib().nb_pack_j(n_j, x_j.data_ptr(), m_j.data_ptr(), xm_out.data_ptr(), _stream_ptr(stream))
    _check(st, "nb_pack_j")
    return xm_out


def force_packed(x_i, xm_j, eps2: float, acc_out=None, pot_out=None, want_pot: bool = True, stream=None):
    """nb_force_packed on CUDA tensors: xm_j is [n_j, 4] = (x, y, z, m) per j-particle."""
    import torch
    _dev_f32(x_i, "x_i", (3,)); _dev_f32(xm_j, "xm_j", (4,))
    n_i, n_j = x_i.shape[0], xm_j.shape[0]
    if acc_out is None:
        acc_out = torch.empty((n_i, 3), dtype=torch.float32, device=x_i.device)
    if pot_out is None and want_pot:
        pot_out = torch.empty((n_i,), dtype=torch.float32, device=x_i.device)
    with torch.cuda.device(x_i.device):
        st = lib().nb_force_packed(n_i, x_i.data_ptr(), n_j, xm_j.data_ptr(), float(eps2), acc_out.data_ptr(),
                                   None if pot_out is None else pot_out.data_ptr(), _stream_ptr(stream))
    _check(st, "nb_force_packed")
    return acc_out, pot_out


def force_eps_i(x_i, eps2_i, x_j, m_j, acc_out=None, pot_out=None, want_pot: bool = True, stream=None):
    """nb_force_eps_i on CUDA tensors: one softening (squared) per i-particle."""
    import torch
    _dev_f32(x_i, "x_i", (3,)); _dev_f32(eps2_i, "eps2_i", ()); _dev_f32(x_j, "x_j", (3,)); _dev_f32(m_j, "m_j", ())
    n_i, n_j = x_i.shape[0], x_j.shape[0]
    if eps2_i.shape[0] != n_i or m_j.shape[0] != n_j:
        raise ValueError("array lengths differ")
    if acc_out is None:
        acc_out = torch.empty((n_i, 3), dtype=torch.float32, device=x_i.device)
    if pot_out is None and want_pot:
        pot_out = torch.empty((n_i,), dtype=torch.float32, device=x_i.device)
    with torch.cuda.device(x_i.device):
        st = lib().nb_force_eps_i(n_i, x_i.data_ptr(), eps2_i.data_ptr(), n_j, x_j.data_ptr(), m_j.data_ptr(),
                                  acc_out.data_ptr(), None if pot_out is None else pot_out.data_ptr(), _stream_ptr(stream))
    _check(st, "nb_force_eps_i")
    return acc_out, pot_out


def force_batched(i_offsets, j_offsets, x_i, x_j, m_j, eps2: float, acc_out=None, pot_out=None, want_pot: bool = True,
                  stream=None):
    """nb_force_batched on CUDA tensors; i_offsets / j_offsets are int32 CUDA tensors of length n_batch + 1."""
    import torch
    _dev_f32(x_i, "x_i", (3,)); _dev_f32(x_j, "x_j", (3,)); _dev_f32(m_j, "m_j", ())
    for t, name in ((i_offsets, "i_offsets"), (j_offsets, "j_offsets")):
        if not isinstance(t, torch.Tensor) or not t.is_cuda or t.dtype != torch.int32 or not t.is_contiguous() or t.dim() != 1:
            raise TypeError(f"{name} must be a contiguous 1-D int32 CUDA tensor")
    if i_offsets.shape[0] != j_offsets.shape[0] or i_offsets.shape[0] < 1:
        raise ValueError("i_offsets and j_offsets must both have n_batch + 1 entries")
    n_batch, n_i, n_j = i_offsets.shape[0] - 1, x_i.shape[0], x_j.shape[0]
    if m_j.shape[0] != n_j:
        raise ValueError("m_j length != n_j")
    if acc_out is None:
        acc_out = torch.zeros((n_i, 3), dtype=torch.float32, device=x_i.device)
    if pot_out is None and want_pot:
        pot_out = torch.zeros((n_i,), dtype=torch.float32, device=x_i.device)
    with torch.cuda.device(x_i.device):
        st = lib().nb_force_batched(n_batch, i_offsets.data_ptr(), j_offsets.data_ptr(), n_i, x_i.data_ptr(), n_j,
                                    x_j.data_ptr(), m_j.data_ptr(), float(eps2), acc_out.data_ptr(),
                                    None if pot_out is None else pot_out.data_ptr(), _stream_ptr(stream))
    _check(st, "nb_force_batched")
    return acc_out, pot_out


def force_batched_packed(i_offsets, j_offsets, x_i, xm_j, eps2: float, acc_out=None, pot_out=None, want_pot: bool = True,
                         stream=None):
    """nb_force_batched_packed on CUDA tensors: the list records as packed (x, y, z, m) rows [n_j_total, 4]."""
    import torch
    _dev_f32(x_i, "x_i", (3,)); _dev_f32(xm_j, "xm_j", (4,))
    for t, name in ((i_offsets, "i_offsets"), (j_offsets, "j_offsets")):
        if not isinstance(t, torch.Tensor) or not t.is_cuda or t.dtype != torch.int32 or not t.is_contiguous() or t.dim() != 1:
            raise TypeError(f"{name} must be a contiguous 1-D int32 CUDA tensor")
    if i_offsets.shape[0] != j_offsets.shape[0] or i_offsets.shape[0] < 1:
        raise ValueError("i_offsets and j_offsets must both have n_batch + 1 entries")
    n_batch, n_i, n_j = i_offsets.shape[0] - 1, x_i.shape[0], xm_j.shape[0]
    if acc_out is None:
        acc_out = torch.zeros((n_i, 3), dtype=torch.float32, device=x_i.device)
    if pot_out is None and want_pot:
        pot_out = torch.zeros((n_i,), dtype=torch.float32, device=x_i.device)
    with torch.cuda.device(x_i.device):
        st = lib().nb_force_batched_packed(n_batch, i_offsets.data_ptr(), j_offsets.data_ptr(), n_i, x_i.data_ptr(), n_j,
                                           xm_j.data_ptr(), float(eps2), acc_out.data_ptr(),
                                           None if pot_out is None else pot_out.data_ptr(), _stream_ptr(stream))
    _check(st, "nb_force_batched_packed")
    return acc_out, pot_out


def force_batched_indexed(i_offsets, j_offsets, x_i, j_index, xm_p, eps2: float, acc_out=None, pot_out=None,
                          want_pot: bool = True, stream=None):
    """nb_force_batched_indexed on CUDA tensors: lists as int32 indices [n_list_total] into packed records xm_p [n_p, 4]."""
    import torch
    _dev_f32(x_i, "x_i", (3,)); _dev_f32(xm_p, "xm_p", (4,))
    for t, name in ((i_offsets, "i_offsets"), (j_offsets, "j_offsets"), (j_index, "j_index")):
        if not isinstance(t, torch.Tensor) or not t.is_cuda or t.dtype != torch.int32 or not t.is_contiguous() or t.dim() != 1:
            raise TypeError(f"{name} must be a contiguous 1-D int32 CUDA tensor")
    if i_offsets.shape[0] != j_offsets.shape[0] or i_offsets.shape[0] < 1:
        raise ValueError("i_offsets and j_offsets must both have n_batch + 1 entries")
    n_batch, n_i = i_offsets.shape[0] - 1, x_i.shape[0]
    if acc_out is None:
        acc_out = torch.zeros((n_i, 3), dtype=torch.float32, device=x_i.device)
    if pot_out is None and want_pot:
        pot_out = torch.zeros((n_i,), dtype=torch.float32, device=x_i.device)
    with torch.cuda.device(x_i.device):
        st = lib().nb_force_batched_indexed(n_batch, i_offsets.data_ptr(), j_offsets.data_ptr(), n_i, x_i.data_ptr(),
                                            j_index.shape[0], j_index.data_ptr(), xm_p.shape[0], xm_p.data_ptr(), float(eps2),
                                            acc_out.data_ptr(), None if pot_out is None else pot_out.data_ptr(), _stream_ptr(stream))
    _check(st, "nb_force_batched_indexed")
    return acc_out, pot_out


def force_jerk_host(x_i, v_i, x_j, v_j, m_j, eps2: float, acc_out=None, jerk_out=None, pot_out=None, want_pot: bool = True):
    """nb_force_jerk_host on numpy float32 arrays (or pinned CPU tensors' numpy views).  Blocking."""
    import numpy as np
    same = x_i is x_j and v_i is v_j
    xj = np.ascontiguousarray(x_j, dtype=np.float32).reshape(-1, 3)
    vj = np.ascontiguousarray(v_j, dtype=np.float32).reshape(-1, 3)
    mj = np.ascontiguousarray(m_j, dtype=np.float32).reshape(-1)
    xi = xj if same else np.ascontiguousarray(x_i, dtype=np.float32).reshape(-1, 3)
    vi = vj if same else np.ascontiguousarray(v_i, dtype=np.float32).reshape(-1, 3)
    n_i, n_j = xi.shape[0], xj.shape[0]
    if vi.shape[0] != n_i or vj.shape[0] != n_j or mj.shape[0] != n_j:
        raise ValueError("array lengths differ")
    if acc_out is None:
        acc_out = np.empty((n_i, 3), dtype=np.float32)
    if jerk_out is None:
        jerk_out = np.empty((n_i, 3), dtype=np.float32)
    if pot_out is None and want_pot:
        pot_out = np.empty((n_i,), dtype=np.float32)
    st = lib().nb_force_jerk_host(n_i, xi.ctypes.data, vi.ctypes.data, n_j, xj.ctypes.data, vj.ctypes.data, mj.ctypes.data,
                                  float(eps2), acc_out.ctypes.data, jerk_out.ctypes.data,
                                  None if pot_out is None else pot_out.ctypes.data)
    _check(st, "nb_force_jerk_host")
    return acc_out, jerk_out, pot_out


def force_host(x_i, x_j, m_j, eps2: float, want_pot: bool = True, acc_out=None, pot_out=None):
    """nb_force_host on numpy float32 arrays (or pinned CPU tensors' numpy views).  Blocking."""
    import numpy as np
    xi = np.ascontiguousarray(x_i, dtype=np.float32).reshape(-1, 3) if x_i is not x_j else None
    xj = np.ascontiguousarray(x_j, dtype=np.float32).reshape(-1, 3)
    mj = np.ascontiguousarray(m_j, dtype=np.float32).reshape(-1)
    if xi is None:
        xi = xj
    n_i, n_j = xi.shape[0], xj.shape[0]
    if mj.shape[0] != n_j:
        raise ValueError("m_j length != n_j")
    if acc_out is None:
        acc_out = np.empty((n_i, 3), dtype=np.float32)
    if pot_out is None and want_pot:
        pot_out = np.empty((n_i,), dtype=np.float32)
    st = lib().nb_force_host(n_i, xi.ctypes.data, n_j, xj.ctypes.data, mj.ctypes.data, float(eps2),
                             acc_out.ctypes.data, None if pot_out is None else pot_out.ctypes.data)
    _check(st, "nb_force_host")
    return acc_out, pot_out


def leapfrog_kdk(x, v, m, eps2: float, dt: float, n_steps: int, acc_io=None, pot_out=None, want_pot: bool = True,
                 stream=None):
    """nb_leapfrog_kdk: x, v updated IN PLACE.  Returns (acc, pot) at the final time."""
    import torch
    _dev_f32(x, "x", (3,)); _dev_f32(v, "v", (3,)); _dev_f32(m, "m", ())
    n = x.shape[0]
    if v.shape[0] != n or m.shape[0] != n:
        raise ValueError("x, v, m lengths differ")
    if acc_io is None:
        acc_io = torch.empty((n, 3), dtype=torch.float32, device=x.device)
    if pot_out is None and want_pot:
        pot_out = torch.empty((n,), dtype=torch.float32, device=x.device)
    with torch.cuda.device(x.device):
        st = lib().nb_leapfrog_kdk(n, x.data_ptr(), v.data_ptr(), m.data_ptr(), float(eps2), float(dt), int(n_steps),
                                   acc_io.data_ptr(), None if pot_out is None else pot_out.data_ptr(),
                                   _stream_ptr(stream))
    _check(st, "nb_leapfrog_kdk")
    return acc_io, pot_out


def hermite4(x, v, m, eps2: float, dt: float, n_steps: int, acc_io=None, jerk_io=None, pot_out=None, want_pot: bool = True,
             stream=None):
    """nb_hermite4: x, v updated IN PLACE.  Returns (acc, jerk, pot) carried out of the last step."""
    import torch
    _dev_f32(x, "x", (3,)); _dev_f32(v, "v", (3,)); _dev_f32(m, "m", ())
    n = x.shape[0]
    if v.shape[0] != n or m.shape[0] != n:
        raise ValueError("x, v, m lengths differ")
    if acc_io is None:
        acc_io = torch.empty((n, 3), dtype=torch.float32, device=x.device)
    if jerk_io is None:
        jerk_io = torch.empty((n, 3), dtype=torch.float32, device=x.device)
    if pot_out is None and want_pot:
        pot_out = torch.empty((n,), dtype=torch.float32, device=x.device)
    with torch.cuda.device(x.device):
        st = lib().nb_hermite4(n, x.data_ptr(), v.data_ptr(), m.data_ptr(), float(eps2), float(dt), int(n_steps),
                               acc_io.data_ptr(), jerk_io.data_ptr(), None if pot_out is None else pot_out.data_ptr(),
                               _stream_ptr(stream))
    _check(st, "nb_hermite4")
    return acc_io, jerk_io, pot_out


def hermite4_block_step(x, v, m, acc_io, jerk_io, t, active, t_now: float, eps2: float, stream=None) -> None:
    """nb_hermite4_block_step: the rows of x, v, acc_io, jerk_io, t listed in ``active`` are updated IN PLACE."""
    import torch
    _dev_f32(x, "x", (3,)); _dev_f32(v, "v", (3,)); _dev_f32(m, "m", ())
    _dev_f32(acc_io, "acc_io", (3,)); _dev_f32(jerk_io, "jerk_io", (3,))
    n = x.shape[0]
    if not (v.shape[0] == m.shape[0] == acc_io.shape[0] == jerk_io.shape[0] == n):
        raise ValueError("x, v, m, acc_io, jerk_io lengths differ")
    if not (t.is_cuda and t.dtype == torch.float64 and t.is_contiguous() and tuple(t.shape) == (n,)):
        raise ValueError("t must be a contiguous CUDA float64 tensor of shape (n,)")
    if not (active.is_cuda and active.dtype == torch.int32 and active.is_contiguous() and active.dim() == 1):
        raise ValueError("active must be a contiguous 1-D CUDA int32 tensor")
    if t.device != x.device or active.device != x.device:
        raise ValueError("tensors live on different devices")
    with torch.cuda.device(x.device):
        st = lib().nb_hermite4_block_step(n, x.data_ptr(), v.data_ptr(), m.data_ptr(), acc_io.data_ptr(),
                                          jerk_io.data_ptr(), t.data_ptr(), int(active.shape[0]),
                                          active.data_ptr() if active.shape[0] else None, float(t_now), float(eps2),
                                          _stream_ptr(stream))
    _check(st, "nb_hermite4_block_step")


def block_schedule(t, dt, t_next_out=None, active_out=None, n_act_out=None, stream=None):
    """nb_block_schedule on CUDA float64 tensors.  Returns (t_next [1] f64, active [n] int32, n_act [1] int32), all on
    the device and asynchronous: only active[:n_act] is meaningful."""
    import torch
    for a, name in ((t, "t"), (dt, "dt")):
        if not (isinstance(a, torch.Tensor) and a.is_cuda and a.dtype == torch.float64 and a.is_contiguous() and a.dim() == 1):
            raise TypeError(f"{name} must be a contiguous 1-D float64 CUDA tensor")
    n = t.shape[0]
    if dt.shape[0] != n or dt.device != t.device:
        raise ValueError("t and dt differ in length or device")
    if t_next_out is None:
        t_next_out = torch.empty((1,), dtype=torch.float64, device=t.device)
    if active_out is None:
        active_out = torch.empty((n,), dtype=torch.int32, device=t.device)
    if n_act_out is None:
        n_act_out = torch.empty((1,), dtype=torch.int32, device=t.device)
    if active_out.dtype != torch.int32 or active_out.numel() < n or not active_out.is_contiguous():
        raise ValueError("active_out must be a contiguous int32 tensor with at least n entries")
    with torch.cuda.device(t.device):
        st = lib().nb_block_schedule(n, t.data_ptr() if n else None, dt.data_ptr() if n else None, t_next_out.data_ptr(),
                                     active_out.data_ptr() if n else None, n_act_out.data_ptr(), _stream_ptr(stream))
    _check(st, "nb_block_schedule")
    return t_next_out, active_out, n_act_out


def block_step_size(a0, j0, a1, j1, h, eta: float, dt_out=None, stream=None):
    """nb_block_step_size on CUDA float32 tensors.  Returns dt [n] float32; asynchronous."""
    import torch
    for z, name in ((a0, "a0"), (j0, "j0"), (a1, "a1"), (j1, "j1")):
        _dev_f32(z, name, (3,))
    _dev_f32(h, "h", ())
    n = a0.shape[0]
    if not (j0.shape[0] == a1.shape[0] == j1.shape[0] == h.shape[0] == n):
        raise ValueError("array lengths differ")
    if dt_out is None:
        dt_out = torch.empty((n,), dtype=torch.float32, device=a0.device)
    _dev_f32(dt_out, "dt_out", ())
    with torch.cuda.device(a0.device):
        st = lib().nb_block_step_size(n, a0.data_ptr(), j0.data_ptr(), a1.data_ptr(), j1.data_ptr(), h.data_ptr(), float(eta),
                                      dt_out.data_ptr(), _stream_ptr(stream))
    _check(st, "nb_block_step_size")
    return dt_out


def kick_drift(x, v, acc, h: float, n_kicks: int, dt: float, stream=None) -> None:
    """nb_kick_drift on CUDA tensors [n, 3]: v += acc h (once or twice), x += v dt; in place."""
    import torch
    _dev_f32(x, "x", (3,)); _dev_f32(v, "v", (3,)); _dev_f32(acc, "acc", (3,))
    with torch.cuda.device(x.device):
        st = lib().nb_kick_drift(x.shape[0], x.data_ptr(), v.data_ptr(), acc.data_ptr(), float(h), int(n_kicks), float(dt), _stream_ptr(stream))
    _check(st, "nb_kick_drift")


def kick(v, acc, h: float, stream=None) -> None:
    """nb_kick on CUDA tensors [n, 3]: v += acc h; in place."""
    import torch
    _dev_f32(v, "v", (3,)); _dev_f32(acc, "acc", (3,))
    with torch.cuda.device(v.device):
        st = lib().nb_kick(v.shape[0], v.data_ptr(), acc.data_ptr(), float(h), _stream_ptr(stream))
    _check(st, "nb_kick")


def plan_query(n_i: int, n_j: int, sm_count: int = 148) -> dict:
    out = (ctypes.c_int64 * 8)()
    _check(lib().nb_plan_query(int(n_i), int(n_j), int(sm_count), out), "nb_plan_query")
    keys = ("K", "WI", "WJ", "S", "tiles_i", "tile_i", "tile_j", "stages")
    return dict(zip(keys, [int(v) for v in out]))


def plan_query_jerk(n_i: int, n_j: int, sm_count: int = 148) -> dict:
    out = (ctypes.c_int64 * 8)()
    _check(lib().nb_plan_query_jerk(int(n_i), int(n_j), int(sm_count), out), "nb_plan_query_jerk")
    keys = ("K", "WI", "WJ", "S", "tiles_i", "tile_i", "tile_j", "stages")
    return dict(zip(keys, [int(v) for v in out]))


def plan_query_small(n_i: int, n_j: int, sm_count: int = 148) -> dict:
    """The small-i-set kernel's decomposition for (n_i, n_j); "default" = nb_force takes that kernel for this shape."""
    out = (ctypes.c_int64 * 8)()
    _check(lib().nb_plan_query_small(int(n_i), int(n_j), int(sm_count), out), "nb_plan_query_small")
    keys = ("NW", "KI", "LJ", "WJ", "S", "CS", "tiles_i", "default")
    d = dict(zip(keys, [int(v) for v in out]))
    d["tile_i"] = (d["NW"] // d["WJ"]) * d["KI"] * (32 // d["LJ"])
    return d


def plan_query_small_jerk(n_i: int, n_j: int, sm_count: int = 148) -> dict:
    """The small-i-set force + jerk kernel's decomposition; "default" = nb_force_jerk takes that kernel for this shape,
    "default_steps" = the Hermite steps do."""
    out = (ctypes.c_int64 * 8)()
    _check(lib().nb_plan_query_small_jerk(int(n_i), int(n_j), int(sm_count), out), "nb_plan_query_small_jerk")
    keys = ("NW", "KI", "LJ", "WJ", "S", "CS", "tiles_i", "default")
    d = dict(zip(keys, [int(v) for v in out]))
    d["default_steps"] = (d["default"] >> 1) & 1        # nb_hermite4 / nb_hermite4_block_step (records already packed)
    d["default"] &= 1                                   # nb_force_jerk
    d["tile_i"] = (d["NW"] // d["WJ"]) * d["KI"] * (32 // d["LJ"])
    return d


def debug_set(key: str, value: Optional[str]) -> None:
    """include/nb_debug.h: a debugging switch of the library (value None restores the default)."""
    _check(lib().nb_debug_set(key.encode(), None if value is None else str(value).encode()), f"nb_debug_set({key})")


def debug_plan_exhaustive(n_i: int, n_j: int, sm_count: int = 148, jerk: bool = False) -> dict:
    out = (ctypes.c_int64 * 8)()
    _check(lib().nb_debug_plan_exhaustive(int(n_i), int(n_j), int(sm_count), 1 if jerk else 0, out), "nb_debug_plan_exhaustive")
    keys = ("K", "WI", "WJ", "S", "tiles_i", "tile_i", "tile_j", "stages")
    return dict(zip(keys, [int(v) for v in out]))


def debug_plans_computed() -> int:
    return int(lib().nb_debug_plans_computed())


def release_stream(stream=None) -> None:
    """nb_release_stream: frees the workspace the library keeps for `stream` (waits for the stream first)."""
    _check(lib().nb_release_stream(_stream_ptr(stream)), "nb_release_stream")


def last_launch_count() -> int:
    return int(lib().nb_last_launch_count())


def profile_enable(on: bool) -> None:
    _check(lib().nb_profile_enable(1 if on else 0), "nb_profile_enable")


def profile_read() -> Tuple[int, float]:
    """(number of force-kernel launches bracketed since the last read, sum of their durations in ms)."""
    n, ms = ctypes.c_int64(0), ctypes.c_double(0.0)
    _check(lib().nb_profile_read(ctypes.byref(n), ctypes.byref(ms)), "nb_profile_read")
    return int(n.value), float(ms.value)


def release_workspace() -> None:
    _check(lib().nb_release_workspace(), "nb_release_workspace")


def status_string(status: int) -> str:
    return lib().nb_status_string(int(status)).decode()


def version() -> int:
    return int(lib().nb_version())
