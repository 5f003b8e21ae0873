"""Thin ctypes binding of libbqc_t.so — argument marshalling only.

Every function has the name of the C entry point it calls (include/bqc_t.h) and takes
torch tensors (device or host, FP64, contiguous) where the C ABI takes pointers.  Nothing is
computed in Python: every step of the (T) path runs in the library's CUDA kernels.  There is no
CPU fallback: a missing library or a failing call raises.
"""
from __future__ import annotations

import ctypes
import os
from ctypes import (POINTER, Structure, byref, c_char_p, c_double, c_int, c_size_t, c_void_p)

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "lib", "libbqc_t.so")


class BqcError(RuntimeError):
    def __init__(self, code, what, detail):
        super().__init__(f"bqc error {code} ({what}): {detail}")
        self.code = code


class bqc_t_opts(Structure):
    _fields_ = [("occ_block", c_int), ("occ_lo", c_int), ("occ_hi", c_int),
                ("shard_rank", c_int), ("shard_count", c_int), ("max_batch", c_int),
                ("flags", c_int), ("workspace_gib", c_int), ("f_ov", c_void_p)]


class bqc_mp2_opts(Structure):
    _fields_ = [("occ_block", c_int), ("shard_rank", c_int), ("shard_count", c_int), ("flags", c_int),
                ("workspace", c_void_p), ("workspace_bytes", c_size_t)]


BQC_T_FLAG_NO_T1 = 1
BQC_T_FLAG_PROFILE = 2
BQC_T_FLAG_ABC_DRIVEN = 4
BQC_T_FLAG_SHARD_BLOCKS = 8

_lib = None


def lib():
    """Load libbqc_t.so (fails loudly if it has not been built: there is no fallback)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2502_17963_b200.build` "
                          "(or __graft_entry__.build()); the CUDA library is the only implementation")
    L = ctypes.CDLL(LIB_PATH)
    dp = c_void_p
    L.bqc_t_num_triplets.restype = c_size_t
    L.bqc_t_num_triplets.argtypes = [c_int]
    L.bqc_t_triplet_index.restype = c_size_t
    L.bqc_t_triplet_index.argtypes = [c_int] * 4
    L.bqc_mp2_workspace_bytes.restype = c_size_t
    L.bqc_mp2_workspace_bytes.argtypes = [c_int] * 3 + [POINTER(bqc_mp2_opts)]
    L.bqc_debug_tiling.restype = c_int
    L.bqc_debug_tiling.argtypes = [c_int, POINTER(c_int), c_int]
    L.bqc_t_triplet_owner.restype = c_int
    L.bqc_t_triplet_owner.argtypes = [c_int] * 5
    L.bqc_t_triplet_owner_ex.restype = c_int
    L.bqc_t_triplet_owner_ex.argtypes = [c_int] * 3 + [POINTER(bqc_t_opts)] + [c_int] * 3
    L.bqc_t_flops.restype = c_double
    L.bqc_t_flops.argtypes = [c_int, c_int, POINTER(bqc_t_opts)]
    L.bqc_t_plan_occ_block.restype = c_int
    L.bqc_t_plan_occ_block.argtypes = [c_int, c_int, c_int, POINTER(bqc_t_opts)]
    L.bqc_t_workspace_bytes.restype = c_size_t
    L.bqc_t_workspace_bytes.argtypes = [c_int, c_int, c_int, POINTER(bqc_t_opts)]
    L.bqc_sum_in_order.restype = c_int
    L.bqc_sum_in_order.argtypes = [dp, c_size_t, POINTER(c_double), c_void_p]
    L.bqc_release_cached.restype = None
    L.bqc_release_cached.argtypes = []
    L.bqc_t_plan_create.restype = c_int
    L.bqc_t_plan_create.argtypes = [c_int] * 3 + [POINTER(bqc_t_opts), c_void_p, c_size_t, POINTER(c_void_p)]
    L.bqc_t_plan_execute.restype = c_int
    L.bqc_t_plan_execute.argtypes = [c_void_p] + [dp] * 8 + [POINTER(c_double), dp, c_void_p]
    L.bqc_t_plan_destroy.restype = None
    L.bqc_t_plan_destroy.argtypes = [c_void_p]
    L.bqc_t_plan_workspace_bytes.restype = c_size_t
    L.bqc_t_plan_workspace_bytes.argtypes = [c_void_p]
    L.bqc_sum_fixed_noalloc.restype = c_int
    L.bqc_sum_fixed_noalloc.argtypes = [dp, c_size_t, dp, c_void_p]
    L.bqc_sum_fixed_noalloc_max.restype = c_size_t
    L.bqc_sum_fixed_noalloc_max.argtypes = []
    L.bqc_last_error.restype = c_int
    L.bqc_error_string.restype = c_char_p
    L.bqc_error_string.argtypes = [c_int]
    L.bqc_error_detail.restype = c_char_p
    L.bqc_version.restype = c_char_p
    L.bqc_t_energy.restype = c_double
    L.bqc_t_energy.argtypes = [c_int] * 3 + [dp] * 7 + [c_void_p]
    L.bqc_t_energy_ex.restype = c_int
    L.bqc_t_energy_ex.argtypes = [c_int] * 3 + [dp] * 7 + [POINTER(bqc_t_opts), c_void_p, c_size_t,
                                                         POINTER(c_double), dp, c_void_p]
    L.bqc_t_last_profile.restype = c_int
    L.bqc_t_last_profile.argtypes = [POINTER(c_double), c_int]
    L.bqc_t_energy_host.restype = c_int
    L.bqc_t_energy_host.argtypes = [c_int] * 3 + [dp] * 7 + [POINTER(bqc_t_opts), POINTER(c_double), dp,
                                                           POINTER(c_size_t), POINTER(c_size_t), c_void_p]
    L.bqc_t_debug_slabs.restype = c_int
    L.bqc_t_debug_slabs.argtypes = [c_int] * 3 + [dp] * 4 + [c_int, c_int] + [dp] * 3 + [c_void_p]
    L.bqc_t_debug_wv.restype = c_int
    L.bqc_t_debug_wv.argtypes = [c_int] * 3 + [dp] * 8 + [c_int] * 3 + [dp] * 2 + [c_void_p]
    L.bqc_dgemm_nt.restype = c_int
    L.bqc_dgemm_nt.argtypes = [c_int] * 3 + [dp, c_int, dp, c_int, dp, c_int, c_void_p]
    L.bqc_fp64_peak_tflops.restype = c_double
    L.bqc_fp64_peak_tflops.argtypes = [c_int, c_double, c_void_p]
    L.bqc_mp2_energy.restype = c_double
    L.bqc_mp2_energy.argtypes = [c_int] * 3 + [dp] * 3 + [c_void_p]
    L.bqc_mp2_energy_ex.restype = c_int
    L.bqc_mp2_energy_ex.argtypes = [c_int] * 3 + [dp] * 3 + [POINTER(bqc_mp2_opts), POINTER(c_double), dp, c_void_p]
    L.bqc_mp2_energy_host.restype = c_int
    L.bqc_mp2_energy_host.argtypes = [c_int] * 3 + [dp] * 3 + [POINTER(bqc_mp2_opts), POINTER(c_double), dp,
                                                             POINTER(c_size_t), POINTER(c_size_t), c_void_p]
    L.bqc_mp2_flops.restype = c_double
    L.bqc_mp2_flops.argtypes = [c_int] * 3
    L.bqc_mp2_plan_occ_block.restype = c_int
    L.bqc_mp2_plan_occ_block.argtypes = [c_int] * 3 + [POINTER(bqc_mp2_opts)]
    L.bqc_mp2_last_profile.restype = c_int
    L.bqc_mp2_last_profile.argtypes = [POINTER(c_double), c_int]
    _lib = L
    return L


# ---------------------------------------------------------------- marshalling helpers
def _check(rc):
    if rc != 0:
        L = lib()
        raise BqcError(rc, L.bqc_error_string(rc).decode(), L.bqc_error_detail().decode())


def _ptr(t, shape, name, device):
    if not isinstance(t, torch.Tensor):
        raise TypeError(f"{name} must be a torch.Tensor")
    if t.dtype != torch.float64 or not t.is_contiguous() or tuple(t.shape) != tuple(shape):
        raise ValueError(f"{name}: need contiguous float64 {tuple(shape)}, got {t.dtype} {tuple(t.shape)}")
    if device and not t.is_cuda:
        raise ValueError(f"{name} must be a CUDA tensor")
    if not device and t.is_cuda:
        raise ValueError(f"{name} must be a host tensor")
    return c_void_p(t.data_ptr())


def _stream():
    return c_void_p(torch.cuda.current_stream().cuda_stream)


def _shapes(nocc, nvir, naux):
    return [(nocc,), (nvir,), (nocc, nvir), (nocc, nocc, nvir, nvir), (naux, nocc, nocc),
            (naux, nocc, nvir), (naux, nvir, nvir)]


_NAMES = ["eps_occ", "eps_vir", "t1", "t2", "B_oo", "B_ov", "B_vv"]


def _inputs(nocc, nvir, naux, arrays, device):
    return [_ptr(t, s, n, device) for t, s, n in zip(arrays, _shapes(nocc, nvir, naux), _NAMES)]


def make_opts(occ_block=0, occ_lo=0, occ_hi=0, shard_rank=0, shard_count=1, max_batch=0, flags=0, f_ov=None,
              workspace_gib=0):
    """`f_ov`: optional [nocc, nvir] float64 tensor (CUDA for bqc_t_energy_ex, host for bqc_t_energy_host);
    the returned struct keeps a reference so the pointer stays valid."""
    o = bqc_t_opts(occ_block, occ_lo, occ_hi, shard_rank, shard_count, max_batch, flags, workspace_gib, None)
    if f_ov is not None:
        if f_ov.dtype != torch.float64 or not f_ov.is_contiguous() or f_ov.dim() != 2:
            raise ValueError("f_ov must be a contiguous float64 [nocc, nvir] tensor")
        o.f_ov = f_ov.data_ptr()
        o._f_ov_keepalive = f_ov
    return o


def _check_f_ov(opts, nocc, nvir, device):
    """opts.f_ov (kept alive by make_opts) must be [nocc, nvir] in the memory space of the entry point."""
    f = getattr(opts, "_f_ov_keepalive", None) if opts is not None else None
    if f is not None:
        _ptr(f, (nocc, nvir), "opts.f_ov", device)


def _optp(opts):
    return byref(opts) if opts is not None else None


# ---------------------------------------------------------------- host-only helpers
def _ntrip_out(nocc, nvir, opts):
    """Length of the per-triplet output: occupied triplets, or virtual triples under BQC_T_FLAG_ABC_DRIVEN."""
    abc = opts is not None and (opts.flags & BQC_T_FLAG_ABC_DRIVEN)
    return bqc_t_num_triplets(nvir if abc else nocc)


def bqc_t_num_triplets(nocc):
    return lib().bqc_t_num_triplets(nocc)


def bqc_t_triplet_index(nocc, i, j, k):
    r = lib().bqc_t_triplet_index(nocc, i, j, k)
    return -1 if r == ctypes.c_size_t(-1).value else r


def bqc_t_triplet_owner(nocc, shard_count, i, j, k):
    return lib().bqc_t_triplet_owner(nocc, shard_count, i, j, k)


def bqc_t_triplet_owner_ex(nocc, nvir, naux, opts, i, j, k):
    return lib().bqc_t_triplet_owner_ex(nocc, nvir, naux, _optp(opts), i, j, k)


def bqc_t_flops(nocc, nvir, opts=None):
    return lib().bqc_t_flops(nocc, nvir, _optp(opts))


def bqc_t_plan_occ_block(nocc, nvir, naux, opts=None):
    return lib().bqc_t_plan_occ_block(nocc, nvir, naux, _optp(opts))


def bqc_t_workspace_bytes(nocc, nvir, naux, opts=None):
    return lib().bqc_t_workspace_bytes(nocc, nvir, naux, _optp(opts))


def bqc_sum_in_order(x):
    """x[0] + x[1] + ... left to right, by the library (host loop or one-thread kernel: same bits).
    `x`: contiguous 1-D float64 tensor, host or CUDA."""
    if not isinstance(x, torch.Tensor) or x.dtype != torch.float64 or x.dim() != 1 or not x.is_contiguous():
        raise ValueError("bqc_sum_in_order: need a contiguous 1-D float64 tensor")
    out = c_double(0.0)
    stream = _stream() if x.is_cuda else None
    _check(lib().bqc_sum_in_order(c_void_p(x.data_ptr()), x.numel(), byref(out), stream))
    return out.value


def bqc_sum_fixed_noalloc(x, out):
    """out[0] = sum(x) by the library's allocation-free two-stage fixed-order sum, enqueued on torch's current
    stream (no synchronisation).  `x`: contiguous 1-D float64 CUDA tensor, `out`: float64 CUDA tensor of 1 element."""
    for t, name in ((x, "x"), (out, "out")):
        if not isinstance(t, torch.Tensor) or t.dtype != torch.float64 or not t.is_cuda or not t.is_contiguous():
            raise ValueError(f"bqc_sum_fixed_noalloc: {name} must be a contiguous float64 CUDA tensor")
    if x.dim() != 1 or out.numel() != 1:
        raise ValueError("bqc_sum_fixed_noalloc: x must be 1-D and out must hold one element")
    _check(lib().bqc_sum_fixed_noalloc(c_void_p(x.data_ptr()), x.numel(), c_void_p(out.data_ptr()), _stream()))
    return out


def bqc_sum_fixed_noalloc_max():
    return lib().bqc_sum_fixed_noalloc_max()


def bqc_last_error():
    return lib().bqc_last_error()


def bqc_error_string(code):
    return lib().bqc_error_string(code).decode()


def bqc_error_detail():
    return lib().bqc_error_detail().decode()


def bqc_version():
    return lib().bqc_version().decode()


# ---------------------------------------------------------------- the (T) energy
def bqc_t_energy(nocc, nvir, naux, eps_occ, eps_vir, t1, t2, B_oo, B_ov, B_vv):
    """E(T) [Hartree] from device tensors, on torch's current CUDA stream."""
    p = _inputs(nocc, nvir, naux, (eps_occ, eps_vir, t1, t2, B_oo, B_ov, B_vv), True)
    e = lib().bqc_t_energy(nocc, nvir, naux, *p, _stream())
    if e != e:
        _check(lib().bqc_last_error() or 6)
    return e


def bqc_t_energy_ex(nocc, nvir, naux, eps_occ, eps_vir, t1, t2, B_oo, B_ov, B_vv, opts=None,
                    workspace=None, e_triplet=None):
    """Returns E (this shard / window).  `workspace`: optional uint8 CUDA tensor;
    `e_triplet`: optional float64 CUDA tensor [num_triplets] filled with e_ijk
    (e_abc over virtual triples, [num_triplets(nvir)], under BQC_T_FLAG_ABC_DRIVEN)."""
    p = _inputs(nocc, nvir, naux, (eps_occ, eps_vir, t1, t2, B_oo, B_ov, B_vv), True)
    _check_f_ov(opts, nocc, nvir, True)
    ws_ptr, ws_bytes = None, 0
    if workspace is not None:
        ws_ptr, ws_bytes = c_void_p(workspace.data_ptr()), workspace.numel() * workspace.element_size()
    et = None
    if e_triplet is not None:
        et = _ptr(e_triplet, (_ntrip_out(nocc, nvir, opts),), "e_triplet", True)
    e = c_double(0.0)
    _check(lib().bqc_t_energy_ex(nocc, nvir, naux, *p, _optp(opts), ws_ptr, ws_bytes, byref(e), et,
                                 _stream()))
    return e.value


def bqc_release_cached():
    lib().bqc_release_cached()


class bqc_t_plan:
    """Handle of bqc_t_plan_create / _execute / _destroy (include/bqc_t.h): marshalling only."""

    def __init__(self, nocc, nvir, naux, opts=None, workspace=None):
        self.nocc, self.nvir, self.naux, self.opts = nocc, nvir, naux, opts
        self._ws = workspace                      # kept alive: the plan uses it until destroyed
        ws_ptr, ws_bytes = None, 0
        if workspace is not None:
            ws_ptr, ws_bytes = c_void_p(workspace.data_ptr()), workspace.numel() * workspace.element_size()
        self._h = c_void_p()
        _check(lib().bqc_t_plan_create(nocc, nvir, naux, _optp(opts), ws_ptr, ws_bytes, byref(self._h)))

    def workspace_bytes(self):
        return lib().bqc_t_plan_workspace_bytes(self._h)

    def execute(self, eps_occ, eps_vir, t1, t2, B_oo, B_ov, B_vv, f_ov=None, e_triplet=None):
        p = _inputs(self.nocc, self.nvir, self.naux, (eps_occ, eps_vir, t1, t2, B_oo, B_ov, B_vv), True)
        f = _ptr(f_ov, (self.nocc, self.nvir), "f_ov", True) if f_ov is not None else None
        et = None
        if e_triplet is not None:
            et = _ptr(e_triplet, (_ntrip_out(self.nocc, self.nvir, self.opts),), "e_triplet", True)
        e = c_double(0.0)
        _check(lib().bqc_t_plan_execute(self._h, *p, f, byref(e), et, _stream()))
        return e.value

    def destroy(self):
        if self._h:
            lib().bqc_t_plan_destroy(self._h)
            self._h = c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def bqc_t_last_profile():
    """Kernel-group timings of the last profiled bqc_t_energy_ex call (see include/bqc_t.h)."""
    buf = (c_double * 9)()
    n = lib().bqc_t_last_profile(buf, 9)
    keys = ["gemm_ms", "gemm_launches", "energy_ms", "energy_launches", "form_ms", "form_blocks",
            "prepare_ms", "total_ms", "kernel_launches"]
    return {k: buf[i] for i, k in enumerate(keys[:n])}


def bqc_t_energy_host(nocc, nvir, naux, eps_occ, eps_vir, t1, t2, B_oo, B_ov, B_vv, opts=None,
                      e_triplet=None):
    """End-to-end call with HOST tensors.  Returns (E, h2d_bytes, d2h_bytes)."""
    p = _inputs(nocc, nvir, naux, (eps_occ, eps_vir, t1, t2, B_oo, B_ov, B_vv), False)
    _check_f_ov(opts, nocc, nvir, False)
    et = None
    if e_triplet is not None:
        et = _ptr(e_triplet, (_ntrip_out(nocc, nvir, opts),), "e_triplet", False)
    e = c_double(0.0)
    h2d, d2h = c_size_t(0), c_size_t(0)
    _check(lib().bqc_t_energy_host(nocc, nvir, naux, *p, _optp(opts), byref(e), et, byref(h2d),
                                   byref(d2h), _stream()))
    return e.value, h2d.value, d2h.value


# ---------------------------------------------------------------- DF-MP2 energy (Eq. (1))
def make_mp2_opts(occ_block=0, shard_rank=0, shard_count=1, flags=0, workspace=None):
    """`workspace`: optional uint8 CUDA tensor of >= bqc_mp2_workspace_bytes (kept alive by the caller)."""
    o = bqc_mp2_opts(occ_block, shard_rank, shard_count, flags, None, 0)
    if workspace is not None:
        o.workspace = workspace.data_ptr()
        o.workspace_bytes = workspace.numel() * workspace.element_size()
    return o


def bqc_mp2_workspace_bytes(nocc, nvir, naux, opts=None):
    return lib().bqc_mp2_workspace_bytes(nocc, nvir, naux, _optp(opts))


def _mp2_inputs(nocc, nvir, naux, eps_occ, eps_vir, B_ov, device):
    return [_ptr(eps_occ, (nocc,), "eps_occ", device), _ptr(eps_vir, (nvir,), "eps_vir", device),
            _ptr(B_ov, (naux, nocc, nvir), "B_ov", device)]


def bqc_mp2_energy(nocc, nvir, naux, eps_occ, eps_vir, B_ov):
    """E_MP2 [Hartree] from device tensors, on torch's current CUDA stream."""
    p = _mp2_inputs(nocc, nvir, naux, eps_occ, eps_vir, B_ov, True)
    e = lib().bqc_mp2_energy(nocc, nvir, naux, *p, _stream())
    if e != e:
        _check(lib().bqc_last_error() or 6)
    return e


def bqc_mp2_energy_ex(nocc, nvir, naux, eps_occ, eps_vir, B_ov, opts=None, e_pair=None):
    """Returns the weighted pair sum of this shard; `e_pair`: optional float64 CUDA [nocc, nocc] filled with e_ij."""
    p = _mp2_inputs(nocc, nvir, naux, eps_occ, eps_vir, B_ov, True)
    ep = _ptr(e_pair, (nocc, nocc), "e_pair", True) if e_pair is not None else None
    e = c_double(0.0)
    _check(lib().bqc_mp2_energy_ex(nocc, nvir, naux, *p, _optp(opts), byref(e), ep, _stream()))
    return e.value


def bqc_mp2_energy_host(nocc, nvir, naux, eps_occ, eps_vir, B_ov, opts=None, e_pair=None):
    """End-to-end call with HOST tensors.  Returns (E, h2d_bytes, d2h_bytes)."""
    p = _mp2_inputs(nocc, nvir, naux, eps_occ, eps_vir, B_ov, False)
    ep = _ptr(e_pair, (nocc, nocc), "e_pair", False) if e_pair is not None else None
    e = c_double(0.0)
    h2d, d2h = c_size_t(0), c_size_t(0)
    _check(lib().bqc_mp2_energy_host(nocc, nvir, naux, *p, _optp(opts), byref(e), ep, byref(h2d), byref(d2h),
                                     _stream()))
    return e.value, h2d.value, d2h.value


def bqc_mp2_flops(nocc, nvir, naux):
    return lib().bqc_mp2_flops(nocc, nvir, naux)


def bqc_mp2_plan_occ_block(nocc, nvir, naux, opts=None):
    return lib().bqc_mp2_plan_occ_block(nocc, nvir, naux, _optp(opts))


def bqc_mp2_last_profile():
    buf = (c_double * 6)()
    n = lib().bqc_mp2_last_profile(buf, 6)
    keys = ["gemm_ms", "gemm_launches", "energy_ms", "energy_launches", "total_ms", "kernel_launches"]
    return {k: buf[i] for i, k in enumerate(keys[:n])}


# ---------------------------------------------------------------- single steps (parity tests)
def bqc_t_debug_slabs(nocc, nvir, naux, t2, B_oo, B_ov, B_vv, x, y, want_I=True, want_O=True, want_J=True):
    sh = _shapes(nocc, nvir, naux)
    p = [_ptr(t, s, n, True) for t, s, n in zip((t2, B_oo, B_ov, B_vv), sh[3:], _NAMES[3:])]
    dev = t2.device
    I = torch.empty((nvir, nvir, nvir), dtype=torch.float64, device=dev) if want_I else None
    O = torch.empty((nocc, nvir), dtype=torch.float64, device=dev) if want_O else None
    J = torch.empty((nvir, nvir), dtype=torch.float64, device=dev) if want_J else None
    q = [c_void_p(t.data_ptr()) if t is not None else None for t in (I, O, J)]
    _check(lib().bqc_t_debug_slabs(nocc, nvir, naux, *p, x, y, *q, _stream()))
    return I, O, J


def bqc_t_debug_wv(nocc, nvir, naux, eps_occ, eps_vir, t1, t2, B_oo, B_ov, B_vv, i, j, k,
                   want_W=True, want_V=True, f_ov=None):
    p = _inputs(nocc, nvir, naux, (eps_occ, eps_vir, t1, t2, B_oo, B_ov, B_vv), True)
    p.append(_ptr(f_ov, (nocc, nvir), "f_ov", True) if f_ov is not None else None)
    dev = t2.device
    W = torch.empty((nvir, nvir, nvir), dtype=torch.float64, device=dev) if want_W else None
    V = torch.empty((nvir, nvir, nvir), dtype=torch.float64, device=dev) if want_V else None
    q = [c_void_p(t.data_ptr()) if t is not None else None for t in (W, V)]
    _check(lib().bqc_t_debug_wv(nocc, nvir, naux, *p, i, j, k, *q, _stream()))
    return W, V


def bqc_debug_tiling(nvir):
    """(column segments [(n0, ntiles, nf)], row segments [(m1_0, tiles_m1, tp, tq)]) of the W-builder GEMM."""
    buf = (c_int * 14)()
    rc = lib().bqc_debug_tiling(nvir, buf, 14)
    if rc < 0:
        _check(lib().bqc_last_error())
    nn, nm = rc // 10, rc % 10
    cols = [tuple(buf[3 * k:3 * k + 3]) for k in range(nn)]
    rows = [tuple(buf[6 + 4 * k:10 + 4 * k]) for k in range(nm)]
    return cols, rows


def bqc_dgemm_nt(A, B, C=None):
    """C[M,N] = A[M,K] @ B[N,K].T with the library's TMA + DMMA kernel (row strides may exceed K)."""
    M, K = A.shape
    N, K2 = B.shape
    assert K == K2 and A.dtype == torch.float64 and B.dtype == torch.float64
    assert A.stride(1) == 1 and B.stride(1) == 1
    if C is None:
        C = torch.empty((M, N), dtype=torch.float64, device=A.device)
    _check(lib().bqc_dgemm_nt(M, N, K, c_void_p(A.data_ptr()), A.stride(0), c_void_p(B.data_ptr()),
                              B.stride(0), c_void_p(C.data_ptr()), C.stride(0), _stream()))
    return C


def bqc_fp64_peak_tflops(kind=0, seconds=1.0):
    r = lib().bqc_fp64_peak_tflops(kind, seconds, _stream())
    if r < 0:
        _check(lib().bqc_last_error() or 6)
    return r
