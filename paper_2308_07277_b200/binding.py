"""Thin ctypes binding of include/qm_hpsi.h -- argument marshalling only.

Every step of the hot path runs in the CUDA kernels of libqm_hpsi.so; PyTorch is used for device
memory and streams.  The functions carry the C names (qm_gspace_create, qm_set_vloc,
qm_set_nonlocal, qm_apply_h, ...).  There is no fallback: a missing library or a failing call
raises.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libqm_hpsi.so")

QM_OK, QM_EINVAL, QM_ENOTSET, QM_EGRID, QM_ECUDA, QM_ENOMEM = 0, -1, -2, -3, -4, -5
_CODES = {QM_EINVAL: "QM_EINVAL", QM_ENOTSET: "QM_ENOTSET", QM_EGRID: "QM_EGRID", QM_ECUDA: "QM_ECUDA",
          QM_ENOMEM: "QM_ENOMEM"}


class QmError(RuntimeError):
    def __init__(self, code: int, text: str):
        super().__init__(f"{_CODES.get(code, code)}: {text}")
        self.code = code


_lib = None
_vp, _i, _d = ctypes.c_void_p, ctypes.c_int, ctypes.c_double
_SIGS = {
    "qm_gspace_create": [_vp, _d, _vp, _vp, _i, ctypes.POINTER(_vp)],
    "qm_gspace_destroy": [_vp],
    "qm_gspace_num_k": [_vp, ctypes.POINTER(_i)],
    "qm_gspace_num_g": [_vp, _i, ctypes.POINTER(_i)],
    "qm_gspace_num_sticks": [_vp, _i, ctypes.POINTER(_i), ctypes.POINTER(_i)],
    "qm_gspace_get_index_map": [_vp, _i, _vp],
    "qm_gspace_get_miller": [_vp, _i, _vp],
    "qm_gspace_get_g2": [_vp, _i, _vp],
    "qm_gspace_alias_free": [_vp, _i, ctypes.POINTER(_i)],
    "qm_fft_size_supported": [_i],
    "qm_set_vloc": [_vp, _vp, _vp],
    "qm_set_nonlocal": [_vp, _i, _vp, _i, _vp, _i, _vp],
    "qm_apply_h": [_vp, _vp, _vp, _i, _i, _vp],
    "qm_reserve": [_vp, _i, _i],
    "qm_batch_plan_create": [_vp, _i, _vp, _vp, _vp, _vp, ctypes.POINTER(_vp)],
    "qm_batch_plan_launch": [_vp, _vp],
    "qm_batch_plan_destroy": [_vp],
    "qm_split_operator_set": [_vp, _vp, _d, _vp],
    "qm_split_operator_propagate": [_vp, _i, _vp, _vp, _i, _vp],
    "qm_mtxel_create": [_vp, _i, _i, _d, ctypes.POINTER(_vp)],
    "qm_mtxel_destroy": [_vp],
    "qm_mtxel_num_g": [_vp, ctypes.POINTER(_i)],
    "qm_mtxel_get_miller": [_vp, _vp],
    "qm_mtxel_get_index_map": [_vp, _vp],
    "qm_matrix_elements": [_vp, _vp, _i, _vp, _i, _vp, _vp],
    "qm_subspace": [_vp, _i, _vp, _i, _vp, _i, _vp, _vp],
    "qm_subspace_static": [_vp, _i, _vp, _i, _i, _vp, _vp],
    "qm_taylor_propagate": [_vp, _i, _vp, _vp, _i, _d, _i, _vp],
    "qm_density_reset": [_vp, _vp],
    "qm_density_accumulate": [_vp, _i, _vp, _i, _vp, _d, _vp],
    "qm_density_get": [_vp, _vp, _d, _vp],
    "qm_apply_h_host": [_vp, _vp, _vp, _i, _i, _vp],
    "qm_apply_h_host_async": [_vp, _vp, _vp, _i, _i, _vp],
    "qm_host_synchronize": [_vp],
    "qm_debug_g2r": [_vp, _vp, _vp, _i, _i, _vp],
    "qm_debug_r2g": [_vp, _vp, _vp, _i, _i, _vp],
    "qm_get_launch_count": [_vp, ctypes.POINTER(ctypes.c_ulonglong)],
    "qm_probe_fp64_tensor_peak": [ctypes.POINTER(_d), ctypes.POINTER(_d)],
    "qm_profile_enable": [_vp, _i],
    "qm_profile_reset": [_vp],
    "qm_profile_read": [_vp, _i, ctypes.POINTER(_d), ctypes.POINTER(ctypes.c_ulonglong)],
}
EXPORTS = sorted(list(_SIGS) + ["qm_last_error", "qm_version", "qm_kernel_name"])
QM_K_COUNT = 11


def load_library():
    """dlopen libqm_hpsi.so (built in-tree by paper_2308_07277_b200/build.py).  Fails loudly."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: run `python __graft_entry__.py` (build()) first; "
                              "there is no CPU fallback")
        lib = ctypes.CDLL(LIB_PATH)
        for name, args in _SIGS.items():
            fn = getattr(lib, name)
            fn.restype = _i
            fn.argtypes = args
        lib.qm_last_error.restype = ctypes.c_char_p
        lib.qm_version.restype = ctypes.c_char_p
        lib.qm_kernel_name.restype = ctypes.c_char_p
        lib.qm_kernel_name.argtypes = [_i]
        _lib = lib
    return _lib


def _check(rc: int):
    if rc != QM_OK:
        raise QmError(rc, load_library().qm_last_error().decode())


def _stream_ptr(stream):
    import torch
    if stream is None:
        stream = torch.cuda.current_stream()
    return ctypes.c_void_p(stream.cuda_stream)


def _dev_ptr(t, dtype, what):
    import torch
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise TypeError(f"{what}: expected a CUDA torch.Tensor")
    if t.dtype != dtype or not t.is_contiguous():
        raise TypeError(f"{what}: expected contiguous {dtype}, got {t.dtype}")
    return ctypes.c_void_p(t.data_ptr())


# ---- C-named functions ---------------------------------------------------------------------------
def qm_version() -> str:
    return load_library().qm_version().decode()


def qm_fft_size_supported(n: int) -> bool:
    return bool(load_library().qm_fft_size_supported(int(n)))


def qm_gspace_create(lattice_bohr, ecutwfc_ry, fft_grid, kpts_cryst=None):
    lib = load_library()
    lat = np.ascontiguousarray(lattice_bohr, dtype=np.float64).reshape(9)
    grid = np.ascontiguousarray(fft_grid, dtype=np.int32).reshape(3)
    if kpts_cryst is None:
        kp, nk, kptr = None, 1, None
    else:
        kp = np.ascontiguousarray(kpts_cryst, dtype=np.float64).reshape(-1, 3)
        nk, kptr = kp.shape[0], kp.ctypes.data
    h = _vp()
    _check(lib.qm_gspace_create(lat.ctypes.data, float(ecutwfc_ry), grid.ctypes.data, kptr, nk, ctypes.byref(h)))
    return h


def qm_gspace_destroy(h):
    _check(load_library().qm_gspace_destroy(h))


def qm_gspace_num_k(h) -> int:
    n = _i()
    _check(load_library().qm_gspace_num_k(h, ctypes.byref(n)))
    return n.value


def qm_gspace_num_g(h, k=0) -> int:
    n = _i()
    _check(load_library().qm_gspace_num_g(h, k, ctypes.byref(n)))
    return n.value


def qm_gspace_num_sticks(h, k=0):
    s, x = _i(), _i()
    _check(load_library().qm_gspace_num_sticks(h, k, ctypes.byref(s), ctypes.byref(x)))
    return s.value, x.value


def qm_gspace_get_index_map(h, k=0) -> np.ndarray:
    out = np.empty(qm_gspace_num_g(h, k), dtype=np.int32)
    _check(load_library().qm_gspace_get_index_map(h, k, out.ctypes.data))
    return out


def qm_gspace_get_miller(h, k=0) -> np.ndarray:
    out = np.empty((qm_gspace_num_g(h, k), 3), dtype=np.int32)
    _check(load_library().qm_gspace_get_miller(h, k, out.ctypes.data))
    return out


def qm_gspace_get_g2(h, k=0) -> np.ndarray:
    out = np.empty(qm_gspace_num_g(h, k), dtype=np.float64)
    _check(load_library().qm_gspace_get_g2(h, k, out.ctypes.data))
    return out


def qm_gspace_alias_free(h, k=0) -> bool:
    f = _i()
    _check(load_library().qm_gspace_alias_free(h, k, ctypes.byref(f)))
    return bool(f.value)


def qm_set_vloc(h, v_r_dev, stream=None):
    import torch
    _check(load_library().qm_set_vloc(h, _dev_ptr(v_r_dev, torch.float64, "V_r"), _stream_ptr(stream)))


def qm_set_nonlocal(h, k, beta_dev, d_dev, stream=None):
    """beta_dev [nproj][ng] complex128 CUDA tensor (or None); d_dev [nblk][db][db] float64 CUDA tensor."""
    import torch
    lib = load_library()
    if beta_dev is None or beta_dev.shape[0] == 0:
        _check(lib.qm_set_nonlocal(h, k, None, 0, None, 0, _stream_ptr(stream)))
        return
    nproj = beta_dev.shape[0]
    if beta_dev.dim() != 2 or beta_dev.shape[1] != qm_gspace_num_g(h, k):
        raise TypeError("beta: expected shape [nproj][ng(k)]")   # wrong basis => error
    if d_dev.dim() != 3 or d_dev.shape[1] != d_dev.shape[2] or d_dev.shape[0] * d_dev.shape[1] != nproj:
        raise TypeError("D: expected shape [nproj/d_block][d_block][d_block]")
    _check(lib.qm_set_nonlocal(h, k, _dev_ptr(beta_dev, torch.complex128, "beta"), nproj,
                               _dev_ptr(d_dev, torch.float64, "D"), int(d_dev.shape[1]), _stream_ptr(stream)))


def _check_block(h, k, t, what):
    ng = qm_gspace_num_g(h, k)
    if t.dim() != 2 or t.shape[1] != ng:
        raise TypeError(f"{what}: expected shape [nbands][{ng}]")     # check_array_type
    return int(t.shape[0])


def qm_apply_h(h, psi_in_dev, psi_out_dev, k=0, stream=None):
    import torch
    nb = _check_block(h, k, psi_in_dev, "psi_in")
    if tuple(psi_out_dev.shape) != tuple(psi_in_dev.shape):
        raise TypeError("psi_out: shape differs from psi_in")
    _check(load_library().qm_apply_h(h, _dev_ptr(psi_in_dev, torch.complex128, "psi_in"),
                                     _dev_ptr(psi_out_dev, torch.complex128, "psi_out"), nb, k,
                                     _stream_ptr(stream)))
    return psi_out_dev


def qm_batch_plan_create(h, items):
    """items: list of (k, psi_in_dev, psi_out_dev) with [nbands][ng(k)] complex128 CUDA tensors (kept alive by the caller)."""
    import torch
    n = len(items)
    ks = (ctypes.c_int * n)(*[int(it[0]) for it in items])
    nbs = (ctypes.c_int * n)()
    pin = (ctypes.c_void_p * n)()
    pout = (ctypes.c_void_p * n)()
    for i, (k, a, b) in enumerate(items):
        nbs[i] = _check_block(h, k, a, "psi_in")
        if tuple(b.shape) != tuple(a.shape):
            raise TypeError("psi_out: shape differs from psi_in")
        pin[i] = _dev_ptr(a, torch.complex128, "psi_in").value
        pout[i] = _dev_ptr(b, torch.complex128, "psi_out").value
    p = _vp()
    _check(load_library().qm_batch_plan_create(h, n, ks, pin, pout, nbs, ctypes.byref(p)))
    return p


def qm_batch_plan_launch(p, stream=None):
    _check(load_library().qm_batch_plan_launch(p, _stream_ptr(stream)))


def qm_batch_plan_destroy(p):
    _check(load_library().qm_batch_plan_destroy(p))


def qm_reserve(h, k, nbands):
    _check(load_library().qm_reserve(h, int(k), int(nbands)))


def qm_split_operator_set(h, v_r_dev, dt, stream=None):
    import torch
    _check(load_library().qm_split_operator_set(h, _dev_ptr(v_r_dev, torch.float64, "V_r"), float(dt), _stream_ptr(stream)))


def qm_split_operator_propagate(h, psi_in_dev, psi_out_dev, k=0, stream=None):
    import torch
    nb = _check_block(h, k, psi_in_dev, "psi_in")
    if tuple(psi_out_dev.shape) != tuple(psi_in_dev.shape):
        raise TypeError("psi_out: shape differs from psi_in")
    _check(load_library().qm_split_operator_propagate(h, k, _dev_ptr(psi_in_dev, torch.complex128, "psi_in"),
                                                      _dev_ptr(psi_out_dev, torch.complex128, "psi_out"), nb,
                                                      _stream_ptr(stream)))
    return psi_out_dev


def qm_mtxel_create(h, k_bra, k_ket, ecut_eps_ry):
    m = _vp()
    _check(load_library().qm_mtxel_create(h, int(k_bra), int(k_ket), float(ecut_eps_ry), ctypes.byref(m)))
    return m


def qm_mtxel_destroy(m):
    _check(load_library().qm_mtxel_destroy(m))


def qm_mtxel_num_g(m) -> int:
    n = _i()
    _check(load_library().qm_mtxel_num_g(m, ctypes.byref(n)))
    return n.value


def qm_mtxel_get_miller(m) -> np.ndarray:
    out = np.empty((qm_mtxel_num_g(m), 3), dtype=np.int32)
    _check(load_library().qm_mtxel_get_miller(m, out.ctypes.data))
    return out


def qm_mtxel_get_index_map(m) -> np.ndarray:
    out = np.empty(qm_mtxel_num_g(m), dtype=np.int32)
    _check(load_library().qm_mtxel_get_index_map(m, out.ctypes.data))
    return out


def qm_matrix_elements(m, h, k_bra, k_ket, bra_dev, ket_dev, out_dev=None, stream=None):
    """out [nbra][nket][ng_eps] = M_{nn'}(G) (include/qm_hpsi.h); h, k_bra, k_ket only check the operand shapes."""
    import torch
    nbra = _check_block(h, k_bra, bra_dev, "bra")
    nket = _check_block(h, k_ket, ket_dev, "ket")
    ng = qm_mtxel_num_g(m)
    if out_dev is None:
        out_dev = torch.empty((nbra, nket, ng), dtype=torch.complex128, device=bra_dev.device)
    if tuple(out_dev.shape) != (nbra, nket, ng):
        raise TypeError("out: expected shape [nbra][nket][ng_eps]")
    _check(load_library().qm_matrix_elements(m, _dev_ptr(bra_dev, torch.complex128, "bra"), nbra,
                                             _dev_ptr(ket_dev, torch.complex128, "ket"), nket,
                                             _dev_ptr(out_dev, torch.complex128, "out"), _stream_ptr(stream)))
    return out_dev


def qm_subspace(h, a_dev, b_dev, s_dev=None, k=0, stream=None):
    """S[i][j] = <a_i|b_j> over the sphere of k-point k (include/qm_hpsi.h); returns the [na][nb] device tensor."""
    import torch
    na = _check_block(h, k, a_dev, "a")
    nb = _check_block(h, k, b_dev, "b")
    if s_dev is None:
        s_dev = torch.empty((na, nb), dtype=torch.complex128, device=a_dev.device)
    if tuple(s_dev.shape) != (na, nb):
        raise TypeError("s: expected shape [na][nb]")
    _check(load_library().qm_subspace(h, k, _dev_ptr(a_dev, torch.complex128, "a"), na,
                                      _dev_ptr(b_dev, torch.complex128, "b"), nb,
                                      _dev_ptr(s_dev, torch.complex128, "s"), _stream_ptr(stream)))
    return s_dev


def qm_subspace_static(a_dev, b_dev, s_dev, stream=None):
    """S[i][j] = <a_i|b_j> written into the caller's s_dev [na][nb], for callers that may not allocate device memory
    (their pool owns the GPU, or a cudaMalloc would stall their other streams): no handle, and the split-K partial sums
    sit in a fixed 16 MiB array inside the library instead of a cudaMalloc'ed buffer (include/qm_hpsi.h).  All three
    tensors are the caller's -- unlike qm_subspace, this wrapper does not create the output either.  Blocks beyond
    1024 x 1024 states (padded to 64) raise QM_EINVAL.  Calls that can overlap on one GPU race on the shared array."""
    import torch
    for t, what in ((a_dev, "a"), (b_dev, "b"), (s_dev, "s")):
        if not isinstance(t, torch.Tensor) or t.dim() != 2:
            raise TypeError(f"{what}: expected a 2-D CUDA torch.Tensor")
    na, ng = a_dev.shape
    nb = b_dev.shape[0]
    if b_dev.shape[1] != ng or tuple(s_dev.shape) != (na, nb):
        raise TypeError("expected a [na][ng], b [nb][ng], s [na][nb]")
    _check(load_library().qm_subspace_static(_dev_ptr(a_dev, torch.complex128, "a"), na,
                                             _dev_ptr(b_dev, torch.complex128, "b"), nb, ng,
                                             _dev_ptr(s_dev, torch.complex128, "s"), _stream_ptr(stream)))
    return s_dev


def qm_taylor_propagate(h, psi_in_dev, psi_out_dev, dt, order, k=0, stream=None):
    import torch
    nb = _check_block(h, k, psi_in_dev, "psi_in")
    if tuple(psi_out_dev.shape) != tuple(psi_in_dev.shape):
        raise TypeError("psi_out: shape differs from psi_in")
    _check(load_library().qm_taylor_propagate(h, k, _dev_ptr(psi_in_dev, torch.complex128, "psi_in"),
                                              _dev_ptr(psi_out_dev, torch.complex128, "psi_out"), nb, float(dt),
                                              int(order), _stream_ptr(stream)))
    return psi_out_dev


def qm_density_reset(h, stream=None):
    _check(load_library().qm_density_reset(h, _stream_ptr(stream)))


def qm_density_accumulate(h, psi_dev, occ_dev, weight=1.0, k=0, stream=None):
    import torch
    nb = _check_block(h, k, psi_dev, "psi")
    if occ_dev.dim() != 1 or occ_dev.shape[0] != nb:
        raise TypeError("occ: expected shape [nbands]")
    _check(load_library().qm_density_accumulate(h, k, _dev_ptr(psi_dev, torch.complex128, "psi"), nb,
                                                _dev_ptr(occ_dev, torch.float64, "occ"), float(weight),
                                                _stream_ptr(stream)))


def qm_density_get(h, rho_dev, scale=1.0, stream=None):
    import torch
    _check(load_library().qm_density_get(h, _dev_ptr(rho_dev, torch.float64, "rho"), float(scale), _stream_ptr(stream)))
    return rho_dev


def _host_call(fn, h, psi_in_host, psi_out_host, k, stream):
    import torch
    nb = _check_block(h, k, psi_in_host, "psi_in")
    if tuple(psi_out_host.shape) != tuple(psi_in_host.shape):
        raise TypeError("psi_out: shape differs from psi_in")
    for t in (psi_in_host, psi_out_host):
        if t.is_cuda or t.dtype != torch.complex128 or not t.is_contiguous():
            raise TypeError("qm_apply_h_host: expected contiguous complex128 host tensors")
    _check(fn(h, ctypes.c_void_p(psi_in_host.data_ptr()), ctypes.c_void_p(psi_out_host.data_ptr()), nb, k,
              _stream_ptr(stream)))
    return psi_out_host


def qm_apply_h_host(h, psi_in_host, psi_out_host, k=0, stream=None):
    """Host (ideally pinned) torch tensors [nb][ng] complex128; copies are done inside the C call."""
    return _host_call(load_library().qm_apply_h_host, h, psi_in_host, psi_out_host, k, stream)


def qm_apply_h_host_async(h, psi_in_host, psi_out_host, k=0, stream=None):
    """Enqueue-only form; results are valid after qm_host_synchronize(h)."""
    return _host_call(load_library().qm_apply_h_host_async, h, psi_in_host, psi_out_host, k, stream)


def qm_host_synchronize(h):
    _check(load_library().qm_host_synchronize(h))


def qm_debug_g2r(h, psi_g_dev, box_r_dev, k=0, stream=None):
    import torch
    nb = _check_block(h, k, psi_g_dev, "psi_g")
    _check(load_library().qm_debug_g2r(h, _dev_ptr(psi_g_dev, torch.complex128, "psi_g"),
                                       _dev_ptr(box_r_dev, torch.complex128, "box_r"), nb, k, _stream_ptr(stream)))
    return box_r_dev


def qm_debug_r2g(h, box_r_dev, psi_g_dev, k=0, stream=None):
    import torch
    nb = _check_block(h, k, psi_g_dev, "psi_g")
    _check(load_library().qm_debug_r2g(h, _dev_ptr(box_r_dev, torch.complex128, "box_r"),
                                       _dev_ptr(psi_g_dev, torch.complex128, "psi_g"), nb, k, _stream_ptr(stream)))
    return psi_g_dev


def qm_get_launch_count(h) -> int:
    c = ctypes.c_ulonglong()
    _check(load_library().qm_get_launch_count(h, ctypes.byref(c)))
    return c.value


def qm_probe_fp64_tensor_peak():
    a, b = _d(), _d()
    _check(load_library().qm_probe_fp64_tensor_peak(ctypes.byref(a), ctypes.byref(b)))
    return a.value, b.value


def qm_profile_enable(h, on: bool):
    _check(load_library().qm_profile_enable(h, int(bool(on))))


def qm_profile_reset(h):
    _check(load_library().qm_profile_reset(h))


def qm_kernel_name(kind: int) -> str:
    return load_library().qm_kernel_name(int(kind)).decode()


def qm_profile_read(h):
    """{kernel name: (total device ms, launches)} since the last reset."""
    out = {}
    for kind in range(QM_K_COUNT):
        ms, n = _d(), ctypes.c_ulonglong()
        _check(load_library().qm_profile_read(h, kind, ctypes.byref(ms), ctypes.byref(n)))
        out[qm_kernel_name(kind)] = (ms.value, n.value)
    return out


class GSpace:
    """Owning wrapper of a qm_gspace handle (the paper's GSpace + KSHam.h_psi)."""

    def __init__(self, lattice_bohr, ecutwfc_ry, fft_grid, kpts_cryst=None):
        self.grid = tuple(int(x) for x in fft_grid)
        self._h = qm_gspace_create(lattice_bohr, ecutwfc_ry, fft_grid, kpts_cryst)
        self.nk = qm_gspace_num_k(self._h)

    def close(self):
        if getattr(self, "_h", None) is not None:
            qm_gspace_destroy(self._h)
            self._h = None

    __del__ = close

    @property
    def handle(self):
        return self._h

    def num_g(self, k=0): return qm_gspace_num_g(self._h, k)
    def num_sticks(self, k=0): return qm_gspace_num_sticks(self._h, k)
    def index_map(self, k=0): return qm_gspace_get_index_map(self._h, k)
    def miller(self, k=0): return qm_gspace_get_miller(self._h, k)
    def g2(self, k=0): return qm_gspace_get_g2(self._h, k)
    def alias_free(self, k=0): return qm_gspace_alias_free(self._h, k)
    def set_vloc(self, v, stream=None): qm_set_vloc(self._h, v, stream)
    def set_nonlocal(self, k, beta, d, stream=None): qm_set_nonlocal(self._h, k, beta, d, stream)

    def apply_h(self, psi_in, psi_out=None, k=0, stream=None):
        import torch
        if psi_out is None:
            psi_out = torch.empty_like(psi_in)
        return qm_apply_h(self._h, psi_in, psi_out, k, stream)

    def subspace(self, a, b, s=None, k=0, stream=None): return qm_subspace(self._h, a, b, s, k, stream)
    def reserve(self, nbands, k=0): qm_reserve(self._h, k, nbands)
    def batch_plan(self, items): return BatchPlan(self, items)
    def split_operator_set(self, v, dt, stream=None): qm_split_operator_set(self._h, v, dt, stream)

    def split_operator_propagate(self, psi_in, psi_out=None, k=0, stream=None):
        import torch
        if psi_out is None:
            psi_out = torch.empty_like(psi_in)
        return qm_split_operator_propagate(self._h, psi_in, psi_out, k, stream)

    def mtxel(self, k_bra, k_ket, ecut_eps_ry): return MatrixElements(self, k_bra, k_ket, ecut_eps_ry)

    def taylor_propagate(self, psi_in, dt, order, psi_out=None, k=0, stream=None):
        import torch
        if psi_out is None:
            psi_out = torch.empty_like(psi_in)
        return qm_taylor_propagate(self._h, psi_in, psi_out, dt, order, k, stream)

    def density_reset(self, stream=None): qm_density_reset(self._h, stream)

    def density_accumulate(self, psi, occ, weight=1.0, k=0, stream=None):
        qm_density_accumulate(self._h, psi, occ, weight, k, stream)

    def density_get(self, rho=None, scale=1.0, stream=None):
        import torch
        if rho is None:
            rho = torch.empty(int(self.grid[0]) * int(self.grid[1]) * int(self.grid[2]), dtype=torch.float64,
                              device=torch.device("cuda", torch.cuda.current_device()))
        return qm_density_get(self._h, rho, scale, stream)

    def apply_h_host(self, psi_in, psi_out, k=0, stream=None):
        return qm_apply_h_host(self._h, psi_in, psi_out, k, stream)

    def apply_h_host_async(self, psi_in, psi_out, k=0, stream=None):
        return qm_apply_h_host_async(self._h, psi_in, psi_out, k, stream)

    def host_synchronize(self): qm_host_synchronize(self._h)

    def g2r(self, psi_g, k=0, stream=None):
        import torch
        box = torch.empty((psi_g.shape[0], int(np.prod(self.grid))), dtype=torch.complex128, device=psi_g.device)
        return qm_debug_g2r(self._h, psi_g, box, k, stream)

    def r2g(self, box_r, k=0, stream=None):
        import torch
        out = torch.empty((box_r.shape[0], self.num_g(k)), dtype=torch.complex128, device=box_r.device)
        return qm_debug_r2g(self._h, box_r, out, k, stream)

    def launch_count(self): return qm_get_launch_count(self._h)


class MatrixElements:
    """Owning wrapper of a qm_mtxel (the paper's matrix_elements step of Epsilon)."""

    def __init__(self, gs: GSpace, k_bra: int, k_ket: int, ecut_eps_ry: float):
        self._gs, self.k_bra, self.k_ket = gs, k_bra, k_ket          # keeps the borrowed handle alive
        self._m = qm_mtxel_create(gs.handle, k_bra, k_ket, ecut_eps_ry)

    def close(self):
        if getattr(self, "_m", None) is not None:
            qm_mtxel_destroy(self._m)
            self._m = None

    __del__ = close

    def num_g(self): return qm_mtxel_num_g(self._m)
    def miller(self): return qm_mtxel_get_miller(self._m)
    def index_map(self): return qm_mtxel_get_index_map(self._m)

    def apply(self, bra, ket, out=None, stream=None):
        return qm_matrix_elements(self._m, self._gs.handle, self.k_bra, self.k_ket, bra, ket, out, stream)


class BatchPlan:
    """Owning wrapper of a qm_batch_plan: a fixed list of (k, psi_in, psi_out) applies launched as one CUDA graph."""

    def __init__(self, gs: GSpace, items):
        self._gs, self._items = gs, list(items)                      # keep the handle and the tensors alive
        self._p = qm_batch_plan_create(gs.handle, self._items)

    def close(self):
        if getattr(self, "_p", None) is not None:
            qm_batch_plan_destroy(self._p)
            self._p = None

    __del__ = close

    def launch(self, stream=None): qm_batch_plan_launch(self._p, stream)
