"""Thin Python binding of the C-ABI in include/wick.h (ctypes; argument marshalling only).

Every step of the path runs inside libwick_b200.so.  PyTorch appears only as the owner of device
memory and streams (tensors are passed as raw pointers).  There is no CPU fallback: if the shared
library is missing or has no CUDA device, the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence, Tuple

import numpy as np

_LIB_PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "libwick_b200.so")
_lib = None

BUILD_IDENTITY_TEST = 1
BUILD_ISOSPIN = 2
CONTRACT_FORCE_FLAT = 1
CONTRACT_NO_STAGED = 2
CONTRACT_COMPLEX_COEFFS = 4
CONTRACT_NO_REG_MINORS = 8
CONTRACT_JACOBI = 16
CONTRACT_JACOBI_UNFUSED = 32

EXPORTED_SYMBOLS = (
    "wick_build_terms", "wick_build_terms_from_list", "wick_terms_get_info", "wick_terms_export_tuples",
    "wick_terms_export_minors", "wick_terms_export_terms", "wick_terms_export_factors",
    "wick_terms_staged_schedule_check", "wick_terms_export_minor_order", "wick_terms_free",
    "wick_contract_min_workspace_bytes", "wick_contract_workspace_bytes", "wick_contract",
    "wick_contract_host", "wick_release_cached_buffers", "wick_minor_dets", "wick_minor_dets_static", "wick_static_scratch_bytes", "wick_terms_minor_table", "wick_launch_count", "wick_launch_count_reset",
    "wick_operator_from_nucleons", "wick_operator_from_raw", "wick_operator_paper", "wick_operator_info", "wick_operator_export",
    "wick_operator_free", "wick_operator_product", "wick_build_block_terms", "wick_block_tensor", "wick_block_tensor_workspace_bytes",
    "wick_combine_two_clusters", "wick_build_terms_matrix", "wick_contract_many", "wick_contract_many_workspace_bytes",
    "wick_last_error", "wick_version", "wick_profile_enable", "wick_profile_read", "wick_measure_fp64_peak",
)


class WickError(RuntimeError):
    pass


class _Nucleon(C.Structure):
    _fields_ = [("kind", C.c_int32), ("gamma", C.c_int32)]


class TermsInfo(C.Structure):
    _fields_ = [
        ("n_u", C.c_int32), ("n_d", C.c_int32),
        ("n_rows_u", C.c_int32), ("n_cols_u", C.c_int32), ("n_rows_d", C.c_int32), ("n_cols_d", C.c_int32),
        ("n_minors_u", C.c_int64), ("n_minors_d", C.c_int64), ("n_terms", C.c_int64),
        ("is_outer_product", C.c_int32), ("n_sink", C.c_int32), ("n_source", C.c_int32),
        ("n_raw", C.c_int64), ("n_identity_merged", C.c_int64),
    ]


class Profile(C.Structure):
    _fields_ = [("ms", C.c_double * 4), ("launches", C.c_int64 * 4)]


def library_path() -> str:
    return _LIB_PATH


def load_library():
    """dlopen libwick_b200.so (built in-tree by paper_2411_08962_b200.build); raises if absent."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise WickError(f"{_LIB_PATH} is missing: run `python -m paper_2411_08962_b200.build` "
                        "(there is no CPU fallback for the CUDA path)")
    lib = C.CDLL(_LIB_PATH)
    vp, i32, i64, u64, u32, sz = C.c_void_p, C.c_int, C.c_int64, C.c_uint64, C.c_uint, C.c_size_t
    lib.wick_build_terms.argtypes = [C.POINTER(_Nucleon), i32, u32, u64, C.POINTER(vp)]
    lib.wick_build_terms_from_list.argtypes = [i32, i32, i64, vp, vp, vp, vp, vp, u32, u64, C.POINTER(vp)]
    lib.wick_terms_get_info.argtypes = [vp, C.POINTER(TermsInfo)]
    lib.wick_terms_export_tuples.argtypes = [vp, vp, vp, vp, vp]
    lib.wick_terms_export_minors.argtypes = [vp, vp, vp, vp, vp]
    lib.wick_terms_export_terms.argtypes = [vp, i64, i64, vp, vp, vp]
    lib.wick_terms_export_factors.argtypes = [vp, vp, vp, vp, vp, vp, vp]
    lib.wick_terms_staged_schedule_check.argtypes = [vp, C.c_int, vp, vp, vp, vp]
    lib.wick_terms_export_minor_order.argtypes = [vp, C.c_int, vp, vp, vp]
    lib.wick_terms_free.argtypes = [vp]
    lib.wick_terms_free.restype = None
    lib.wick_release_cached_buffers.restype = None
    lib.wick_release_cached_buffers.argtypes = []
    for f in (lib.wick_contract_min_workspace_bytes, lib.wick_contract_workspace_bytes):
        f.argtypes = [vp, i32, i32, i32]
        f.restype = sz
    lib.wick_contract.argtypes = [vp, vp, vp, vp, i32, i32, i32, vp, vp, vp, sz, u32, vp]
    lib.wick_contract_host.argtypes = [vp, vp, vp, vp, i32, i32, i32, vp, vp, u32]
    lib.wick_minor_dets.argtypes = [vp, i64, i32, vp, vp, i64, vp, vp]
    lib.wick_minor_dets_static.argtypes = [vp, i64, i32, vp, vp, i64, vp, vp]
    lib.wick_static_scratch_bytes.argtypes = []
    lib.wick_static_scratch_bytes.restype = sz
    lib.wick_terms_minor_table.argtypes = [vp, i64, vp, i32, u32, vp, vp]
    lib.wick_operator_from_nucleons.argtypes = [C.POINTER(_Nucleon), i32, C.POINTER(vp)]
    lib.wick_operator_from_raw.argtypes = [i32, i64, vp, vp, vp, C.POINTER(vp)]
    lib.wick_operator_paper.argtypes = [i32, i32, C.POINTER(vp)]
    lib.wick_operator_info.argtypes = [vp, C.POINTER(C.c_int32), C.POINTER(C.c_int32), C.POINTER(i64)]
    lib.wick_operator_export.argtypes = [vp, vp, vp, vp]
    lib.wick_operator_free.argtypes = [vp]
    lib.wick_operator_free.restype = None
    lib.wick_operator_product.argtypes = [vp, vp, C.POINTER(vp)]
    lib.wick_build_block_terms.argtypes = [vp, C.POINTER(vp)]
    lib.wick_block_tensor_workspace_bytes.argtypes = [vp, i32]
    lib.wick_block_tensor_workspace_bytes.restype = sz
    lib.wick_block_tensor.argtypes = [vp, vp, vp, vp, i32, i32, vp, vp, sz, u32, vp]
    lib.wick_combine_two_clusters.argtypes = [vp, vp, vp, vp, vp, i32, vp]
    lib.wick_build_terms_matrix.argtypes = [C.POINTER(vp), i32, u32, C.POINTER(vp)]
    lib.wick_contract_many_workspace_bytes.argtypes = [vp, i32, i32, i32, i32]
    lib.wick_contract_many_workspace_bytes.restype = sz
    lib.wick_contract_many.argtypes = [vp, vp, C.POINTER(vp), i32, vp, i32, i32, i32, vp, vp, vp, sz, u32, vp]
    lib.wick_profile_enable.argtypes = [i32]
    lib.wick_profile_read.argtypes = [C.POINTER(Profile)]
    lib.wick_measure_fp64_peak.argtypes = [C.POINTER(C.c_double), vp]
    lib.wick_launch_count.restype = i64
    lib.wick_launch_count_reset.restype = i64
    lib.wick_last_error.restype = C.c_char_p
    lib.wick_version.restype = C.c_char_p
    _lib = lib
    return lib


def _check(rc: int, what: str):
    if rc != 0:
        raise WickError(f"{what} failed ({rc}): {load_library().wick_last_error().decode()}")


def _np_ptr(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


class Terms:
    """Handle of a canonical term list + unique-minor tables (wick_terms*)."""

    def __init__(self, handle):
        self._h = C.c_void_p(handle)
        info = TermsInfo()
        _check(load_library().wick_terms_get_info(self._h, C.byref(info)), "wick_terms_get_info")
        self.info = info

    def __del__(self):
        h, self._h = getattr(self, "_h", None), None
        if h and _lib is not None:
            _lib.wick_terms_free(h)

    # -- exports (host numpy arrays) --
    def tuples(self):
        i = self.info
        out = [np.zeros((i.n_rows_u, i.n_u), np.uint8), np.zeros((i.n_cols_u, i.n_u), np.uint8),
               np.zeros((i.n_rows_d, i.n_d), np.uint8), np.zeros((i.n_cols_d, i.n_d), np.uint8)]
        _check(_lib.wick_terms_export_tuples(self._h, *[_np_ptr(a) for a in out]), "wick_terms_export_tuples")
        return tuple(out)

    def minors(self):
        i = self.info
        out = [np.zeros(i.n_minors_u, np.int32), np.zeros(i.n_minors_u, np.int32),
               np.zeros(i.n_minors_d, np.int32), np.zeros(i.n_minors_d, np.int32)]
        _check(_lib.wick_terms_export_minors(self._h, *[_np_ptr(a) for a in out]), "wick_terms_export_minors")
        return tuple(out)

    def terms(self, first: int = 0, count: Optional[int] = None):
        count = self.info.n_terms - first if count is None else count
        uid, did = np.zeros(count, np.int32), np.zeros(count, np.int32)
        w = np.zeros(count, np.complex128)
        _check(_lib.wick_terms_export_terms(self._h, first, count, _np_ptr(uid), _np_ptr(did), _np_ptr(w)),
               "wick_terms_export_terms")
        return uid, did, w

    def factors(self):
        i = self.info
        sru, srd = np.zeros(i.n_sink, np.int32), np.zeros(i.n_sink, np.int32)
        qcu, qcd = np.zeros(i.n_source, np.int32), np.zeros(i.n_source, np.int32)
        sc, qc = np.zeros(i.n_sink, np.complex128), np.zeros(i.n_source, np.complex128)
        _check(_lib.wick_terms_export_factors(self._h, _np_ptr(sru), _np_ptr(srd), _np_ptr(sc),
                                              _np_ptr(qcu), _np_ptr(qcd), _np_ptr(qc)), "wick_terms_export_factors")
        return sru, srd, sc, qcu, qcd, qc

    def minor_order(self, flavour: int):
        """(minor_id [n_minors], proc_cols [n_minors][n], negate [n_minors]): the order in which the minors kernel walks this
        flavour's unique minors and takes their columns (flavour 0 = u, 1 = d)."""
        i = self.info
        nm, n = (i.n_minors_u, i.n_u) if flavour == 0 else (i.n_minors_d, i.n_d)
        mid, pc, neg = np.zeros(nm, np.int32), np.zeros((nm, n), np.uint8), np.zeros(nm, np.uint8)
        _check(_lib.wick_terms_export_minor_order(self._h, flavour, _np_ptr(mid), _np_ptr(pc), _np_ptr(neg)),
               "wick_terms_export_minor_order")
        return mid, pc, neg

    def staged_schedule_check(self, n_bins: int):
        """Host-only self-check of the staged-reduction schedule; returns (batches, pairs covered, max MD block, max rows)."""
        out = [C.c_int64(0) for _ in range(4)]
        _check(_lib.wick_terms_staged_schedule_check(self._h, n_bins, *[C.byref(o) for o in out]),
               "wick_terms_staged_schedule_check")
        return tuple(int(o.value) for o in out)

    def term_tuples(self, first: int = 0, count: Optional[int] = None):
        """Flat terms as index tuples (a_u, b_u, a_d, b_d, w) -- what an oracle consumes."""
        ur, uc, dr, dc = self.tuples()
        umr, umc, dmr, dmc = self.minors()
        uid, did, w = self.terms(first, count)
        return ur[umr[uid]], uc[umc[uid]], dr[dmr[did]], dc[dmc[did]], w


def build_terms(nucleus: Sequence[Tuple[str, int]], flags: int = 0, seed: int = 0) -> Terms:
    """nucleus: sequence of ('p' | 'n', gamma) in product order -> canonical term list."""
    lib = load_library()
    arr = (_Nucleon * max(len(nucleus), 1))()
    for k, (kind, gamma) in enumerate(nucleus):
        if kind not in ("p", "n"):
            raise WickError(f"nucleon kind must be 'p' or 'n', got {kind!r}")
        arr[k].kind = 0 if kind == "p" else 1
        arr[k].gamma = int(gamma)
    h = C.c_void_p()
    _check(lib.wick_build_terms(arr, len(nucleus), flags, seed, C.byref(h)), "wick_build_terms")
    return Terms(h.value)


def build_terms_from_list(a_u, b_u, a_d, b_d, w, flags: int = 0, seed: int = 0) -> Terms:
    lib = load_library()
    a_u, b_u, a_d, b_d = (np.ascontiguousarray(x, dtype=np.uint8) for x in (a_u, b_u, a_d, b_d))
    w = np.ascontiguousarray(w, dtype=np.complex128)
    n_raw = len(w)
    n_u = a_u.shape[1] if a_u.ndim == 2 else 0
    n_d = a_d.shape[1] if a_d.ndim == 2 else 0
    h = C.c_void_p()
    _check(lib.wick_build_terms_from_list(n_u, n_d, n_raw, _np_ptr(a_u), _np_ptr(b_u), _np_ptr(a_d), _np_ptr(b_d),
                                          _np_ptr(w), flags, seed, C.byref(h)), "wick_build_terms_from_list")
    return Terms(h.value)


OP_DEUTERON_EQ20 = 1
OP_HELIUM3_EQ21 = 2


class Operator:
    """Handle of an interpolator in canonical form (wick_operator*): monomial (u tuple, d tuple) -> coefficient."""

    def __init__(self, handle):
        self._h = C.c_void_p(handle)
        nu, nd, nt = C.c_int32(0), C.c_int32(0), C.c_int64(0)
        _check(load_library().wick_operator_info(self._h, C.byref(nu), C.byref(nd), C.byref(nt)), "wick_operator_info")
        self.n_u, self.n_d, self.n_terms = int(nu.value), int(nd.value), int(nt.value)

    def __del__(self):
        h, self._h = getattr(self, "_h", None), None
        if h and _lib is not None:
            _lib.wick_operator_free(h)

    def terms(self):
        """(u_tuples [n_terms][n_u], d_tuples [n_terms][n_d], coefficients [n_terms])."""
        u = np.zeros((self.n_terms, self.n_u), np.uint8)
        d = np.zeros((self.n_terms, self.n_d), np.uint8)
        c = np.zeros(self.n_terms, np.complex128)
        _check(_lib.wick_operator_export(self._h, _np_ptr(u), _np_ptr(d), _np_ptr(c)), "wick_operator_export")
        return u, d, c


def operator_from_nucleons(nucleus: Sequence[Tuple[str, int]]) -> Operator:
    lib = load_library()
    arr = (_Nucleon * max(len(nucleus), 1))()
    for k, (kind, gamma) in enumerate(nucleus):
        if kind not in ("p", "n"):
            raise WickError(f"nucleon kind must be 'p' or 'n', got {kind!r}")
        arr[k].kind = 0 if kind == "p" else 1
        arr[k].gamma = int(gamma)
    h = C.c_void_p()
    _check(lib.wick_operator_from_nucleons(arr, len(nucleus), C.byref(h)), "wick_operator_from_nucleons")
    return Operator(h.value)


def operator_from_raw(flavour, chi, coef) -> Operator:
    """flavour, chi: [n_raw][n_quarks] (0 = u, 1 = d; chi = 3*spin + colour) in operator order; coef [n_raw] complex."""
    lib = load_library()
    flavour = np.ascontiguousarray(flavour, dtype=np.uint8)
    chi = np.ascontiguousarray(chi, dtype=np.uint8)
    coef = np.ascontiguousarray(coef, dtype=np.complex128)
    n_raw = len(coef)
    n_q = flavour.shape[1] if flavour.ndim == 2 else 0
    h = C.c_void_p()
    _check(lib.wick_operator_from_raw(n_q, n_raw, _np_ptr(flavour), _np_ptr(chi), _np_ptr(coef), C.byref(h)), "wick_operator_from_raw")
    return Operator(h.value)


def operator_paper(which: int, J: int = 0) -> Operator:
    """The paper's interpolators: OP_DEUTERON_EQ20 (Eq. 20) or OP_HELIUM3_EQ21 (Eq. 21, open index J)."""
    h = C.c_void_p()
    _check(load_library().wick_operator_paper(which, J, C.byref(h)), "wick_operator_paper")
    return Operator(h.value)


def operator_product(a: Operator, b: Operator) -> Operator:
    """The ordered product A.B of two interpolators (Grassmann product, canonical form)."""
    h = C.c_void_p()
    _check(load_library().wick_operator_product(a._h, b._h, C.byref(h)), "wick_operator_product")
    return Operator(h.value)


def build_block_terms(cluster: Operator) -> Terms:
    """Block handle of one cluster of a cluster sink (wick_build_block_terms): rows = the cluster's row tuples, columns =
    every subset of the 12 source indices."""
    h = C.c_void_p()
    _check(load_library().wick_build_block_terms(cluster._h, C.byref(h)), "wick_build_block_terms")
    return Terms(h.value)


def block_tensor(U, D, block_terms: Terms, momentum, L: int, T: int, flags: int = 0, stream=None):
    """B[t][S_u][S_d] = sum_x e^{ip.x} sum_i c_i det U_x[a_u(i), S_u] det D_x[a_d(i), S_d] on the device
    (wick_block_tensor).  Returns CUDA complex128 [T][C(12,n_u)][C(12,n_d)]."""
    import torch
    lib = load_library()
    V = L ** 3
    _check_dev(U, "U", (T, V, 12, 12))
    _check_dev(D, "D", (T, V, 12, 12))
    mom = np.ascontiguousarray(momentum, dtype=np.int32).reshape(3)
    i = block_terms.info
    with torch.cuda.device(U.device), torch.cuda.stream(torch.cuda.current_stream() if stream is None else stream):
        ws = torch.empty(int(lib.wick_block_tensor_workspace_bytes(block_terms._h, L)), dtype=torch.uint8, device=U.device)
        out = torch.empty((T, i.n_cols_u, i.n_cols_d), dtype=torch.complex128, device=U.device)
        rc = lib.wick_block_tensor(U.data_ptr(), D.data_ptr(), block_terms._h, _np_ptr(mom), L, T, out.data_ptr(), ws.data_ptr(),
                                   ws.numel(), flags, _stream_ptr(stream))
    _check(rc, "wick_block_tensor")
    return out


def combine_two_clusters(a: Operator, b: Operator, source: Operator, BA, BB) -> np.ndarray:
    """C[t] from the two block tensors (host numpy complex128 [T][..][..]) and the source operator (wick_combine_two_clusters)."""
    BA = np.ascontiguousarray(BA, dtype=np.complex128)
    BB = np.ascontiguousarray(BB, dtype=np.complex128)
    T = BA.shape[0]
    out = np.zeros(T, np.complex128)
    _check(load_library().wick_combine_two_clusters(a._h, b._h, source._h, _np_ptr(BA), _np_ptr(BB), T, _np_ptr(out)),
           "wick_combine_two_clusters")
    return out


def two_cluster_correlator(U, D, a: Operator, b: Operator, mom_a, mom_b, L: int, T: int, source: Optional[Operator] = None):
    """Cluster-sink correlator C[t] = sum_{x,y} e^{ip_A.x} e^{ip_B.y} <O_A(x) O_B(y) Obar_source(0)>  (the
    plane-wave sink of Eq. 8 for single nucleons): two block tensors on the device, combined on the host."""
    source = operator_product(a, b) if source is None else source
    BA = block_tensor(U, D, build_block_terms(a), mom_a, L, T).cpu().numpy()
    BB = block_tensor(U, D, build_block_terms(b), mom_b, L, T).cpu().numpy()
    return combine_two_clusters(a, b, source, BA, BB)


def build_terms_matrix(ops: Sequence[Operator], flags: int = 0):
    """K operators -> K x K nested list of Terms, [k][k'] = (operator k at the sink) x conj(operator k' at the source),
    all over one pair of unique-minor tables (for contract_many)."""
    lib = load_library()
    K = len(ops)
    arr = (C.c_void_p * max(K, 1))(*[o._h for o in ops])
    out = (C.c_void_p * max(K * K, 1))()
    _check(lib.wick_build_terms_matrix(arr, K, flags, out), "wick_build_terms_matrix")
    return [[Terms(out[k * K + kp]) for kp in range(K)] for k in range(K)]


def contract_many(U, D, terms_list: Sequence[Terms], momenta, L: int, T: int, want_sigma: bool = False, flags: int = 0,
                  stream=None):
    """C[list][p][t] for term lists that share their unique-minor tables (wick_contract_many): the determinants are
    evaluated once per site for all lists.  Returns C (CUDA complex128 [n_lists][n_mom][T]) or (C, sigma [n_lists][T][L^3])."""
    import torch
    lib = load_library()
    V = L ** 3
    _check_dev(U, "U", (T, V, 12, 12))
    _check_dev(D, "D", (T, V, 12, 12))
    mom = np.ascontiguousarray(momenta, dtype=np.int32).reshape(-1, 3)
    n_mom, n = mom.shape[0], len(terms_list)
    arr = (C.c_void_p * max(n, 1))(*[t._h for t in terms_list])
    with torch.cuda.device(U.device), torch.cuda.stream(torch.cuda.current_stream() if stream is None else stream):
        ws = torch.empty(int(lib.wick_contract_many_workspace_bytes(terms_list[0]._h, n, L, T, n_mom)), dtype=torch.uint8, device=U.device)
        Cout = torch.empty((n, n_mom, T), dtype=torch.complex128, device=U.device)
        sigma = torch.empty((n, T, V), dtype=torch.complex128, device=U.device) if want_sigma else None
        rc = lib.wick_contract_many(U.data_ptr(), D.data_ptr(), arr, n, _np_ptr(mom), n_mom, L, T, Cout.data_ptr(),
                                    None if sigma is None else sigma.data_ptr(), ws.data_ptr(), ws.numel(), flags, _stream_ptr(stream))
    _check(rc, "wick_contract_many")
    return (Cout, sigma) if want_sigma else Cout


def _stream_ptr(stream):
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def _check_dev(t, name, shape=None):
    import torch
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.complex128 and t.is_contiguous()):
        raise WickError(f"{name} must be a contiguous CUDA complex128 tensor")
    if shape is not None and tuple(t.shape) != tuple(shape):
        raise WickError(f"{name} must have shape {tuple(shape)}, got {tuple(t.shape)}")


def contract_workspace_bytes(terms: Terms, L: int, T: int, n_mom: int, minimum: bool = False) -> int:
    lib = load_library()
    f = lib.wick_contract_min_workspace_bytes if minimum else lib.wick_contract_workspace_bytes
    return int(f(terms._h, L, T, n_mom))


def contract(U, D, terms: Terms, momenta, L: int, T: int, workspace=None, want_sigma: bool = False,
             flags: int = 0, stream=None, out=None):
    """C[p][t] on the device (wick_contract).  U, D: CUDA complex128 [T][L^3][12][12].
    Returns C (CUDA complex128 [n_mom][T]) or (C, sigma [T][L^3]) if want_sigma."""
    import torch
    lib = load_library()
    V = L ** 3
    _check_dev(U, "U", (T, V, 12, 12))
    _check_dev(D, "D", (T, V, 12, 12))
    mom = np.ascontiguousarray(momenta, dtype=np.int32).reshape(-1, 3)
    n_mom = mom.shape[0]
    if out is not None:
        _check_dev(out, "out", (n_mom, T))
    if workspace is not None and not (isinstance(workspace, torch.Tensor) and workspace.is_cuda and workspace.is_contiguous()):
        raise WickError("workspace must be a contiguous CUDA tensor")
    # buffers created here are allocated on the stream the work is enqueued on, so the caching allocator cannot hand
    # them to another stream's allocation while the kernels still run
    with torch.cuda.device(U.device), torch.cuda.stream(torch.cuda.current_stream() if stream is None else stream):
        if workspace is None:
            workspace = torch.empty(contract_workspace_bytes(terms, L, T, n_mom), dtype=torch.uint8, device=U.device)
        Cout = torch.empty((n_mom, T), dtype=torch.complex128, device=U.device) if out is None else out
        sigma = torch.empty((T, V), dtype=torch.complex128, device=U.device) if want_sigma else None
        rc = lib.wick_contract(U.data_ptr(), D.data_ptr(), terms._h, _np_ptr(mom), n_mom, L, T, Cout.data_ptr(),
                               None if sigma is None else sigma.data_ptr(), workspace.data_ptr(),
                               workspace.numel() * workspace.element_size(), flags, _stream_ptr(stream))
    _check(rc, "wick_contract")
    return (Cout, sigma) if want_sigma else Cout


def contract_host(U: np.ndarray, D: np.ndarray, terms: Terms, momenta, L: int, T: int, want_sigma: bool = False,
                  flags: int = 0):
    """Same from HOST arrays (numpy complex128 or pinned torch CPU tensors); copies are inside the call."""
    lib = load_library()
    V = L ** 3

    def host_ptr(a, name):
        if isinstance(a, np.ndarray):
            if a.dtype != np.complex128 or not a.flags.c_contiguous or a.shape != (T, V, 12, 12):
                raise WickError(f"{name} must be a C-contiguous complex128 array [T][L^3][12][12]")
            return a.ctypes.data_as(C.c_void_p)
        import torch
        if tuple(a.shape) != (T, V, 12, 12) or not a.is_contiguous() or a.is_cuda or a.dtype != torch.complex128:
            raise WickError(f"{name} must be a contiguous CPU complex128 tensor [T][L^3][12][12]")
        return C.c_void_p(a.data_ptr())

    mom = np.ascontiguousarray(momenta, dtype=np.int32).reshape(-1, 3)
    Cout = np.zeros((mom.shape[0], T), np.complex128)
    sigma = np.zeros((T, V), np.complex128) if want_sigma else None
    rc = lib.wick_contract_host(host_ptr(U, "U"), host_ptr(D, "D"), terms._h, _np_ptr(mom), mom.shape[0], L, T,
                                _np_ptr(Cout), _np_ptr(sigma), flags)
    _check(rc, "wick_contract_host")
    return (Cout, sigma) if want_sigma else Cout


def minor_dets(P, rows, cols, stream=None):
    """Step a4 alone: out[m][s] = det P[s][rows[m], cols[m]].  P: CUDA complex128 [n_sites][12][12]."""
    import torch
    lib = load_library()
    _check_dev(P, "P")
    rows = np.ascontiguousarray(rows, dtype=np.uint8)
    cols = np.ascontiguousarray(cols, dtype=np.uint8)
    n_minors, n = rows.shape
    n_sites = P.shape[0]
    out = torch.empty((n_minors, n_sites), dtype=torch.complex128, device=P.device)
    with torch.cuda.device(P.device):
        rc = lib.wick_minor_dets(P.data_ptr(), n_sites, n, _np_ptr(rows), _np_ptr(cols), n_minors, out.data_ptr(),
                                 _stream_ptr(stream))
    _check(rc, "wick_minor_dets")
    return out


def minor_dets_static(P, rows, cols, out, stream=None):
    """wick_minor_dets_static: step a4 with no allocation inside the library (scratch in a static device array).  The caller
    passes the output too: out CUDA complex128 [n_minors][n_sites]."""
    lib = load_library()
    _check_dev(P, "P")
    rows = np.ascontiguousarray(rows, dtype=np.uint8)
    cols = np.ascontiguousarray(cols, dtype=np.uint8)
    n_minors, n = rows.shape
    n_sites = P.shape[0]
    _check_dev(out, "out", (n_minors, n_sites))
    import torch
    with torch.cuda.device(P.device):
        rc = lib.wick_minor_dets_static(P.data_ptr(), n_sites, n, _np_ptr(rows), _np_ptr(cols), n_minors, out.data_ptr(),
                                        _stream_ptr(stream))
    _check(rc, "wick_minor_dets_static")
    return out


def static_scratch_bytes() -> int:
    return int(load_library().wick_static_scratch_bytes())


def minor_table(P, terms: Terms, flavour: int, flags: int = 0, stream=None):
    """Unique-minor table of one flavour (0 = u, 1 = d) for the matrices P [n_sites][12][12], through the kernels
    wick_contract uses for this handle.  Returns CUDA complex128 [n_minors][n_sites]."""
    import torch
    lib = load_library()
    _check_dev(P, "P")
    n_sites = P.shape[0]
    n_pad = (n_sites + 31) // 32 * 32
    nm = terms.info.n_minors_u if flavour == 0 else terms.info.n_minors_d
    out = torch.zeros((nm, n_pad), dtype=torch.complex128, device=P.device)
    with torch.cuda.device(P.device):
        rc = lib.wick_terms_minor_table(P.data_ptr(), n_sites, terms._h, flavour, flags, out.data_ptr(), _stream_ptr(stream))
    _check(rc, "wick_terms_minor_table")
    return out[:, :n_sites]


def release_cached_buffers() -> None:
    """Free the device buffers contract_host keeps between calls (this thread)."""
    _lib.wick_release_cached_buffers()


def launch_count(reset: bool = False) -> int:
    lib = load_library()
    return int(lib.wick_launch_count_reset() if reset else lib.wick_launch_count())


def profile_enable(on: bool = True) -> None:
    _check(load_library().wick_profile_enable(1 if on else 0), "wick_profile_enable")


def profile_read():
    """Per-class device time (ms) and launch counts recorded since the last read:
    {'minors_u': (ms, n), 'minors_d': ..., 'reduce': ..., 'project': ...}."""
    p = Profile()
    _check(load_library().wick_profile_read(C.byref(p)), "wick_profile_read")
    names = ("minors_u", "minors_d", "reduce", "project")
    return {k: (float(p.ms[i]), int(p.launches[i])) for i, k in enumerate(names)}


def measure_fp64_peak(stream=None) -> float:
    """TFLOP/s of a register-only DFMA stream on all SMs."""
    out = C.c_double(0.0)
    _check(load_library().wick_measure_fp64_peak(C.byref(out), _stream_ptr(stream)), "wick_measure_fp64_peak")
    return float(out.value)
