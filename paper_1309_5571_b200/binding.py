"""Thin ctypes binding of libdmrg_b200.so (include/dmrg_b200.h) -- argument marshalling only.

Every step of the hot path runs in the CUDA kernels of the library; PyTorch is used for device
memory (``torch.empty(..., device='cuda')``), ``data_ptr()`` and the current stream.  There is
no CPU fallback: importing works without a GPU (so the symbol table can be checked), but every
compute call needs the built library and a CUDA device and fails loudly otherwise.
"""
from __future__ import annotations
import ctypes as C
import os
from typing import Optional, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libdmrg_b200.so")

DMRG_OK, DMRG_NOT_CONVERGED = 0, 1
DMRG_E_INVALID_ARG, DMRG_E_SECTOR, DMRG_E_ALLOC, DMRG_E_CUDA, DMRG_E_NUMERIC = -1, -2, -3, -4, -5
DMRG_HEISENBERG, DMRG_HUBBARD = 1, 2

EXPORTS = [
    "dmrg_plan_create", "dmrg_plan_destroy", "dmrg_get_layout", "dmrg_get_stats", "dmrg_get_diag",
    "dmrg_last_error", "dmrg_apply_H", "dmrg_davidson_init", "dmrg_davidson_step", "dmrg_davidson_step_host", "dmrg_davidson_poll", "dmrg_get_small",
    "dmrg_set_small", "dmrg_ritz_vector", "dmrg_lowest_eigenpair", "dmrg_gemv_trans", "dmrg_gemv_sub",
    "dmrg_probe_fp64_peak", "dmrg_probe_hbm_read", "dmrg_set_timing", "dmrg_get_timing", "dmrg_get_unit_trace", "dmrg_version",
    "dmrg_apply_H_multi", "dmrg_block_init", "dmrg_block_step", "dmrg_block_ritz", "dmrg_block_get_small",
    "dmrg_block_lowest_eigenpairs",
    "dmrg_plan_create_l11r", "dmrg_partition_outputs", "dmrg_get_shard", "dmrg_davidson_step_given_w",
    "dmrg_density_matrix", "dmrg_sector_eig", "dmrg_select_states", "dmrg_rotate_op", "dmrg_infinite_heisenberg",
    "dmrg_gemv_trans_static",
]


class DmrgError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"dmrg_b200 error {code}: {msg}")
        self.code = code


class _Sectors(C.Structure):
    _fields_ = [("n_labels", C.c_int32), ("n_sectors", C.c_int32),
                ("labels", C.POINTER(C.c_int32)), ("dims", C.POINTER(C.c_int32))]


class _IdmrgOptions(C.Structure):
    _fields_ = [("n_sites", C.c_int32), ("m_keep", C.c_int32), ("J", C.c_double), ("Delta", C.c_double), ("tol", C.c_double),
                ("k_max", C.c_int32), ("max_iter", C.c_int32)]


class _BlockOp(C.Structure):
    _fields_ = [("n_blocks", C.c_int32), ("src", C.POINTER(C.c_int32)), ("dst", C.POINTER(C.c_int32)),
                ("offset", C.POINTER(C.c_int64)), ("ld", C.POINTER(C.c_int32)), ("data", C.c_void_p)]


class _ProblemL11r(C.Structure):
    _fields_ = [("J", C.c_double), ("Delta", C.c_double), ("left", _Sectors), ("right", _Sectors),
                ("H_l", _BlockOp), ("Sz_l", _BlockOp), ("Sp_l", _BlockOp), ("H_r", _BlockOp), ("Sz_r", _BlockOp), ("Sp_r", _BlockOp),
                ("target_twice_sz", C.c_int32)]


_OP_NAMES = ["H_L", "H_R", "Sz_L", "Sp_L", "Sz_R", "Sp_R", "Cup_L", "Cdn_L", "Cup_R", "Cdn_R", "D_L", "D_R"]


class _Problem(C.Structure):
    _fields_ = ([("model", C.c_int32), ("J", C.c_double), ("Delta", C.c_double), ("t", C.c_double),
                 ("U", C.c_double), ("left", _Sectors), ("right", _Sectors)]
                + [(nm, _BlockOp) for nm in _OP_NAMES] + [("target", C.POINTER(C.c_int32))])


class _Options(C.Structure):
    _fields_ = [("k_max", C.c_int32), ("tol", C.c_double), ("max_iter", C.c_int32), ("reorth", C.c_int32),
                ("seed", C.c_uint64), ("tile", C.c_int32), ("check_every", C.c_int32), ("reserve_basis", C.c_int32),
                ("shard_rank", C.c_int32), ("shard_count", C.c_int32), ("max_rhs", C.c_int32)]


class Stats(C.Structure):
    _fields_ = [("n", C.c_int64), ("n_pairs", C.c_int32), ("n_records", C.c_int32), ("n_gemms", C.c_int32),
                ("flop_per_apply", C.c_int64), ("operator_elems", C.c_int64), ("apply_bytes", C.c_int64),
                ("stage1_units", C.c_int32), ("stage2_units", C.c_int32), ("stage2_split_tiles", C.c_int32),
                ("pool_bytes", C.c_int64), ("workspace_bytes", C.c_int64), ("device_bytes", C.c_int64),
                ("kernel_launches_per_apply", C.c_int32), ("kernel_launches_per_step", C.c_int32),
                ("flop_stage1", C.c_int64), ("flop_stage2", C.c_int64), ("launches", C.c_int64)]

    def as_dict(self):
        return {f: getattr(self, f) for f, _ in self._fields_}


_lib = None


def load_library():
    """dlopen the C-ABI library and declare the signatures.  Raises if it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_1309_5571_b200.build` "
                          "(nvcc, sm_100a).  There is no CPU fallback.")
    lib = C.CDLL(LIB_PATH)
    vp, i32, i64, dbl = C.c_void_p, C.c_int32, C.c_int64, C.c_double
    pi32, pi64, pdbl = C.POINTER(i32), C.POINTER(i64), C.POINTER(dbl)
    sig = {
        "dmrg_plan_create": [C.POINTER(_Problem), C.POINTER(_Options), C.POINTER(vp)],
        "dmrg_plan_destroy": [vp],
        "dmrg_get_layout": [vp, pi64, pi32, pi32, pi32, pi64],
        "dmrg_get_stats": [vp, C.POINTER(Stats)],
        "dmrg_get_diag": [vp, vp, vp],
        "dmrg_apply_H": [vp, vp, vp, vp],
        "dmrg_davidson_init": [vp, vp, i32, vp, vp, i64, vp],
        "dmrg_davidson_step": [vp, vp, vp, i64, pi32, pdbl, pdbl, pi32, vp],
        "dmrg_davidson_step_host": [vp, vp, vp, i64, pi32, vp, vp, pdbl, pdbl, pi32, vp],
        "dmrg_davidson_poll": [vp, pdbl, pdbl, pi32, pi32, vp],
        "dmrg_get_small": [vp, pdbl, pdbl, vp],
        "dmrg_set_small": [vp, pdbl, vp],
        "dmrg_ritz_vector": [vp, vp, i64, i32, vp, vp],
        "dmrg_lowest_eigenpair": [vp, vp, i32, vp, pdbl, pdbl, pi32, vp],
        "dmrg_gemv_trans": [vp, vp, i64, i32, vp, vp, vp],
        "dmrg_gemv_trans_static": [vp, i64, i64, i32, vp, vp, vp],
        "dmrg_gemv_sub": [vp, vp, i64, i32, vp, vp, vp, vp],
        "dmrg_probe_fp64_peak": [i32, i32, pdbl, vp],
        "dmrg_probe_hbm_read": [i64, i32, pdbl, vp],
        "dmrg_set_timing": [vp, i32],
        "dmrg_get_timing": [vp, pdbl],
        "dmrg_get_unit_trace": [vp, C.POINTER(C.c_uint64), i32, pi32],
        "dmrg_version": [],
        "dmrg_apply_H_multi": [vp, i32, vp, i64, vp, i64, vp],
        "dmrg_block_init": [vp, i32, vp, i64, vp, vp, i64, vp],
        "dmrg_block_step": [vp, vp, vp, i64, pi32, pi32, i32, pdbl, pdbl, pi32, vp],
        "dmrg_block_ritz": [vp, vp, vp, i64, i32, i32, vp, i64, vp],
        "dmrg_block_get_small": [vp, i32, pdbl, pdbl, vp],
        "dmrg_block_lowest_eigenpairs": [vp, i32, vp, i64, vp, i64, pdbl, pdbl, pi32, pi32, vp],
        "dmrg_plan_create_l11r": [C.POINTER(_ProblemL11r), C.POINTER(_Options), C.POINTER(vp)],
        "dmrg_partition_outputs": [i32, pi64, i32, pi32],
        "dmrg_get_shard": [vp, pi32],
        "dmrg_davidson_step_given_w": [vp, vp, vp, i64, pi32, pdbl, pdbl, pi32, vp],
        "dmrg_density_matrix": [vp, vp, i32, vp, vp],
        "dmrg_sector_eig": [i32, pi32, vp, vp, vp, vp],
        "dmrg_select_states": [i32, pi32, pdbl, i32, pi32, pdbl],
        "dmrg_rotate_op": [i32, pi32, pi32, vp, C.POINTER(_BlockOp), vp, pi64, pi64, vp],
        "dmrg_infinite_heisenberg": [C.POINTER(_IdmrgOptions), i32, pi32, pi32, pdbl, pdbl, pdbl, pi64, pi32, vp],
    }
    for name, args in sig.items():
        fn = getattr(lib, name)
        fn.argtypes = args
        fn.restype = C.c_int
    lib.dmrg_last_error.argtypes = [vp]
    lib.dmrg_last_error.restype = C.c_char_p
    _lib = lib
    return lib


def partition_outputs(cost, n_ranks: int):
    """dmrg_partition_outputs: LPT owner table (host only; works without a GPU)."""
    lib = load_library()
    c = np.ascontiguousarray(np.asarray(cost, dtype=np.int64))
    own = np.zeros(len(c), dtype=np.int32)
    rc = lib.dmrg_partition_outputs(len(c), c.ctypes.data_as(C.POINTER(C.c_int64)), int(n_ranks), own.ctypes.data_as(C.POINTER(C.c_int32)))
    if rc != DMRG_OK:
        raise DmrgError(rc, (lib.dmrg_last_error(None) or b"").decode())
    return own


def sector_eig(dims, rho, stream=None):
    """All eigenpairs of the sector blocks in `rho` (flat CUDA tensor, destroyed): (U flat, w flat), descending per sector."""
    torch = _torch()
    lib = load_library()
    d = np.ascontiguousarray(np.asarray(dims, dtype=np.int32))
    U = torch.empty_like(rho)
    w = torch.empty(max(int(d.sum()), 1), dtype=torch.float64, device=rho.device)
    rc = lib.dmrg_sector_eig(len(d), d.ctypes.data_as(C.POINTER(C.c_int32)), _ptr(rho), _ptr(U), _ptr(w), _stream_ptr(stream))
    if rc != DMRG_OK:
        raise DmrgError(rc, (lib.dmrg_last_error(None) or b"").decode())
    return U, w[:int(d.sum())]


def select_states(dims, w_host, m: int):
    """-> (m_keep per sector, discarded weight)"""
    lib = load_library()
    d = np.ascontiguousarray(np.asarray(dims, dtype=np.int32)); w = np.ascontiguousarray(np.asarray(w_host, dtype=np.float64))
    mk = np.zeros(len(d), dtype=np.int32); disc = C.c_double()
    rc = lib.dmrg_select_states(len(d), d.ctypes.data_as(C.POINTER(C.c_int32)), w.ctypes.data_as(C.POINTER(C.c_double)), int(m),
                                mk.ctypes.data_as(C.POINTER(C.c_int32)), C.byref(disc))
    if rc != DMRG_OK:
        raise DmrgError(rc, (lib.dmrg_last_error(None) or b"").decode())
    return mk, float(disc.value)


def infinite_heisenberg(n_sites: int, m_keep: int, J: float = 1.0, Delta: float = 1.0, tol: float = 1e-10, k_max: int = 20,
                        max_iter: int = 4000, stream=None):
    """dmrg_infinite_heisenberg: list of dicts(n_sites, energy, discarded, n, davidson_iters), one per DMRG iteration."""
    _torch()
    lib = load_library()
    cap = n_sites // 2
    o = _IdmrgOptions(int(n_sites), int(m_keep), float(J), float(Delta), float(tol), int(k_max), int(max_iter))
    nr = C.c_int32(); ns = (C.c_int32 * cap)(); e = (C.c_double * cap)(); dl = (C.c_double * cap)(); dr = (C.c_double * cap)()
    td = (C.c_int64 * cap)(); it = (C.c_int32 * cap)()
    rc = lib.dmrg_infinite_heisenberg(C.byref(o), cap, C.byref(nr), ns, e, dl, dr, td, it, _stream_ptr(stream))
    if rc != DMRG_OK:
        raise DmrgError(rc, (lib.dmrg_last_error(None) or b"").decode())
    return [dict(n_sites=int(ns[q]), energy=float(e[q]), discarded=(float(dl[q]), float(dr[q])), n=int(td[q]), davidson_iters=int(it[q]))
            for q in range(nr.value)]


def gemv_trans_static(V, k: int, w, out, n: Optional[int] = None, stream=None):
    """dmrg_gemv_trans_static: out[0..k) = V(:,0..k)^T w without a plan and without any allocation (scratch in a file-scope device
    array; k <= 32; calls that overlap on the GPU race).  V: (>= k, ldv) or flat float64 CUDA tensor, rows = basis vectors; w: n
    doubles; out: k doubles, caller-allocated (this wrapper allocates nothing either)."""
    torch = _torch()
    lib = load_library()
    n = int(w.numel() if n is None else n)
    for t, name in ((V, "V"), (w, "w"), (out, "out")):
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64):
            raise TypeError(f"{name}: need a float64 CUDA tensor")
    if V.dim() == 2 and V.stride(1) != 1 or not w.is_contiguous() or not out.is_contiguous():
        raise TypeError("gemv_trans_static: rows of V, w and out must be contiguous")
    ldv = V.stride(0) if V.dim() == 2 else n
    rows = V.shape[0] if V.dim() == 2 else V.numel() // max(n, 1)
    if 1 <= k <= 32 and (rows < k or out.numel() < k or w.numel() < n or (V.dim() == 2 and V.shape[1] < n)):
        raise ValueError("gemv_trans_static: V, w or out smaller than (k, n) asks for")
    rc = lib.dmrg_gemv_trans_static(C.c_void_p(_ptr(V)), C.c_int64(int(ldv)), C.c_int64(n), C.c_int32(int(k)), C.c_void_p(_ptr(w)),
                                    C.c_void_p(_ptr(out)), C.c_void_p(_stream_ptr(stream)))
    if rc != DMRG_OK:
        raise DmrgError(rc, (lib.dmrg_last_error(None) or b"").decode())
    return out


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("paper_1309_5571_b200 needs a CUDA device (B200, sm_100a); there is no CPU fallback")
    return torch


def _stream_ptr(stream=None) -> int:
    torch = _torch()
    s = stream if stream is not None else torch.cuda.current_stream()
    return int(s.cuda_stream)


def _ptr(t) -> int:
    return 0 if t is None else int(t.data_ptr())


def _check_vec(t, n: int, name: str):
    torch = _torch()
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
        raise TypeError(f"{name}: need a contiguous float64 CUDA tensor")
    if t.numel() < n:
        raise ValueError(f"{name}: needs at least {n} elements")


class Plan:
    """Owns a dmrg_handle_t plus the device copies of the operator blocks."""

    def __init__(self, problem, k_max: int = 20, tol: float = 1e-10, max_iter: int = 2000, reorth: int = 1,
                 seed: int = 1, check_every: int = 8, max_rhs: int = 1, reserve_basis: bool = False, shard_rank: int = 0, shard_count: int = 0,
                 device: Optional[str] = None):
        torch = _torch()
        self._lib = load_library()
        self._keep = []
        self.device = torch.device(device or "cuda:0")
        torch.cuda.set_device(self.device)
        pr = _Problem()
        model = problem.model
        pr.model = {"heisenberg": DMRG_HEISENBERG, "hubbard": DMRG_HUBBARD}.get(model, model)
        pr.J, pr.Delta, pr.t, pr.U = float(problem.J), float(problem.Delta), float(problem.t), float(problem.U)
        pr.left = self._sectors(problem.left)
        pr.right = self._sectors(problem.right)
        for nm in _OP_NAMES:
            setattr(pr, nm, self._block_op(problem.ops.get(nm)))
        tgt = np.ascontiguousarray(np.asarray(problem.target, dtype=np.int32).ravel())
        self._keep.append(tgt)
        pr.target = tgt.ctypes.data_as(C.POINTER(C.c_int32))
        opt = _Options(int(k_max), float(tol), int(max_iter), int(reorth), int(seed), 0, int(check_every), int(bool(reserve_basis)), int(shard_rank), int(shard_count), int(max_rhs))
        h = C.c_void_p()
        rc = self._lib.dmrg_plan_create(C.byref(pr), C.byref(opt), C.byref(h))
        self._finish(rc, h, k_max)

    @classmethod
    def from_l11r(cls, left_block, right_block, J: float, Delta: float, target_twice_sz: int = 0, k_max: int = 20, tol: float = 1e-10,
                  max_iter: int = 2000, reorth: int = 1, max_rhs: int = 1, device: Optional[str] = None):
        """Plan of the l-1-1-r strategy (dmrg_plan_create_l11r).  Blocks: objects with .sectors (labels = 2 S_z, dims) and the
        sector-blocked operators .H, .Sz, .Sp of the UN-enlarged block (dmrg_inputs containers)."""
        torch = _torch()
        self = cls.__new__(cls)
        self._lib = load_library(); self._keep = []
        self.device = torch.device(device or "cuda:0")
        torch.cuda.set_device(self.device)
        pr = _ProblemL11r()
        pr.J, pr.Delta, pr.target_twice_sz = float(J), float(Delta), int(target_twice_sz)
        pr.left, pr.right = self._sectors(left_block.sectors), self._sectors(right_block.sectors)
        pr.H_l, pr.Sz_l, pr.Sp_l = self._block_op(left_block.H), self._block_op(left_block.Sz), self._block_op(left_block.Sp)
        pr.H_r, pr.Sz_r, pr.Sp_r = self._block_op(right_block.H), self._block_op(right_block.Sz), self._block_op(right_block.Sp)
        opt = _Options(int(k_max), float(tol), int(max_iter), int(reorth), 1, 0, 8, 0, 0, 0, int(max_rhs))
        h = C.c_void_p()
        rc = self._lib.dmrg_plan_create_l11r(C.byref(pr), C.byref(opt), C.byref(h))
        self._finish(rc, h, k_max)
        return self

    def _finish(self, rc, h, k_max):
        if rc != DMRG_OK:
            raise DmrgError(rc, (self._lib.dmrg_last_error(None) or b"").decode())
        self._h = h
        self.k_max = int(k_max)
        n, npairs = C.c_int64(), C.c_int32()
        self._lib.dmrg_get_layout(self._h, C.byref(n), C.byref(npairs), None, None, None)
        self.n, self.n_pairs = int(n.value), int(npairs.value)
        ls = np.zeros(self.n_pairs, np.int32); rs = np.zeros(self.n_pairs, np.int32); off = np.zeros(self.n_pairs, np.int64)
        self._lib.dmrg_get_layout(self._h, None, None, ls.ctypes.data_as(C.POINTER(C.c_int32)),
                                  rs.ctypes.data_as(C.POINTER(C.c_int32)), off.ctypes.data_as(C.POINTER(C.c_int64)))
        self.left_sector, self.right_sector, self.seg_offset = ls, rs, off

    # ---- marshalling helpers
    def _sectors(self, s) -> _Sectors:
        labels = np.ascontiguousarray(np.asarray(s.labels, dtype=np.int32).reshape(len(s.dims), -1))
        dims = np.ascontiguousarray(np.asarray(s.dims, dtype=np.int32))
        self._keep += [labels, dims]
        return _Sectors(labels.shape[1], dims.shape[0], labels.ctypes.data_as(C.POINTER(C.c_int32)),
                        dims.ctypes.data_as(C.POINTER(C.c_int32)))

    def _block_op(self, op) -> _BlockOp:
        torch = _torch()
        if op is None or len(op.blocks) == 0:
            return _BlockOp(0, None, None, None, None, None)
        src = np.ascontiguousarray(np.asarray(op.src, dtype=np.int32))
        dst = np.ascontiguousarray(np.asarray(op.dst, dtype=np.int32))
        sizes = np.array([b.size for b in op.blocks], dtype=np.int64)
        offset = np.ascontiguousarray(np.concatenate([[0], np.cumsum(sizes)[:-1]]).astype(np.int64))
        ld = np.ascontiguousarray(np.array([b.shape[1] for b in op.blocks], dtype=np.int32))
        flat = np.concatenate([np.ascontiguousarray(b, dtype=np.float64).ravel() for b in op.blocks]) \
            if sizes.sum() > 0 else np.zeros(1)
        data = torch.from_numpy(flat).to(self.device)
        self._keep += [src, dst, offset, ld, data]
        ip = C.POINTER(C.c_int32)
        return _BlockOp(len(op.blocks), src.ctypes.data_as(ip), dst.ctypes.data_as(ip),
                        offset.ctypes.data_as(C.POINTER(C.c_int64)), ld.ctypes.data_as(ip), C.c_void_p(data.data_ptr()))

    def _check(self, rc: int):
        if rc < 0:
            raise DmrgError(rc, (self._lib.dmrg_last_error(self._h) or b"").decode())
        return rc

    # ---- plan queries
    def stats(self) -> dict:
        s = Stats()
        self._check(self._lib.dmrg_get_stats(self._h, C.byref(s)))
        return s.as_dict()

    def diag(self):
        torch = _torch()
        d = torch.empty(self.n, dtype=torch.float64, device=self.device)
        self._check(self._lib.dmrg_get_diag(self._h, _ptr(d), _stream_ptr()))
        return d

    def new_basis(self, ldv: Optional[int] = None):
        """Allocates V, W as (k_max, ldv) row-major tensors = column-contiguous n x k_max."""
        torch = _torch()
        ldv = int(ldv) if ldv is not None else (self.n + 15) // 16 * 16
        V = torch.zeros((self.k_max, ldv), dtype=torch.float64, device=self.device)
        W = torch.zeros((self.k_max, ldv), dtype=torch.float64, device=self.device)
        return V, W

    # ---- hot path (same names as the C entry points, without the prefix)
    def apply_H(self, x, y=None, stream=None):
        torch = _torch()
        _check_vec(x, self.n, "x")
        if y is None:
            y = torch.empty(self.n, dtype=torch.float64, device=self.device)
        _check_vec(y, self.n, "y")
        self._check(self._lib.dmrg_apply_H(self._h, _ptr(x), _ptr(y), _stream_ptr(stream)))
        return y

    # ---- several vectors at once (block Davidson).  Blocks of vectors are (nb, ld) row-major tensors =
    #      column-contiguous n x nb, like V and W.
    def _check_block(self, X, nb: int, name: str) -> int:
        if X.dim() != 2 or X.shape[0] < nb or X.stride(1) != 1 or X.stride(0) < self.n or not X.is_cuda or X.dtype != _torch().float64:
            raise ValueError(f"{name}: need a float64 CUDA tensor of shape (>= {nb}, ld >= n) with contiguous rows")
        return int(X.stride(0))

    def apply_H_multi(self, X, Y=None, stream=None):
        torch = _torch()
        nb = X.shape[0]
        ldx = self._check_block(X, nb, "X")
        if Y is None:
            Y = torch.empty((nb, (self.n + 15) // 16 * 16), dtype=torch.float64, device=self.device)
        ldy = self._check_block(Y, nb, "Y")
        self._check(self._lib.dmrg_apply_H_multi(self._h, int(nb), _ptr(X), ldx, _ptr(Y), ldy, _stream_ptr(stream)))
        return Y

    def block_init(self, V, W, X0, stream=None):
        nb = X0.shape[0]
        ldx = self._check_block(X0, nb, "X0")
        self._check_basis(V, W)
        self._check(self._lib.dmrg_block_init(self._h, int(nb), _ptr(X0), ldx, _ptr(V), _ptr(W), int(V.stride(0)), _stream_ptr(stream)))
        return nb, nb

    def block_step(self, V, W, k: int, na: int, nb: int, stream=None):
        """-> (k, na, theta[nb], resnorm[nb], converged)"""
        self._check_basis(V, W)
        kk, nn, conv = C.c_int32(int(k)), C.c_int32(int(na)), C.c_int32()
        th = (C.c_double * nb)(); rho = (C.c_double * nb)()
        self._check(self._lib.dmrg_block_step(self._h, _ptr(V), _ptr(W), int(V.stride(0)), C.byref(kk), C.byref(nn), int(nb),
                                              th, rho, C.byref(conv), _stream_ptr(stream)))
        return int(kk.value), int(nn.value), np.array(th[:]), np.array(rho[:]), bool(conv.value)

    def block_ritz(self, V, W, k: int, nb: int, stream=None):
        torch = _torch()
        X = torch.empty((nb, (self.n + 15) // 16 * 16), dtype=torch.float64, device=self.device)
        self._check(self._lib.dmrg_block_ritz(self._h, _ptr(V), _ptr(W), int(V.stride(0)), int(k), int(nb), _ptr(X), int(X.stride(0)),
                                              _stream_ptr(stream)))
        return X[:, :self.n]

    def block_get_small(self, nb: int, stream=None):
        G = np.zeros((self.k_max, self.k_max)); Y = np.zeros((self.k_max, nb))
        self._check(self._lib.dmrg_block_get_small(self._h, int(nb), G.ctypes.data_as(C.POINTER(C.c_double)),
                                                   Y.ctypes.data_as(C.POINTER(C.c_double)), _stream_ptr(stream)))
        return G, Y

    def block_lowest_eigenpairs(self, X0, stream=None):
        """-> (rc, theta[nb], X (nb, n), resnorm[nb], block iterations, applies)"""
        torch = _torch()
        nb = X0.shape[0]
        ldx = self._check_block(X0, nb, "X0")
        X = torch.empty((nb, (self.n + 15) // 16 * 16), dtype=torch.float64, device=self.device)
        th = (C.c_double * nb)(); rho = (C.c_double * nb)(); it = C.c_int32(); ap = C.c_int32()
        rc = self._lib.dmrg_block_lowest_eigenpairs(self._h, int(nb), _ptr(X0), ldx, _ptr(X), int(X.stride(0)), th, rho,
                                                    C.byref(it), C.byref(ap), _stream_ptr(stream))
        if rc < 0:
            self._check(rc)
        return rc, np.array(th[:]), X[:, :self.n], np.array(rho[:]), int(it.value), int(ap.value)

    # ---- the steps either side of the path (Alg. 1 lines 5-7)
    def density_matrix(self, x, side: int, dims, stream=None):
        """rho of side 0 (left) / 1 (right): flat CUDA tensor, sector s at offset sum_{t<s} d_t^2, row-major d_s x d_s."""
        torch = _torch()
        _check_vec(x, self.n, "x")
        tot = int(sum(int(d) * int(d) for d in dims))
        rho = torch.empty(max(tot, 1), dtype=torch.float64, device=self.device)
        self._check(self._lib.dmrg_density_matrix(self._h, _ptr(x), int(side), _ptr(rho), _stream_ptr(stream)))
        return rho[:tot]

    def rotate_op(self, op, dims, m_keep, U, stream=None):
        """-> (out_data CUDA tensor, out_offset np.int64 [n_blocks]) for a dmrg_inputs BlockOp."""
        torch = _torch()
        bo = self._block_op(op)
        d = np.ascontiguousarray(np.asarray(dims, dtype=np.int32)); mk = np.ascontiguousarray(np.asarray(m_keep, dtype=np.int32))
        off = np.zeros(max(len(op.blocks), 1), dtype=np.int64); ne = C.c_int64()
        args = (len(d), d.ctypes.data_as(C.POINTER(C.c_int32)), mk.ctypes.data_as(C.POINTER(C.c_int32)), _ptr(U), C.byref(bo))
        self._check(self._lib.dmrg_rotate_op(*args, None, off.ctypes.data_as(C.POINTER(C.c_int64)), C.byref(ne), _stream_ptr(stream)))
        out = torch.empty(max(int(ne.value), 1), dtype=torch.float64, device=self.device)
        self._check(self._lib.dmrg_rotate_op(*args, _ptr(out), off.ctypes.data_as(C.POINTER(C.c_int64)), C.byref(ne), _stream_ptr(stream)))
        return out[:int(ne.value)], off[:len(op.blocks)]

    def _check_basis(self, V, W):
        """a wrong-shaped basis must not reach the kernels (they would write out of bounds)."""
        t = _torch()
        for nm, B in (("V", V), ("W", W)):
            if not (isinstance(B, t.Tensor) and B.is_cuda and B.dtype == t.float64 and B.dim() == 2 and B.shape[0] >= self.k_max
                    and B.stride(1) == 1 and B.stride(0) >= self.n):
                raise ValueError(f"{nm}: need a float64 CUDA tensor of shape (>= k_max, ld >= n) with contiguous rows "
                                 f"(column-contiguous n x k_max), got {tuple(B.shape) if hasattr(B, 'shape') else type(B)}")
        if V.stride(0) != W.stride(0):
            raise ValueError("V and W must have the same column stride")

    def _check_cols(self, V, k: int):
        t = _torch()
        if not (isinstance(V, t.Tensor) and V.is_cuda and V.dtype == t.float64 and V.dim() == 2 and V.shape[0] >= k
                and V.stride(1) == 1 and V.stride(0) >= self.n):
            raise ValueError(f"V: need a float64 CUDA tensor of shape (>= {k}, ld >= n) with contiguous rows")

    def davidson_init(self, V, W, x0=None, start_at_argmin_diag: bool = False, stream=None):
        self._check_basis(V, W)
        if x0 is not None:
            _check_vec(x0, self.n, "x0")
        ldv = V.stride(0) if V.dim() == 2 else self.n
        self._check(self._lib.dmrg_davidson_init(self._h, _ptr(x0), int(bool(start_at_argmin_diag)), _ptr(V), _ptr(W),
                                                 int(ldv), _stream_ptr(stream)))

    def davidson_enqueue(self, V, W, k: int, stream=None) -> int:
        """dmrg_davidson_step with NULL outputs: enqueue only, returns the next basis size; see davidson_poll."""
        self._check_basis(V, W)
        kk = C.c_int32(int(k))
        ldv = V.stride(0) if V.dim() == 2 else self.n
        self._check(self._lib.dmrg_davidson_step(self._h, _ptr(V), _ptr(W), int(ldv), C.byref(kk), None, None, None,
                                                 _stream_ptr(stream)))
        return int(kk.value)

    def davidson_step_given_w(self, V, W, k: int, stream=None) -> Tuple[int, float, float, bool]:
        """Lines 3-14 of Alg. 3 with W(:,k-1) already formed by the caller (output-sharded projection + all-reduce)."""
        self._check_basis(V, W)
        kk = C.c_int32(int(k)); lam = C.c_double(); rho = C.c_double(); conv = C.c_int32()
        self._check(self._lib.dmrg_davidson_step_given_w(self._h, _ptr(V), _ptr(W), int(V.stride(0)), C.byref(kk), C.byref(lam),
                                                         C.byref(rho), C.byref(conv), _stream_ptr(stream)))
        return int(kk.value), float(lam.value), float(rho.value), bool(conv.value)

    def shard_owner(self):
        own = np.zeros(self.n_pairs, dtype=np.int32)
        self._check(self._lib.dmrg_get_shard(self._h, own.ctypes.data_as(C.POINTER(C.c_int32))))
        return own

    def davidson_poll(self, stream=None) -> Tuple[float, float, bool, int]:
        """(lambda, rho, converged, executed iterations) after a stream synchronisation."""
        lam, rho, conv, it = C.c_double(), C.c_double(), C.c_int32(), C.c_int32()
        self._check(self._lib.dmrg_davidson_poll(self._h, C.byref(lam), C.byref(rho), C.byref(conv), C.byref(it),
                                                 _stream_ptr(stream)))
        return float(lam.value), float(rho.value), bool(conv.value), int(it.value)

    def davidson_step_host(self, V, W, k: int, v_in_host=None, w_out_host=None, stream=None) -> Tuple[int, float, float, bool]:
        """dmrg_davidson_step_host: v_in_host / w_out_host are CPU float64 tensors of n elements (pinned for overlap)."""
        self._check_basis(V, W)
        for nm, t in (("v_in_host", v_in_host), ("w_out_host", w_out_host)):
            if t is not None and (t.is_cuda or t.dtype != _torch().float64 or t.numel() != self.n or not t.is_contiguous()):
                raise ValueError(f"{nm} must be a contiguous CPU float64 tensor of {self.n} elements")
        kk, lam, rho, conv = C.c_int32(int(k)), C.c_double(), C.c_double(), C.c_int32()
        ldv = V.stride(0) if V.dim() == 2 else self.n
        self._check(self._lib.dmrg_davidson_step_host(
            self._h, _ptr(V), _ptr(W), int(ldv), C.byref(kk), _ptr(v_in_host), _ptr(w_out_host),
            C.byref(lam), C.byref(rho), C.byref(conv), _stream_ptr(stream)))
        return int(kk.value), float(lam.value), float(rho.value), bool(conv.value)

    def davidson_step(self, V, W, k: int, stream=None) -> Tuple[int, float, float, bool]:
        self._check_basis(V, W)
        kk, lam, rho, conv = C.c_int32(int(k)), C.c_double(), C.c_double(), C.c_int32()
        ldv = V.stride(0) if V.dim() == 2 else self.n
        self._check(self._lib.dmrg_davidson_step(self._h, _ptr(V), _ptr(W), int(ldv), C.byref(kk), C.byref(lam),
                                                 C.byref(rho), C.byref(conv), _stream_ptr(stream)))
        return int(kk.value), float(lam.value), float(rho.value), bool(conv.value)

    def get_small(self):
        B = np.zeros((self.k_max, self.k_max)); y = np.zeros(self.k_max)
        pd = C.POINTER(C.c_double)
        self._check(self._lib.dmrg_get_small(self._h, B.ctypes.data_as(pd), y.ctypes.data_as(pd), _stream_ptr()))
        return B, y

    def set_small(self, B):
        B = np.ascontiguousarray(B, dtype=np.float64)
        assert B.shape == (self.k_max, self.k_max)
        self._check(self._lib.dmrg_set_small(self._h, B.ctypes.data_as(C.POINTER(C.c_double)), _stream_ptr()))

    def ritz_vector(self, V, k: int, stream=None):
        self._check_cols(V, k)
        torch = _torch()
        x = torch.empty(self.n, dtype=torch.float64, device=self.device)
        ldv = V.stride(0) if V.dim() == 2 else self.n
        self._check(self._lib.dmrg_ritz_vector(self._h, _ptr(V), int(ldv), int(k), _ptr(x), _stream_ptr(stream)))
        return x

    def lowest_eigenpair(self, x0=None, start_at_argmin_diag: bool = False, x_out=None, stream=None):
        """Returns (rc, lambda, x, resnorm, iters); rc is DMRG_OK or DMRG_NOT_CONVERGED."""
        torch = _torch()
        if x0 is not None:
            _check_vec(x0, self.n, "x0")
        if x_out is None:
            x_out = torch.empty(self.n, dtype=torch.float64, device=self.device)
        lam, rho, it = C.c_double(), C.c_double(), C.c_int32()
        rc = self._check(self._lib.dmrg_lowest_eigenpair(self._h, _ptr(x0), int(bool(start_at_argmin_diag)), _ptr(x_out),
                                                         C.byref(lam), C.byref(rho), C.byref(it), _stream_ptr(stream)))
        return rc, float(lam.value), x_out, float(rho.value), int(it.value)

    def gemv_trans(self, V, k: int, w, out=None, stream=None):
        self._check_cols(V, k)
        torch = _torch()
        if out is None:
            out = torch.empty(k, dtype=torch.float64, device=self.device)
        ldv = V.stride(0) if V.dim() == 2 else self.n
        self._check(self._lib.dmrg_gemv_trans(self._h, _ptr(V), int(ldv), int(k), _ptr(w), _ptr(out), _stream_ptr(stream)))
        return out

    def gemv_sub(self, V, k: int, s, t, nrm2=None, stream=None):
        self._check_cols(V, k)
        torch = _torch()
        if nrm2 is None:
            nrm2 = torch.empty(1, dtype=torch.float64, device=self.device)
        ldv = V.stride(0) if V.dim() == 2 else self.n
        self._check(self._lib.dmrg_gemv_sub(self._h, _ptr(V), int(ldv), int(k), _ptr(s), _ptr(t), _ptr(nrm2), _stream_ptr(stream)))
        return nrm2

    # ---- host-buffer entry (end-to-end measurement: H2D of x, apply, D2H of y)
    def apply_H_host(self, x_host, y_host, x_dev=None, y_dev=None, stream=None):
        """x_host, y_host: pinned CPU float64 tensors of n elements.  Copies x to the device, applies H
        through the C ABI and copies y back on the same stream; synchronises before returning."""
        torch = _torch()
        if x_dev is None:
            x_dev = torch.empty(self.n, dtype=torch.float64, device=self.device)
        if y_dev is None:
            y_dev = torch.empty(self.n, dtype=torch.float64, device=self.device)
        x_dev.copy_(x_host, non_blocking=True)
        self.apply_H(x_dev, y_dev, stream)
        y_host.copy_(y_dev, non_blocking=True)
        (stream or torch.cuda.current_stream()).synchronize()
        return y_host

    def set_timing(self, enable: bool):
        self._check(self._lib.dmrg_set_timing(self._h, int(bool(enable))))

    def get_timing(self):
        ms = np.zeros(8)
        self._check(self._lib.dmrg_get_timing(self._h, ms.ctypes.data_as(C.POINTER(C.c_double))))
        return ms

    def unit_trace(self):
        """Diagnostics (plan created with DMRG_TRACE set): (rows, 4) uint64 array of the last apply: one row per work
        unit in ticket order, then one row of phase stamps per CTA slot (include/dmrg_b200.h)."""
        st = self.stats()
        cap = st["stage1_units"] + st["stage2_units"] + 8 * 256
        buf = np.zeros((max(cap, 1), 4), dtype=np.uint64)
        nu = C.c_int32()
        self._check(self._lib.dmrg_get_unit_trace(self._h, buf.ctypes.data_as(C.POINTER(C.c_uint64)), cap, C.byref(nu)))
        return buf[: nu.value]

    def close(self):
        if getattr(self, "_h", None):
            self._lib.dmrg_plan_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


# ---- module-level functions with the names of the C entry points ---------------------------
def dmrg_plan_create(problem, **opts) -> Plan:
    return Plan(problem, **opts)


def dmrg_apply_H(plan: Plan, x, y=None, stream=None):
    return plan.apply_H(x, y, stream)


def dmrg_davidson_step(plan: Plan, V, W, k: int, stream=None):
    return plan.davidson_step(V, W, k, stream)


def dmrg_lowest_eigenpair(plan: Plan, x0=None, start_at_argmin_diag: bool = False, x_out=None, stream=None):
    return plan.lowest_eigenpair(x0, start_at_argmin_diag, x_out, stream)


def dmrg_probe_fp64_peak(kind: int = 1, reps: int = 3) -> float:
    lib = load_library(); _torch()
    v = C.c_double()
    rc = lib.dmrg_probe_fp64_peak(int(kind), int(reps), C.byref(v), _stream_ptr())
    if rc != DMRG_OK:
        raise DmrgError(rc, (lib.dmrg_last_error(None) or b"").decode())
    return float(v.value)


def dmrg_probe_hbm_read(nbytes: int = 1 << 31, reps: int = 3) -> float:
    lib = load_library(); _torch()
    v = C.c_double()
    rc = lib.dmrg_probe_hbm_read(int(nbytes), int(reps), C.byref(v), _stream_ptr())
    if rc != DMRG_OK:
        raise DmrgError(rc, (lib.dmrg_last_error(None) or b"").decode())
    return float(v.value)
