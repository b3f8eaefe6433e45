"""ctypes binding of libnolsm.so.  Names follow include/nolsm.h one to one:
Context.build_neighbours / build_submatrices / sign_batched / scatter_density / solve_mu /
sign_dense_batched.  torch is used for device memory and streams only."""
import ctypes as C
import os

HERE = os.path.dirname(os.path.abspath(__file__))
FP16_FP32, FP32 = 0, 1
MAT_S, MAT_H, MAT_SINV, MAT_B, MAT_X = 0, 1, 2, 3, 4
FLAG_SIMT_ONLY = 1
FLAG_PAIR = 2
FLAG_SINGLE = 8
FLAG_UNIT_SCALE = 16
FLAG_ORDER3 = 32
FLAG_NO_PREDICT = 64
FLAG_LOWDIN = 128
FLAG_NO_RESCALE = 256
STATUS = {0: "NOLSM_OK", 1: "NOLSM_EINVAL", 2: "NOLSM_ENOMEM", 3: "NOLSM_ECUDA", 4: "NOLSM_ENOTSPD",
          5: "NOLSM_ENOCONV", 6: "NOLSM_EBRACKET"}

EXPORTED_SYMBOLS = [
    "nolsm_create", "nolsm_destroy", "nolsm_last_error", "nolsm_version", "nolsm_build_neighbours",
    "nolsm_build_submatrices", "nolsm_batch_capacity", "nolsm_release_batch", "nolsm_sign_batched",
    "nolsm_scatter_density", "nolsm_solve_mu", "nolsm_solve_mu_host", "nolsm_sign_dense_batched", "nolsm_batch_read",
    "nolsm_batch_size", "nolsm_batch_ld", "nolsm_gemm_batched", "nolsm_launch_count",
    "nolsm_scatter_energy", "nolsm_evaluate", "nolsm_set_model", "nolsm_combine_submatrices",
    "nolsm_build_submatrices_grouped", "nolsm_union_pattern", "nolsm_expand_store",
    "nolsm_static_setup", "nolsm_build_neighbours_static",
]


class NolsmError(RuntimeError):
    def __init__(self, status, message):
        super().__init__(f"{STATUS.get(status, status)}: {message}")
        self.status = status


class Config(C.Structure):
    _fields_ = [("precision", C.c_int32), ("tol", C.c_float), ("max_iter", C.c_int32), ("fixed_iter", C.c_int32),
                ("inv_tol", C.c_float), ("inv_max_iter", C.c_int32), ("inv_refine", C.c_int32),
                ("workspace_bytes", C.c_int64), ("group", C.c_int32), ("flags", C.c_int32),
                ("gap_hint", C.c_float), ("cache_bytes", C.c_int64)]

    def __init__(self, precision=FP16_FP32, tol=0.0, max_iter=0, fixed_iter=0, inv_tol=0.0, inv_max_iter=0,
                 inv_refine=-1, workspace_bytes=0, group=0, flags=0, cache_bytes=0, gap_hint=0.0):
        super().__init__(precision, tol, max_iter, fixed_iter, inv_tol, inv_max_iter, inv_refine,
                         workspace_bytes, group, flags, gap_hint, cache_bytes)


class _Bsr(C.Structure):
    _fields_ = [("n_mol", C.c_int32), ("bs", C.c_int32), ("row_ptr", C.c_void_p), ("col_idx", C.c_void_p),
                ("val", C.c_void_p)]


class _Model(C.Structure):
    _fields_ = [("pos_q", C.c_void_p), ("n_mol", C.c_int32), ("box_q", C.c_int32 * 3), ("rc_q", C.c_int32),
                ("unit_per_grid", C.c_double), ("site_offset", (C.c_double * 3) * 3), ("orb_site", C.c_int32 * 6),
                ("orb_energy", C.c_double * 6), ("s_ampl", C.c_double), ("h_ampl", C.c_double),
                ("h_len", C.c_double), ("eval_fp32", C.c_int32)]


class _Groups(C.Structure):
    _fields_ = [("n_groups", C.c_int32), ("own_ptr", C.c_void_p), ("own_idx", C.c_void_p), ("list_ptr", C.c_void_p),
                ("list_idx", C.c_void_p)]


class SignStats(C.Structure):
    _fields_ = [("n_sub", C.c_int32), ("iter_min", C.c_int32), ("iter_max", C.c_int32), ("iter_sum", C.c_int64),
                ("n_unconverged", C.c_int32), ("worst_residual", C.c_float), ("gemms", C.c_int64),
                ("flops_sign", C.c_double), ("flops_sign_padded", C.c_double), ("flops_prepare", C.c_double),
                ("inv_iter_max", C.c_int32), ("inv_worst_residual", C.c_float), ("ms_chain", C.c_float),
                ("chain_mcycles", C.c_float)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


class SolveStats(C.Structure):
    _fields_ = [("mu_steps", C.c_int32), ("n_batches", C.c_int32), ("resident", C.c_int32), ("cached", C.c_int32),
                ("mu_lo", C.c_double), ("mu_hi", C.c_double), ("ne_diag", C.c_double), ("last", SignStats),
                ("flops_sign_total", C.c_double), ("flops_prepare_total", C.c_double),
                ("ms_gather", C.c_float), ("ms_prepare", C.c_float), ("ms_sign", C.c_float),
                ("ms_density", C.c_float), ("ms_chain", C.c_float), ("chain_launches", C.c_int32)]

    def as_dict(self):
        d = {k: getattr(self, k) for k, _ in self._fields_ if k != "last"}
        d["last"] = self.last.as_dict()
        return d


def library_path():
    return os.path.join(HERE, "libnolsm.so")


_LIB = None


def load_library():
    """dlopen libnolsm.so (built by paper_2104_08245_b200.build).  Raises if it is missing: there is
    no other implementation to fall back to."""
    global _LIB
    if _LIB is not None:
        return _LIB
    path = library_path()
    if not os.path.exists(path):
        raise NolsmError(3, f"{path} not built; run `python -m paper_2104_08245_b200.build`")
    lib = C.CDLL(path)
    vp, i32, i64, f32, f64 = C.c_void_p, C.c_int32, C.c_int64, C.c_float, C.c_double
    P = C.POINTER
    lib.nolsm_create.argtypes = [P(vp), P(Config)]
    lib.nolsm_create.restype = i32
    lib.nolsm_destroy.argtypes = [vp]
    lib.nolsm_destroy.restype = None
    lib.nolsm_last_error.argtypes = [vp]
    lib.nolsm_last_error.restype = C.c_char_p
    lib.nolsm_version.restype = i32
    lib.nolsm_launch_count.argtypes = [vp]
    lib.nolsm_launch_count.restype = i64
    lib.nolsm_build_neighbours.argtypes = [vp, i32, vp, P(i32), i32, vp, vp, i64, P(i64), vp]
    lib.nolsm_build_neighbours.restype = i32
    lib.nolsm_build_neighbours_static.argtypes = [vp, i32, vp, P(i32), i32, vp, vp, i64, P(i64), vp]
    lib.nolsm_build_neighbours_static.restype = i32
    lib.nolsm_static_setup.argtypes = []
    lib.nolsm_static_setup.restype = i32
    lib.nolsm_set_model.argtypes = [vp, P(_Model)]
    lib.nolsm_set_model.restype = i32
    lib.nolsm_build_submatrices.argtypes = [vp, P(_Bsr), P(_Bsr), i32, i32, i32, P(vp), vp]
    lib.nolsm_build_submatrices.restype = i32
    lib.nolsm_batch_capacity.argtypes = [vp, P(_Bsr), i32, i32, vp]
    lib.nolsm_batch_capacity.restype = i32
    lib.nolsm_release_batch.argtypes = [vp, vp]
    lib.nolsm_release_batch.restype = None
    lib.nolsm_sign_batched.argtypes = [vp, vp, f64, i32, f32, i32, i32, P(SignStats), vp]
    lib.nolsm_sign_batched.restype = i32
    lib.nolsm_scatter_energy.argtypes = [vp, vp, P(_Bsr), P(_Bsr), P(_Bsr), vp, vp]
    lib.nolsm_scatter_energy.restype = i32
    lib.nolsm_evaluate.argtypes = [vp, P(_Bsr), P(_Bsr), f64, i32, P(_Bsr), P(_Bsr), P(f64), P(f64), vp,
                                   P(SolveStats), vp]
    lib.nolsm_evaluate.restype = i32
    lib.nolsm_scatter_density.argtypes = [vp, vp, P(_Bsr), P(_Bsr), vp, vp, vp, vp]
    lib.nolsm_scatter_density.restype = i32
    lib.nolsm_solve_mu.argtypes = [vp, P(_Bsr), P(_Bsr), f64, f64, f64, f64, i32, i32, P(_Bsr), P(f64), P(f64),
                                   vp, P(SolveStats), vp]
    lib.nolsm_solve_mu.restype = i32
    lib.nolsm_solve_mu_host.argtypes = [vp, i32, vp, vp, vp, vp, f64, f64, f64, f64, i32, i32, vp, P(f64), P(f64),
                                        P(SolveStats), P(i64), P(i64), vp]
    lib.nolsm_solve_mu_host.restype = i32
    lib.nolsm_sign_dense_batched.argtypes = [vp, vp, vp, i32, i32, i32, f32, i32, i32, vp, P(SignStats), vp]
    lib.nolsm_sign_dense_batched.restype = i32
    lib.nolsm_batch_read.argtypes = [vp, vp, i32, i32, vp, i64, P(i32), vp]
    lib.nolsm_batch_read.restype = i32
    lib.nolsm_batch_size.argtypes = [vp]
    lib.nolsm_batch_size.restype = i32
    lib.nolsm_batch_ld.argtypes = [vp]
    lib.nolsm_batch_ld.restype = i32
    lib.nolsm_gemm_batched.argtypes = [vp, i32, i32, f32, f32, vp, vp, vp, vp, vp, i32, i32, vp]
    lib.nolsm_gemm_batched.restype = i32
    lib.nolsm_combine_submatrices.argtypes = [i32, vp, vp, P(i32), vp, vp, vp, vp, i64, P(i64)]
    lib.nolsm_combine_submatrices.restype = i32
    lib.nolsm_build_submatrices_grouped.argtypes = [vp, P(_Bsr), P(_Bsr), P(_Groups), i32, i32, i32, P(vp), vp]
    lib.nolsm_build_submatrices_grouped.restype = i32
    lib.nolsm_union_pattern.argtypes = [i32, vp, vp, vp, vp, vp, vp, i64, P(i64)]
    lib.nolsm_union_pattern.restype = i32
    lib.nolsm_expand_store.argtypes = [vp, P(_Bsr), vp, vp, vp, vp]
    lib.nolsm_expand_store.restype = i32
    _LIB = lib
    return lib


def _torch():
    import torch
    return torch


def _ptr(t, dtype=None):
    """Device pointer of a contiguous CUDA tensor (None -> NULL)."""
    if t is None:
        return None
    torch = _torch()
    if not t.is_cuda:
        raise NolsmError(1, "tensor must live on the CUDA device")
    if not t.is_contiguous():
        raise NolsmError(1, "tensor must be contiguous")
    if dtype is not None and t.dtype != dtype:
        raise NolsmError(1, f"tensor dtype {t.dtype}, expected {dtype}")
    return C.c_void_p(t.data_ptr())


def _stream(stream):
    torch = _torch()
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


class BlockSparse:
    """CSR of 6x6 FP32 blocks on the device (nolsm_bsr).  row_ptr/col_idx int32, val float32 [nnzb,6,6]."""

    def __init__(self, row_ptr, col_idx, val):
        torch = _torch()
        self.row_ptr, self.col_idx, self.val = row_ptr, col_idx, val
        self.n_mol = int(row_ptr.numel()) - 1
        self._c = _Bsr(self.n_mol, 6, _ptr(row_ptr, torch.int32).value, _ptr(col_idx, torch.int32).value,
                       _ptr(val, torch.float32).value)

    @classmethod
    def from_numpy(cls, row_ptr, col_idx, val, device="cuda"):
        torch = _torch()
        return cls(torch.as_tensor(row_ptr, dtype=torch.int32).to(device),
                   torch.as_tensor(col_idx, dtype=torch.int32).to(device),
                   torch.as_tensor(val, dtype=torch.float32).contiguous().to(device))

    def like(self):
        torch = _torch()
        return BlockSparse(self.row_ptr, self.col_idx, torch.zeros_like(self.val))

    def ref(self):
        return C.byref(self._c)


class Batch:
    def __init__(self, ctx, handle):
        self.ctx, self.handle = ctx, handle

    @property
    def size(self):
        return self.ctx.lib.nolsm_batch_size(self.handle)

    @property
    def ld(self):
        return self.ctx.lib.nolsm_batch_ld(self.handle)

    def read(self, local, which, stream=None):
        """Row-major n_j x n_j FP32 copy of one matrix of the batch (tests)."""
        torch = _torch()
        ld = self.ld
        buf = torch.empty(ld * ld, dtype=torch.float32, device="cuda")
        n = C.c_int32(0)
        self.ctx._check(self.ctx.lib.nolsm_batch_read(self.ctx.handle, self.handle, local, which, _ptr(buf),
                                                      buf.numel(), C.byref(n), _stream(stream)))
        return buf[: n.value * n.value].view(n.value, n.value)


def combine_submatrices(row_ptr, col_idx):
    """nolsm_combine_submatrices on host int32 numpy arrays (the heuristic is host work: no device, no context).
    Returns (own_ptr, own_idx, list_ptr, list_idx) as numpy int32 arrays."""
    import numpy as np
    lib = load_library()
    row_ptr = np.ascontiguousarray(row_ptr, dtype=np.int32)
    col_idx = np.ascontiguousarray(col_idx, dtype=np.int32)
    n = int(row_ptr.shape[0]) - 1
    own_ptr = np.zeros(n + 1, dtype=np.int32)
    own_idx = np.zeros(max(n, 1), dtype=np.int32)
    list_ptr = np.zeros(n + 1, dtype=np.int32)
    list_idx = np.zeros(max(int(col_idx.shape[0]), 1), dtype=np.int32)
    ng, ll = C.c_int32(0), C.c_int64(0)
    st = lib.nolsm_combine_submatrices(n, row_ptr.ctypes.data, col_idx.ctypes.data, C.byref(ng), own_ptr.ctypes.data,
                                       own_idx.ctypes.data, list_ptr.ctypes.data, list_idx.ctypes.data,
                                       int(list_idx.shape[0]), C.byref(ll))
    if st != 0:
        raise NolsmError(st, "nolsm_combine_submatrices")
    g = ng.value
    return own_ptr[:g + 1].copy(), own_idx[:n].copy(), list_ptr[:g + 1].copy(), list_idx[:ll.value].copy()


def union_pattern(row_ptr_a, col_idx_a, row_ptr_b, col_idx_b):
    """nolsm_union_pattern on host int32 numpy arrays. Returns (row_ptr, col_idx) of the merged pattern."""
    import numpy as np
    lib = load_library()
    a_rp, a_ci, b_rp, b_ci = (np.ascontiguousarray(x, dtype=np.int32) for x in (row_ptr_a, col_idx_a, row_ptr_b, col_idx_b))
    n = int(a_rp.shape[0]) - 1
    rp = np.zeros(n + 1, dtype=np.int32)
    cap = int(a_ci.shape[0] + b_ci.shape[0])
    ci = np.zeros(max(cap, 1), dtype=np.int32)
    nnzb = C.c_int64(0)
    st = lib.nolsm_union_pattern(n, a_rp.ctypes.data, a_ci.ctypes.data, b_rp.ctypes.data, b_ci.ctypes.data,
                                 rp.ctypes.data, ci.ctypes.data, cap, C.byref(nnzb))
    if st != 0:
        raise NolsmError(st, "nolsm_union_pattern")
    return rp, ci[:nnzb.value].copy()


class Groups:
    """Device copy of the combined submatrices (nolsm_groups)."""

    def __init__(self, own_ptr, own_idx, list_ptr, list_idx):
        torch = _torch()
        self.n_groups = int(len(own_ptr)) - 1
        self.own_ptr, self.own_idx, self.list_ptr, self.list_idx = (
            torch.as_tensor(x, dtype=torch.int32).contiguous().cuda() for x in (own_ptr, own_idx, list_ptr, list_idx))
        self._ref = _Groups(self.n_groups, self.own_ptr.data_ptr(), self.own_idx.data_ptr(), self.list_ptr.data_ptr(),
                            self.list_idx.data_ptr())

    def ref(self):
        return C.byref(self._ref)


class Context:
    """nolsm_ctx.  Raises NolsmError when the library or a CUDA device is missing."""

    def __init__(self, config=None):
        self.lib = load_library()
        self.handle = C.c_void_p()
        self.config = config if config is not None else Config()
        st = self.lib.nolsm_create(C.byref(self.handle), C.byref(self.config))
        if st != 0:
            msg = self.lib.nolsm_last_error(None)
            self.handle = None
            raise NolsmError(st, msg.decode() if msg else "")

    def close(self):
        if getattr(self, "handle", None):
            self.lib.nolsm_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, st):
        if st != 0:
            msg = self.lib.nolsm_last_error(self.handle)
            raise NolsmError(st, msg.decode() if msg else "")

    @property
    def launch_count(self):
        return int(self.lib.nolsm_launch_count(self.handle))

    # a0 -----------------------------------------------------------------------------------------
    def build_neighbours(self, pos_q, box_q, rc_q, cap=None, stream=None):
        """pos_q: int32 CUDA tensor [n_mol,3]; box_q: 3 ints (host).  Returns (row_ptr, col_idx)."""
        torch = _torch()
        n_mol = int(pos_q.shape[0])
        row_ptr = torch.empty(n_mol + 1, dtype=torch.int32, device=pos_q.device)
        box = (C.c_int32 * 3)(*[int(x) for x in box_q])
        nnzb = C.c_int64(0)
        if cap is None:
            st = self.lib.nolsm_build_neighbours(self.handle, n_mol, _ptr(pos_q, torch.int32), box, int(rc_q),
                                                 _ptr(row_ptr), None, 0, C.byref(nnzb), _stream(stream))
            if st not in (0, 2):
                self._check(st)
            cap = nnzb.value
        col_idx = torch.empty(max(cap, 1), dtype=torch.int32, device=pos_q.device)
        self._check(self.lib.nolsm_build_neighbours(self.handle, n_mol, _ptr(pos_q, torch.int32), box, int(rc_q),
                                                    _ptr(row_ptr), _ptr(col_idx), cap, C.byref(nnzb),
                                                    _stream(stream)))
        return row_ptr, col_idx[: nnzb.value]

    def build_neighbours_static(self, pos_q, box_q, rc_q, row_ptr, col_idx, stream=None):
        """nolsm_build_neighbours_static: the caller passes the outputs (row_ptr int32 [n_mol+1], col_idx int32 [cap]);
        no device memory is allocated.  Returns nnzb; the list is col_idx[:nnzb]."""
        torch = _torch()
        n_mol = int(pos_q.shape[0])
        box = (C.c_int32 * 3)(*[int(x) for x in box_q])
        nnzb = C.c_int64(0)
        self._check(self.lib.nolsm_build_neighbours_static(self.handle, n_mol, _ptr(pos_q, torch.int32), box,
                                                           int(rc_q), _ptr(row_ptr, torch.int32),
                                                           _ptr(col_idx, torch.int32), int(col_idx.numel()),
                                                           C.byref(nnzb), _stream(stream)))
        return nnzb.value

    # a1' ----------------------------------------------------------------------------------------
    def set_model(self, pos_q=None, box_q=None, rc_q=0, unit_per_grid=1.0, site_offset=None, orb_site=None,
                  orb_energy=None, s_ampl=0.0, h_ampl=0.0, h_len=1.0, eval_fp32=False):
        """Attach the two-centre model of nolsm.h (nolsm_model): submatrix builds then evaluate the elements
        from pos_q (int32 CUDA tensor [n_mol,3], kept alive here) instead of gathering.  pos_q=None detaches."""
        if pos_q is None:
            self._model_pos = None
            self._check(self.lib.nolsm_set_model(self.handle, None))
            return
        torch = _torch()
        m = _Model()
        m.pos_q = _ptr(pos_q, torch.int32)
        m.n_mol = int(pos_q.shape[0])
        m.rc_q = int(rc_q)
        m.unit_per_grid = float(unit_per_grid)
        for i in range(3):
            m.box_q[i] = int(box_q[i])
            for k in range(3):
                m.site_offset[i][k] = float(site_offset[i][k])
        for o in range(6):
            m.orb_site[o] = int(orb_site[o])
            m.orb_energy[o] = float(orb_energy[o])
        m.s_ampl, m.h_ampl, m.h_len = float(s_ampl), float(h_ampl), float(h_len)
        m.eval_fp32 = 1 if eval_fp32 else 0
        self._check(self.lib.nolsm_set_model(self.handle, C.byref(m)))
        self._model_pos = pos_q

    # a1 -----------------------------------------------------------------------------------------
    def build_submatrices(self, H, S, mol_begin, mol_count, slot=0, stream=None):
        h = C.c_void_p()
        self._check(self.lib.nolsm_build_submatrices(self.handle, H.ref(), S.ref(), mol_begin, mol_count, slot,
                                                     C.byref(h), _stream(stream)))
        return Batch(self, h)

    def build_submatrices_grouped(self, H, S, groups, grp_begin, grp_count, slot=0, stream=None):
        """groups: a Groups object (device arrays of the combined submatrices)."""
        h = C.c_void_p()
        self._check(self.lib.nolsm_build_submatrices_grouped(self.handle, H.ref(), S.ref(), groups.ref(), grp_begin,
                                                             grp_count, slot, C.byref(h), _stream(stream)))
        return Batch(self, h)

    def expand_store(self, src, row_ptr, col_idx, stream=None):
        """src (BlockSparse) laid out on the (larger) device pattern (row_ptr, col_idx): a new BlockSparse."""
        torch = _torch()
        val = torch.empty((int(col_idx.numel()), 6, 6), dtype=torch.float32, device="cuda")
        self._check(self.lib.nolsm_expand_store(self.handle, src.ref(), _ptr(row_ptr, torch.int32), _ptr(col_idx, torch.int32),
                                                _ptr(val, torch.float32), _stream(stream)))
        return BlockSparse(row_ptr, col_idx, val)

    def batch_capacity(self, H, mol_begin=0, n_slots=1, stream=None):
        r = self.lib.nolsm_batch_capacity(self.handle, H.ref(), mol_begin, n_slots, _stream(stream))
        if r < 0:
            self._check(-r)
        return r

    # a2-a4 --------------------------------------------------------------------------------------
    def sign_batched(self, batch, mu, precision=-1, tol=0.0, max_iter=0, fixed_iter=-1, want_stats=True,
                     stream=None):
        stats = SignStats() if want_stats else None
        self._check(self.lib.nolsm_sign_batched(self.handle, batch.handle, float(mu), precision, tol, max_iter,
                                                fixed_iter, C.byref(stats) if want_stats else None,
                                                _stream(stream)))
        return stats

    # a5-a7 --------------------------------------------------------------------------------------
    def scatter_density(self, batch, S, D, ne_partial, q_mol=None, ne_diag=None, stream=None):
        torch = _torch()
        self._check(self.lib.nolsm_scatter_density(self.handle, batch.handle, S.ref(), D.ref(),
                                                   _ptr(ne_partial, torch.float64), _ptr(q_mol, torch.float64),
                                                   _ptr(ne_diag, torch.float64), _stream(stream)))

    def scatter_energy(self, batch, H, D, W=None, e_partial=None, stream=None):
        """Own columns of W = D H0 D into W (optional) and Tr(D H0) of the batch's molecules added to e_partial."""
        torch = _torch()
        self._check(self.lib.nolsm_scatter_energy(self.handle, batch.handle, H.ref(), D.ref() if D is not None else None,
                                                  W.ref() if W is not None else None, _ptr(e_partial, torch.float64),
                                                  _stream(stream)))

    # whole path -----------------------------------------------------------------------------------
    def evaluate(self, H, S, mu, precision=-1, D=None, W=None, want_w=True, q_mol=None, stream=None):
        """One evaluation at a given mu. Returns (n_electrons, E_elec, D, W, stats)."""
        torch = _torch()
        if D is None:
            D = S.like()
        if W is None and want_w:
            W = S.like()
        ne, e = C.c_double(0.0), C.c_double(0.0)
        stats = SolveStats()
        st = self.lib.nolsm_evaluate(self.handle, H.ref(), S.ref(), float(mu), precision, D.ref(),
                                     W.ref() if W is not None else None, C.byref(ne), C.byref(e),
                                     _ptr(q_mol, torch.float64), C.byref(stats), _stream(stream))
        self._check(st)
        return ne.value, e.value, D, W, stats

    def solve_mu(self, H, S, n_electrons, mu_lo, mu_hi, tol_ne_per_mol=1e-3, max_steps=40, precision=-1, D=None,
                 q_mol=None, want_stats=True, stream=None):
        """Returns (mu, n_electrons(mu), D, stats)."""
        torch = _torch()
        if D is None:
            D = S.like()
        mu, ne = C.c_double(0.0), C.c_double(0.0)
        stats = SolveStats() if want_stats else None
        st = self.lib.nolsm_solve_mu(self.handle, H.ref(), S.ref(), float(n_electrons), float(mu_lo), float(mu_hi),
                                     float(tol_ne_per_mol), int(max_steps), precision, D.ref(), C.byref(mu),
                                     C.byref(ne), _ptr(q_mol, torch.float64),
                                     C.byref(stats) if want_stats else None, _stream(stream))
        self._check(st)
        return mu.value, ne.value, D, stats

    def solve_mu_host(self, row_ptr, col_idx, h_val, s_val, d_val, n_electrons, mu_lo, mu_hi, tol_ne_per_mol=1e-3,
                      max_steps=40, precision=-1, want_stats=True, stream=None):
        """HOST tensors (CPU torch tensors, ideally pinned): pattern int32, blocks float32.  d_val is
        overwritten with the density blocks.  Returns (mu, n_electrons(mu), stats, h2d_bytes, d2h_bytes)."""
        torch = _torch()
        for t, dt in ((row_ptr, torch.int32), (col_idx, torch.int32), (h_val, torch.float32),
                      (s_val, torch.float32), (d_val, torch.float32)):
            if t.is_cuda or not t.is_contiguous() or t.dtype != dt:
                raise NolsmError(1, "solve_mu_host takes contiguous CPU tensors (int32 pattern, float32 blocks)")
        mu, ne = C.c_double(0.0), C.c_double(0.0)
        h2d, d2h = C.c_int64(0), C.c_int64(0)
        stats = SolveStats() if want_stats else None
        st = self.lib.nolsm_solve_mu_host(self.handle, int(row_ptr.numel()) - 1, C.c_void_p(row_ptr.data_ptr()),
                                          C.c_void_p(col_idx.data_ptr()), C.c_void_p(h_val.data_ptr()),
                                          C.c_void_p(s_val.data_ptr()), float(n_electrons), float(mu_lo),
                                          float(mu_hi), float(tol_ne_per_mol), int(max_steps), precision,
                                          C.c_void_p(d_val.data_ptr()), C.byref(mu), C.byref(ne),
                                          C.byref(stats) if want_stats else None, C.byref(h2d), C.byref(d2h),
                                          _stream(stream))
        self._check(st)
        return mu.value, ne.value, stats, h2d.value, d2h.value

    # dense microbench -------------------------------------------------------------------------------
    def sign_dense_batched(self, a, scale=None, precision=-1, tol=0.0, max_iter=0, fixed_iter=-1, out=None,
                           want_stats=True, stream=None):
        """a: float32 CUDA tensor [batch,n,n] row-major.  Returns (sign(a) [batch,n,n], stats)."""
        torch = _torch()
        batch, n = int(a.shape[0]), int(a.shape[1])
        if out is None:
            out = torch.empty_like(a)
        stats = SignStats() if want_stats else None
        self._check(self.lib.nolsm_sign_dense_batched(self.handle, _ptr(a, torch.float32), _ptr(scale, torch.float32),
                                                      n, batch, precision, tol, max_iter, fixed_iter,
                                                      _ptr(out, torch.float32),
                                                      C.byref(stats) if want_stats else None, _stream(stream)))
        return out, stats

    # GEMM building block (tests) ---------------------------------------------------------------------
    def gemm_batched(self, kind, a, b, cin=None, ident=False, alpha=1.0, beta=0.0, stream=None):
        torch = _torch()
        batch, n = int(a.shape[0]), int(a.shape[1])
        c = torch.empty_like(a)
        resid2 = torch.zeros(batch, dtype=torch.float32, device=a.device)
        self._check(self.lib.nolsm_gemm_batched(self.handle, kind, 1 if ident else 0, alpha, beta,
                                                _ptr(a, torch.float32), _ptr(b, torch.float32),
                                                _ptr(cin, torch.float32), _ptr(c, torch.float32), _ptr(resid2), n,
                                                batch, _stream(stream)))
        return c, resid2
