"""ctypes binding of libdmrgk.so — same names as include/dmrgk.h (and include/dmrgk_harness.h), argument marshalling only.

Every step of the hot path runs in the library's CUDA kernels; this module converts Python ints,
NumPy arrays (host metadata) and device pointers (``torch.Tensor.data_ptr()``) into the C types of
the ABI, checks the returned status and raises ``DmrgkError`` with ``dmrgk_last_error()``.
There is no fallback of any kind: if the shared library is missing, ``load()`` raises.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "_build", "libdmrgk.so")

OK, EINVAL, ESHAPE, ECHARGE, EALIGN, ENOMEM, ECUDA, ENOTCONV, ESTATE = 0, -1, -2, -3, -4, -5, -6, -7, -8
TRANS_L, TRANS_R, IDENT_L, IDENT_R, HC_OF_PREV = 1, 2, 4, 8, 16

_STATUS_NAMES = {0: "OK", -1: "EINVAL", -2: "ESHAPE", -3: "ECHARGE", -4: "EALIGN", -5: "ENOMEM",
                 -6: "ECUDA", -7: "ENOTCONV", -8: "ESTATE"}


class DmrgkError(RuntimeError):
    def __init__(self, status, message):
        super().__init__(f"dmrgk status {status} ({_STATUS_NAMES.get(status, '?')}): {message}")
        self.status = status
        self.message = message


class RenormOpts(C.Structure):
    _fields_ = [("t_chunk_bytes", C.c_int64), ("kernel", C.c_int32), ("reserved", C.c_int32 * 5)]


class HeffOpts(C.Structure):
    _fields_ = [("t_chunk_bytes", C.c_int64), ("ring_bytes", C.c_int64), ("kernel", C.c_int32),
                ("split_waves", C.c_int32), ("order_policy", C.c_int32), ("per_pair_output", C.c_int32),
                ("reserved", C.c_int32 * 2)]


_p, _i32, _i64, _u64, _f64 = C.c_void_p, C.c_int32, C.c_int64, C.c_uint64, C.c_double
_pp = C.POINTER(C.c_void_p)
_pi32, _pi64, _pf64 = C.POINTER(C.c_int32), C.POINTER(C.c_int64), C.POINTER(C.c_double)

# name -> (restype, argtypes); the list of symbols include/dmrgk.h and include/dmrgk_harness.h declare.
SIGNATURES = {
    "dmrgk_last_error": (C.c_char_p, []),
    "dmrgk_version": (C.c_char_p, []),
    "dmrgk_launch_count": (_i64, [_i32]),
    "dmrgk_ctx_create": (_i32, [_i32, _pp]),
    "dmrgk_ctx_destroy": (None, [_p]),
    "dmrgk_ctx_query": (_i32, [_p, _pi32, _pi64, _pi64]),
    "dmrgk_space_create": (_i32, [_p, _i32, _i32, _p, _p, _pp]),
    "dmrgk_space_destroy": (None, [_p]),
    "dmrgk_layout_create": (_i32, [_p, _p, _p, _p, _pp]),
    "dmrgk_layout_destroy": (None, [_p]),
    "dmrgk_layout_query": (_i32, [_p, _pi64, _pi64, _pi64]),
    "dmrgk_layout_blocks": (_i32, [_p, _p, _p, _p, _p, _p, _p]),
    "dmrgk_layout_pack": (_i32, [_p, _p, _p]),
    "dmrgk_layout_unpack": (_i32, [_p, _p, _p]),
    "dmrgk_op_create": (_i32, [_p, _p, _p, _i32, _pp]),
    "dmrgk_op_destroy": (None, [_p]),
    "dmrgk_op_query": (_i32, [_p, _pi64, _pi64, _pi64]),
    "dmrgk_op_blocks": (_i32, [_p, _p, _p, _p, _p, _p, _p]),
    "dmrgk_op_pack": (_i32, [_p, _p, _p]),
    "dmrgk_op_unpack": (_i32, [_p, _p, _p]),
    "dmrgk_block_size": (_i64, [_i32, _i32]),
    "dmrgk_block_unpack": (_i32, [_i32, _i32, _p, _p]),
    "dmrgk_block_padding_is_zero": (_i32, [_i32, _i32, _p]),
    "dmrgk_op_bind_device": (_i32, [_p, _p]),
    "dmrgk_op_bind_pinned": (_i32, [_p, _p]),
    "dmrgk_heff_create": (_i32, [_p, _p, _i64, _p, _p, _p, _p, _p, _pp]),
    "dmrgk_heff_create_blockcoef": (_i32, [_p, _p, _i64, _p, _p, _p, _p, _p, _p, _pp]),
    "dmrgk_heff_destroy": (None, [_p]),
    "dmrgk_heff_query": (_i32, [_p, _pi64, _pf64, _pf64, _pi64, _pi64, _pi64, _pi64]),
    "dmrgk_heff_apply": (_i32, [_p, _p, _p, _p, _p, _p]),
    "dmrgk_heff_expect": (_i32, [_p, _p, _p, _p, _p, _p]),
    "dmrgk_heff_apply_host": (_i32, [_p, _p, _p, _p, _p, _p, _p, _p]),
    "dmrgk_heff_diag": (_i32, [_p, _p, _p, _p, _p]),
    "dmrgk_heff_profile": (_i32, [_p, _i32]),
    "dmrgk_heff_profile_read": (_i32, [_p, _p, _p]),
    "dmrgk_iso_create": (_i32, [_p, _p, _p, _pp]),
    "dmrgk_iso_destroy": (None, [_p]),
    "dmrgk_iso_query": (_i32, [_p, _pi64, _pi64, _pi64]),
    "dmrgk_iso_blocks": (_i32, [_p, _p, _p, _p, _p, _p, _p]),
    "dmrgk_iso_pack": (_i32, [_p, _p, _p]),
    "dmrgk_iso_bind_device": (_i32, [_p, _p]),
    "dmrgk_iso_fill_normal": (_i32, [_p, _p, _u64, _u64, _p]),
    "dmrgk_renorm_create": (_i32, [_p, _p, _i64, _p, _p, _p, _pp]),
    "dmrgk_renorm_destroy": (None, [_p]),
    "dmrgk_renorm_query": (_i32, [_p, _pi64, _pf64, _pi64, _pi64]),
    "dmrgk_renorm_apply": (_i32, [_p, _p, _p]),
    "dmrgk_enlarge_create": (_i32, [_p, _p, _p, _i32, _p, _i32, _i64, _p, _i64, _p, _p, _p, _p, _p, _pp]),
    "dmrgk_enlarge_destroy": (None, [_p]),
    "dmrgk_enlarge_query": (_i32, [_p, _pi64, _pi64, _pi64, _pi64]),
    "dmrgk_enlarge_apply": (_i32, [_p, _p]),
    "dmrgk_vec_scratch_bytes": (_i64, [_i32]),
    "dmrgk_vec_multi_dot": (_i32, [_p, _i64, _i32, _p, _i64, _p, _p, _p, _p]),
    "dmrgk_vec_multi_dot_noalloc": (_i32, [_p, _i64, _i32, _p, _i64, _p, _p, _p]),
    "dmrgk_vec_multi_axpy": (_i32, [_p, _i64, _i32, _p, _i64, _p, _f64, _f64, _p, _p]),
    "dmrgk_vec_axpby": (_i32, [_p, _i64, _f64, _p, _f64, _p, _p]),
    "dmrgk_vec_dot": (_i32, [_p, _i64, _p, _p, _p, _p, _p]),
    "dmrgk_vec_nrm2": (_i32, [_p, _i64, _p, _p, _p, _p]),
    "dmrgk_vec_axpy": (_i32, [_p, _i64, _f64, _p, _p, _p]),
    "dmrgk_vec_scal": (_i32, [_p, _i64, _f64, _p, _p]),
    "dmrgk_vec_scal_dev": (_i32, [_p, _i64, _p, _i32, _p, _p, _p]),
    "dmrgk_vec_residual": (_i32, [_p, _i64, _i32, _p, _p, _i64, _p, _p, _p, _p, _p]),
    "dmrgk_vec_precond": (_i32, [_p, _i64, _p, _p, _p, _p, _p]),
    "dmrgk_davidson_extra_bytes": (_i64, [_i32, _i64]),
    "dmrgk_davidson_create": (_i32, [_p, _i32, _f64, _i32, _p, _p, _p, _p, _p, _p, _pp]),
    "dmrgk_davidson_destroy": (None, [_p]),
    "dmrgk_davidson_start": (_i32, [_p, _p]),
    "dmrgk_davidson_step": (_i32, [_p, _pf64, _pf64, _pi32]),
    "dmrgk_davidson_solve": (_i32, [_p, _pf64, _pf64, _p, _pi32]),
    "dmrgk_davidson_query": (_i32, [_p, _pi32, _pi32]),
    "dmrgk_davidson_set_allreduce": (_i32, [_p, _p, _p]),
    "dmrgk_op_fill_normal": (_i32, [_p, _p, _u64, _u64, _i32, _i32, _p]),
    "dmrgk_layout_fill_normal": (_i32, [_p, _p, _u64, _u64, _p]),
    "dmrgk_probe_fp64": (_i32, [_p, _i32, _i64, _p, _pf64, _p]),
    "dmrgk_plan_tile_cuts": (_i32, [_i32, _i32, _p, _i32]),
    "dmrgk_plan_tile_cost": (_i32, [_i32, _i32]),
}

_lib = None


def load(path=None):
    """dlopen libdmrgk.so and declare every prototype.  Raises if the library is not built."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    path = path or LIB_PATH
    if not os.path.exists(path):
        raise FileNotFoundError(
            f"{path} not found: build it with `python -m paper_2311_14106_b200.build` "
            "(dmrgk has no CPU or PyTorch fallback)")
    if path == LIB_PATH:
        # a binary built from other sources than the ones beside it must not be loaded silently
        # (mtimes mean nothing after a checkout or a copy): rebuild it, or fail
        from . import build as _build
        if _build.built_hash() != _build.source_hash():
            _build.build()
    lib = C.CDLL(path)
    for name, (res, args) in SIGNATURES.items():
        fn = getattr(lib, name)
        fn.restype = res
        fn.argtypes = args
    if path == LIB_PATH:
        from . import build as _build
        have = lib.dmrgk_version().decode().rsplit("src:", 1)[-1]
        if have != _build.source_hash():
            raise RuntimeError(f"{path} was built from sources {have}, the tree holds {_build.source_hash()}: "
                               "rebuild with `python -m paper_2311_14106_b200.build --force`")
    _lib = lib
    return lib


def source_hash():
    """The source hash compiled into the loaded library (dmrgk_version)."""
    return load().dmrgk_version().decode().rsplit("src:", 1)[-1]


def last_error():
    return load().dmrgk_last_error().decode("utf-8", "replace")


def check(status):
    if status != OK:
        raise DmrgkError(status, last_error())


def _dev(t):
    """Device pointer of a torch tensor (or a raw int / None)."""
    if t is None:
        return None
    if isinstance(t, int):
        return t
    return t.data_ptr()


def _stream(s):
    if s is None:
        return None
    if isinstance(s, int):
        return s
    return s.cuda_stream


def _i32arr(x):
    return np.ascontiguousarray(np.asarray(x, dtype=np.int32))


class Ctx:
    def __init__(self, device=0):
        self.lib = load()
        h = C.c_void_p()
        check(self.lib.dmrgk_ctx_create(device, C.byref(h)))
        self.h = h
        self.device = device

    def query(self):
        n_sm, l2, hbm = C.c_int32(), C.c_int64(), C.c_int64()
        check(self.lib.dmrgk_ctx_query(self.h, C.byref(n_sm), C.byref(l2), C.byref(hbm)))
        return n_sm.value, l2.value, hbm.value

    def __del__(self):
        if getattr(self, "h", None):
            self.lib.dmrgk_ctx_destroy(self.h)
            self.h = None


class Space:
    """dmrgk_space: sectors = [(charge tuple, dim)]."""

    def __init__(self, ctx, n_charges, sectors):
        self.ctx, self.lib = ctx, ctx.lib
        self.sectors = list(sectors)
        q = _i32arr([list(s[0]) for s in sectors]).reshape(-1)
        d = _i32arr([s[1] for s in sectors])
        h = C.c_void_p()
        check(self.lib.dmrgk_space_create(ctx.h, n_charges, len(sectors), q.ctypes.data, d.ctypes.data, C.byref(h)))
        self.h = h
        self.n_charges = n_charges

    def __del__(self):
        if getattr(self, "h", None):
            self.lib.dmrgk_space_destroy(self.h)
            self.h = None


class _Blocked:
    """Shared query helpers of Layout and Op (block table as NumPy arrays)."""
    _query = _blocks = None

    def query(self):
        nb, ne, npad = C.c_int64(), C.c_int64(), C.c_int64()
        check(getattr(self.lib, self._query)(self.h, C.byref(nb), C.byref(ne), C.byref(npad)))
        return nb.value, ne.value, npad.value

    def blocks(self):
        nb = self.query()[0]
        r, c, rows, cols, ld = (np.zeros(nb, np.int32) for _ in range(5))
        off = np.zeros(nb, np.int64)
        check(getattr(self.lib, self._blocks)(self.h, r.ctypes.data, c.ctypes.data, rows.ctypes.data,
                                              cols.ctypes.data, ld.ctypes.data, off.ctypes.data))
        return r, c, rows, cols, ld, off


class Layout(_Blocked):
    _query, _blocks = "dmrgk_layout_query", "dmrgk_layout_blocks"

    def __init__(self, ctx, A, B, target):
        self.ctx, self.lib, self.A, self.B = ctx, ctx.lib, A, B
        t = _i32arr(list(target))
        h = C.c_void_p()
        check(self.lib.dmrgk_layout_create(ctx.h, A.h, B.h, t.ctypes.data, C.byref(h)))
        self.h = h
        self.n_blocks, self.n_elems, self.n_padded = self.query()

    def pack(self, unpadded):
        u = np.ascontiguousarray(unpadded, dtype=np.float64)
        assert u.size == self.n_elems
        p = np.zeros(self.n_padded, np.float64)
        check(self.lib.dmrgk_layout_pack(self.h, u.ctypes.data, p.ctypes.data))
        return p

    def unpack(self, packed):
        p = np.ascontiguousarray(packed, dtype=np.float64)
        assert p.size == self.n_padded
        u = np.zeros(self.n_elems, np.float64)
        check(self.lib.dmrgk_layout_unpack(self.h, p.ctypes.data, u.ctypes.data))
        return u

    def fill_normal(self, arena, seed, stream_id, stream=None):
        check(self.lib.dmrgk_layout_fill_normal(self.h, _dev(arena), seed, stream_id, _stream(stream)))

    def __del__(self):
        if getattr(self, "h", None):
            self.lib.dmrgk_layout_destroy(self.h)
            self.h = None


class Op(_Blocked):
    _query, _blocks = "dmrgk_op_query", "dmrgk_op_blocks"

    def __init__(self, ctx, space, dq, parity):
        self.ctx, self.lib, self.space = ctx, ctx.lib, space
        d = _i32arr(list(dq))
        h = C.c_void_p()
        check(self.lib.dmrgk_op_create(ctx.h, space.h, d.ctypes.data, int(parity), C.byref(h)))
        self.h = h
        self.n_blocks, self.n_elems, self.n_padded = self.query()
        self._keep = None

    def pack(self, unpadded):
        u = np.ascontiguousarray(unpadded, dtype=np.float64)
        assert u.size == self.n_elems
        p = np.zeros(self.n_padded, np.float64)
        check(self.lib.dmrgk_op_pack(self.h, u.ctypes.data, p.ctypes.data))
        return p

    def bind_device(self, arena):
        check(self.lib.dmrgk_op_bind_device(self.h, _dev(arena)))
        self._keep = arena

    def bind_pinned(self, arena):
        check(self.lib.dmrgk_op_bind_pinned(self.h, _dev(arena)))
        self._keep = arena

    def fill_normal(self, arena, seed, stream_id, scale_mode, symmetric, stream=None):
        check(self.lib.dmrgk_op_fill_normal(self.h, _dev(arena), seed, stream_id, int(scale_mode),
                                            int(bool(symmetric)), _stream(stream)))

    def __del__(self):
        if getattr(self, "h", None):
            self.lib.dmrgk_op_destroy(self.h)
            self.h = None


class Enlarge:
    """dmrgk_enlarge: out[i] = Σ_j coef_j (X_j P^π_j) ⊗ y_j.
    terms = [(index into out_ops, X Op or None, transposed, site_odd, coef, y (d×d array))].
    site_major=False: left block, kept ⊗ site, the kept-parity sign is applied when site_odd;
    site_major=True: right block, site ⊗ kept, y already carries P_s^{π_x} (blockops.fold_site_parity)."""

    def __init__(self, ctx, kept, enlarged, site_charges, out_ops, terms, site_major=False):
        self.lib, self.ctx = ctx.lib, ctx
        sc = np.ascontiguousarray(site_charges, dtype=np.int32).reshape(len(site_charges), -1)
        d = sc.shape[0]
        n_out, n_terms = len(out_ops), len(terms)
        oarr = (C.c_void_p * max(n_out, 1))(*[o.h for o in out_ops])
        xarr = (C.c_void_p * max(n_terms, 1))()
        t_out = np.zeros(max(n_terms, 1), np.int32)
        t_flags = np.zeros(max(n_terms, 1), np.uint32)
        t_coef = np.zeros(max(n_terms, 1), np.float64)
        t_y = np.zeros((max(n_terms, 1), d, d), np.float64)
        for j, (o, X, trans, odd, coef, y) in enumerate(terms):
            t_out[j], t_coef[j] = o, coef
            xarr[j] = X.h if X is not None else None
            t_flags[j] = (1 if trans else 0) | ((4 if site_major else 2) if odd else 0)
            t_y[j] = np.asarray(y, dtype=np.float64)
        self._keep = (out_ops, [t[1] for t in terms], kept, enlarged)
        h = C.c_void_p()
        check(self.lib.dmrgk_enlarge_create(ctx.h, kept.h, enlarged.h, d, sc.ctypes.data, int(bool(site_major)), n_out, oarr, n_terms,
                                            t_out.ctypes.data, xarr, t_flags.ctypes.data, t_coef.ctypes.data,
                                            t_y.ctypes.data, C.byref(h)))
        self.h = h
        a, b, c_, d_ = (C.c_int64() for _ in range(4))
        check(self.lib.dmrgk_enlarge_query(self.h, C.byref(a), C.byref(b), C.byref(c_), C.byref(d_)))
        self.n_tiles, self.n_sources, self.bytes_read, self.bytes_written = a.value, b.value, c_.value, d_.value

    def apply(self, stream=None):
        check(self.lib.dmrgk_enlarge_apply(self.h, _stream(stream)))

    def __del__(self):
        if getattr(self, "h", None):
            self.lib.dmrgk_enlarge_destroy(self.h)
            self.h = None


def block_size(rows, cols):
    """Doubles a rows×cols block occupies in the panel layout."""
    return load().dmrgk_block_size(int(rows), int(cols))


def block_unpack(packed, rows, cols):
    """Dense rows×cols array of ONE block from its packed (panel-layout) doubles."""
    p = np.ascontiguousarray(packed, dtype=np.float64)
    assert p.size >= block_size(rows, cols)
    out = np.zeros((int(rows), int(cols)), np.float64)
    check(load().dmrgk_block_unpack(int(rows), int(cols), p.ctypes.data, out.ctypes.data))
    return out


def block_padding_is_zero(packed, rows, cols):
    p = np.ascontiguousarray(packed, dtype=np.float64)
    assert p.size >= block_size(rows, cols)
    st = load().dmrgk_block_padding_is_zero(int(rows), int(cols), p.ctypes.data)
    if st < 0:
        check(st)
    return st == 0


class Iso(_Blocked):
    """dmrgk_iso: the kept basis Φ (kept space → enlarged space)."""
    _query, _blocks = "dmrgk_iso_query", "dmrgk_iso_blocks"

    def __init__(self, ctx, enlarged, kept):
        self.ctx, self.lib, self.enlarged, self.kept = ctx, ctx.lib, enlarged, kept
        h = C.c_void_p()
        check(self.lib.dmrgk_iso_create(ctx.h, enlarged.h, kept.h, C.byref(h)))
        self.h = h
        self.n_blocks, self.n_elems, self.n_padded = self.query()
        self._keep = None

    def pack(self, unpadded):
        u = np.ascontiguousarray(unpadded, dtype=np.float64)
        assert u.size == self.n_elems
        p = np.zeros(self.n_padded, np.float64)
        check(self.lib.dmrgk_iso_pack(self.h, u.ctypes.data, p.ctypes.data))
        return p

    def bind_device(self, arena):
        check(self.lib.dmrgk_iso_bind_device(self.h, _dev(arena)))
        self._keep = arena

    def fill_normal(self, arena, seed, stream_id, stream=None):
        check(self.lib.dmrgk_iso_fill_normal(self.h, _dev(arena), seed, stream_id, _stream(stream)))

    def __del__(self):
        if getattr(self, "h", None):
            self.lib.dmrgk_iso_destroy(self.h)
            self.h = None


class Renorm:
    """dmrgk_renorm: out[i] = Φᵀ in[i] Φ for lists of bound operators."""

    def __init__(self, ctx, phi, ops_in, ops_out, t_chunk_bytes=0, kernel=0):
        self.ctx, self.lib = ctx, ctx.lib
        n = len(ops_in)
        assert len(ops_out) == n
        a_in = (C.c_void_p * max(n, 1))()
        a_out = (C.c_void_p * max(n, 1))()
        for i in range(n):
            a_in[i], a_out[i] = ops_in[i].h, ops_out[i].h
        opts = RenormOpts(int(t_chunk_bytes), int(kernel))
        h = C.c_void_p()
        check(self.lib.dmrgk_renorm_create(ctx.h, phi.h, n, a_in, a_out, C.byref(opts), C.byref(h)))
        self.h = h
        self._keep = (phi, list(ops_in), list(ops_out))
        nt, wb, nl, fl = C.c_int64(), C.c_int64(), C.c_int64(), C.c_double()
        check(self.lib.dmrgk_renorm_query(self.h, C.byref(nt), C.byref(fl), C.byref(wb), C.byref(nl)))
        self.n_tasks, self.flops, self.workspace_bytes, self.n_launches = nt.value, fl.value, wb.value, nl.value

    def apply(self, workspace, stream=None):
        check(self.lib.dmrgk_renorm_apply(self.h, _dev(workspace), _stream(stream)))

    def __del__(self):
        if getattr(self, "h", None):
            self.lib.dmrgk_renorm_destroy(self.h)
            self.h = None


class Heff:
    """dmrgk_heff: terms = [(L Op or None, R Op or None, coef, trans_L, trans_R)]."""

    def __init__(self, ctx, layout, terms, t_chunk_bytes=0, ring_bytes=0, kernel=0, split_waves=0, order_policy=0, per_pair_output=0,
                 block_coef=None):
        self.ctx, self.lib, self.layout = ctx, ctx.lib, layout
        K = len(terms)
        Larr = (C.c_void_p * max(K, 1))()
        Rarr = (C.c_void_p * max(K, 1))()
        coef = np.zeros(max(K, 1), np.float64)
        flags = np.zeros(max(K, 1), np.uint32)
        self._ops = []
        for k, (L, R, c, tL, tR) in enumerate(terms):
            coef[k] = c
            if tL == "hc":                    # (None, None, coef, "hc", "hc"): the h.c. of the previous pair
                Larr[k] = Rarr[k] = None
                flags[k] = HC_OF_PREV
                continue
            Larr[k] = L.h if L is not None else None
            Rarr[k] = R.h if R is not None else None
            flags[k] = ((TRANS_L if tL else 0) | (TRANS_R if tR else 0) |
                        (IDENT_L if L is None else 0) | (IDENT_R if R is None else 0))
            self._ops += [L, R]
        opts = HeffOpts(int(t_chunk_bytes), int(ring_bytes), int(kernel), int(split_waves), int(order_policy), int(per_pair_output))
        h = C.c_void_p()
        if block_coef is None:
            check(self.lib.dmrgk_heff_create(ctx.h, layout.h, K, Larr, Rarr, coef.ctypes.data, flags.ctypes.data,
                                             C.byref(opts), C.byref(h)))
        else:       # [K][n_blocks] recoupling scalars per (pair, input block)
            bc = np.ascontiguousarray(block_coef, dtype=np.float64).reshape(max(K, 1), -1)
            assert bc.shape[1] == layout.n_blocks
            check(self.lib.dmrgk_heff_create_blockcoef(ctx.h, layout.h, K, Larr, Rarr, coef.ctypes.data, bc.ctypes.data,
                                                       flags.ctypes.data, C.byref(opts), C.byref(h)))
        self.h = h
        q = self.query()
        self.n_tasks, self.flops_alg, self.flops_exec = q["n_tasks"], q["flops_alg"], q["flops_exec"]
        self.op_bytes, self.workspace_bytes = q["op_bytes"], q["workspace_bytes"]
        self.n_chunks, self.n_launches = q["n_chunks"], q["n_launches"]

    def query(self):
        nt, ob, wb, nc, nl = (C.c_int64() for _ in range(5))
        fa, fe = C.c_double(), C.c_double()
        check(self.lib.dmrgk_heff_query(self.h, C.byref(nt), C.byref(fa), C.byref(fe), C.byref(ob), C.byref(wb),
                                        C.byref(nc), C.byref(nl)))
        return {"n_tasks": nt.value, "flops_alg": fa.value, "flops_exec": fe.value, "op_bytes": ob.value,
                "workspace_bytes": wb.value, "n_chunks": nc.value, "n_launches": nl.value}

    def apply(self, psi, sigma, workspace, stream_main=None, stream_copy=None):
        check(self.lib.dmrgk_heff_apply(self.h, _dev(psi), _dev(sigma), _dev(workspace), _stream(stream_main),
                                        _stream(stream_copy)))

    def expect(self, psi, out, workspace, stream_main=None, stream_copy=None):
        """out[k] = ⟨ψ, c_k (L_k ⊗ R_k) ψ⟩ for every pair (plan created with per_pair_output=1)."""
        check(self.lib.dmrgk_heff_expect(self.h, _dev(psi), _dev(out), _dev(workspace), _stream(stream_main),
                                         _stream(stream_copy)))

    def apply_host(self, psi_host, sigma_host, psi, sigma, workspace, stream_main=None, stream_copy=None):
        check(self.lib.dmrgk_heff_apply_host(self.h, _dev(psi_host), _dev(sigma_host), _dev(psi), _dev(sigma),
                                             _dev(workspace), _stream(stream_main), _stream(stream_copy)))

    def profile(self, enable=1):
        """0 off, 1 whole-apply span with normal overlap, 2 serialised per-launch timing."""
        check(self.lib.dmrgk_heff_profile(self.h, int(enable)))

    def profile_read(self):
        """({"p1","p2","reduce","apply"} → ms, same → launch counts) accumulated since profile()."""
        ms = np.zeros(4, np.float64)
        ln = np.zeros(4, np.int64)
        check(self.lib.dmrgk_heff_profile_read(self.h, ms.ctypes.data, ln.ctypes.data))
        names = ("p1", "p2", "reduce", "apply")
        return dict(zip(names, ms.tolist())), dict(zip(names, ln.tolist()))

    def diag(self, diag, workspace, stream_main=None, stream_copy=None):
        check(self.lib.dmrgk_heff_diag(self.h, _dev(diag), _dev(workspace), _stream(stream_main),
                                       _stream(stream_copy)))

    def __del__(self):
        if getattr(self, "h", None):
            self.lib.dmrgk_heff_destroy(self.h)
            self.h = None


class Davidson:
    def __init__(self, heff, m_max, tol, max_iter, V, W, diag, workspace, stream_main=None, stream_copy=None):
        self.lib, self.heff = heff.lib, heff
        self._keep = (V, W, diag, workspace, stream_main, stream_copy)
        h = C.c_void_p()
        check(self.lib.dmrgk_davidson_create(heff.h, m_max, tol, max_iter, _dev(V), _dev(W), _dev(diag),
                                             _dev(workspace), _stream(stream_main), _stream(stream_copy),
                                             C.byref(h)))
        self.h = h

    def start(self, x0):
        check(self.lib.dmrgk_davidson_start(self.h, _dev(x0)))

    def step(self):
        th, rn, cv = C.c_double(), C.c_double(), C.c_int32()
        check(self.lib.dmrgk_davidson_step(self.h, C.byref(th), C.byref(rn), C.byref(cv)))
        return th.value, rn.value, bool(cv.value)

    def solve(self, x=None):
        th, rn, na = C.c_double(), C.c_double(), C.c_int32()
        st = self.lib.dmrgk_davidson_solve(self.h, C.byref(th), C.byref(rn), _dev(x), C.byref(na))
        if st not in (OK, ENOTCONV):
            check(st)
        return th.value, rn.value, na.value, st == OK

    def query(self):
        m, na = C.c_int32(), C.c_int32()
        check(self.lib.dmrgk_davidson_query(self.h, C.byref(m), C.byref(na)))
        return m.value, na.value

    def set_allreduce(self, fn):
        """fn(device pointer, n doubles) -> 0: called after every apply of the driver (k-sharding hook), with
        the solver's main stream made torch's current stream for the duration of the call.  A non-zero return
        or an exception in fn makes the driver fail with ESTATE."""
        if fn is None:
            self._reduce_cb = None
            check(self.lib.dmrgk_davidson_set_allreduce(self.h, None, None))
            return
        proto = C.CFUNCTYPE(C.c_int32, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p)

        def trampoline(ptr, n, stream, user):
            # fn runs with the solver's main stream as torch's current stream, whatever stream the caller
            # has made current since: a collective issued by fn is then ordered after the apply that wrote
            # the vector.  An exception must not unwind through the C frames: it becomes a non-zero
            # status, which the driver reports as DMRGK_ESTATE.
            try:
                import torch
                s = torch.cuda.ExternalStream(int(stream)) if stream else torch.cuda.default_stream()
                with torch.cuda.stream(s):
                    return int(fn(int(ptr), int(n)))
            except BaseException:          # noqa: BLE001 — nothing may propagate into ctypes
                import traceback
                traceback.print_exc()
                return -1

        self._reduce_cb = proto(trampoline)
        check(self.lib.dmrgk_davidson_set_allreduce(self.h, C.cast(self._reduce_cb, C.c_void_p), None))

    def __del__(self):
        if getattr(self, "h", None):
            self.lib.dmrgk_davidson_destroy(self.h)
            self.h = None


def launch_count(reset=False):
    return load().dmrgk_launch_count(int(bool(reset)))


def davidson_extra_bytes(m_max, n_padded):
    return load().dmrgk_davidson_extra_bytes(m_max, n_padded)


def vec_scratch_bytes(nv):
    return load().dmrgk_vec_scratch_bytes(nv)


def vec_multi_dot(ctx, n, nv, X, stride, y, out, scratch, stream=None):
    check(ctx.lib.dmrgk_vec_multi_dot(ctx.h, n, nv, _dev(X), stride, _dev(y), _dev(out), _dev(scratch), _stream(stream)))


def vec_multi_dot_noalloc(ctx, n, nv, X, stride, y, out, stream=None):
    """vec_multi_dot without the scratch tensor, for callers that cannot allocate device memory (HBM already
    full of operators, no allocator of their own, or a cudaMalloc would stall the overlapped operator copies):
    the partial sums use a fixed array inside libdmrgk.so.  nv ≤ 64; one array per GPU, so calls that may
    overlap on the GPU race; make the first call on a device before any stream capture (include/dmrgk.h)."""
    check(ctx.lib.dmrgk_vec_multi_dot_noalloc(ctx.h, n, nv, _dev(X), stride, _dev(y), _dev(out), _stream(stream)))


def vec_multi_axpy(ctx, n, nv, X, stride, coef, alpha, beta, y, stream=None):
    check(ctx.lib.dmrgk_vec_multi_axpy(ctx.h, n, nv, _dev(X), stride, _dev(coef), alpha, beta, _dev(y), _stream(stream)))


def vec_dot(ctx, n, x, y, out, scratch, stream=None):
    check(ctx.lib.dmrgk_vec_dot(ctx.h, n, _dev(x), _dev(y), _dev(out), _dev(scratch), _stream(stream)))


def vec_nrm2(ctx, n, x, out, scratch, stream=None):
    check(ctx.lib.dmrgk_vec_nrm2(ctx.h, n, _dev(x), _dev(out), _dev(scratch), _stream(stream)))


def vec_axpy(ctx, n, alpha, x, y, stream=None):
    check(ctx.lib.dmrgk_vec_axpy(ctx.h, n, alpha, _dev(x), _dev(y), _stream(stream)))


def vec_scal(ctx, n, alpha, x, stream=None):
    check(ctx.lib.dmrgk_vec_scal(ctx.h, n, alpha, _dev(x), _stream(stream)))


def vec_axpby(ctx, n, alpha, x, beta, y, stream=None):
    check(ctx.lib.dmrgk_vec_axpby(ctx.h, n, alpha, _dev(x), beta, _dev(y), _stream(stream)))


def vec_scal_dev(ctx, n, alpha_dev, mode, x, y, stream=None):
    check(ctx.lib.dmrgk_vec_scal_dev(ctx.h, n, _dev(alpha_dev), mode, _dev(x), _dev(y), _stream(stream)))


def vec_residual(ctx, n, m, V, W, stride, coef, r, out, scratch, stream=None):
    check(ctx.lib.dmrgk_vec_residual(ctx.h, n, m, _dev(V), _dev(W), stride, _dev(coef), _dev(r), _dev(out),
                                     _dev(scratch), _stream(stream)))


def vec_precond(ctx, n, r, diag, theta_dev, t, stream=None):
    check(ctx.lib.dmrgk_vec_precond(ctx.h, n, _dev(r), _dev(diag), _dev(theta_dev), _dev(t), _stream(stream)))


def probe_fp64(ctx, kind, iters, sink, stream=None):
    fl = C.c_double()
    check(ctx.lib.dmrgk_probe_fp64(ctx.h, kind, iters, _dev(sink), C.byref(fl), _stream(stream)))
    return fl.value


def plan_tile_cuts(extent, tile_max=64):
    """Tile boundaries of a block dimension (host only): [0, …, extent]."""
    lib = load()
    out = np.zeros(extent // 16 + 3, np.int32)
    n = lib.dmrgk_plan_tile_cuts(int(extent), int(tile_max), out.ctypes.data, len(out))
    if n < 0:
        raise DmrgkError(n, last_error())
    return [int(x) for x in out[:n + 1]]


def plan_tile_cost(rows, cols):
    lib = load()
    c = lib.dmrgk_plan_tile_cost(int(rows), int(cols))
    if c < 0:
        raise DmrgkError(c, last_error())
    return int(c)
