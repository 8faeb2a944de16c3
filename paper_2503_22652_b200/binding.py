"""Thin ctypes binding of librchfsi.so (include/rchfsi.h): argument marshalling only.

Every step of the filter path runs in the library's CUDA kernels.  PyTorch is used for device
memory (torch tensors own the buffers whose data_ptr() crosses the C ABI) and for the stream.
There is no CPU fallback: a missing or unloadable library raises at import / first use.
"""
import ctypes as C
import os

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "librchfsi.so")

OK, EINVAL, ENOMEM, ECUDA, ENOTCONVERGED, EBREAKDOWN = range(6)
OP_DENSE, OP_CSR, OP_FE = 0, 1, 2
FP64, FP32, TF32, BF16 = 0, 1, 2, 3
METHOD_CHFSI, METHOD_RCHFSI = 0, 1
USE_FILTER, USE_RAYLEIGH_RITZ, USE_SOLVE, USE_FILTER_HOST, USE_BOUNDS, USE_FILTER_NULL_G = 1, 2, 4, 8, 16, 32
PREC = {"fp64": FP64, "fp32": FP32, "tf32": TF32, "bf16": BF16}
STATUS_NAME = {0: "OK", 1: "EINVAL", 2: "ENOMEM", 3: "ECUDA", 4: "ENOTCONVERGED", 5: "EBREAKDOWN"}


class RchfsiOperator(C.Structure):
    _fields_ = [("kind", C.c_int32), ("m", C.c_int64), ("dense", C.c_void_p), ("lda", C.c_int64),
                ("rowptr", C.c_void_p), ("colind", C.c_void_p), ("vals", C.c_void_p), ("nnz", C.c_int64),
                ("n_cells", C.c_int64), ("n_loc", C.c_int32), ("cell_shared", C.c_int32),
                ("cell_mats", C.c_void_p), ("cell_mats_f32", C.c_void_p), ("conn", C.c_void_p)]


class RchfsiOptions(C.Structure):
    _fields_ = [("apply_prec", C.c_int32), ("store_prec", C.c_int32),
                ("normalize_columns_before_rr", C.c_int32), ("adaptive_bounds", C.c_int32),
                ("noise_eps", C.c_double), ("noise_seed", C.c_uint64),
                ("allow_high_degree", C.c_int32), ("g_input_f32", C.c_int32)]


class RchfsiBounds(C.Structure):
    _fields_ = [("lam_max", C.c_double), ("lanczos_max", C.c_double), ("lanczos_theta_max", C.c_double),
                ("lanczos_theta_min", C.c_double), ("gershgorin_max", C.c_double), ("fe_cellwise_max", C.c_double),
                ("lanczos_steps", C.c_int32)]


# every symbol include/rchfsi.h declares: name -> (restype, argtypes)
SYMBOLS = {
    "rchfsi_version": (C.c_char_p, []),
    "rchfsi_default_options": (None, [C.POINTER(RchfsiOptions)]),
    "rchfsi_create": (C.c_int, [C.POINTER(C.c_void_p), C.POINTER(RchfsiOperator), C.POINTER(RchfsiOperator),
                                C.c_void_p, C.c_int32, C.POINTER(RchfsiOptions), C.c_void_p]),
    "rchfsi_destroy": (C.c_int, [C.c_void_p]),
    "rchfsi_operator_changed": (C.c_int, [C.c_void_p]),
    "rchfsi_last_error": (C.c_char_p, [C.c_void_p]),
    "rchfsi_workspace_bytes": (C.c_size_t, [C.POINTER(RchfsiOperator), C.POINTER(RchfsiOperator), C.c_int32,
                                            C.POINTER(RchfsiOptions), C.c_int32, C.c_int32]),
    "rchfsi_add_workspace": (C.c_int, [C.c_void_p, C.c_void_p, C.c_size_t]),
    "rchfsi_workspace_shortfall": (C.c_size_t, [C.c_void_p]),
    "rchfsi_workspace_used": (C.c_size_t, [C.c_void_p]),
    "rchfsi_filter": (C.c_int, [C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32,
                                C.c_double, C.c_double, C.c_double]),
    "rchfsi_filter_begin": (C.c_int, [C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32,
                                      C.c_double, C.c_double, C.c_double]),
    "rchfsi_filter_step": (C.c_int, [C.c_void_p]),
    "rchfsi_filter_end": (C.c_int, [C.c_void_p]),
    "rchfsi_filter_steps_left": (C.c_int32, [C.c_void_p]),
    "rchfsi_interface_save": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int32]),
    "rchfsi_interface_pack": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int32, C.c_int32, C.c_void_p]),
    "rchfsi_interface_apply": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int32, C.c_int32, C.c_void_p, C.c_void_p]),
    "rchfsi_filter_host": (C.c_int, [C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32,
                                     C.c_double, C.c_double, C.c_double]),
    "rchfsi_rayleigh_ritz": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]),
    "rchfsi_rotate": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p]),
    "rchfsi_solve": (C.c_int, [C.c_void_p, C.c_int32, C.c_void_p, C.c_int32, C.c_int32, C.c_double, C.c_double,
                               C.c_double, C.c_double, C.c_int32, C.c_void_p, C.c_void_p,
                               C.POINTER(C.c_int32), C.c_void_p]),
    "rchfsi_estimate_bounds": (C.c_int, [C.c_void_p, C.c_int32, C.c_int32, C.c_uint64, C.POINTER(RchfsiBounds)]),
    "rchfsi_apply": (C.c_int, [C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p]),
    "rchfsi_launch_count": (C.c_int64, [C.c_void_p]),
    "rchfsi_last_filter_step_ms": (C.c_int, [C.c_void_p, C.POINTER(C.c_float), C.POINTER(C.c_int32)]),
    "rchfsi_static_setup": (C.c_int, []),
    "rchfsi_residual_static": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64, C.c_int32, C.c_void_p,
                                         C.c_void_p, C.c_void_p]),
    "rchfsi_static_last_error": (C.c_char_p, []),
}
STATIC_MAX_N = 4096          # RCHFSI_STATIC_MAX_N

_lib = None


def load_library():
    """dlopen librchfsi.so and type every exported symbol.  Raises if the library is missing
    (build it with `python -m paper_2503_22652_b200.build`): there is no fallback path."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError("librchfsi.so is not built (%s); run python -m paper_2503_22652_b200.build"
                           % LIB_PATH)
    lib = C.CDLL(LIB_PATH, mode=C.RTLD_GLOBAL)
    for name, (res, args) in SYMBOLS.items():
        fn = getattr(lib, name)
        fn.restype = res
        fn.argtypes = args
    _lib = lib
    return lib


class RchfsiError(RuntimeError):
    def __init__(self, status, message):
        super().__init__("%s: %s" % (STATUS_NAME.get(status, status), message))
        self.status = status


def _ptr(t):
    return C.c_void_p(t.data_ptr()) if t is not None else C.c_void_p(0)


def _check_dev(t, dtype, name):
    import torch
    if not isinstance(t, torch.Tensor) or not t.is_cuda or t.dtype != dtype or not t.is_contiguous():
        raise TypeError("%s must be a contiguous CUDA tensor of %s" % (name, dtype))
    return t


def make_operator(spec, keep):
    """spec: dict(kind='dense', A=tensor) | dict(kind='csr', rowptr, colind, vals) |
    dict(kind='fe', conn, cell_mats=None, cell_mats_f32=None, shared=False, m=...)  (CUDA tensors).
    `keep` collects the tensors so they outlive the handle."""
    import torch
    op = RchfsiOperator()
    kind = spec["kind"]
    if kind == "dense":
        A = _check_dev(spec["A"], torch.float64, "A")
        op.kind, op.m, op.dense, op.lda = OP_DENSE, A.shape[0], A.data_ptr(), A.shape[1]
        keep.append(A)
    elif kind == "csr":
        rp = _check_dev(spec["rowptr"], torch.int64, "rowptr")
        ci = _check_dev(spec["colind"], torch.int32, "colind")
        va = _check_dev(spec["vals"], torch.float64, "vals")
        op.kind, op.m = OP_CSR, rp.numel() - 1
        op.rowptr, op.colind, op.vals, op.nnz = rp.data_ptr(), ci.data_ptr(), va.data_ptr(), va.numel()
        keep += [rp, ci, va]
    elif kind == "fe":
        conn = _check_dev(spec["conn"], torch.int32, "conn")
        op.kind, op.m = OP_FE, int(spec["m"])
        op.n_cells, op.n_loc = conn.shape[0], conn.shape[1]
        op.cell_shared = 1 if spec.get("shared") else 0
        op.conn = conn.data_ptr()
        keep.append(conn)
        if spec.get("cell_mats") is not None:
            cm = _check_dev(spec["cell_mats"], torch.float64, "cell_mats")
            op.cell_mats = cm.data_ptr()
            keep.append(cm)
        if spec.get("cell_mats_f32") is not None:
            cf = _check_dev(spec["cell_mats_f32"], torch.float32, "cell_mats_f32")
            op.cell_mats_f32 = cf.data_ptr()
            keep.append(cf)
    else:
        raise ValueError(kind)
    return op


class Rchfsi:
    """Handle wrapper.  Method names mirror the C entry points (rchfsi_filter -> .filter, ...).

    Device memory: the library allocates none.  `workspace=None` (default): torch tensors are handed to the handle
    on demand -- a call that returns ENOMEM has not changed any caller block, so the binding adds a segment of
    rchfsi_workspace_shortfall() bytes (torch.empty) and repeats the call.  `workspace=<uint8 CUDA tensor>`: that
    single buffer only (size it with Rchfsi.workspace_bytes); running out raises."""

    def __init__(self, A, B=None, dinv=None, block_N=1, apply_prec="fp64", store_prec="fp64",
                 normalize_columns_before_rr=True, adaptive_bounds=False, noise_eps=0.0, noise_seed=0,
                 allow_high_degree=False, g_input_f32=False, stream=None, workspace=None):
        import torch
        self.lib = load_library()
        self._keep = []
        self.opA = make_operator(A, self._keep)
        self.opB = make_operator(B, self._keep) if B is not None else None
        if dinv is not None:
            self._keep.append(_check_dev(dinv, torch.float64, "dinv"))
        opt = RchfsiOptions()
        self.lib.rchfsi_default_options(C.byref(opt))
        opt.apply_prec = PREC[apply_prec] if isinstance(apply_prec, str) else apply_prec
        opt.store_prec = PREC[store_prec] if isinstance(store_prec, str) else store_prec
        opt.normalize_columns_before_rr = int(normalize_columns_before_rr)
        opt.adaptive_bounds = int(adaptive_bounds)
        opt.noise_eps = float(noise_eps)
        opt.noise_seed = int(noise_seed)
        opt.allow_high_degree = int(allow_high_degree)
        opt.g_input_f32 = int(g_input_f32)
        self.opt = opt
        self.m, self.N = int(self.opA.m), int(block_N)
        self.stream = stream if stream is not None else torch.cuda.current_stream()
        h = C.c_void_p()
        st = self.lib.rchfsi_create(C.byref(h), C.byref(self.opA),
                                    C.byref(self.opB) if self.opB is not None else None,
                                    _ptr(dinv), self.N, C.byref(opt), C.c_void_p(self.stream.cuda_stream))
        if st == ENOMEM or st == OK:
            self.h = h
        if st != OK and st != ENOMEM:
            raise RchfsiError(st, (self.lib.rchfsi_last_error(None) or b"").decode())
        self._ws = []
        self._grow = workspace is None
        if workspace is not None:
            _check_dev(workspace, torch.uint8, "workspace")
            self.add_workspace(workspace)

    @staticmethod
    def workspace_bytes(A, B=None, block_N=1, uses=USE_FILTER, max_degree=64, **opts):
        """rchfsi_workspace_bytes for operator specs as the constructor takes them."""
        lib = load_library()
        keep = []
        opA = make_operator(A, keep)
        opB = make_operator(B, keep) if B is not None else None
        opt = RchfsiOptions()
        lib.rchfsi_default_options(C.byref(opt))
        for k, v in opts.items():
            setattr(opt, k, PREC[v] if isinstance(v, str) else int(v))
        return int(lib.rchfsi_workspace_bytes(C.byref(opA), C.byref(opB) if opB is not None else None, block_N,
                                              C.byref(opt), uses, max_degree))

    def add_workspace(self, t):
        """rchfsi_add_workspace: hand a uint8 CUDA tensor to the handle (kept alive here)."""
        st = self.lib.rchfsi_add_workspace(self.h, C.c_void_p(t.data_ptr()), t.numel())
        if st != OK:
            self._raise(st)
        self._ws.append(t)

    def workspace_used(self):
        return int(self.lib.rchfsi_workspace_used(self.h))

    def _call(self, fn, *args):
        """Call an entry point; on ENOMEM (workspace exhausted, nothing of the caller's changed) add a torch-owned
        segment of the missing size and repeat."""
        import torch
        for _attempt in range(64):     # an entry point owns a few dozen buffers at most: more retries mean a bug
            st = fn(self.h, *args)
            if st != ENOMEM or not self._grow:
                return st
            need = int(self.lib.rchfsi_workspace_shortfall(self.h))
            if need <= 0:
                return st
            # small requests share a 1 MiB segment: fewer, larger torch tensors
            self.add_workspace(torch.empty(max(need, 1 << 20), dtype=torch.uint8,
                                           device=torch.device("cuda", torch.cuda.current_device())))
        return ENOMEM

    def _raise(self, st):
        raise RchfsiError(st, (self.lib.rchfsi_last_error(self.h) or b"").decode())

    def close(self):
        if getattr(self, "h", None):
            self.lib.rchfsi_destroy(self.h)     # synchronises the stream: the segments may go after it
            self.h = None
            self._ws = []

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def operator_changed(self):
        """rchfsi_operator_changed: the caller rewrote A / dinv in place; drop the reduced-precision copies."""
        st = self.lib.rchfsi_operator_changed(self.h)
        if st != OK:
            self._raise(st)

    def _block(self, t, name):
        import torch
        _check_dev(t, torch.float64, name)
        if tuple(t.shape) != (self.m, self.N):
            raise ValueError("%s must have shape (%d, %d)" % (name, self.m, self.N))
        return t

    def filter(self, method, X, ritz, G, degree, lam_min, lam_T, lam_max):
        """rchfsi_filter: X [m][N] CUDA float64 is overwritten by the filtered block Y_p."""
        import torch
        self._block(X, "X")
        if G is not None:
            if self.opt.g_input_f32:
                _check_dev(G, torch.float32, "G")
                if tuple(G.shape) != (self.m, self.N):
                    raise ValueError("G must have shape (%d, %d)" % (self.m, self.N))
            else:
                self._block(G, "G")
        if ritz is not None:
            _check_dev(ritz, torch.float64, "ritz")
        st = self._call(self.lib.rchfsi_filter, method, _ptr(X), _ptr(ritz), _ptr(G), degree, lam_min, lam_T, lam_max)
        if st != OK:
            self._raise(st)
        return X

    # ---- step-wise filter and interface exchange (row-sharded multi-GPU filter; see sharding.py)
    def filter_begin(self, method, X, ritz, G, degree, lam_min, lam_T, lam_max):
        self._block(X, "X")
        st = self._call(self.lib.rchfsi_filter_begin, method, _ptr(X), _ptr(ritz), _ptr(G), degree, lam_min, lam_T, lam_max)
        if st != OK:
            self._raise(st)

    def filter_step(self):
        st = self._call(self.lib.rchfsi_filter_step)
        if st != OK:
            self._raise(st)

    def filter_end(self):
        st = self._call(self.lib.rchfsi_filter_end)
        if st != OK:
            self._raise(st)

    def filter_steps_left(self):
        return int(self.lib.rchfsi_filter_steps_left(self.h))

    def interface_save(self, rows):
        st = self._call(self.lib.rchfsi_interface_save, _ptr(rows), rows.numel())
        if st != OK:
            self._raise(st)

    def interface_pack(self, rows, wire, send):
        st = self._call(self.lib.rchfsi_interface_pack, _ptr(rows), rows.numel(), PREC[wire], _ptr(send))
        if st != OK:
            self._raise(st)

    def interface_apply(self, rows, wire, own, nbr):
        st = self._call(self.lib.rchfsi_interface_apply, _ptr(rows), rows.numel(), PREC[wire], _ptr(own), _ptr(nbr))
        if st != OK:
            self._raise(st)

    def filter_host(self, method, X_host, ritz_host, G_host, degree, lam_min, lam_T, lam_max):
        """rchfsi_filter_host: numpy / CPU-tensor buffers (float64, C-contiguous); X_host is
        overwritten with Y_p.  Host<->device copies happen inside the call."""
        import numpy as np

        def hp(a, name, shape, f32=False):
            if a is None:
                return C.c_void_p(0)
            if hasattr(a, "data_ptr"):      # CPU torch tensor
                import torch
                ok = (not a.is_cuda and a.is_contiguous() and tuple(a.shape) == shape
                      and a.dtype == (torch.float32 if f32 else torch.float64))
                ptr = a.data_ptr()
            else:
                ok = (isinstance(a, np.ndarray) and a.flags["C_CONTIGUOUS"] and a.shape == shape
                      and a.dtype == (np.float32 if f32 else np.float64))
                ptr = a.ctypes.data if ok else 0
            if not ok:
                raise TypeError("%s must be a C-contiguous host array of shape %s, %s" %
                                (name, shape, "float32" if f32 else "float64"))
            return C.c_void_p(ptr)
        blk = (self.m, self.N)
        st = self._call(self.lib.rchfsi_filter_host, method, hp(X_host, "X_host", blk), hp(ritz_host, "ritz_host", (self.N,)),
                        hp(G_host, "G_host", blk, f32=bool(self.opt.g_input_f32)), degree, lam_min, lam_T, lam_max)
        if st != OK:
            self._raise(st)
        return X_host

    def rayleigh_ritz(self, Y, want_G=True):
        """rchfsi_rayleigh_ritz: returns (ritz, X (= Y overwritten), G or None, resnorm)."""
        import torch
        self._block(Y, "Y")
        ritz = torch.empty(self.N, dtype=torch.float64, device=Y.device)
        res = torch.empty(self.N, dtype=torch.float64, device=Y.device)
        G = torch.empty_like(Y) if want_G else None
        st = self._call(self.lib.rchfsi_rayleigh_ritz, _ptr(Y), _ptr(ritz), _ptr(G), _ptr(res))
        if st != OK:
            self._raise(st)
        return ritz, Y, G, res

    def rotate(self, Y, E_colmajor):
        """rchfsi_rotate: Y <- Y E in place; E_colmajor is a contiguous [N][N] CUDA tensor holding E COLUMN-major
        (i.e. E.T.contiguous() of a row-major E)."""
        import torch
        self._block(Y, "Y")
        _check_dev(E_colmajor, torch.float64, "E")
        if tuple(E_colmajor.shape) != (self.N, self.N):
            raise ValueError("E must be [N][N]")
        st = self._call(self.lib.rchfsi_rotate, _ptr(Y), _ptr(E_colmajor))
        if st != OK:
            self._raise(st)
        return Y

    def solve(self, method, X, n_wanted, degree, lam_min, lam_T, lam_max, tol=1e-8, max_iter=50,
              raise_on_not_converged=False):
        """rchfsi_solve: returns dict(evals, resnorm, iters, history, converged); X overwritten."""
        import numpy as np
        self._block(X, "X")
        evals = np.empty(self.N)
        res = np.empty(self.N)
        hist = np.full(max_iter, np.nan)
        iters = C.c_int32(0)
        st = self._call(self.lib.rchfsi_solve, method, _ptr(X), n_wanted, degree, lam_min, lam_T, lam_max, tol,
                        max_iter, C.c_void_p(evals.ctypes.data), C.c_void_p(res.ctypes.data),
                        C.byref(iters), C.c_void_p(hist.ctypes.data))
        if st not in (OK, ENOTCONVERGED) or (st == ENOTCONVERGED and raise_on_not_converged):
            self._raise(st)
        return dict(evals=evals, resnorm=res, iters=iters.value, history=hist[:iters.value],
                    converged=(st == OK))

    def estimate_bounds(self, lanczos_steps=20, fe_cell_stride=0, seed=0):
        """rchfsi_estimate_bounds: dict of the estimates (lam_max = the recommended upper bound)."""
        b = RchfsiBounds()
        st = self._call(self.lib.rchfsi_estimate_bounds, lanczos_steps, fe_cell_stride, seed, C.byref(b))
        if st != OK:
            self._raise(st)
        return {name: getattr(b, name) for name, _ in RchfsiBounds._fields_}

    def apply(self, which, V):
        """rchfsi_apply: exact FP64 A V (which=0) or B V (which=1)."""
        import torch
        self._block(V, "V")
        out = torch.empty_like(V)
        st = self._call(self.lib.rchfsi_apply, which, _ptr(V), _ptr(out))
        if st != OK:
            self._raise(st)
        return out

    def launch_count(self):
        return int(self.lib.rchfsi_launch_count(self.h))

    def last_filter_step_ms(self):
        ms, n = C.c_float(0), C.c_int32(0)
        st = self.lib.rchfsi_last_filter_step_ms(self.h, C.byref(ms), C.byref(n))
        if st != OK:
            self._raise(st)
        return ms.value, n.value


# ------------------------------------------------------------------------- allocation-free entry point
def static_setup():
    """rchfsi_static_setup on the current device (needed before a CUDA graph capture; otherwise lazy)."""
    lib = load_library()
    st = lib.rchfsi_static_setup()
    if st != OK:
        raise RchfsiError(st, (lib.rchfsi_static_last_error() or b"").decode())


def residual_static(AX, BX, ritz, G_out=None, resnorm_out=None, stream=None):
    """rchfsi_residual_static: G_out = AX - BX diag(ritz), resnorm_out[j] = ||G_j||_2, written into the CALLER's
    tensors ([m][N] / [N], FP64, contiguous, CUDA); the library allocates nothing (static device scratch, N <= 4096).
    Marshalling only: no tensor is created here."""
    import torch
    lib = load_library()
    _check_dev(AX, torch.float64, "AX")
    _check_dev(BX, torch.float64, "BX")
    _check_dev(ritz, torch.float64, "ritz")
    if AX.dim() != 2 or BX.shape != AX.shape or ritz.numel() != AX.shape[1]:
        raise ValueError("AX, BX must be [m][N] and ritz [N]")
    if G_out is not None and (_check_dev(G_out, torch.float64, "G_out").shape != AX.shape):
        raise ValueError("G_out must be [m][N]")
    if resnorm_out is not None and _check_dev(resnorm_out, torch.float64, "resnorm_out").numel() != AX.shape[1]:
        raise ValueError("resnorm_out must be [N]")
    s = torch.cuda.current_stream().cuda_stream if stream is None else int(stream)
    st = lib.rchfsi_residual_static(_ptr(AX), _ptr(BX), _ptr(ritz), AX.shape[0], AX.shape[1], _ptr(G_out),
                                    _ptr(resnorm_out), C.c_void_p(s))
    if st != OK:
        raise RchfsiError(st, (lib.rchfsi_static_last_error() or b"").decode())
