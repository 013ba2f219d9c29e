"""Thin ctypes binding of libcola.so (include/cola.h): argument marshalling only.

Every step of the hot path runs in the CUDA library; torch is used for device memory and streams.
There is no CPU fallback: if libcola.so is missing or cannot be loaded, importing this module raises.
"""
from __future__ import annotations

import ctypes
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libcola.so")   # the in-tree library, nothing else: no environment variables are read

COLA_OK, COLA_EINVAL, COLA_ECUDA, COLA_ENOTREADY, COLA_ENOCONV, COLA_ENOMEM = range(6)
COLA_F64, COLA_F32, COLA_F32_H16, COLA_F32_R8 = 0, 1, 2, 3
COLA_EVEN, COLA_ODD = 0, 1
COLA_FEAT_FULL_M, COLA_FEAT_H16, COLA_FEAT_R8, COLA_FEAT_A72, COLA_FEAT_ALL = 1, 2, 4, 8, 15
COLA_CGNR, COLA_BICGSTAB = 0, 1
_METHOD = {"cgnr": COLA_CGNR, "bicgstab": COLA_BICGSTAB, COLA_CGNR: COLA_CGNR, COLA_BICGSTAB: COLA_BICGSTAB}
STATUS_NAMES = {0: "COLA_OK", 1: "COLA_EINVAL", 2: "COLA_ECUDA", 3: "COLA_ENOTREADY", 4: "COLA_ENOCONV", 5: "COLA_ENOMEM"}

EXPORTS = [
    "cola_create", "cola_destroy", "cola_last_error", "cola_set_stream", "cola_spinor_bytes",
    "cola_workspace_bytes", "cola_set_workspace", "cola_gauge_upload", "cola_gauge_upload_dev",
    "cola_gauge_info", "cola_clover_unpack", "cola_spinor_pack", "cola_spinor_unpack",
    "cola_spinor_convert", "cola_dslash_apply", "cola_fermion_matrix_apply", "cola_schur_apply",
    "cola_cg_solve", "cola_dslash_apply_host", "cola_fermion_matrix_apply_host", "cola_cg_solve_host",
    "cola_launch_count",
    "cola_mrhs_workspace_bytes", "cola_set_mrhs_workspace", "cola_dslash_apply_mrhs", "cola_fermion_matrix_apply_mrhs",
    "cola_schur_apply_mrhs", "cola_cg_solve_mrhs", "cola_set_l2_budget", "cola_selftest_host", "cola_cg_solve_history", "cola_profile_kernel", "cola_profile_result",
    "cola_set_features", "cola_clover_info", "cola_set_staging", "cola_set_compact", "cola_gauge_info_r8",
    "cola_eig_workspace_bytes", "cola_eig_lowest", "cola_cg_solve_deflated",
    "cola_spinor_norm2", "cola_spinor_norm2_static",
]


class ColaParams(ctypes.Structure):
    _fields_ = [
        ("dims", ctypes.c_int * 4), ("kappa", ctypes.c_double), ("csw", ctypes.c_double),
        ("bc", ctypes.c_int * 4), ("compress12", ctypes.c_int), ("trace_sub", ctypes.c_int),
        ("device", ctypes.c_int), ("stream", ctypes.c_void_p),
    ]


class ColaSolveParams(ctypes.Structure):
    _fields_ = [("tol", ctypes.c_double), ("max_iter", ctypes.c_int), ("even_odd", ctypes.c_int),
                ("mixed", ctypes.c_int), ("delta", ctypes.c_double), ("method", ctypes.c_int)]


class ColaSolveInfo(ctypes.Structure):
    _fields_ = [("iters", ctypes.c_int), ("reliable_updates", ctypes.c_int),
                ("iterated_residual", ctypes.c_double), ("true_residual", ctypes.c_double),
                ("seconds", ctypes.c_double), ("op_flops", ctypes.c_double)]


class ColaEigParams(ctypes.Structure):
    _fields_ = [("n_ev", ctypes.c_int), ("n_kr", ctypes.c_int), ("tol", ctypes.c_double), ("max_restarts", ctypes.c_int),
                ("cheb_order", ctypes.c_int), ("cheb_lo", ctypes.c_double), ("cheb_hi", ctypes.c_double), ("seed", ctypes.c_uint)]


class ColaEigInfo(ctypes.Structure):
    _fields_ = [("restarts", ctypes.c_int), ("op_applications", ctypes.c_int), ("cheb_lo", ctypes.c_double),
                ("cheb_hi", ctypes.c_double), ("seconds", ctypes.c_double)]


def lib_path() -> str:
    return _LIB_PATH


def _load():
    if not os.path.exists(_LIB_PATH):
        raise ImportError(
            f"{_LIB_PATH} is missing: build it with `python -m paper_2302_00850_b200.build` "
            "(there is no CPU fallback for the COLA hot path)")
    lib = ctypes.CDLL(_LIB_PATH)
    vp, ci, cd = ctypes.c_void_p, ctypes.c_int, ctypes.c_double
    lib.cola_create.argtypes = [ctypes.POINTER(vp), ctypes.POINTER(ColaParams)]
    lib.cola_destroy.argtypes = [vp]
    lib.cola_last_error.argtypes = [vp]
    lib.cola_last_error.restype = ctypes.c_char_p
    lib.cola_set_stream.argtypes = [vp, vp]
    lib.cola_set_l2_budget.argtypes = [vp, ctypes.c_size_t]
    lib.cola_selftest_host.argtypes = [ctypes.c_char_p, ctypes.c_size_t]
    lib.cola_profile_kernel.argtypes = [vp, ci]
    lib.cola_profile_result.argtypes = [vp, ctypes.POINTER(cd), ctypes.POINTER(ci), ctypes.POINTER(ci)]
    lib.cola_cg_solve_history.argtypes = [vp, ctypes.POINTER(ColaSolveParams), vp, vp, ctypes.POINTER(ColaSolveInfo), ctypes.POINTER(cd), ci,
                                          ctypes.POINTER(ci), ci]
    lib.cola_set_features.argtypes = [vp, ctypes.c_uint]
    lib.cola_set_staging.argtypes = [vp, ci]
    lib.cola_set_compact.argtypes = [vp, ci]
    lib.cola_gauge_info_r8.argtypes = [vp, ctypes.POINTER(cd)]
    lib.cola_eig_workspace_bytes.argtypes = [vp, ctypes.POINTER(ColaEigParams)]
    lib.cola_eig_workspace_bytes.restype = ctypes.c_size_t
    lib.cola_eig_lowest.argtypes = [vp, ctypes.POINTER(ColaEigParams), vp, ctypes.c_size_t, ctypes.POINTER(cd), ctypes.POINTER(cd), vp,
                                    ctypes.POINTER(ColaEigInfo)]
    lib.cola_cg_solve_deflated.argtypes = [vp, ctypes.POINTER(ColaSolveParams), vp, vp, ctypes.POINTER(ColaSolveInfo), vp, ctypes.POINTER(cd), ci]
    lib.cola_clover_info.argtypes = [vp, ctypes.POINTER(cd)]
    lib.cola_spinor_norm2.argtypes = [vp, ci, vp, ci, vp]
    lib.cola_spinor_norm2_static.argtypes = [ci, vp, ci, vp, ctypes.c_size_t, vp]
    lib.cola_spinor_bytes.argtypes = [vp, ci, ci]
    lib.cola_spinor_bytes.restype = ctypes.c_size_t
    lib.cola_workspace_bytes.argtypes = [vp]
    lib.cola_workspace_bytes.restype = ctypes.c_size_t
    lib.cola_set_workspace.argtypes = [vp, vp, ctypes.c_size_t]
    lib.cola_gauge_upload.argtypes = [vp, vp]
    lib.cola_gauge_upload_dev.argtypes = [vp, vp]
    lib.cola_gauge_info.argtypes = [vp, ctypes.POINTER(cd)]
    lib.cola_clover_unpack.argtypes = [vp, ci, vp]
    lib.cola_spinor_pack.argtypes = [vp, ci, vp, vp]
    lib.cola_spinor_unpack.argtypes = [vp, ci, vp, vp]
    lib.cola_spinor_convert.argtypes = [vp, ci, vp, vp, ci]
    lib.cola_dslash_apply.argtypes = [vp, ci, ci, vp, vp]
    lib.cola_fermion_matrix_apply.argtypes = [vp, ci, ci, vp, vp]
    lib.cola_schur_apply.argtypes = [vp, ci, ci, vp, vp]
    lib.cola_cg_solve.argtypes = [vp, ctypes.POINTER(ColaSolveParams), vp, vp, ctypes.POINTER(ColaSolveInfo)]
    lib.cola_dslash_apply_host.argtypes = [vp, ci, ci, vp, vp]
    lib.cola_fermion_matrix_apply_host.argtypes = [vp, ci, ci, vp, vp]
    lib.cola_cg_solve_host.argtypes = [vp, ctypes.POINTER(ColaSolveParams), vp, vp, ctypes.POINTER(ColaSolveInfo)]
    lib.cola_launch_count.argtypes = [vp]
    lib.cola_launch_count.restype = ctypes.c_ulonglong
    lib.cola_mrhs_workspace_bytes.argtypes = [vp, ci, ci]
    lib.cola_mrhs_workspace_bytes.restype = ctypes.c_size_t
    lib.cola_set_mrhs_workspace.argtypes = [vp, vp, ctypes.c_size_t, ci]
    lib.cola_dslash_apply_mrhs.argtypes = [vp, ci, ci, ci, vp, vp]
    lib.cola_fermion_matrix_apply_mrhs.argtypes = [vp, ci, ci, ci, vp, vp]
    lib.cola_schur_apply_mrhs.argtypes = [vp, ci, ci, ci, vp, vp]
    lib.cola_cg_solve_mrhs.argtypes = [vp, ctypes.POINTER(ColaSolveParams), ci, vp, vp, ctypes.POINTER(ColaSolveInfo)]
    for name in EXPORTS:
        fn = getattr(lib, name)
        if name not in ("cola_last_error", "cola_spinor_bytes", "cola_workspace_bytes", "cola_launch_count", "cola_mrhs_workspace_bytes",
                        "cola_eig_workspace_bytes"):
            fn.restype = ci
    return lib


_lib = _load()


def selftest_host() -> str:
    """cola_selftest_host: host-side index machinery (no GPU).  Returns "ok" or raises with the first failure."""
    buf = ctypes.create_string_buffer(256)
    st = _lib.cola_selftest_host(buf, 256)
    if st != COLA_OK:
        raise RuntimeError(buf.value.decode())
    return buf.value.decode()


COLA_STATIC_SCRATCH_BYTES = 16384
COLA_STATIC_MAX_SITES = 1 << 25


def spinor_norm2_static(v: torch.Tensor, out: torch.Tensor | None = None, stream=None) -> torch.Tensor:
    """cola_spinor_norm2_static: |v|^2 of an internal spinor buffer without a context, a workspace or any allocation
    inside the library (its reduction scratch is a fixed 16 KB array in the library's device image, shared by every
    call in the process).  For callers that own device pointers but may not allocate.  `out`: a CUDA float64 tensor of
    one element to receive the result (allocated here with torch when omitted -- pass it if even that is not allowed).
    At most COLA_STATIC_MAX_SITES sites; the first call on a device should happen outside stream capture; calls that
    overlap on one GPU race on the shared scratch."""
    if not (v.is_cuda and v.is_contiguous() and v.dtype in (torch.float64, torch.float32)) or v.numel() % 24:
        raise ValueError("v must be a contiguous CUDA float64 / float32 internal buffer (24 reals per site)")
    if out is None:
        out = torch.empty(1, dtype=torch.float64, device=v.device)
    if not (out.is_cuda and out.dtype == torch.float64 and out.numel() >= 1 and out.device == v.device):
        raise ValueError("out must be a CUDA float64 tensor on v's device")
    if stream is None:
        stream = torch.cuda.current_stream(v.device).cuda_stream
    st = _lib.cola_spinor_norm2_static(v.device.index, ctypes.c_void_p(stream or 0), _PREC[v.dtype], ctypes.c_void_p(v.data_ptr()),
                                       v.numel() // 24, ctypes.c_void_p(out.data_ptr()))
    if st != COLA_OK:
        raise ColaError(st, _lib.cola_last_error(None).decode())
    return out


class ColaError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"{STATUS_NAMES.get(status, status)}: {message}")
        self.status = status


_PREC = {torch.float64: COLA_F64, torch.float32: COLA_F32, torch.complex128: COLA_F64, torch.complex64: COLA_F32,
         "f64": COLA_F64, "f32": COLA_F32, COLA_F64: COLA_F64, COLA_F32: COLA_F32}
_REAL = {COLA_F64: torch.float64, COLA_F32: torch.float32}
_CPLX = {COLA_F64: torch.complex128, COLA_F32: torch.complex64}


class Cola:
    """One lattice context.  Method names mirror the C entry points (cola_<name>)."""

    def __init__(self, dims, kappa, csw, bc=(1, 1, 1, -1), compress12=True, trace_sub=True, device=0, stream=None, features=None):
        self.dims = tuple(int(d) for d in dims)
        self.device = torch.device("cuda", device)
        self._h = ctypes.c_void_p()
        self._ws = None
        self._mws = None
        self._mws_nrhs = 0
        self._mws_solver = False
        p = ColaParams()
        p.dims[:] = self.dims
        p.kappa, p.csw = float(kappa), float(csw)
        p.bc[:] = [int(b) for b in bc]
        p.compress12, p.trace_sub, p.device = int(bool(compress12)), int(bool(trace_sub)), int(device)
        if stream is None and torch.cuda.is_available():
            stream = torch.cuda.current_stream(self.device).cuda_stream
        p.stream = ctypes.c_void_p(stream or 0)
        st = _lib.cola_create(ctypes.byref(self._h), ctypes.byref(p))
        if st != COLA_OK:
            raise ColaError(st, _lib.cola_last_error(None).decode())
        lx, ly, lz, lt = self.dims
        self.V = lx * ly * lz * lt
        self.Vh = self.V // 2
        self.kappa, self.csw = float(kappa), float(csw)
        if features is not None:
            self.set_features(features)

    # ---- plumbing
    def _ck(self, st, ok=(COLA_OK,)):
        if st not in ok:
            raise ColaError(st, _lib.cola_last_error(self._h).decode())
        return st

    def close(self):
        if self._h:
            _lib.cola_destroy(self._h)
            self._h = ctypes.c_void_p()
            self._ws = None
            self._mws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def profile_kernel(self, enable: bool = True):
        """Bracket later launches of the fused dslash+clover+xpay kernel (fp32 / 16-bit) with CUDA event pairs."""
        self._ck(_lib.cola_profile_kernel(self._h, int(bool(enable))))

    def profile_result(self):
        """(average ms of the launches that did work, their count, speculative launches that returned at once)."""
        ms, n, sk = ctypes.c_double(), ctypes.c_int(), ctypes.c_int()
        self._ck(_lib.cola_profile_result(self._h, ctypes.byref(ms), ctypes.byref(n), ctypes.byref(sk)))
        return ms.value, n.value, sk.value

    def set_l2_budget(self, nbytes: int = 0):
        """Bytes of L2 the sweep order counts on for neighbour reuse (0: default 40 MB); tuning only, results unchanged."""
        self._ck(_lib.cola_set_l2_budget(self._h, int(nbytes)))

    def set_staging(self, mode: int):
        """0: neighbour spinors through L1; 1: staged in shared memory per 4-D tile (fp32 / 16-bit single-rhs kernels)."""
        self._ck(_lib.cola_set_staging(self._h, int(mode)))

    def set_compact(self, mask: int):
        """bit 0: COLA_F32_R8 reads the 8-real links; bit 1: the fp32 operators read A in its 48-real form (else 72 reals)."""
        self._ck(_lib.cola_set_compact(self._h, int(mask)))

    def gauge_info_r8(self) -> float:
        """Smallest |U00| over the links of the last upload (COLA_F32_R8 needs >= 0.1)."""
        v = ctypes.c_double()
        self._ck(_lib.cola_gauge_info_r8(self._h, ctypes.byref(v)))
        return v.value

    def set_features(self, features: int):
        """COLA_FEAT_* parts of the workspace to carve; call before set_workspace / gauge_upload."""
        self._ck(_lib.cola_set_features(self._h, int(features)))
        self._ws = None

    def clover_info(self) -> float:
        """Smallest Gauss-Jordan pivot of the 6x6 inverses of the last upload."""
        v = ctypes.c_double()
        self._ck(_lib.cola_clover_info(self._h, ctypes.byref(v)))
        return v.value

    def set_stream(self, stream):
        self._ck(_lib.cola_set_stream(self._h, ctypes.c_void_p(stream)))

    def spinor_bytes(self, prec, full=True) -> int:
        return int(_lib.cola_spinor_bytes(self._h, _PREC[prec], int(full)))

    def workspace_bytes(self) -> int:
        return int(_lib.cola_workspace_bytes(self._h))

    def set_workspace(self, tensor: torch.Tensor | None = None):
        """Lend a device buffer to the context (allocated here with torch if not given)."""
        if tensor is None:
            tensor = torch.empty(self.workspace_bytes(), dtype=torch.uint8, device=self.device)
        self._ck(_lib.cola_set_workspace(self._h, ctypes.c_void_p(tensor.data_ptr()), tensor.numel() * tensor.element_size()))
        self._ws = tensor
        return tensor

    def launch_count(self) -> int:
        return int(_lib.cola_launch_count(self._h))

    # ---- internal buffers (torch owns the memory; shapes mirror the SoA layout)
    def empty_internal(self, prec, full=True) -> torch.Tensor:
        pr = _PREC[prec]
        n = 2 if pr == COLA_F64 else 4
        shape = (2, 24 // n, self.Vh, n) if full else (24 // n, self.Vh, n)
        return torch.empty(shape, dtype=_REAL[pr], device=self.device)

    # ---- H0-H2
    def gauge_upload(self, links: torch.Tensor):
        """links: complex128 [t][z][y][x][4][3][3]; a CPU tensor goes through cola_gauge_upload,
        a CUDA tensor through cola_gauge_upload_dev."""
        if self._ws is None:
            self.set_workspace()
        if links.dtype != torch.complex128 or links.numel() != self.V * 36:
            raise ValueError("links must be complex128 with 4*V*9 entries")
        links = links.contiguous()
        if links.is_cuda:
            self._ck(_lib.cola_gauge_upload_dev(self._h, ctypes.c_void_p(links.data_ptr())))
        else:
            self._ck(_lib.cola_gauge_upload(self._h, ctypes.c_void_p(links.data_ptr())))

    def gauge_upload_dev(self, links: torch.Tensor):
        assert links.is_cuda
        self.gauge_upload(links)

    def gauge_info(self) -> float:
        v = ctypes.c_double()
        self._ck(_lib.cola_gauge_info(self._h, ctypes.byref(v)))
        return v.value

    def clover_unpack(self, which: int) -> torch.Tensor:
        lx, ly, lz, lt = self.dims
        out = torch.empty((lt, lz, ly, lx, 12, 12), dtype=torch.complex128, device=self.device)
        self._ck(_lib.cola_clover_unpack(self._h, int(which), ctypes.c_void_p(out.data_ptr())))
        return out

    # ---- layout
    def spinor_pack(self, canon: torch.Tensor) -> torch.Tensor:
        pr = _PREC[canon.dtype]
        canon = canon.contiguous()
        assert canon.is_cuda and canon.numel() == self.V * 12
        out = self.empty_internal(pr, full=True)
        self._ck(_lib.cola_spinor_pack(self._h, pr, ctypes.c_void_p(canon.data_ptr()), ctypes.c_void_p(out.data_ptr())))
        return out

    def spinor_unpack(self, internal: torch.Tensor) -> torch.Tensor:
        pr = _PREC[internal.dtype]
        assert internal.is_cuda and internal.is_contiguous() and internal.numel() == self.V * 24
        lx, ly, lz, lt = self.dims
        out = torch.empty((lt, lz, ly, lx, 4, 3), dtype=_CPLX[pr], device=self.device)
        self._ck(_lib.cola_spinor_unpack(self._h, pr, ctypes.c_void_p(internal.data_ptr()), ctypes.c_void_p(out.data_ptr())))
        return out

    def spinor_convert(self, src: torch.Tensor, dst_prec) -> torch.Tensor:
        dp = _PREC[dst_prec]
        assert src.is_cuda and src.is_contiguous()
        full = src.dim() == 4
        out = self.empty_internal(dp, full=full)
        self._ck(_lib.cola_spinor_convert(self._h, dp, ctypes.c_void_p(src.data_ptr()), ctypes.c_void_p(out.data_ptr()), 2 if full else 1))
        return out

    def spinor_norm2(self, v: torch.Tensor, out: torch.Tensor | None = None) -> torch.Tensor:
        """|v|^2 (fp64, deterministic) of a half-lattice or full internal buffer; returns a CUDA float64 tensor of one element."""
        assert v.is_cuda and v.is_contiguous() and v.numel() in (self.Vh * 24, self.V * 24)
        if out is None:
            out = torch.empty(1, dtype=torch.float64, device=self.device)
        self._ck(_lib.cola_spinor_norm2(self._h, _PREC[v.dtype], ctypes.c_void_p(v.data_ptr()), v.numel() // (self.Vh * 24), ctypes.c_void_p(out.data_ptr())))
        return out

    # ---- H3-H8.  fp32 tensors only: h16=True (or fmt="h16") selects COLA_F32_H16, the operator that reads 16-bit links and
    # fp16 clover; fmt="r8" selects COLA_F32_R8 (8-real links, 48-real A)
    @staticmethod
    def _op_prec(t: torch.Tensor, h16: bool, fmt=None) -> int:
        pr = _PREC[t.dtype]
        if fmt not in (None, "h16", "r8"):
            raise ValueError("fmt must be None, 'h16' or 'r8'")
        if h16 or fmt is not None:
            if pr != COLA_F32:
                raise ValueError("h16 / r8 operators take fp32 spinors")
            return COLA_F32_R8 if fmt == "r8" else COLA_F32_H16
        return pr

    def dslash_apply(self, out_parity: int, inp: torch.Tensor, out: torch.Tensor | None = None, h16=False, fmt=None) -> torch.Tensor:
        pr = self._op_prec(inp, h16, fmt)
        assert inp.is_cuda and inp.is_contiguous() and inp.numel() == self.Vh * 24
        if out is None:
            out = self.empty_internal(inp.dtype, full=False)
        self._ck(_lib.cola_dslash_apply(self._h, pr, int(out_parity), ctypes.c_void_p(inp.data_ptr()), ctypes.c_void_p(out.data_ptr())))
        return out

    def fermion_matrix_apply(self, inp: torch.Tensor, dagger=False, out: torch.Tensor | None = None, h16=False, fmt=None) -> torch.Tensor:
        pr = self._op_prec(inp, h16, fmt)
        assert inp.is_cuda and inp.is_contiguous() and inp.numel() == self.V * 24
        if out is None:
            out = self.empty_internal(inp.dtype, full=True)
        self._ck(_lib.cola_fermion_matrix_apply(self._h, pr, int(bool(dagger)), ctypes.c_void_p(inp.data_ptr()), ctypes.c_void_p(out.data_ptr())))
        return out

    def schur_apply(self, inp: torch.Tensor, dagger=False, out: torch.Tensor | None = None, h16=False, fmt=None) -> torch.Tensor:
        pr = self._op_prec(inp, h16, fmt)
        assert inp.is_cuda and inp.is_contiguous() and inp.numel() == self.Vh * 24
        if out is None:
            out = self.empty_internal(inp.dtype, full=False)
        self._ck(_lib.cola_schur_apply(self._h, pr, int(bool(dagger)), ctypes.c_void_p(inp.data_ptr()), ctypes.c_void_p(out.data_ptr())))
        return out

    # ---- H9-H12
    @staticmethod
    def _solve_params(tol, max_iter, even_odd, mixed, delta, method="cgnr"):
        sp = ColaSolveParams()
        sp.tol, sp.max_iter, sp.even_odd, sp.mixed, sp.delta = float(tol), int(max_iter), int(bool(even_odd)), int(mixed), float(delta)
        sp.method = _METHOD[method]
        return sp

    @staticmethod
    def _info_dict(info, st):
        return dict(iters=info.iters, reliable_updates=info.reliable_updates, iterated_residual=info.iterated_residual,
                    true_residual=info.true_residual, seconds=info.seconds, op_flops=info.op_flops, converged=(st == COLA_OK))

    def cg_solve(self, b: torch.Tensor, tol=1e-10, max_iter=20000, even_odd=True, mixed=False, delta=0.1, x: torch.Tensor | None = None, method="cgnr"):
        """b: canonical complex128 [t][z][y][x][4][3].  A CUDA tensor goes through cola_cg_solve, a CPU
        tensor (ideally pinned) through cola_cg_solve_host.  Returns (x, info dict)."""
        assert b.dtype == torch.complex128 and b.numel() == self.V * 12
        b = b.contiguous()
        if x is None:
            x = torch.empty_like(b, pin_memory=True) if not b.is_cuda else torch.empty_like(b)
        sp = self._solve_params(tol, max_iter, even_odd, mixed, delta, method)
        info = ColaSolveInfo()
        fn = _lib.cola_cg_solve if b.is_cuda else _lib.cola_cg_solve_host
        st = fn(self._h, ctypes.byref(sp), ctypes.c_void_p(b.data_ptr()), ctypes.c_void_p(x.data_ptr()), ctypes.byref(info))
        self._ck(st, ok=(COLA_OK, COLA_ENOCONV))
        return x, self._info_dict(info, st)

    def cg_solve_history(self, b: torch.Tensor, tol=1e-10, max_iter=20000, even_odd=True, mixed=False, delta=0.1, hist_len=4096, method="cgnr"):
        """cg_solve on a device source that also returns the residual history |r_{k+1}|/|b| of the recurrence."""
        assert b.is_cuda and b.dtype == torch.complex128 and b.numel() == self.V * 12
        b = b.contiguous()
        x = torch.empty_like(b)
        sp = self._solve_params(tol, max_iter, even_odd, mixed, delta, method)
        info = ColaSolveInfo()
        hist = (ctypes.c_double * hist_len)()
        upd = (ctypes.c_int * 256)()
        st = _lib.cola_cg_solve_history(self._h, ctypes.byref(sp), ctypes.c_void_p(b.data_ptr()), ctypes.c_void_p(x.data_ptr()), ctypes.byref(info),
                                        hist, hist_len, upd, 256)
        self._ck(st, ok=(COLA_OK, COLA_ENOCONV))
        d = self._info_dict(info, st)
        d["history"] = [hist[k] for k in range(min(info.iters, hist_len))]
        d["update_iters"] = [upd[k] for k in range(min(info.reliable_updates, 256))]
        return x, d

    def cg_solve_host(self, b: torch.Tensor, **kw):
        assert not b.is_cuda
        return self.cg_solve(b, **kw)

    def dslash_apply_host(self, out_parity: int, inp: torch.Tensor, out: torch.Tensor | None = None) -> torch.Tensor:
        pr = _PREC[inp.dtype]
        assert not inp.is_cuda and inp.is_contiguous() and inp.numel() == self.V * 12
        if out is None:
            out = torch.empty_like(inp, pin_memory=True)
        self._ck(_lib.cola_dslash_apply_host(self._h, pr, int(out_parity), ctypes.c_void_p(inp.data_ptr()), ctypes.c_void_p(out.data_ptr())))
        return out

    def fermion_matrix_apply_host(self, inp: torch.Tensor, dagger=False, out: torch.Tensor | None = None) -> torch.Tensor:
        pr = _PREC[inp.dtype]
        assert not inp.is_cuda and inp.is_contiguous() and inp.numel() == self.V * 12
        if out is None:
            out = torch.empty_like(inp, pin_memory=True)
        self._ck(_lib.cola_fermion_matrix_apply_host(self._h, pr, int(bool(dagger)), ctypes.c_void_p(inp.data_ptr()), ctypes.c_void_p(out.data_ptr())))
        return out

    # ---- low modes of S^+ S and the deflated start
    @staticmethod
    def _eig_params(n_ev, n_kr, tol, max_restarts, cheb_order, cheb_lo, cheb_hi, seed):
        ep = ColaEigParams()
        ep.n_ev, ep.n_kr, ep.tol, ep.max_restarts = int(n_ev), int(n_kr), float(tol), int(max_restarts)
        ep.cheb_order, ep.cheb_lo, ep.cheb_hi, ep.seed = int(cheb_order), float(cheb_lo), float(cheb_hi), int(seed)
        return ep

    def eig_workspace_bytes(self, n_ev, n_kr=0) -> int:
        ep = self._eig_params(n_ev, n_kr, 0, 0, 0, 0, 0, 0)
        return int(_lib.cola_eig_workspace_bytes(self._h, ctypes.byref(ep)))

    def eig_lowest(self, n_ev, n_kr=0, tol=0.0, max_restarts=0, cheb_order=0, cheb_lo=0.0, cheb_hi=0.0, seed=0):
        """The n_ev smallest eigenpairs of S^+ S.  Returns (evals list, evecs tensor (n_ev, 12, Vh, 2) fp64 internal even
        half-lattice vectors, info dict with the true residuals)."""
        ep = self._eig_params(n_ev, n_kr, tol, max_restarts, cheb_order, cheb_lo, cheb_hi, seed)
        nb = int(_lib.cola_eig_workspace_bytes(self._h, ctypes.byref(ep)))
        if nb == 0:
            raise ValueError("n_ev must be 1..32")
        work = torch.empty(nb, dtype=torch.uint8, device=self.device)
        evecs = torch.empty((int(n_ev), 12, self.Vh, 2), dtype=torch.float64, device=self.device)
        ev, rs = (ctypes.c_double * n_ev)(), (ctypes.c_double * n_ev)()
        info = ColaEigInfo()
        st = _lib.cola_eig_lowest(self._h, ctypes.byref(ep), ctypes.c_void_p(work.data_ptr()), nb, ev, rs, ctypes.c_void_p(evecs.data_ptr()),
                                  ctypes.byref(info))
        self._ck(st, ok=(COLA_OK, COLA_ENOCONV))
        return list(ev), evecs, dict(residuals=list(rs), restarts=info.restarts, op_applications=info.op_applications, cheb_lo=info.cheb_lo,
                                     cheb_hi=info.cheb_hi, seconds=info.seconds, converged=(st == COLA_OK))

    def cg_solve_deflated(self, b: torch.Tensor, evals, evecs: torch.Tensor, tol=1e-10, max_iter=20000, mixed=True, delta=0.1):
        """cg_solve (even-odd CGNR) started from the guess deflated with eigenpairs of S^+ S (eig_lowest's output)."""
        assert b.is_cuda and b.dtype == torch.complex128 and b.numel() == self.V * 12
        assert evecs.is_cuda and evecs.is_contiguous() and evecs.dtype == torch.float64 and evecs.numel() == len(evals) * self.Vh * 24
        b = b.contiguous()
        x = torch.empty_like(b)
        sp = self._solve_params(tol, max_iter, True, mixed, delta)
        info = ColaSolveInfo()
        ev = (ctypes.c_double * len(evals))(*[float(v) for v in evals])
        st = _lib.cola_cg_solve_deflated(self._h, ctypes.byref(sp), ctypes.c_void_p(b.data_ptr()), ctypes.c_void_p(x.data_ptr()), ctypes.byref(info),
                                         ctypes.c_void_p(evecs.data_ptr()), ev, len(evals))
        self._ck(st, ok=(COLA_OK, COLA_ENOCONV))
        return x, self._info_dict(info, st)

    # ---- multi-right-hand-side operators and batched solver
    def mrhs_workspace_bytes(self, nrhs: int, for_solver: bool = True) -> int:
        return int(_lib.cola_mrhs_workspace_bytes(self._h, int(nrhs), int(bool(for_solver))))

    def set_mrhs_workspace(self, nrhs: int, tensor: torch.Tensor | None = None, for_solver: bool = True):
        """Lend the per-right-hand-side workspace (allocated here with torch if not given); for_solver=False sizes it for
        the multi-rhs operators only."""
        if tensor is None:
            self.release_mrhs_workspace()
            tensor = torch.empty(self.mrhs_workspace_bytes(nrhs, for_solver), dtype=torch.uint8, device=self.device)
        self._ck(_lib.cola_set_mrhs_workspace(self._h, ctypes.c_void_p(tensor.data_ptr()), tensor.numel() * tensor.element_size(), int(nrhs)))
        self._mws, self._mws_nrhs = tensor, int(nrhs)
        self._mws_solver = tensor.numel() * tensor.element_size() >= self.mrhs_workspace_bytes(nrhs, True)
        return tensor

    def release_mrhs_workspace(self):
        self._ck(_lib.cola_set_mrhs_workspace(self._h, None, 0, 0))
        self._mws, self._mws_nrhs, self._mws_solver = None, 0, False

    def _need_mrhs(self, nrhs, for_solver=False):
        if self._mws is None or self._mws_nrhs < nrhs or (for_solver and not self._mws_solver):
            self.set_mrhs_workspace(nrhs, for_solver=for_solver)

    def empty_internal_mrhs(self, nrhs, prec, full=True) -> torch.Tensor:
        """nrhs internal buffers back to back: shape (nrhs,) + the shape of empty_internal."""
        one = self.empty_internal(prec, full=full)
        return torch.empty((int(nrhs),) + tuple(one.shape), dtype=one.dtype, device=self.device)

    def dslash_apply_mrhs(self, out_parity: int, inp: torch.Tensor, out: torch.Tensor | None = None, h16=False, fmt=None) -> torch.Tensor:
        pr, nrhs = self._op_prec(inp, h16, fmt), inp.shape[0]
        assert inp.is_cuda and inp.is_contiguous() and inp.numel() == nrhs * self.Vh * 24
        self._need_mrhs(nrhs)
        if out is None:
            out = torch.empty_like(inp)
        self._ck(_lib.cola_dslash_apply_mrhs(self._h, pr, int(out_parity), nrhs, ctypes.c_void_p(inp.data_ptr()), ctypes.c_void_p(out.data_ptr())))
        return out

    def fermion_matrix_apply_mrhs(self, inp: torch.Tensor, dagger=False, out: torch.Tensor | None = None, h16=False, fmt=None) -> torch.Tensor:
        pr, nrhs = self._op_prec(inp, h16, fmt), inp.shape[0]
        assert inp.is_cuda and inp.is_contiguous() and inp.numel() == nrhs * self.V * 24
        self._need_mrhs(nrhs)
        if out is None:
            out = torch.empty_like(inp)
        self._ck(_lib.cola_fermion_matrix_apply_mrhs(self._h, pr, int(bool(dagger)), nrhs, ctypes.c_void_p(inp.data_ptr()), ctypes.c_void_p(out.data_ptr())))
        return out

    def schur_apply_mrhs(self, inp: torch.Tensor, dagger=False, out: torch.Tensor | None = None, h16=False, fmt=None) -> torch.Tensor:
        pr, nrhs = self._op_prec(inp, h16, fmt), inp.shape[0]
        assert inp.is_cuda and inp.is_contiguous() and inp.numel() == nrhs * self.Vh * 24
        self._need_mrhs(nrhs)
        if out is None:
            out = torch.empty_like(inp)
        self._ck(_lib.cola_schur_apply_mrhs(self._h, pr, int(bool(dagger)), nrhs, ctypes.c_void_p(inp.data_ptr()), ctypes.c_void_p(out.data_ptr())))
        return out

    def cg_solve_mrhs(self, b: torch.Tensor, tol=1e-10, max_iter=20000, delta=0.1, x: torch.Tensor | None = None, mixed=1, method="cgnr"):
        """b: nrhs canonical complex128 sources, shape (nrhs, t, z, y, x, 4, 3), on the device.
        method: "cgnr" or "bicgstab" (both on the Schur system, mixed precision).  Returns (x, [info dict per system])."""
        assert b.is_cuda and b.dtype == torch.complex128 and b.dim() == 7 and b[0].numel() == self.V * 12
        b = b.contiguous()
        nrhs = b.shape[0]
        self._need_mrhs(nrhs, for_solver=True)
        if x is None:
            x = torch.empty_like(b)
        sp = self._solve_params(tol, max_iter, True, mixed, delta, method)
        infos = (ColaSolveInfo * nrhs)()
        st = _lib.cola_cg_solve_mrhs(self._h, ctypes.byref(sp), nrhs, ctypes.c_void_p(b.data_ptr()), ctypes.c_void_p(x.data_ptr()), infos)
        self._ck(st, ok=(COLA_OK, COLA_ENOCONV))
        out = []
        for n in range(nrhs):
            d = self._info_dict(infos[n], COLA_OK)
            d["converged"] = bool(d["iterated_residual"] <= tol) or st == COLA_OK
            out.append(d)
        return x, out
