"""ctypes binding of libwz.so (include/wz.h).  Argument marshalling only: every
step of the path runs in the CUDA kernels behind the C ABI.  PyTorch is used for
device memory and streams.  There is no CPU fallback: a missing library or a
missing GPU raises.
"""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libwz.so")
_lib = None

WZ_C64, WZ_C128 = 0, 1
WZ_NKINDS = 9
WZ_OK, WZ_EINVAL, WZ_EUNSUPPORTED, WZ_ENOMEM, WZ_ECUDA, WZ_ENOTCONVERGED = range(6)

EXPORTS = [
    "wz_status_string", "wz_last_error", "wz_version", "wz_plan_create", "wz_plan_destroy",
    "wz_supported", "wz_plan_workspace_bytes", "wz_fft4d", "wz_apply_M", "wz_apply_MdagM",
    "wz_cg_solve", "wz_plan_launch_count", "wz_plan_reset_launch_count",
    "wz_plan_profile", "wz_plan_profile_read", "wz_kind_name",
    "wz_apply_M0inv", "wz_apply_MtdagMt", "wz_cg_solve_pc", "wz_apply_Dslash", "wz_locality_profile",
    "wz_cg_solve_shift", "wz_cg_solve_shift_pc", "wz_rational_apply",
    "wz_plan_set_graph", "wz_plan_cg_history", "wz_plan_set_block",
    "wz_cg_solve_multishift", "wz_rational_apply_multishift", "wz_cg_solve_dc", "wz_apply_MdagM_noalloc", "wz_cg_solve_dc_half", "wz_cg_solve_half",
]


class WZError(RuntimeError):
    def __init__(self, status: int, text: str):
        super().__init__(text)
        self.status = status


class _CGInfo(ctypes.Structure):
    _fields_ = [("iterations", ctypes.c_int), ("reliable_updates", ctypes.c_int),
                ("converged", ctypes.c_int), ("rel_residual_recursive", ctypes.c_double),
                ("rel_residual_true", ctypes.c_double)]


@dataclass
class CGInfo:
    iterations: int
    reliable_updates: int
    converged: bool
    rel_residual_recursive: float
    rel_residual_true: float


def lib() -> ctypes.CDLL:
    """Load libwz.so (built by paper_1005_3276_b200.build); fail loudly if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise WZError(-1, "libwz.so not found at %s: run `python -m paper_1005_3276_b200.build` "
                              "(there is no CPU fallback)" % LIB_PATH)
        L = ctypes.CDLL(LIB_PATH)
        vp, ci, cd = ctypes.c_void_p, ctypes.c_int, ctypes.c_double
        d2 = ctypes.POINTER(ctypes.c_double)
        L.wz_status_string.restype = ctypes.c_char_p
        L.wz_status_string.argtypes = [ci]
        L.wz_last_error.restype = ctypes.c_char_p
        L.wz_version.restype = ctypes.c_char_p
        L.wz_plan_create.argtypes = [ctypes.POINTER(vp), ci, ci, ci, ci, ci, ci, vp]
        L.wz_plan_destroy.argtypes = [vp]
        L.wz_supported.argtypes = [ci, ci, ci, ci, ci]
        L.wz_plan_workspace_bytes.restype = ctypes.c_ulonglong
        L.wz_plan_workspace_bytes.argtypes = [vp]
        L.wz_plan_launch_count.restype = ctypes.c_ulonglong
        L.wz_plan_launch_count.argtypes = [vp]
        L.wz_plan_reset_launch_count.restype = None
        L.wz_plan_reset_launch_count.argtypes = [vp]
        L.wz_fft4d.argtypes = [vp, ci, ci, vp, vp, ci]
        L.wz_apply_M.argtypes = [vp, ci, vp, d2, d2, cd, vp, vp, ci]
        L.wz_apply_MdagM.argtypes = [vp, vp, d2, d2, cd, vp, vp, ci]
        L.wz_cg_solve.argtypes = [vp, vp, vp, vp, d2, d2, cd, cd, ci, ci, ctypes.POINTER(_CGInfo)]
        L.wz_cg_solve_pc.argtypes = L.wz_cg_solve.argtypes
        L.wz_cg_solve_half.argtypes = L.wz_cg_solve.argtypes
        L.wz_cg_solve_shift.argtypes = [vp, vp, vp, vp, d2, d2, cd, cd, cd, ci, ci, ctypes.POINTER(_CGInfo)]
        L.wz_cg_solve_shift_pc.argtypes = L.wz_cg_solve_shift.argtypes
        L.wz_rational_apply.argtypes = [vp, vp, vp, vp, d2, d2, cd, cd, d2, d2, ci, cd, cd, ci, ci,
                                        ctypes.POINTER(_CGInfo)]
        L.wz_rational_apply_multishift.argtypes = L.wz_rational_apply.argtypes
        L.wz_cg_solve_multishift.argtypes = [vp, vp, vp, vp, d2, d2, cd, d2, ci, cd, ci, ci, ctypes.POINTER(_CGInfo)]
        L.wz_cg_solve_dc.argtypes = [vp, vp, vp, vp, d2, d2, cd, cd, cd, ci, ci, ctypes.POINTER(_CGInfo)]
        L.wz_cg_solve_dc_half.argtypes = L.wz_cg_solve_dc.argtypes
        L.wz_apply_MdagM_noalloc.argtypes = [ci, ci, ci, ci, ci, vp, d2, d2, cd, vp, vp, ci, vp]
        L.wz_apply_M0inv.argtypes = [vp, ci, d2, cd, vp, vp, ci]
        L.wz_apply_MtdagMt.argtypes = [vp, vp, d2, d2, cd, vp, vp, ci]
        L.wz_apply_Dslash.argtypes = [vp, cd, vp, vp, ci]
        L.wz_locality_profile.argtypes = [vp, cd, ci, d2, ci]
        L.wz_plan_profile.argtypes = [vp, ci]
        L.wz_plan_profile_read.argtypes = [vp, d2, ctypes.POINTER(ctypes.c_ulonglong)]
        L.wz_plan_set_graph.argtypes = [vp, ci]
        L.wz_plan_set_block.argtypes = [vp, ci]
        L.wz_plan_cg_history.argtypes = [vp, ci, ctypes.POINTER(ci), d2, ci]
        L.wz_kind_name.restype = ctypes.c_char_p
        L.wz_kind_name.argtypes = [ci]
        _lib = L
    return _lib


def _check(status: int):
    if status != WZ_OK:
        L = lib()
        text = L.wz_status_string(status).decode()
        extra = L.wz_last_error().decode()
        raise WZError(status, "wz: %s%s" % (text, (" [" + extra + "]") if extra else ""))


def _c2(z):
    z = complex(z)
    return (ctypes.c_double * 2)(z.real, z.imag)


def supported(dims, dtype="c64") -> bool:
    T, L1, L2, L3 = [int(d) for d in dims]
    return bool(lib().wz_supported(T, L1, L2, L3, WZ_C64 if dtype == "c64" else WZ_C128))


class Plan:
    """wz_plan for a T x L1 x L2 x L3 lattice; dtype 'c64' or 'c128'."""

    def __init__(self, dims, dtype: str = "c64", max_batch: int = 1, device="cuda:0", stream=None):
        if not torch.cuda.is_available():
            raise WZError(-1, "wz needs a CUDA device (no CPU fallback)")
        self.dims = tuple(int(d) for d in dims)
        self.dtype = dtype
        self.tdtype = torch.complex64 if dtype == "c64" else torch.complex128
        self.device = torch.device(device)
        if self.device.index is None:
            self.device = torch.device("cuda", torch.cuda.current_device())
        self.max_batch = int(max_batch)
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        h = ctypes.c_void_p()
        T, L1, L2, L3 = self.dims
        with torch.cuda.device(self.device):  # the plan lives on the device current at creation
            _check(lib().wz_plan_create(ctypes.byref(h), T, L1, L2, L3,
                                        WZ_C64 if dtype == "c64" else WZ_C128, self.max_batch,
                                        ctypes.c_void_p(self.stream.cuda_stream)))
        self._h = h

    def close(self):
        if getattr(self, "_h", None):
            lib().wz_plan_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- helpers --
    def _spinor(self, t: torch.Tensor, dtype=None, nb=None):
        """Validate a spinor batch (dtype, device, layout, shape); returns its batch count.
        nb given: the batch count it must have (outputs must match their inputs)."""
        dtype = dtype or self.tdtype
        shape = (4,) + self.dims
        if t.dtype != dtype or not t.is_cuda or not t.is_contiguous():
            raise ValueError("expected a contiguous CUDA tensor of dtype %s" % dtype)
        if t.device != self.device:
            raise ValueError("tensor is on %s, the plan lives on %s" % (t.device, self.device))
        if tuple(t.shape) == shape:
            n = 1
        elif t.dim() == 6 and tuple(t.shape[1:]) == shape:
            n = int(t.shape[0])
        else:
            raise ValueError("expected shape [nbatch,]4,T,L1,L2,L3 = %s, got %s" % (shape, tuple(t.shape)))
        if nb is not None and n != nb:
            raise ValueError("output holds %d spinor(s), input %d" % (n, nb))
        return n

    def _phi(self, phi: torch.Tensor):
        if phi.dtype != self.tdtype or not phi.is_cuda or not phi.is_contiguous() or \
                tuple(phi.shape) != self.dims or phi.device != self.device:
            raise ValueError("phi must be a contiguous tensor on %s of shape %s, dtype %s"
                             % (self.device, self.dims, self.tdtype))

    @property
    def workspace_bytes(self) -> int:
        return int(lib().wz_plan_workspace_bytes(self._h))

    @property
    def launch_count(self) -> int:
        return int(lib().wz_plan_launch_count(self._h))

    def reset_launch_count(self):
        lib().wz_plan_reset_launch_count(self._h)

    def set_graph(self, enable: bool):
        """CUDA-graph replay of the iteration chunks on (default) or off (wz_plan_set_graph)."""
        _check(lib().wz_plan_set_graph(self._h, int(bool(enable))))

    def set_block(self, sources_per_block: int):
        """Sources per block of a batched solve (wz_plan_set_block); 0 = whole batch in lock step."""
        _check(lib().wz_plan_set_block(self._h, int(sources_per_block)))

    def cg_history(self, source: int = 0):
        """[(iteration, ||r||/||b||)] of the last solve as the host saw it (wz_plan_cg_history)."""
        n = lib().wz_plan_cg_history(self._h, int(source), None, None, 0)
        if n < 0:
            raise ValueError("no history for source %d" % source)
        it = (ctypes.c_int * max(n, 1))()
        rr = (ctypes.c_double * max(n, 1))()
        lib().wz_plan_cg_history(self._h, int(source), it, rr, n)
        return [(int(it[i]), float(rr[i])) for i in range(n)]

    def profile(self, enable: bool):
        _check(lib().wz_plan_profile(self._h, int(bool(enable))))

    def profile_read(self) -> dict:
        """{kind: (total_ms, launches)} of the launches recorded since profile(True)."""
        ms = (ctypes.c_double * WZ_NKINDS)()
        cnt = (ctypes.c_ulonglong * WZ_NKINDS)()
        _check(lib().wz_plan_profile_read(self._h, ms, cnt))
        return {lib().wz_kind_name(k).decode(): (ms[k], int(cnt[k])) for k in range(WZ_NKINDS) if cnt[k]}

    # -- the calls of include/wz.h --
    def fft4d(self, inp, direction: int, antiperiodic_time: bool = True, out=None):
        nb = self._spinor(inp)
        if out is None:
            out = torch.empty_like(inp)
        self._spinor(out, nb=nb)
        _check(lib().wz_fft4d(self._h, int(direction), int(bool(antiperiodic_time)),
                              inp.data_ptr(), out.data_ptr(), nb))
        return out

    def apply_M(self, phi, psi, m, g, rho: float = 1.0, dagger: bool = False, out=None):
        nb = self._spinor(psi)
        self._phi(phi)
        if out is None:
            out = torch.empty_like(psi)
        self._spinor(out, nb=nb)
        _check(lib().wz_apply_M(self._h, int(bool(dagger)), phi.data_ptr(), _c2(m), _c2(g), float(rho),
                                psi.data_ptr(), out.data_ptr(), nb))
        return out

    def apply_MdagM(self, phi, psi, m, g, rho: float = 1.0, out=None):
        nb = self._spinor(psi)
        self._phi(phi)
        if out is None:
            out = torch.empty_like(psi)
        self._spinor(out, nb=nb)
        _check(lib().wz_apply_MdagM(self._h, phi.data_ptr(), _c2(m), _c2(g), float(rho),
                                    psi.data_ptr(), out.data_ptr(), nb))
        return out

    def apply_Dslash(self, psi, rho: float = 1.0, out=None):
        nb = self._spinor(psi)
        if out is None:
            out = torch.empty_like(psi)
        self._spinor(out, nb=nb)
        _check(lib().wz_apply_Dslash(self._h, float(rho), psi.data_ptr(), out.data_ptr(), nb))
        return out

    def locality_profile(self, spin: int = 0, rho: float = 1.0):
        """f(r) of Eq. (3.11) as a list of floats, r = 0 .. sum(L_mu // 2)."""
        nf = 1 + sum(d // 2 for d in self.dims)
        f = (ctypes.c_double * nf)()
        _check(lib().wz_locality_profile(self._h, float(rho), int(spin), f, nf))
        return list(f)

    def apply_M0inv(self, psi, m, rho: float = 1.0, dagger: bool = False, out=None):
        nb = self._spinor(psi)
        if out is None:
            out = torch.empty_like(psi)
        self._spinor(out, nb=nb)
        _check(lib().wz_apply_M0inv(self._h, int(bool(dagger)), _c2(m), float(rho), psi.data_ptr(),
                                    out.data_ptr(), nb))
        return out

    def apply_MtdagMt(self, phi, psi, m, g, rho: float = 1.0, out=None):
        nb = self._spinor(psi)
        self._phi(phi)
        if out is None:
            out = torch.empty_like(psi)
        self._spinor(out, nb=nb)
        _check(lib().wz_apply_MtdagMt(self._h, phi.data_ptr(), _c2(m), _c2(g), float(rho),
                                      psi.data_ptr(), out.data_ptr(), nb))
        return out

    def cg_solve(self, phi, b, m, g, rho: float = 1.0, tol: float = 1e-6, max_iter: int = 100000,
                 out=None, raise_on_fail: bool = True, precondition: bool = False, sigma=None,
                 half_storage: bool = False):
        """Solve M^dag M x = b per source (precondition=True: through the free-inverse
        preconditioned system, wz_cg_solve_pc; sigma given: the shifted system
        (M^dag M + sigma) x = b, wz_cg_solve_shift; both: Eq. 7.14, wz_cg_solve_shift_pc).
        Returns (x complex128, [CGInfo])."""
        nb = self._spinor(b)
        self._phi(phi)
        if out is None:
            out = torch.empty(b.shape, dtype=torch.complex128, device=b.device)
        self._spinor(out, torch.complex128, nb=nb)
        infos = (_CGInfo * nb)()
        if sigma is not None:
            if half_storage:
                raise ValueError("half_storage: plain system only")
            fn = lib().wz_cg_solve_shift_pc if precondition else lib().wz_cg_solve_shift
            st = fn(self._h, phi.data_ptr(), b.data_ptr(), out.data_ptr(), _c2(m), _c2(g),
                    float(rho), float(sigma), float(tol), int(max_iter), nb, infos)
        else:
            fn = lib().wz_cg_solve_pc if precondition else lib().wz_cg_solve
            if half_storage:  # binary16 storage of t, chi, r, p (wz_cg_solve_half); plain system only
                if precondition:
                    raise ValueError("half_storage: plain system only")
                fn = lib().wz_cg_solve_half
            st = fn(self._h, phi.data_ptr(), b.data_ptr(), out.data_ptr(), _c2(m), _c2(g),
                    float(rho), float(tol), int(max_iter), nb, infos)
        if st != WZ_OK and not (st == WZ_ENOTCONVERGED and not raise_on_fail):
            _check(st)
        res = [CGInfo(i.iterations, i.reliable_updates, bool(i.converged), i.rel_residual_recursive,
                      i.rel_residual_true) for i in infos]
        return out, res


    def cg_solve_dc(self, phi, b, m, g, rho: float = 1.0, tol: float = 1e-10, inner_tol: float = 1e-3,
                    max_iter: int = 100000, out=None, raise_on_fail: bool = True, half_storage: bool = False):
        """Defect correction: complex128 outer loop, complex64 inner solves (wz_cg_solve_dc; 'c64' plans).
        Returns (x complex128, [CGInfo]) with iterations = inner iterations, reliable_updates = outer steps."""
        nb = self._spinor(b)
        self._phi(phi)
        if out is None:
            out = torch.empty(b.shape, dtype=torch.complex128, device=b.device)
        self._spinor(out, torch.complex128, nb=nb)
        infos = (_CGInfo * nb)()
        fn = lib().wz_cg_solve_dc_half if half_storage else lib().wz_cg_solve_dc  # half_storage: binary16 storage of t, chi, r, p
        st = fn(self._h, phi.data_ptr(), b.data_ptr(), out.data_ptr(), _c2(m), _c2(g), float(rho),
                float(tol), float(inner_tol), int(max_iter), nb, infos)
        if st != WZ_OK and not (st == WZ_ENOTCONVERGED and not raise_on_fail):
            _check(st)
        return out, [CGInfo(i.iterations, i.reliable_updates, bool(i.converged), i.rel_residual_recursive,
                            i.rel_residual_true) for i in infos]

    def cg_solve_multishift(self, phi, b, m, g, sigmas, rho: float = 1.0, tol: float = 1e-6, max_iter: int = 100000,
                            out=None, raise_on_fail: bool = True):
        """All (M^dag M + sigma_i) x_i = b from one Krylov space (wz_cg_solve_multishift).
        Returns (x complex128 [nshift, nbatch, 4, T, L1, L2, L3], infos[shift][source])."""
        nb = self._spinor(b)
        self._phi(phi)
        d = len(sigmas)
        shape = (d, nb, 4) + self.dims
        if out is None:
            out = torch.empty(shape, dtype=torch.complex128, device=b.device)
        if out.dtype != torch.complex128 or tuple(out.shape) != shape or not out.is_contiguous() or out.device != self.device:
            raise ValueError("out must be a contiguous complex128 tensor of shape %s on %s" % (shape, self.device))
        cs = (ctypes.c_double * max(d, 1))(*[float(v) for v in sigmas])
        infos = (_CGInfo * max(d * nb, 1))()
        st = lib().wz_cg_solve_multishift(self._h, phi.data_ptr(), b.data_ptr(), out.data_ptr(), _c2(m), _c2(g),
                                          float(rho), cs, d, float(tol), int(max_iter), nb, infos)
        if st != WZ_OK and not (st == WZ_ENOTCONVERGED and not raise_on_fail):
            _check(st)
        res = [[CGInfo(infos[i * nb + j].iterations, infos[i * nb + j].reliable_updates,
                       bool(infos[i * nb + j].converged), infos[i * nb + j].rel_residual_recursive,
                       infos[i * nb + j].rel_residual_true) for j in range(nb)] for i in range(d)]
        return out, res

    def rational_apply(self, phi, eta, m, g, alpha0, alphas, betas, rho: float = 1.0, tol: float = 1e-6,
                       max_iter: int = 100000, pc_cutoff: float = 100.0, out=None, raise_on_fail: bool = True,
                       multishift: bool = False):
        """out = alpha0 eta + sum_i alphas[i] (M^dag M + betas[i])^-1 eta (wz_rational_apply, Eq. 7.6-7.7;
        multishift=True: wz_rational_apply_multishift, one multi-shift solve for the shifts above pc_cutoff).
        Returns (out complex128, infos[shift][source])."""
        nb = self._spinor(eta)
        self._phi(phi)
        if out is None:
            out = torch.empty(eta.shape, dtype=torch.complex128, device=eta.device)
        self._spinor(out, torch.complex128, nb=nb)
        d = len(alphas)
        assert len(betas) == d
        ca = (ctypes.c_double * max(d, 1))(*[float(a) for a in alphas])
        cb = (ctypes.c_double * max(d, 1))(*[float(b) for b in betas])
        infos = (_CGInfo * max(d * nb, 1))()
        fn = lib().wz_rational_apply_multishift if multishift else lib().wz_rational_apply
        st = fn(self._h, phi.data_ptr(), eta.data_ptr(), out.data_ptr(), _c2(m), _c2(g),
                                     float(rho), float(alpha0), ca, cb, d, float(pc_cutoff), float(tol),
                                     int(max_iter), nb, infos)
        if st != WZ_OK and not (st == WZ_ENOTCONVERGED and not raise_on_fail):
            _check(st)
        res = [[CGInfo(infos[i * nb + j].iterations, infos[i * nb + j].reliable_updates,
                       bool(infos[i * nb + j].converged), infos[i * nb + j].rel_residual_recursive,
                       infos[i * nb + j].rel_residual_true) for j in range(nb)] for i in range(d)]
        return out, res


NOALLOC_MAX_BYTES = 8 << 20  # WZ_NOALLOC_MAX_BYTES of include/wz.h


def apply_MdagM_noalloc(phi, psi, m, g, rho: float = 1.0, out=None, stream=None):
    """out = M^dag M psi through wz_apply_MdagM_noalloc: no plan, no device allocation inside the call (its
    scratch is a static device array of NOALLOC_MAX_BYTES inside libwz.so, shared by all calls: overlapping
    calls race).  `out` must be given if the caller may not allocate.  Lattice and dtype are taken from phi."""
    if not (phi.is_cuda and psi.is_cuda and phi.is_contiguous() and psi.is_contiguous()):
        raise ValueError("expected contiguous CUDA tensors")
    if phi.dtype not in (torch.complex64, torch.complex128) or psi.dtype != phi.dtype or phi.dim() != 4:
        raise ValueError("phi: [T, L1, L2, L3] complex64 or complex128; psi of the same dtype")
    dims = tuple(int(d) for d in phi.shape)
    if tuple(psi.shape) == (4,) + dims:
        nb = 1
    elif psi.dim() == 6 and tuple(psi.shape[1:]) == (4,) + dims:
        nb = int(psi.shape[0])
    else:
        raise ValueError("expected psi of shape [nbatch,]4,T,L1,L2,L3")
    if out is None:
        out = torch.empty_like(psi)
    if out.shape != psi.shape or out.dtype != psi.dtype or out.device != psi.device or not out.is_contiguous() \
            or phi.device != psi.device:
        raise ValueError("out must match psi; phi, psi, out on one device")
    with torch.cuda.device(psi.device):
        st = stream if stream is not None else torch.cuda.current_stream(psi.device)
        _check(lib().wz_apply_MdagM_noalloc(dims[0], dims[1], dims[2], dims[3],
                                            WZ_C64 if phi.dtype == torch.complex64 else WZ_C128,
                                            phi.data_ptr(), _c2(m), _c2(g), float(rho), psi.data_ptr(),
                                            out.data_ptr(), nb, ctypes.c_void_p(st.cuda_stream)))
    return out


# module-level aliases with the C names
def wz_plan_create(dims, dtype="c64", max_batch=1, device="cuda:0", stream=None) -> Plan:
    return Plan(dims, dtype, max_batch, device, stream)


def wz_fft4d(plan: Plan, direction, antiperiodic_time, inp, out=None):
    return plan.fft4d(inp, direction, antiperiodic_time, out)


def wz_apply_M(plan: Plan, dagger, phi, m, g, rho, inp, out=None):
    return plan.apply_M(phi, inp, m, g, rho, dagger, out)


def wz_apply_MdagM(plan: Plan, phi, m, g, rho, inp, out=None):
    return plan.apply_MdagM(phi, inp, m, g, rho, out)


def wz_cg_solve(plan: Plan, phi, b, m, g, rho, tol, max_iter=100000, out=None):
    return plan.cg_solve(phi, b, m, g, rho, tol, max_iter, out)
