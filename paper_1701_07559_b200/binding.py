"""Thin ctypes binding of include/mdwf.h: same names, argument marshalling only.

PyTorch appears here only as the owner of device memory (tensor.data_ptr()) and streams.
There is no CPU fallback: lib() raises if libmdwf_b200.so has not been built, and every compute
call returns the library's error code (raised as MdwfError) when no CUDA device is present.
"""
import ctypes
import os

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libmdwf_b200.so")

MDWF_OK, MDWF_EARG, MDWF_ENOGAUGE, MDWF_ECUDA, MDWF_ENOCONV, MDWF_ENOMEM = 0, -1, -2, -3, -4, -5
OP_MPC, OP_MPCDAG, OP_MDAGM, OP_D, OP_DDAG, OP_MPC_SYM, OP_MPCDAG_SYM = 0, 1, 2, 3, 4, 5, 6

EXPORTS = ["mdwf_create", "mdwf_destroy", "mdwf_set_option", "mdwf_load_gauge", "mdwf_load_gauge_host",
           "mdwf_apply", "mdwf_solve", "mdwf_solve_host", "mdwf_blas_norm2", "mdwf_blas_redot", "mdwf_blas_axpy",
           "mdwf_get_stat", "mdwf_last_error", "mdwf_flops_per_site", "mdwf_time_op", "mdwf_fma_rates",
           "mdwf_half_encode", "mdwf_half_decode", "mdwf_l2_rates", "mdwf_wall_source", "mdwf_wall_project", "mdwf_gradient_flow", "mdwf_plaquette",
           "mdwf_apply_batch", "mdwf_time_op_batch", "mdwf_blas_norm2_noalloc", "mdwf_noalloc_setup", "mdwf_noalloc_max_n", "mdwf_noalloc_last_error"]

_lib = None


class MdwfError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("mdwf error %d: %s" % (code, msg))
        self.code = code


def lib():
    """Load the C-ABI library; fail loudly if it is missing (no fallback)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError("libmdwf_b200.so is not built: run `python -m paper_1701_07559_b200.build` "
                               "(or __graft_entry__.build()); there is no CPU fallback")
        L = ctypes.CDLL(LIB_PATH)
        P, I, D, LL = ctypes.c_void_p, ctypes.c_int, ctypes.c_double, ctypes.c_longlong
        L.mdwf_create.argtypes = [ctypes.POINTER(P), I, I, I, I, I, D, D, D, D]
        L.mdwf_destroy.argtypes = [P]
        L.mdwf_set_option.argtypes = [P, ctypes.c_char_p, ctypes.c_char_p]
        L.mdwf_load_gauge.argtypes = [P, P, I]
        L.mdwf_load_gauge_host.argtypes = [P, P, I]
        L.mdwf_apply.argtypes = [P, I, P, P, I]
        L.mdwf_solve.argtypes = [P, P, P, D, I, ctypes.POINTER(I), ctypes.POINTER(D)]
        L.mdwf_solve_host.argtypes = [P, P, P, D, I, ctypes.POINTER(I), ctypes.POINTER(D)]
        L.mdwf_blas_norm2.argtypes = [P, P, LL, I, ctypes.POINTER(D)]
        L.mdwf_blas_redot.argtypes = [P, P, P, LL, I, ctypes.POINTER(D)]
        L.mdwf_blas_norm2_noalloc.argtypes = [P, LL, I, P, P]
        L.mdwf_apply_batch.argtypes = [P, I, I, P, P, I]
        L.mdwf_time_op_batch.argtypes = [P, I, ctypes.c_char_p, I, I, I, ctypes.POINTER(D)]
        L.mdwf_noalloc_setup.argtypes = []
        L.mdwf_noalloc_max_n.argtypes = []
        L.mdwf_noalloc_max_n.restype = LL
        L.mdwf_noalloc_last_error.argtypes = []
        L.mdwf_noalloc_last_error.restype = ctypes.c_char_p
        L.mdwf_blas_axpy.argtypes = [P, D, P, P, LL, I]
        L.mdwf_get_stat.argtypes = [P, ctypes.c_char_p, ctypes.POINTER(D)]
        L.mdwf_last_error.argtypes = [P]
        L.mdwf_last_error.restype = ctypes.c_char_p
        L.mdwf_flops_per_site.argtypes = [P]
        L.mdwf_time_op.argtypes = [P, I, ctypes.c_char_p, I, I, ctypes.POINTER(D)]
        L.mdwf_fma_rates.argtypes = [P, ctypes.POINTER(D)]
        L.mdwf_l2_rates.argtypes = [P, ctypes.POINTER(D)]
        L.mdwf_half_encode.argtypes = [P, P, I, I, P, P]
        L.mdwf_wall_source.argtypes = [P, P, P, I, I]
        L.mdwf_gradient_flow.argtypes = [P, P, D, I, I, ctypes.POINTER(D)]
        L.mdwf_plaquette.argtypes = [P, P, ctypes.POINTER(D)]
        L.mdwf_wall_project.argtypes = [P, P, P, I, I]
        L.mdwf_half_decode.argtypes = [P, P, P, P, I]
        _lib = L
    return _lib


# ---- same-name functions on raw pointers / integers ---------------------------------------------
def mdwf_create(Lx, Ly, Lz, Lt, L5, M5, b5, c5, m_f):
    h = ctypes.c_void_p()
    rc = lib().mdwf_create(ctypes.byref(h), Lx, Ly, Lz, Lt, L5, M5, b5, c5, m_f)
    if rc != MDWF_OK:
        raise MdwfError(rc, "mdwf_create: bad argument")
    return h


def _check(h, rc, allow=()):
    if rc != MDWF_OK and rc not in allow:
        raise MdwfError(rc, lib().mdwf_last_error(h).decode())
    return rc


def blas_norm2_noalloc(x, out, stream=None):
    """||x||^2 of the device tensor x into the one-element fp64 device tensor `out`, through the entry point that allocates
    nothing (include/mdwf.h); queued on `stream` (a raw cudaStream_t handle, default stream if None), not synchronised."""
    n = x.numel() * (2 if x.is_complex() else 1)
    rb = Mdwf._rb(x)
    rc = lib().mdwf_blas_norm2_noalloc(x.data_ptr(), n, rb, out.data_ptr(), stream)
    if rc != MDWF_OK:
        raise MdwfError(rc, lib().mdwf_noalloc_last_error().decode())
    return rc


def noalloc_setup():
    rc = lib().mdwf_noalloc_setup()
    if rc != MDWF_OK:
        raise MdwfError(rc, lib().mdwf_noalloc_last_error().decode())


def noalloc_max_n():
    return int(lib().mdwf_noalloc_max_n())


def mdwf_destroy(h):
    return lib().mdwf_destroy(h)


def mdwf_set_option(h, key, value):
    return _check(h, lib().mdwf_set_option(h, key.encode(), str(value).encode()))


def mdwf_load_gauge(h, U_ptr, real_bytes):
    return _check(h, lib().mdwf_load_gauge(h, U_ptr, real_bytes))


def mdwf_load_gauge_host(h, U_ptr, real_bytes):
    return _check(h, lib().mdwf_load_gauge_host(h, U_ptr, real_bytes))


def mdwf_apply(h, op, in_ptr, out_ptr, real_bytes):
    return _check(h, lib().mdwf_apply(h, op, in_ptr, out_ptr, real_bytes))


def mdwf_solve(h, src_ptr, sol_ptr, tol, maxiter, host=False):
    it, tr = ctypes.c_int(0), ctypes.c_double(0.0)
    fn = lib().mdwf_solve_host if host else lib().mdwf_solve
    rc = _check(h, fn(h, src_ptr, sol_ptr, tol, maxiter, ctypes.byref(it), ctypes.byref(tr)), allow=(MDWF_ENOCONV,))
    return rc, it.value, tr.value


def mdwf_get_stat(h, key):
    v = ctypes.c_double(0.0)
    _check(h, lib().mdwf_get_stat(h, key.encode(), ctypes.byref(v)))
    return v.value


def mdwf_flops_per_site(h):
    return lib().mdwf_flops_per_site(h)


def mdwf_time_op(h, op, precision, reps, warmup):
    """Average device milliseconds per application (CUDA events on the context's stream) of op
    0 Mpc / 1 Mpc^dagger in the given precision on library-owned buffers; also per-kernel times."""
    out = (ctypes.c_double * 4)()
    _check(h, lib().mdwf_time_op(h, op, precision.encode(), reps, warmup, out))
    return dict(ms=out[0], ms_k1=out[1], ms_k2=out[2], launches=out[3])


# ---- convenience wrapper on torch tensors (marshalling only) ------------------------------------
class Mdwf:
    def __init__(self, L, L5, M5, b5, c5, mf):
        self.L, self.L5 = tuple(L), L5
        self.h = mdwf_create(L[0], L[1], L[2], L[3], L5, M5, b5, c5, mf)

    def close(self):
        if self.h is not None:
            mdwf_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_option(self, key, value):
        mdwf_set_option(self.h, key, value)

    @staticmethod
    def _rb(t):
        import torch
        return 8 if t.dtype in (torch.complex128, torch.float64) else 4

    def load_gauge(self, U):
        assert U.is_contiguous()
        if U.is_cuda:
            mdwf_load_gauge(self.h, U.data_ptr(), self._rb(U))
        else:
            mdwf_load_gauge_host(self.h, U.data_ptr(), self._rb(U))

    def apply(self, op, x):
        import torch
        assert x.is_cuda and x.is_contiguous()
        out = torch.empty_like(x)
        mdwf_apply(self.h, op, x.data_ptr(), out.data_ptr(), self._rb(x))
        return out

    def gradient_flow(self, U, eps, nsteps, action="wilson"):
        """flow the canonical fp64 gauge field U in place; returns the mean plaquette of the flowed field  (mdwf_gradient_flow)"""
        import torch
        assert U.is_cuda and U.is_contiguous() and U.dtype == torch.complex128
        out = ctypes.c_double()
        _check(self.h, lib().mdwf_gradient_flow(self.h, U.data_ptr(), float(eps), int(nsteps), {"wilson": 0, "symanzik": 1}[action],
                                                ctypes.byref(out)))
        return out.value

    def plaquette(self, U):
        import torch
        assert U.is_cuda and U.is_contiguous() and U.dtype == torch.complex128
        out = ctypes.c_double()
        _check(self.h, lib().mdwf_plaquette(self.h, U.data_ptr(), ctypes.byref(out)))
        return out.value

    def wall_source(self, eta, lift=False):
        """4D field eta[t][z][y][x][4][3] -> 5D wall source (lift: with D_- applied)  (mdwf_wall_source)"""
        import torch
        assert eta.is_cuda and eta.is_contiguous()
        out = torch.empty((self.L5,) + tuple(eta.shape), dtype=eta.dtype, device=eta.device)
        _check(self.h, lib().mdwf_wall_source(self.h, eta.data_ptr(), out.data_ptr(), self._rb(eta), int(lift)))
        return out

    def wall_project(self, psi, midpoint=False):
        """5D field -> q(x) on the walls (or the midpoint field)  (mdwf_wall_project)"""
        import torch
        assert psi.is_cuda and psi.is_contiguous()
        out = torch.empty(tuple(psi.shape[1:]), dtype=psi.dtype, device=psi.device)
        _check(self.h, lib().mdwf_wall_project(self.h, psi.data_ptr(), out.data_ptr(), self._rb(psi), int(midpoint)))
        return out

    def solve(self, src, tol=1e-10, maxiter=20000):
        import torch
        assert src.is_contiguous() and src.dtype == torch.complex128
        sol = torch.empty_like(src)
        rc, it, tr = mdwf_solve(self.h, src.data_ptr(), sol.data_ptr(), tol, maxiter, host=not src.is_cuda)
        return sol, it, tr, rc

    def stat(self, key):
        return mdwf_get_stat(self.h, key)

    def flops_per_site(self):
        return mdwf_flops_per_site(self.h)

    def time_op(self, op, precision, reps=20, warmup=3):
        return mdwf_time_op(self.h, op, precision, reps, warmup)

    def fma_rates(self):
        """(FFMA, FFMA2) rates of this device in 1e12 FMA/s (mdwf_fma_rates)."""
        out = (ctypes.c_double * 2)()
        _check(self.h, lib().mdwf_fma_rates(self.h, out))
        return out[0], out[1]

    def l2_rates(self):
        """GB/s: (LDG from L2, bulk copies from L2, LDG DRAM stream, bulk-copy DRAM stream) (mdwf_l2_rates)."""
        out = (ctypes.c_double * 4)()
        _check(self.h, lib().mdwf_l2_rates(self.h, out))
        return tuple(out)

    def half_encode(self, x, via_fp64=False):
        """parity spinor [L5][Vh][4][3] -> (uint16 words [L5][Vh][24], fp32 scales [L5][Vh]) as the 16-bit format stores them"""
        import torch
        assert x.is_cuda and x.is_contiguous()
        words = torch.empty(x.shape[0], x.shape[1], 24, dtype=torch.int16, device=x.device)
        scales = torch.empty(x.shape[0], x.shape[1], dtype=torch.float32, device=x.device)
        _check(self.h, lib().mdwf_half_encode(self.h, x.data_ptr(), self._rb(x), int(via_fp64), words.data_ptr(), scales.data_ptr()))
        return words, scales

    def half_decode(self, words, scales, dtype=None):
        import torch
        dtype = dtype or torch.complex64
        out = torch.empty(words.shape[0], words.shape[1], 4, 3, dtype=dtype, device=words.device)
        _check(self.h, lib().mdwf_half_decode(self.h, words.data_ptr(), scales.data_ptr(), out.data_ptr(), self._rb(out)))
        return out

    def apply_batch(self, op, x):
        """x: (nrhs, Vh, L5, 4, 3) complex device tensor of parity vectors; returns Mpc / Mpc^dagger of each (NEXT-2)"""
        import torch
        assert x.is_contiguous() and x.is_cuda
        out = torch.empty_like(x)
        _check(self.h, lib().mdwf_apply_batch(self.h, op, x.shape[0], x.data_ptr(), out.data_ptr(), self._rb(x)))
        return out

    def time_op_batch(self, op, prec, nrhs, reps=10, warmup=3):
        o = (ctypes.c_double * 2)()
        _check(self.h, lib().mdwf_time_op_batch(self.h, op, prec.encode(), nrhs, reps, warmup, o))
        return {"ms": o[0], "launches": o[1]}

    def norm2(self, x):
        v = ctypes.c_double(0.0)
        n = x.numel() * (2 if x.is_complex() else 1)
        _check(self.h, lib().mdwf_blas_norm2(self.h, x.data_ptr(), n, self._rb(x), ctypes.byref(v)))
        return v.value

    def redot(self, x, y):
        v = ctypes.c_double(0.0)
        n = x.numel() * (2 if x.is_complex() else 1)
        _check(self.h, lib().mdwf_blas_redot(self.h, x.data_ptr(), y.data_ptr(), n, self._rb(x), ctypes.byref(v)))
        return v.value

    def axpy(self, a, x, y):
        n = x.numel() * (2 if x.is_complex() else 1)
        _check(self.h, lib().mdwf_blas_axpy(self.h, float(a), x.data_ptr(), y.data_ptr(), n, self._rb(x)))
