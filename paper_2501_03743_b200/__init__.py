"""paper_2501_03743_b200 -- thin Python binding of the C-ABI library libsstepcg.so (include/sstep_cg.h).

Argument marshalling only: every step of the hot path (Jacobi-fused CSR SpMV / matrix-powers kernel, fused
Gram blocks, on-device s x s solves, fused block updates, graph-captured solve loop) runs in the hand-written
sm_100a kernels under csrc/.  PyTorch is used for device memory and streams.  There is no CPU fallback: if the
library is missing or no B200-class device is present, the calls raise.

Block conventions of the Python face: an n x s block is a torch tensor of shape (s, n) whose row j is column j
of the paper's block.  The R / AR blocks are passed to the kernels as they are ("column-major");
P / AP are transposed to the interleaved (n, s) layout the kernels use.
"""
from __future__ import annotations

import ctypes as C
import os

from .build import LIB, build_library

__all__ = ["SStepCG", "SStepCGError", "load_library", "STATUS_NAMES", "EXPORTED_SYMBOLS"]

SMAX = 16
STATUS_NAMES = {0: "converged", 1: "maxit", 2: "breakdown"}
EXPORTED_SYMBOLS = [
    "sstep_cg_create", "sstep_cg_setup", "sstep_cg_set_option", "sstep_cg_get_info", "sstep_cg_solve",
    "sstep_cg_solve_begin", "sstep_cg_iterate", "sstep_cg_solve_end", "sstep_cg_solve_peek", "sstep_cg_profile_outer",
    "sstep_cg_measure_bandwidth", "sstep_cg_test_small_solve_carried", "sstep_cg_test_division", "sstep_cg_solve_host", "sstep_cg_destroy",
    "sstep_cg_last_error", "sstep_cg_test_spmv", "sstep_cg_test_mpk", "sstep_cg_test_mpk_moments", "sstep_cg_test_sw",
    "sstep_cg_test_gram",
    "sstep_cg_test_small_solve", "sstep_cg_test_update", "sstep_cg_test_read_state",
    "sstep_cg_get_permutation", "sstep_cg_gram_noalloc",
]


class SStepCGError(RuntimeError):
    pass


class _Result(C.Structure):
    _fields_ = [("status", C.c_int32), ("outer_iters", C.c_int32), ("cg_equiv_iters", C.c_int64),
                ("relres", C.c_double), ("r0_norm", C.c_double), ("solve_seconds", C.c_double),
                ("kernel_launches", C.c_int64)]

    def as_dict(self):
        d = {k: getattr(self, k) for k, _ in self._fields_}
        d["status_name"] = STATUS_NAMES.get(d["status"], str(d["status"]))
        return d


_lib = None


def load_library(build: bool = True):
    """dlopen libsstepcg.so (building it with nvcc first if it is missing or stale) and declare the prototypes."""
    global _lib
    if _lib is not None:
        return _lib
    if build:
        build_library()
    if not os.path.exists(LIB):
        raise SStepCGError(f"{LIB} is missing: run `python -c 'import __graft_entry__ as g; g.build()'`")
    lib = C.CDLL(LIB)
    vp, i64, i32, dbl = C.c_void_p, C.c_int64, C.c_int, C.c_double
    lib.sstep_cg_create.argtypes = [C.POINTER(vp), i32, vp]
    lib.sstep_cg_setup.argtypes = [vp, i64, i64, vp, vp, vp, i32]
    lib.sstep_cg_set_option.argtypes = [vp, C.c_char_p, i64]
    lib.sstep_cg_get_info.argtypes = [vp, C.c_char_p, C.POINTER(i64)]
    lib.sstep_cg_solve.argtypes = [vp, vp, vp, vp, dbl, i32, C.POINTER(_Result)]
    lib.sstep_cg_solve_begin.argtypes = [vp, vp, vp, dbl]
    lib.sstep_cg_iterate.argtypes = [vp, i32]
    lib.sstep_cg_solve_end.argtypes = [vp, vp, C.POINTER(_Result)]
    lib.sstep_cg_solve_peek.argtypes = [vp, C.POINTER(_Result)]
    lib.sstep_cg_profile_outer.argtypes = [vp, i32, C.POINTER(dbl)]
    lib.sstep_cg_measure_bandwidth.argtypes = [vp, i32, i64, i32, i32, C.POINTER(dbl)]
    lib.sstep_cg_test_small_solve_carried.argtypes = [vp] + [vp] * 9
    lib.sstep_cg_test_division.argtypes = [vp, C.c_int64, vp, vp, vp]
    lib.sstep_cg_solve_host.argtypes = [vp, i64, i64, vp, vp, vp, vp, vp, vp, i32, dbl, i32, C.POINTER(_Result)]
    lib.sstep_cg_destroy.argtypes = [vp]
    lib.sstep_cg_last_error.argtypes = [vp]
    lib.sstep_cg_last_error.restype = C.c_char_p
    lib.sstep_cg_test_spmv.argtypes = [vp, vp, vp, vp]
    lib.sstep_cg_test_mpk.argtypes = [vp, vp, vp, vp]
    lib.sstep_cg_test_mpk_moments.argtypes = [vp, vp, vp, vp, vp]
    lib.sstep_cg_test_sw.argtypes = [vp, vp, i32, vp, vp, vp, vp]
    lib.sstep_cg_test_gram.argtypes = [vp] + [vp] * 7
    lib.sstep_cg_test_small_solve.argtypes = [vp] + [vp] * 8
    lib.sstep_cg_test_update.argtypes = [vp] + [vp] * 9
    lib.sstep_cg_test_read_state.argtypes = [vp, C.c_char_p, vp, i64]
    lib.sstep_cg_get_permutation.argtypes = [vp, vp]
    lib.sstep_cg_gram_noalloc.argtypes = [vp, i64, i32] + [vp] * 7
    for name in EXPORTED_SYMBOLS:
        if name != "sstep_cg_last_error":
            getattr(lib, name).restype = C.c_int
    _lib = lib
    return lib


def _torch():
    import torch
    return torch


class SStepCG:
    """One solver handle (sstep_cg_create ... sstep_cg_destroy)."""

    def __init__(self, device: int = 0, stream: int | None = None, **options):
        torch = _torch()
        if not torch.cuda.is_available():
            raise SStepCGError("no CUDA device: the s-step PCG path has no CPU fallback")
        self._lib = load_library()
        self.device = device
        if stream is None:
            stream = torch.cuda.current_stream(device).cuda_stream
        self._h = C.c_void_p()
        rc = self._lib.sstep_cg_create(C.byref(self._h), device, C.c_void_p(stream))
        if rc:
            self._h = None
            raise SStepCGError(f"sstep_cg_create failed ({rc}): needs an sm_100 device")
        self._keep = []
        self.n = self.s = None
        for k, v in options.items():
            self.set_option(k, v)

    # ------------------------------------------------------------------ helpers
    def _check(self, rc, what):
        if rc < 0:
            raise SStepCGError(f"{what} failed ({rc}): {self._lib.sstep_cg_last_error(self._h).decode()}")
        return rc

    def _dev(self, t, dtype, name, numel=None):
        torch = _torch()
        if t is None:
            return None
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == dtype and t.is_contiguous()):
            raise SStepCGError(f"{name}: need a contiguous CUDA tensor of dtype {dtype}")
        if numel is not None and t.numel() != numel:
            raise SStepCGError(f"{name}: expected {numel} elements, got {t.numel()}")
        return t

    @staticmethod
    def _ptr(t):
        return C.c_void_p(0 if t is None else t.data_ptr())

    def close(self):
        if getattr(self, "_h", None):
            self._lib.sstep_cg_destroy(self._h)
            self._h = None
            self._keep = []

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    # ------------------------------------------------------------------ API (same names as the C ABI)
    def set_option(self, key: str, value: int):
        self._check(self._lib.sstep_cg_set_option(self._h, key.encode(), int(value)), "sstep_cg_set_option")

    def get_info(self, key: str) -> int:
        v = C.c_int64(0)
        self._check(self._lib.sstep_cg_get_info(self._h, key.encode(), C.byref(v)), "sstep_cg_get_info")
        return v.value

    def setup(self, rowptr, colidx, vals, s: int):
        torch = _torch()
        rowptr = self._dev(rowptr, torch.int32, "rowptr")
        colidx = self._dev(colidx, torch.int32, "colidx")
        vals = self._dev(vals, torch.float64, "vals", colidx.numel())
        n, nnz = rowptr.numel() - 1, colidx.numel()
        self._check(self._lib.sstep_cg_setup(self._h, n, nnz, self._ptr(rowptr), self._ptr(colidx), self._ptr(vals), int(s)),
                    "sstep_cg_setup")
        self._keep = [rowptr, colidx, vals]  # borrowed by the library until the next setup / destroy
        self.n, self.nnz, self.s = n, nnz, int(s)

    def get_permutation(self):
        """perm[i'] = the caller's index of the solver's row i' (identity unless setup reordered the matrix)."""
        torch = _torch()
        perm = torch.empty(self.n, dtype=torch.int32, device=f"cuda:{self.device}")
        self._check(self._lib.sstep_cg_get_permutation(self._h, self._ptr(perm)), "sstep_cg_get_permutation")
        return perm

    def solve(self, b, x0=None, rtol: float = 1e-8, maxit: int = 2000, out=None):
        """sstep_cg_solve; `out` = the tensor that receives x (may be x0 itself: the ABI allows the alias)."""
        torch = _torch()
        b = self._dev(b, torch.float64, "b", self.n)
        x0 = self._dev(x0, torch.float64, "x0", self.n)
        x = torch.empty_like(b) if out is None else self._dev(out, torch.float64, "out", self.n)
        res = _Result()
        self._check(self._lib.sstep_cg_solve(self._h, self._ptr(b), self._ptr(x0), self._ptr(x), float(rtol), int(maxit),
                                             C.byref(res)), "sstep_cg_solve")
        return x, res.as_dict()

    def solve_begin(self, b, x0=None, rtol: float = 0.0):
        torch = _torch()
        b = self._dev(b, torch.float64, "b", self.n)
        x0 = self._dev(x0, torch.float64, "x0", self.n)
        self._check(self._lib.sstep_cg_solve_begin(self._h, self._ptr(b), self._ptr(x0), float(rtol)), "sstep_cg_solve_begin")
        self._solve_keep = [b, x0]

    def iterate(self, k_outer: int):
        self._check(self._lib.sstep_cg_iterate(self._h, int(k_outer)), "sstep_cg_iterate")

    def solve_peek(self):
        """Where the solve in progress stands (status -1 = still running); the solve goes on."""
        res = _Result()
        self._check(self._lib.sstep_cg_solve_peek(self._h, C.byref(res)), "sstep_cg_solve_peek")
        d = res.as_dict()
        d["status_name"] = "running" if d["status"] == -1 else d["status_name"]
        return d

    def measure_bandwidth(self, variant: int, nbytes: int, passes: int = 1, reps: int = 5):
        """(best, mean) GB/s of the library's streaming kernels (see sstep_cg.h): 0 ldg reads, 1 / 3 bulk reads, 2 copy."""
        out = (C.c_double * 2)()
        self._check(self._lib.sstep_cg_measure_bandwidth(self._h, int(variant), int(nbytes), int(passes), int(reps), out),
                    "sstep_cg_measure_bandwidth")
        return float(out[0]), float(out[1])

    def profile_outer(self, reps: int):
        """Per-kernel-class device milliseconds of `reps` un-graphed outer iterations: (spmv, gram, update)."""
        ms = (C.c_double * 3)()
        self._check(self._lib.sstep_cg_profile_outer(self._h, int(reps), ms), "sstep_cg_profile_outer")
        return float(ms[0]), float(ms[1]), float(ms[2])

    def solve_end(self, want_x: bool = True):
        torch = _torch()
        x = torch.empty(self.n, dtype=torch.float64, device=f"cuda:{self.device}") if want_x else None
        res = _Result()
        self._check(self._lib.sstep_cg_solve_end(self._h, self._ptr(x), C.byref(res)), "sstep_cg_solve_end")
        return x, res.as_dict()

    def solve_host(self, rowptr, colidx, vals, b, s: int, x0=None, rtol: float = 1e-8, maxit: int = 2000, x_out=None):
        """End-to-end call with HOST buffers (CPU torch tensors, ideally pinned)."""
        torch = _torch()

        def host(t, dtype, name):
            if t is None:
                return None
            if not (isinstance(t, torch.Tensor) and not t.is_cuda and t.dtype == dtype and t.is_contiguous()):
                raise SStepCGError(f"{name}: need a contiguous CPU tensor of dtype {dtype}")
            return t
        rowptr, colidx = host(rowptr, torch.int32, "rowptr"), host(colidx, torch.int32, "colidx")
        vals, b, x0 = host(vals, torch.float64, "vals"), host(b, torch.float64, "b"), host(x0, torch.float64, "x0")
        n, nnz = rowptr.numel() - 1, colidx.numel()
        x = x_out if x_out is not None else torch.empty(n, dtype=torch.float64)
        res = _Result()
        self._check(self._lib.sstep_cg_solve_host(self._h, n, nnz, self._ptr(rowptr), self._ptr(colidx), self._ptr(vals),
                                                  self._ptr(b), self._ptr(x0), self._ptr(x), int(s), float(rtol), int(maxit),
                                                  C.byref(res)), "sstep_cg_solve_host")
        self.n, self.nnz, self.s = n, nnz, int(s)
        return x, res.as_dict()

    # ------------------------------------------------------------------ test hooks
    def test_spmv(self, x, jacobi: bool = True):
        torch = _torch()
        x = self._dev(x, torch.float64, "x", self.n)
        y = torch.empty_like(x)
        yjac = torch.empty_like(x) if jacobi else None
        self._check(self._lib.sstep_cg_test_spmv(self._h, self._ptr(x), self._ptr(y), self._ptr(yjac)), "sstep_cg_test_spmv")
        return y, yjac

    def test_mpk(self, r):
        torch = _torch()
        r = self._dev(r, torch.float64, "r", self.n)
        R = torch.empty((self.s, self.n), dtype=torch.float64, device=r.device)
        AR = torch.empty_like(R)
        self._check(self._lib.sstep_cg_test_mpk(self._h, self._ptr(r), self._ptr(R), self._ptr(AR)), "sstep_cg_test_mpk")
        return R, AR

    def test_mpk_moments(self, r):
        """Moment form: R, AR as in test_mpk plus the 2s moments vm[k] = mu^k left by the SpMV epilogues."""
        torch = _torch()
        r = self._dev(r, torch.float64, "r", self.n)
        R = torch.empty((self.s, self.n), dtype=torch.float64, device=r.device)
        AR = torch.empty_like(R)
        vm = torch.empty(2 * self.s, dtype=torch.float64, device=r.device)
        self._check(self._lib.sstep_cg_test_mpk_moments(self._h, self._ptr(r), self._ptr(R), self._ptr(AR), self._ptr(vm)),
                    "sstep_cg_test_mpk_moments")
        return R, AR, vm

    def test_sw(self, vm, alpha_prev=None, W_prev=None):
        """Alg. 6: (status, beta, alpha, W); alpha_prev / W_prev None = first outer iteration."""
        torch = _torch()
        s = self.s
        vm = self._dev(vm, torch.float64, "vm", 2 * s)
        first = alpha_prev is None
        alpha = torch.zeros(s, dtype=torch.float64, device=vm.device) if first else self._dev(alpha_prev, torch.float64, "alpha", s).clone()
        W = torch.zeros((s, s), dtype=torch.float64, device=vm.device) if first else self._dev(W_prev, torch.float64, "W", s * s).clone()
        beta = torch.zeros((s, s), dtype=torch.float64, device=vm.device)
        st = torch.zeros(1, dtype=torch.int32, device=vm.device)
        self._check(self._lib.sstep_cg_test_sw(self._h, self._ptr(vm), 1 if first else 0, self._ptr(beta), self._ptr(alpha),
                                               self._ptr(W), self._ptr(st)), "sstep_cg_test_sw")
        return int(st.item()), beta, alpha, W

    def test_gram(self, R, AR, AP, r):
        torch = _torch()
        ns = self.n * self.s
        R, AR = self._dev(R, torch.float64, "R", ns), self._dev(AR, torch.float64, "AR", ns)
        AP_il = self._dev(AP, torch.float64, "AP", ns).t().contiguous()      # (s, n) -> interleaved (n, s)
        r = self._dev(r, torch.float64, "r", self.n)
        s = self.s
        M = torch.empty((s, s), dtype=torch.float64, device=r.device)
        Cm = torch.empty_like(M)
        m = torch.empty(s, dtype=torch.float64, device=r.device)
        self._check(self._lib.sstep_cg_test_gram(self._h, self._ptr(R), self._ptr(AR), self._ptr(AP_il), self._ptr(r),
                                                 self._ptr(M), self._ptr(Cm), self._ptr(m)), "sstep_cg_test_gram")
        return M, Cm, m

    def gram_noalloc(self, R, AR, AP_il, r, M, Cm, m):
        """sstep_cg_gram_noalloc: a2 on the library's static scratch -- no allocation anywhere (the caller passes every
        buffer, AP already in the interleaved (n, s) layout; outputs M, Cm (s, s) and m (s) are filled asynchronously on
        the handle's stream).  Works after create alone; s <= 8."""
        torch = _torch()
        s, n = R.shape
        ns = n * s
        R, AR = self._dev(R, torch.float64, "R", ns), self._dev(AR, torch.float64, "AR", ns)
        AP_il = self._dev(AP_il, torch.float64, "AP_il", ns)
        r = self._dev(r, torch.float64, "r", n)
        M, Cm = self._dev(M, torch.float64, "M", s * s), self._dev(Cm, torch.float64, "C", s * s)
        m = self._dev(m, torch.float64, "m", s)
        self._check(self._lib.sstep_cg_gram_noalloc(self._h, n, s, self._ptr(R), self._ptr(AR), self._ptr(AP_il), self._ptr(r),
                                                    self._ptr(M), self._ptr(Cm), self._ptr(m)), "sstep_cg_gram_noalloc")

    def test_small_solve(self, M, Cm, m, Wprev):
        torch = _torch()
        s = self.s
        M, Cm, Wprev = (self._dev(t, torch.float64, nm, s * s) for t, nm in ((M, "M"), (Cm, "C"), (Wprev, "Wprev")))
        m = self._dev(m, torch.float64, "m", s)
        beta = torch.zeros((s, s), dtype=torch.float64, device=M.device)
        alpha = torch.zeros(s, dtype=torch.float64, device=M.device)
        W = torch.zeros_like(beta)
        st = torch.zeros(1, dtype=torch.int32, device=M.device)
        self._check(self._lib.sstep_cg_test_small_solve(self._h, self._ptr(M), self._ptr(Cm), self._ptr(m), self._ptr(Wprev),
                                                        self._ptr(beta), self._ptr(alpha), self._ptr(W), self._ptr(st)),
                    "sstep_cg_test_small_solve")
        return int(st.item()), beta, alpha, W

    def test_small_solve_carried(self, M, Cm, m, Lprev):
        """a3 with the carried Cholesky factor: (status, beta, alpha, W, L)."""
        torch = _torch()
        s = self.s
        M, Cm, Lprev = (self._dev(t, torch.float64, nm, s * s) for t, nm in ((M, "M"), (Cm, "C"), (Lprev, "Lprev")))
        m = self._dev(m, torch.float64, "m", s)
        beta = torch.zeros((s, s), dtype=torch.float64, device=M.device)
        alpha = torch.zeros(s, dtype=torch.float64, device=M.device)
        W, L = torch.zeros_like(beta), torch.zeros_like(beta)
        st = torch.zeros(1, dtype=torch.int32, device=M.device)
        self._check(self._lib.sstep_cg_test_small_solve_carried(self._h, self._ptr(M), self._ptr(Cm), self._ptr(m), self._ptr(Lprev),
                                                                self._ptr(beta), self._ptr(alpha), self._ptr(W), self._ptr(L),
                                                                self._ptr(st)), "sstep_cg_test_small_solve_carried")
        return int(st.item()), beta, alpha, W, L

    def test_division(self, a, b):
        """q = a / b elementwise by the prepared-divisor division of the register-resident solves (see sstep_cg.h)."""
        torch = _torch()
        n = a.numel()
        a, b = self._dev(a, torch.float64, "a", n), self._dev(b, torch.float64, "b", n)
        q = torch.empty(n, dtype=torch.float64, device=a.device)
        self._check(self._lib.sstep_cg_test_division(self._h, n, self._ptr(a), self._ptr(b), self._ptr(q)), "sstep_cg_test_division")
        return q

    def test_read_state(self, name: str):
        """One internal array of the current solve state (see sstep_cg.h): blocks come back as (s, n) tensors."""
        torch = _torch()
        s, n = self.s, self.n
        shape = {"R": (s, n), "AR": (s, n), "P": (n, s), "AP": (n, s), "x": (n,), "r": (n,), "M": (s, s), "C": (s, s),
                 "W": (s, s), "beta": (s, s), "m": (s,), "alpha": (s,)}[name]
        out = torch.empty(shape, dtype=torch.float64, device=f"cuda:{self.device}")
        self._check(self._lib.sstep_cg_test_read_state(self._h, name.encode(), self._ptr(out), out.numel()),
                    "sstep_cg_test_read_state")
        return out.t().contiguous() if name in ("P", "AP") else out

    def test_update(self, R, AR, P, AP, x, r, beta, alpha):
        """Returns new (P, AP, x, r) as (s, n)/(n,) tensors plus R1 = D^-1 r_new and rho = ||r_new||^2; inputs are not modified."""
        torch = _torch()
        ns, s = self.n * self.s, self.s
        R = self._dev(R, torch.float64, "R", ns).clone()
        AR = self._dev(AR, torch.float64, "AR", ns)
        P_il = self._dev(P, torch.float64, "P", ns).t().contiguous()
        AP_il = self._dev(AP, torch.float64, "AP", ns).t().contiguous()
        x = self._dev(x, torch.float64, "x", self.n).clone()
        r = self._dev(r, torch.float64, "r", self.n).clone()
        beta = self._dev(beta, torch.float64, "beta", s * s)
        alpha = self._dev(alpha, torch.float64, "alpha", s)
        rho = torch.zeros(1, dtype=torch.float64, device=x.device)
        self._check(self._lib.sstep_cg_test_update(self._h, self._ptr(R), self._ptr(AR), self._ptr(P_il), self._ptr(AP_il),
                                                   self._ptr(x), self._ptr(r), self._ptr(beta), self._ptr(alpha), self._ptr(rho)),
                    "sstep_cg_test_update")
        return P_il.t().contiguous(), AP_il.t().contiguous(), x, r, R[0].clone(), float(rho.item())
