"""ctypes face of oracle/sstep_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this package.  It never imports the CUDA
package and the CUDA package never imports it.

Layouts: n x s blocks are column-major numpy arrays of shape (s, n) in C
order (row j of the numpy array = column j of the paper's block); small
matrices are (s, s) C-order numpy arrays.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sstep_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
SMAX = 16


def build(force: bool = False) -> str:
    """Compile the oracle with gcc -O2 (no fast-math, no contraction)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-ffp-contract=off", "-fPIC", "-shared",
                               "-o", _LIB, _SRC, "-lm"])
    return _LIB


_LIB_OMP = os.path.join(_HERE, "liboracle_omp.so")


def build_omp(force: bool = False) -> str:
    """The same source once more with -fopenmp: the all-core timing leg of bench.py's cpu_baseline (never used for
    parity -- its inner products are summed in another order)."""
    if force or not os.path.exists(_LIB_OMP) or os.path.getmtime(_LIB_OMP) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared",
                               "-o", _LIB_OMP, _SRC, "-lm"])
    return _LIB_OMP


_lib = None
_lib_omp = None


def lib(omp: bool = False):
    global _lib, _lib_omp
    if omp:
        if _lib_omp is None:
            _lib_omp = C.CDLL(build_omp())
        return _lib_omp
    if _lib is None:
        _lib = C.CDLL(build())
    return _lib


def omp_threads() -> int:
    """Threads the OpenMP build will use (OMP_NUM_THREADS or all cores this process may run on)."""
    return int(lib(omp=True).omp_get_max_threads())


def _p(a, ty=C.c_double):
    return None if a is None else a.ctypes.data_as(C.POINTER(ty))


def _f64(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64)


def _csr(rowptr, colidx, vals):
    rp = np.ascontiguousarray(rowptr, dtype=np.int32)
    ci = np.ascontiguousarray(colidx, dtype=np.int32)
    v = np.ascontiguousarray(vals, dtype=np.float64)
    return rp, ci, v


def spmv(rowptr, colidx, vals, x):
    rp, ci, v = _csr(rowptr, colidx, vals)
    n = rp.size - 1
    x = _f64(x)
    y = np.empty(n)
    lib().orc_spmv(C.c_int64(n), _p(rp, C.c_int32), _p(ci, C.c_int32), _p(v), _p(x), _p(y))
    return y


def dinv(rowptr, colidx, vals):
    rp, ci, v = _csr(rowptr, colidx, vals)
    n = rp.size - 1
    d = np.empty(n)
    rc = lib().orc_dinv(C.c_int64(n), _p(rp, C.c_int32), _p(ci, C.c_int32), _p(v), _p(d))
    if rc:
        raise ValueError("missing or non-positive diagonal entry")
    return d


def mpk(rowptr, colidx, vals, dinv_, r, s, basis=0):
    """Alg. 4: returns R, AR as (s, n) arrays (row j = column j of the block)."""
    rp, ci, v = _csr(rowptr, colidx, vals)
    n = rp.size - 1
    R = np.empty((s, n)); AR = np.empty((s, n))
    d = _f64(dinv_); r = _f64(r)
    lib().orc_mpk(C.c_int64(n), _p(rp, C.c_int32), _p(ci, C.c_int32), _p(v), _p(d), _p(r),
                  C.c_int(s), C.c_int(basis), _p(R), _p(AR))
    return R, AR


def gram(R, AR, AP, r):
    """M = R^T AR, C = AP^T R, m = R^T r (AP None -> C = 0)."""
    R = _f64(R); AR = _f64(AR); AP = _f64(AP); r = _f64(r)
    s, n = R.shape
    M = np.empty((s, s)); Cm = np.empty((s, s)); m = np.empty(s)
    lib().orc_gram(C.c_int64(n), C.c_int(s), _p(R), _p(AR), _p(AP), _p(r), _p(M), _p(Cm), _p(m))
    return M, Cm, m


def cvm(R, AR, r):
    R = _f64(R); AR = _f64(AR); r = _f64(r)
    s, n = R.shape
    vm = np.empty(2 * s)
    lib().orc_cvm(C.c_int64(n), C.c_int(s), _p(R), _p(AR), _p(r), _p(vm))
    return vm


def cvm_fused(R, AR, r):
    """The 2s moments where the MPK produces them: mu^0 = R_1.r, mu^{2j-1} = R_j.AR_j, mu^{2j} = R_{j+1}.AR_j."""
    R = _f64(R); AR = _f64(AR); r = _f64(r)
    s, n = R.shape
    vm = np.empty(2 * s)
    lib().orc_cvm_fused(C.c_int64(n), C.c_int(s), _p(R), _p(AR), _p(r), _p(vm))
    return vm


def chol(W):
    W = _f64(W); s = W.shape[0]
    L = np.empty((s, s))
    st = lib().orc_chol(C.c_int(s), _p(W), _p(L))
    return st, L


def chol_solve(L, B):
    L = _f64(L); s = L.shape[0]
    B2 = _f64(B).reshape(s, -1)
    X = np.empty_like(B2)
    lib().orc_chol_solve(C.c_int(s), _p(L), C.c_int(B2.shape[1]), _p(B2), _p(X))
    return X.reshape(np.shape(B))


def small_solve(M, Cm, m, Wprev, first=False):
    """Returns status, beta, alpha, W (Gram-form scalar work)."""
    M = _f64(M); Cm = _f64(Cm); m = _f64(m); Wprev = _f64(Wprev)
    s = M.shape[0]
    beta = np.empty((s, s)); alpha = np.empty(s); W = np.empty((s, s))
    st = lib().orc_small_solve(C.c_int(s), C.c_int(1 if first else 0), _p(M), _p(Cm), _p(m), _p(Wprev),
                               _p(beta), _p(alpha), _p(W))
    return st, beta, alpha, W


def sw(vm, alpha_prev, W_prev):
    """Alg. 6: returns status, beta, alpha, W from the 2s moments and the previous alpha, W."""
    vm = _f64(vm); s = vm.size // 2
    alpha = _f64(alpha_prev).copy(); W = _f64(W_prev).copy(); beta = np.empty((s, s))
    st = lib().orc_sw(C.c_int(s), _p(vm), _p(alpha), _p(beta), _p(W))
    return st, beta, alpha, W


def update(R, AR, P, AP, x, r, beta, alpha):
    """Alg. 3 l.17-21; returns new (P, AP, x, r) -- inputs are not modified."""
    R = _f64(R); AR = _f64(AR)
    P = _f64(P).copy(); AP = _f64(AP).copy(); x = _f64(x).copy(); r = _f64(r).copy()
    beta = _f64(beta); alpha = _f64(alpha)
    s, n = R.shape
    lib().orc_update(C.c_int64(n), C.c_int(s), _p(R), _p(AR), _p(P), _p(AP), _p(x), _p(r), _p(beta), _p(alpha))
    return P, AP, x, r


def _solver_common(fn, rowptr, colidx, vals, b, x0, rtol, maxit, pre_args, history, xhist_cap):
    rp, ci, v = _csr(rowptr, colidx, vals)
    n = rp.size - 1
    b = _f64(b); x0 = _f64(x0)
    x = np.empty(n)
    iters = C.c_int(0); relres = C.c_double(0.0)
    hist = np.full(maxit, np.nan) if history else None
    xh = np.empty((xhist_cap, n)) if xhist_cap else None
    st = fn(C.c_int64(n), _p(rp, C.c_int32), _p(ci, C.c_int32), _p(v), _p(b), _p(x0), *pre_args,
            C.c_double(rtol), C.c_int(maxit), _p(x), C.byref(iters), C.byref(relres), _p(hist), _p(xh),
            C.c_int(xhist_cap))
    out = dict(status=int(st), x=x, iters=iters.value, relres=relres.value)
    if history:
        out["hist"] = hist[:iters.value]
    if xhist_cap:
        out["xhist"] = xh[:min(iters.value, xhist_cap)]
    return out


def pcg(rowptr, colidx, vals, b, x0=None, rtol=1e-8, maxit=2000, history=False, xhist_cap=0):
    """Alg. 1 PCG-HS with B = diag(A)."""
    return _solver_common(lib().orc_pcg, rowptr, colidx, vals, b, x0, rtol, maxit, (), history, xhist_cap)


def pfcg(rowptr, colidx, vals, b, x0=None, rtol=1e-8, maxit=2000, history=False, xhist_cap=0):
    """Alg. 2 PFCG-NN with B = diag(A)."""
    return _solver_common(lib().orc_pfcg, rowptr, colidx, vals, b, x0, rtol, maxit, (), history, xhist_cap)


def sstep_timed(rowptr, colidx, vals, b, s, iters, omp=False, basis=0):
    """bench.py's cpu_baseline: `iters` outer iterations of orc_sstep (Gram form, rtol = 0) with the wall clock taken
    inside the C loop; returns (seconds per outer iteration without the start-up, start-up seconds, result dict).
    omp = True runs the -fopenmp build of the same source on all host cores."""
    import time
    L = lib(omp)
    tlog = np.zeros(iters + 1)
    L.orc_set_time_log(_p(tlog), C.c_int(iters + 1))
    t0 = time.perf_counter()
    try:
        out = _solver_common(L.orc_sstep, rowptr, colidx, vals, b, None, 0.0, iters, (C.c_int(s), C.c_int(0), C.c_int(basis)),
                             False, 0)
    finally:
        L.orc_set_time_log(None, C.c_int(0))
    total = time.perf_counter() - t0
    assert out["iters"] == iters, out
    per = (tlog[iters] - tlog[0]) / iters
    return per, total - per * iters, out


def sstep(rowptr, colidx, vals, b, s, x0=None, rtol=1e-8, maxit=2000, form="gram", basis=0,
          history=False, xhist_cap=0, replace_every=0):
    """Alg. 3 PCGs; form 'gram' (O2), 'moment' (O3, Alg. 5 + Alg. 6) or 'moment_fused' (O3 with the moments taken
    in the MPK, cvm_fused); iters = outer iterations.  replace_every = R > 0: residual replacement every R outer
    iterations (orc_sstep_rr; with history, hist[k] is the replaced residual on those iterations)."""
    f = {"gram": 0, "moment": 1, "moment_fused": 2}[form]
    if replace_every:
        return _solver_common(lib().orc_sstep_rr, rowptr, colidx, vals, b, x0, rtol, maxit,
                              (C.c_int(s), C.c_int(f), C.c_int(basis), C.c_int(replace_every)), history, xhist_cap)
    return _solver_common(lib().orc_sstep, rowptr, colidx, vals, b, x0, rtol, maxit,
                          (C.c_int(s), C.c_int(f), C.c_int(basis)), history, xhist_cap)
