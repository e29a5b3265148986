"""Pins for the per-step oracle functions (oracle/sstep_oracle.c) against what
the mathematics fixes: dense definitions on tiny systems, the closed-form
eigenpairs of the Poisson stencils, the closed-form inverse of the Hilbert
matrix, library routines (numpy.linalg, scipy CSR) and the invariants the
paper states.  No GPU, no CUDA code."""
from math import comb

import numpy as np
import pytest
import scipy.sparse as sp

import sstep_inputs as gen


def dense_of(rp, ci, v):
    n = rp.size - 1
    return sp.csr_matrix((v, ci, rp), shape=(n, n)).toarray()


def poisson7_eigvec(N, ix, iy, iz):
    k = np.arange(1, N + 1)
    sx, sy, sz = (np.sin(i * k * np.pi / (N + 1)) for i in (ix, iy, iz))
    vec = (sz[:, None, None] * sy[None, :, None] * sx[None, None, :]).ravel()
    lam = 6 - 2 * sum(np.cos(i * np.pi / (N + 1)) for i in (ix, iy, iz))
    return vec, lam


# ------------------------------------------------------------------ SpMV / Jacobi
def test_spmv_vs_dense_and_scipy(oracle_mod):
    rp, ci, v, A = gen.random_spd_csr(64, 0.15, 1, max_row=50)
    x = np.random.default_rng(2).uniform(-1, 1, 64)
    y = oracle_mod.spmv(rp, ci, v, x)
    scale = np.abs(A) @ np.abs(x)
    assert np.all(np.abs(y - A @ x) <= 1e-15 * scale)
    ysp = sp.csr_matrix((v, ci, rp), shape=(64, 64)) @ x
    assert np.all(np.abs(y - ysp) <= 1e-15 * scale)
    assert np.allclose(oracle_mod.dinv(rp, ci, v), 1.0 / np.diag(A), rtol=1e-16)


@pytest.mark.parametrize("N,idx", [(9, (1, 1, 1)), (9, (2, 5, 9)), (16, (3, 1, 7))])
def test_spmv_poisson_eigenvector(oracle_mod, N, idx):
    rp, ci, v = gen.poisson7(N)
    vec, lam = poisson7_eigvec(N, *idx)
    y = oracle_mod.spmv(rp, ci, v, vec)
    assert np.abs(y - lam * vec).max() <= 2e-14 * np.abs(vec).max()


def test_spmv_poisson27_eigenvector(oracle_mod):
    N = 8
    rp, ci, v = gen.poisson27(N)
    k = np.arange(1, N + 1)
    idx = (2, 3, 1)
    s3 = [np.sin(i * k * np.pi / (N + 1)) for i in idx]
    vec = (s3[2][:, None, None] * s3[1][None, :, None] * s3[0][None, None, :]).ravel()
    lam = 27 - np.prod([1 + 2 * np.cos(i * np.pi / (N + 1)) for i in idx])
    y = oracle_mod.spmv(rp, ci, v, vec)
    assert np.abs(y - lam * vec).max() <= 1e-13


def test_dinv_rejects_bad_diagonal(oracle_mod):
    rp = np.array([0, 1, 2], dtype=np.int32)
    ci = np.array([1, 0], dtype=np.int32)
    with pytest.raises(ValueError):
        oracle_mod.dinv(rp, ci, np.array([1.0, 1.0]))


# ------------------------------------------------------------------ MPK (Alg. 4)
@pytest.mark.parametrize("s", [1, 2, 4, 8])
def test_mpk_eigenvector_closed_form(oracle_mod, s):
    N = 10
    rp, ci, v = gen.poisson7(N)
    vec, lam = poisson7_eigvec(N, 2, 3, 4)
    d = 6.0
    R, AR = oracle_mod.mpk(rp, ci, v, oracle_mod.dinv(rp, ci, v), vec, s)
    for j in range(s):
        Rj = (lam / d) ** j * vec / d
        # a rounding perturbation is not an eigenvector: each application can amplify it by ||A||/lam <= 12/lam
        # relative to the shrinking exact vector (the monomial-basis growth PAPER.md:154-156 warns about)
        tol = 4e-16 * (12.0 / lam) ** (j + 1)
        assert np.abs(R[j] - Rj).max() <= tol * np.abs(Rj).max()
        assert np.abs(AR[j] - lam * Rj).max() <= tol * np.abs(lam * Rj).max()


def test_mpk_column_relations_dense(oracle_mod):
    rp, ci, v, A = gen.random_spd_csr(48, 0.2, 3)
    r = np.random.default_rng(4).uniform(-1, 1, 48)
    dinv = 1.0 / np.diag(A)
    s = 5
    R, AR = oracle_mod.mpk(rp, ci, v, dinv, r, s)
    Z = np.diag(dinv) @ A                      # B^{-1} A
    for j in range(s):
        Rj = np.linalg.matrix_power(Z, j) @ (dinv * r)   # (B^-1 A)^j B^-1 r
        assert np.allclose(R[j], Rj, rtol=1e-12, atol=1e-14)
        assert np.allclose(AR[j], A @ Rj, rtol=1e-12, atol=1e-14)


def test_mpk_chebyshev_basis_dense(oracle_mod):
    rp, ci, v, A = gen.random_spd_csr(40, 0.2, 5)
    r = np.random.default_rng(6).uniform(-1, 1, 40)
    dinv = 1.0 / np.diag(A)
    s = 6
    R, AR = oracle_mod.mpk(rp, ci, v, dinv, r, s, basis=1)
    Z = np.diag(dinv) @ A - np.eye(40)
    T = [dinv * r, Z @ (dinv * r)]
    for j in range(2, s):
        T.append(2 * Z @ T[-1] - T[-2])       # Chebyshev three-term recurrence on [-1, 1]
    for j in range(s):
        assert np.allclose(R[j], T[j], rtol=1e-12, atol=1e-14)
        assert np.allclose(AR[j], A @ T[j], rtol=1e-12, atol=1e-14)


# ------------------------------------------------------------------ Gram blocks
def test_gram_dense_definition(oracle_mod):
    rng = np.random.default_rng(7)
    n, s = 257, 4
    R, AR, AP = (rng.uniform(-1, 1, (s, n)) for _ in range(3))
    r = rng.uniform(-1, 1, n)
    M, C, m = oracle_mod.gram(R, AR, AP, r)
    # float128 evaluation of the definitions (not the oracle's loop)
    Rl, ARl, APl, rl = (a.astype(np.longdouble) for a in (R, AR, AP, r))
    assert np.allclose(M, (Rl @ ARl.T).astype(float), rtol=0, atol=1e-14 * n)
    assert np.allclose(C, (APl @ Rl.T).astype(float), rtol=0, atol=1e-14 * n)
    assert np.allclose(m, (Rl @ rl).astype(float), rtol=0, atol=1e-14 * n)
    # C is NOT symmetric for generic inputs: a transposed operand would fail here
    assert np.abs(C - C.T).max() > 1e-3
    M0, C0, m0 = oracle_mod.gram(R, AR, None, r)
    assert np.all(C0 == 0) and np.array_equal(M0, M) and np.array_equal(m0, m)


@pytest.mark.parametrize("s", [2, 4])
def test_gram_eigenvector_closed_form_and_hankel(oracle_mod, s):
    N = 9
    rp, ci, v = gen.poisson7(N)
    vec, lam = poisson7_eigvec(N, 1, 2, 3)
    dinv = oracle_mod.dinv(rp, ci, v)
    R, AR = oracle_mod.mpk(rp, ci, v, dinv, vec, s)
    M, C, m = oracle_mod.gram(R, AR, None, vec)
    nr2 = vec @ vec
    for i in range(s):
        assert np.isclose(m[i], lam ** i / 6.0 ** (i + 1) * nr2, rtol=1e-12)     # mu^{i}
        for j in range(s):
            assert np.isclose(M[i, j], lam ** (i + j + 1) / 6.0 ** (i + j + 2) * nr2, rtol=1e-12)
    # generic residual: M symmetric Hankel in the moments (Eq. 4); cvm picks its last column
    r = np.random.default_rng(8).uniform(-1, 1, N ** 3)
    R, AR = oracle_mod.mpk(rp, ci, v, dinv, r, s)
    M, C, m = oracle_mod.gram(R, AR, None, r)
    vm = oracle_mod.cvm(R, AR, r)
    assert np.allclose(vm[:s], m, rtol=1e-15) and np.allclose(vm[s:], M[:, s - 1], rtol=1e-15)
    for i in range(s):
        for j in range(s):
            assert np.isclose(M[i, j], vm[i + j + 1], rtol=1e-12)   # M(i,j) = vm(i+j), 1-based


# ------------------------------------------------------------------ small solves
def hilbert_inverse(n):
    H = np.empty((n, n))
    for i in range(1, n + 1):
        for j in range(1, n + 1):
            H[i - 1, j - 1] = ((-1) ** (i + j) * (i + j - 1) * comb(n + i - 1, n - j) * comb(n + j - 1, n - i)
                               * comb(i + j - 2, i - 1) ** 2)
    return H


@pytest.mark.parametrize("s", [1, 2, 4, 8])
def test_cvm_fused_closed_form_and_symmetry(oracle_mod, s):
    """The moments taken in the MPK epilogues (cvm_fused): (a) closed form for an eigenvector input,
    mu^k = lam^k ||r||^2 / d^(k+1); (b) for a general r they equal Alg. 5's moments (cvm) because A is symmetric
    (Eq. 4) -- two different sets of inner products, so a wrong index or column fails here."""
    N = 9
    rp, ci, v = gen.poisson7(N)
    vec, lam = poisson7_eigvec(N, 1, 2, 3)
    dinv = oracle_mod.dinv(rp, ci, v)
    R, AR = oracle_mod.mpk(rp, ci, v, dinv, vec, s)
    vm = oracle_mod.cvm_fused(R, AR, vec)
    expect = np.array([lam ** k * (vec @ vec) / 6.0 ** (k + 1) for k in range(2 * s)])
    assert np.allclose(vm, expect, rtol=1e-12, atol=0)
    c = gen.make_config(5, N=7)                        # variable diagonal, permuted: D^-1 does not commute with A
    rp, ci, v = c["rowptr"], c["colidx"], c["vals"]
    dinv = oracle_mod.dinv(rp, ci, v)
    r = np.random.default_rng(9).uniform(-1, 1, c["n"])
    R, AR = oracle_mod.mpk(rp, ci, v, dinv, r, s)
    a, b = oracle_mod.cvm_fused(R, AR, r), oracle_mod.cvm(R, AR, r)
    assert np.allclose(a, b, rtol=1e-10, atol=0)


@pytest.mark.parametrize("s", [1, 2, 3, 4, 5, 6])
def test_cholesky_hilbert_closed_form(oracle_mod, s):
    H = 1.0 / (np.arange(1, s + 1)[:, None] + np.arange(1, s + 1)[None, :] - 1.0)
    st, L = oracle_mod.chol(H)
    assert st == 0 and np.allclose(L @ L.T, H, rtol=1e-14) and np.allclose(L, np.tril(L))
    X = oracle_mod.chol_solve(L, np.eye(s))
    cond = np.linalg.cond(H)
    assert np.abs(X - hilbert_inverse(s)).max() <= 50 * cond * 1e-16 * np.abs(hilbert_inverse(s)).max()


def test_cholesky_random_spd_and_breakdown(oracle_mod):
    rng = np.random.default_rng(9)
    for s in (1, 3, 8, 16):
        G = rng.normal(size=(s, s + 3))
        W = G @ G.T
        B = rng.normal(size=(s, 5))
        st, L = oracle_mod.chol(W)
        assert st == 0
        assert np.allclose(oracle_mod.chol_solve(L, B), np.linalg.solve(W, B), rtol=1e-9, atol=1e-11)
        # reads only the lower triangle (implicit symmetrisation, reading A10)
        Wu = W.copy(); Wu[np.triu_indices(s, 1)] = 123.0
        assert np.array_equal(oracle_mod.chol(Wu)[1], L)
    assert oracle_mod.chol(np.array([[1.0, 2.0], [2.0, 1.0]]))[0] == 2      # indefinite
    assert oracle_mod.chol(np.array([[np.nan]]))[0] == 2


def test_small_solve_definitions(oracle_mod):
    rng = np.random.default_rng(10)
    s = 4
    G = rng.normal(size=(s, s + 2)); Wp = G @ G.T
    G2 = rng.normal(size=(s, s + 2)); M = G2 @ G2.T + 10 * np.eye(s)
    Cm = 0.1 * rng.normal(size=(s, s)); m = rng.normal(size=s)
    st, beta, alpha, W = oracle_mod.small_solve(M, Cm, m, Wp)
    assert st == 0
    assert np.allclose(Wp @ beta + Cm, 0, atol=1e-12)            # W_{i-1} beta + c_i = 0
    assert np.allclose(W, M + Cm.T @ beta, rtol=1e-13)           # W_i = M_i - c_i beta_{i-1}
    assert np.allclose(W @ alpha, m, atol=1e-12)                 # Eq. 3
    st, beta0, alpha0, W0 = oracle_mod.small_solve(M, Cm, m, Wp, first=True)
    assert st == 0 and np.all(beta0 == 0) and np.array_equal(W0, M) and np.allclose(M @ alpha0, m, atol=1e-12)


# ------------------------------------------------------------------ block updates (Alg. 3 l.17-21)
def test_update_definition(oracle_mod):
    rng = np.random.default_rng(12)
    n, s = 101, 3
    R, AR, P, AP = (rng.uniform(-1, 1, (s, n)) for _ in range(4))
    x, r = rng.uniform(-1, 1, n), rng.uniform(-1, 1, n)
    beta, alpha = rng.normal(size=(s, s)), rng.normal(size=s)
    Pn, APn, xn, rn = oracle_mod.update(R, AR, P, AP, x, r, beta, alpha)
    # matrix form with blocks as n x s: P2 = R + P1 beta ; x += P2 alpha ; r -= AP2 alpha
    assert np.allclose(Pn.T, R.T + P.T @ beta, rtol=1e-14, atol=1e-15)
    assert np.allclose(APn.T, AR.T + AP.T @ beta, rtol=1e-14, atol=1e-15)
    assert np.allclose(xn, x + Pn.T @ alpha, rtol=1e-14, atol=1e-15)
    assert np.allclose(rn, r - APn.T @ alpha, rtol=1e-14, atol=1e-15)


@pytest.mark.parametrize("s,basis", [(1, 0), (2, 0), (3, 0), (4, 0), (6, 1)])
def test_one_step_invariants(oracle_mod, s, basis):
    """Two composed outer iterations on a dense-checkable system: A-conjugacy of
    successive direction blocks, r_new orthogonal to the new
    directions, W = P^T A P, r = b - A x."""
    rp, ci, v, A = gen.random_spd_csr(60, 0.12, 13)
    n = 60
    b = np.random.default_rng(14).uniform(-1, 1, n)
    dinv = oracle_mod.dinv(rp, ci, v)
    x = np.zeros(n); r = b.copy()
    P = np.zeros((s, n)); AP = np.zeros((s, n)); W = np.eye(s)
    for k in range(3):
        R, AR = oracle_mod.mpk(rp, ci, v, dinv, r, s, basis)
        M, C, m = oracle_mod.gram(R, AR, AP if k else None, r)
        st, beta, alpha, Wn = oracle_mod.small_solve(M, C, m, W, first=(k == 0))
        assert st == 0
        Pold, APold = P, AP
        P, AP, x, r = oracle_mod.update(R, AR, P, AP, x, r, beta, alpha)
        scaleW = np.sqrt(np.outer(np.diag(P @ A @ P.T), np.diag(P @ A @ P.T)))
        assert np.allclose(AP, P @ A, rtol=1e-9, atol=1e-12)                  # AP really is A P
        assert np.abs(P @ A @ P.T - Wn).max() <= 1e-9 * scaleW.max()          # W = P^T A P
        if k:
            cross = Pold @ A @ P.T
            assert np.abs(cross).max() <= 1e-9 * scaleW.max()                 # A-conjugacy
        assert np.abs(P @ r).max() <= 1e-9 * np.linalg.norm(P, axis=1).max() * np.linalg.norm(b)
        assert np.linalg.norm(b - A @ x - r) <= 1e-12 * np.linalg.norm(b)
        W = Wn
