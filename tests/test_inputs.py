"""Pins for the seeded input generators (sstep_inputs): closed forms that fix
the stencils, orderings and the variable-coefficient / permuted recipe
(SURVEY.md §8c "What pins each part": matrix generators)."""
import numpy as np
import pytest

import sstep_inputs as gen


def _dense(rp, ci, v):
    n = rp.size - 1
    A = np.zeros((n, n))
    for i in range(n):
        A[i, ci[rp[i]:rp[i + 1]]] = v[rp[i]:rp[i + 1]]
    return A


@pytest.mark.parametrize("N", [3, 5, 8])
def test_poisson7_closed_forms(N):
    rp, ci, v = gen.poisson7(N)
    n = N ** 3
    assert rp.dtype == np.int32 and ci.dtype == np.int32 and v.dtype == np.float64
    assert rp[-1] == 7 * N ** 3 - 6 * N ** 2          # nnz closed form
    for i in range(n):                                 # sorted columns, diagonal present
        cols = ci[rp[i]:rp[i + 1]]
        assert np.all(np.diff(cols) > 0) and i in cols
    A = _dense(rp, ci, v)
    assert np.array_equal(A, A.T)
    # row sum = number of missing (Dirichlet) neighbours
    x, y, z = [a.ravel() for a in np.meshgrid(np.arange(N), np.arange(N), np.arange(N), indexing="ij")][::-1]
    missing = sum(((c == 0).astype(int) + (c == N - 1).astype(int)) for c in (x, y, z))
    assert np.array_equal(A.sum(axis=1), missing.astype(float))
    # spectrum: lambda = 6 - 2 sum_d cos(i_d pi/(N+1))
    k = np.arange(1, N + 1)
    c = 2 * np.cos(k * np.pi / (N + 1))
    lam = (6 - (c[:, None, None] + c[None, :, None] + c[None, None, :])).ravel()
    assert np.allclose(np.sort(np.linalg.eigvalsh(A)), np.sort(lam), rtol=0, atol=1e-12)


@pytest.mark.parametrize("N", [3, 4, 6])
def test_poisson27_closed_forms(N):
    rp, ci, v = gen.poisson27(N)
    assert rp[-1] == (3 * N - 2) ** 3
    A = _dense(rp, ci, v)
    assert np.array_equal(A, A.T)
    assert np.all(np.diag(A) == 26.0)
    # A = 27 I - S x S x S with S = tridiag(1,1,1): lambda = 27 - prod(1 + 2cos(i_d pi/(N+1)))
    k = np.arange(1, N + 1)
    c = 1 + 2 * np.cos(k * np.pi / (N + 1))
    lam = (27 - c[:, None, None] * c[None, :, None] * c[None, None, :]).ravel()
    assert np.allclose(np.sort(np.linalg.eigvalsh(A)), np.sort(lam), rtol=0, atol=1e-11)


@pytest.mark.parametrize("N", [4, 7])
def test_stencil_apply_matches_csr(N):
    rng = np.random.default_rng(11)
    x = rng.uniform(-1, 1, N ** 3)
    for build, apply in ((gen.poisson7, gen.apply_poisson7), (gen.poisson27, gen.apply_poisson27)):
        A = _dense(*build(N))
        assert np.allclose(A @ x, apply(N, x), rtol=0, atol=1e-13)


def test_varcoef_reduces_to_poisson_and_flux_form():
    N = 5
    rp, ci, v = gen.varcoef7(N, np.ones(N ** 3))
    rp7, ci7, v7 = gen.poisson7(N)
    assert np.array_equal(rp, rp7) and np.array_equal(ci, ci7) and np.array_equal(v, v7)
    k = gen.varcoef_cells(N, 4)
    assert np.all(k > 0)
    A = _dense(*gen.varcoef7(N, k))
    assert np.allclose(A, A.T, rtol=0, atol=0)
    assert np.all(np.linalg.eigvalsh(A) > 0)
    x = np.random.default_rng(3).uniform(-1, 1, N ** 3)
    assert np.allclose(A @ x, gen.apply_varcoef7(N, k, x), rtol=1e-13, atol=1e-12)
    # interior face coefficient is the harmonic mean of the two cells
    i, j = 0, 1
    assert np.isclose(-A[i, j], 2 * k[i] * k[j] / (k[i] + k[j]))


def test_symmetric_permutation():
    N = 4
    k = gen.varcoef_cells(N, 4)
    rp, ci, v = gen.varcoef7(N, k)
    perm = np.random.default_rng(5).permutation(N ** 3)
    rp2, ci2, v2 = gen.symmetric_permute(rp, ci, v, perm)
    A, A2 = _dense(rp, ci, v), _dense(rp2, ci2, v2)
    assert np.array_equal(A2, A[np.ix_(perm, perm)])
    for i in range(N ** 3):
        assert np.all(np.diff(ci2[rp2[i]:rp2[i + 1]]) > 0)
    assert np.array_equal(A2, A2.T)


def test_random_spd_is_spd_and_irregular():
    rp, ci, v, A = gen.random_spd_csr(60, 0.1, 7, max_row=40)
    assert np.array_equal(_dense(rp, ci, v), A)
    assert np.all(np.linalg.eigvalsh(A) > 0)
    lens = np.diff(rp)
    assert lens.max() >= 30 and lens.min() <= 10


def test_random_structure_matrices_meet_the_csr_contract():
    """random_structure_spd_csr: every structure kind gives a symmetric, strictly diagonally dominant matrix with the
    diagonal present once and positive, columns ascending and unique in a row, seeded (same seed, same matrix); the
    kinds differ in what they are for -- long rows, ragged boxes, rows of one entry."""
    for k, kind in enumerate(gen.STRUCTURE_KINDS):
        for n in (1, 2, 33, 700):
            rp, ci, v, kind_out, n_out = gen.random_structure_spd_csr(40 + k, kind, n)
            assert kind_out == kind and rp.size == n_out + 1 and rp[-1] == ci.size == v.size
            assert rp.dtype == np.int32 and ci.dtype == np.int32 and v.dtype == np.float64
            if kind not in ("box7", "box27"):
                assert n_out == n
            A = _dense(rp, ci, v)
            assert np.array_equal(A, A.T)
            d = np.diag(A)
            assert np.all(d > 0) and np.all(d > np.abs(A).sum(axis=1) - d)
            for i in range(n_out):
                row = ci[rp[i]:rp[i + 1]]
                assert np.all(np.diff(row) > 0) and np.count_nonzero(row == i) == 1
            again = gen.random_structure_spd_csr(40 + k, kind, n)
            assert np.array_equal(again[0], rp) and np.array_equal(again[1], ci) and np.array_equal(again[2], v)
    lens = lambda kind: np.diff(gen.random_structure_spd_csr(3, kind, 5000)[0])
    assert lens("stencil_long_rows").max() > 1000 and lens("power_law").max() > 200 and lens("near_diagonal").min() == 1
    assert lens("box27").max() == 27 and lens("box7").max() == 7
    kinds = {gen.random_structure_spd_csr(seed, n=50)[3] for seed in range(40)}
    assert kinds == set(gen.STRUCTURE_KINDS)


def test_configs_are_seeded_and_consistent():
    a = gen.make_config(1, N=6)
    b = gen.make_config(1, N=6)
    assert np.array_equal(a["b"], b["b"]) and a["s"] == 2 and a["rtol"] == 1e-6
    assert np.allclose(_dense(a["rowptr"], a["colidx"], a["vals"]) @ a["xstar"], a["b"], atol=1e-13)
    c5 = gen.make_config(5, N=5)
    assert c5["s"] == 8 and c5["nnz"] == 7 * 125 - 6 * 25
    c6 = gen.make_config(6, N=5)
    assert np.all(c6["b"] == 1.0) and c6["rtol"] == 1e-6


def test_poisson7_box_matches_cube_and_definition():
    rp, ci, v = gen.poisson7_box(5, 5, 5)
    rp7, ci7, v7 = gen.poisson7(5)
    assert np.array_equal(rp, rp7) and np.array_equal(ci, ci7) and np.array_equal(v, v7)
    nx, ny, nz = 6, 4, 3
    A = _dense(*gen.poisson7_box(nx, ny, nz))
    assert np.array_equal(A, A.T) and A.shape[0] == nx * ny * nz
    x = np.random.default_rng(2).uniform(-1, 1, nx * ny * nz)
    assert np.allclose(A @ x, gen.apply_poisson7_box(nx, ny, nz, x), rtol=0, atol=1e-13)
    kx, ky, kz = (np.arange(1, m + 1) for m in (nx, ny, nz))
    lam = (6 - 2 * (np.cos(kz * np.pi / (nz + 1))[:, None, None] + np.cos(ky * np.pi / (ny + 1))[None, :, None]
                    + np.cos(kx * np.pi / (nx + 1))[None, None, :])).ravel()
    assert np.allclose(np.sort(np.linalg.eigvalsh(A)), np.sort(lam), atol=1e-12)
