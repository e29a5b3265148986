"""Random-STRUCTURE parity: the fixed parity cases of test_gpu_parity.py are stencils plus one irregular matrix; here the
sparsity structure itself is drawn (sstep_inputs.random_structure_spd_csr: banded, uniform row lengths, a stencil with
rows of thousands of entries, boxes with random edge lengths incl. 1, 27-point boxes, power-law row lengths, almost
diagonal; 1 .. 3e5 rows) and every way of running step a1 -- Jacobi-fused SpMV, Alg. 4, PAPER.md:166-190 -- is put on
it: the automatic choice, the generic kernel at every lane count, the per-warp bulk-staged kernel at every tile shape,
the CTA pipeline, with and without the moment partials.  A forced kernel may refuse a matrix at setup (its tile does not
hold the rows); the automatic choice and the generic kernel must take everything; whatever runs must match the oracle's
SpMV at the per-row bar of north_star.  Whole solves (Alg. 3) on the same matrices against the oracle:
outer-iteration count within +-1, x within 1e-8, true residual -- on the graph path and, where it fits, the resident path.
A working-file sweep of the same shape (4 seeds x 300 matrices, 2e4 SpMV runs, 500 solves) found no failure in round 2.
"""
import numpy as np
import pytest

import sstep_inputs as gen

pytestmark = pytest.mark.gpu

TOL_ROW = 1e-13
SEEDS = list(range(100, 128))


@pytest.fixture(scope="module")
def torch_mod():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return torch


@pytest.fixture(scope="module")
def cg_mod():
    import paper_2501_03743_b200 as cg
    cg.load_library()
    return cg


def dev(torch, a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def abs_spmv(rp, ci, v, x):
    import scipy.sparse as sp
    n = rp.size - 1
    return sp.csr_matrix((np.abs(v), ci, rp), shape=(n, n)) @ np.abs(x)


WAYS = [(0, 0), (3, 0)] + [(variant, lanes) for variant in (1, 2) for lanes in (0, 1, 2, 4, 8, 32)]


@pytest.mark.parametrize("seed", SEEDS)
def test_spmv_every_kernel_on_random_structure(oracle_mod, cg_mod, torch_mod, seed):
    rp, ci, v, kind, n = gen.random_structure_spd_csr(seed)
    x = np.random.default_rng(seed).uniform(-1, 1, n)
    y_ref = oracle_mod.spmv(rp, ci, v, x)
    dinv = oracle_mod.dinv(rp, ci, v)
    scale = abs_spmv(rp, ci, v, x)
    t = lambda a: dev(torch_mod, a)
    drp, dci, dv, dx = t(rp), t(ci), t(v), t(x)
    ran = refused = 0
    for variant, lanes in WAYS:
        for form in (0, 1):
            opts = {"spmv_variant": variant, "form": form}
            if lanes:
                opts["lanes"] = lanes
            try:
                with cg_mod.SStepCG(0, **opts) as h:
                    h.setup(drp, dci, dv, 2)
                    y, yj = h.test_spmv(dx)
                    shape = (h.get_info("spmv_cta"), h.get_info("spmv_bulk"), h.get_info("lanes"))
            except cg_mod.SStepCGError:
                assert variant in (2, 3), (kind, n, opts)          # only a FORCED staged kernel may refuse a matrix
                refused += 1
                continue
            ran += 1
            y, yj = y.cpu().numpy(), yj.cpu().numpy()
            assert np.all(np.abs(y - y_ref) <= TOL_ROW * scale), (kind, n, opts, shape)
            assert np.all(np.abs(yj - dinv * y_ref) <= TOL_ROW * dinv * scale), (kind, n, opts, shape)
    assert ran >= 2 * 7                                             # auto + the generic kernel at six lane settings, both forms


@pytest.mark.parametrize("seed", SEEDS[:16])
def test_solve_on_random_structure(oracle_mod, cg_mod, torch_mod, seed):
    rng = np.random.default_rng(seed + 5000)
    n_req = int(rng.choice([33, 257, 1000, 4097, 20000, 65537]))
    rp, ci, v, kind, n = gen.random_structure_spd_csr(seed, n=n_req)
    b = rng.uniform(-1, 1, n)
    basis = int(rng.integers(0, 2))
    s = int(rng.integers(1, 7 if basis else 4))                    # monomial: s <= 3 (parity pinned); Chebyshev: s <= 6
    rtol = 1e-8
    ref = oracle_mod.sstep(rp, ci, v, b, s, rtol=rtol, maxit=2000, basis=basis)
    assert ref["status"] == 0, (kind, n, s, basis)
    t = lambda a: dev(torch_mod, a)
    for resident in (1, 0):                                          # 1 = graph path; 0 = auto (resident where it fits)
        with cg_mod.SStepCG(0, basis=basis, resident=resident) as h:
            h.setup(t(rp), t(ci), t(v), s)
            x, res = h.solve(t(b), rtol=rtol, maxit=2000)
            assert res["status"] == 0 and abs(res["outer_iters"] - ref["iters"]) <= 1, (kind, n, s, basis, res, ref["iters"])
            if res["outer_iters"] != ref["iters"]:
                x, res = h.solve(t(b), rtol=0.0, maxit=ref["iters"])
        x = x.cpu().numpy()
        assert np.linalg.norm(x - ref["x"]) <= 1e-8 * np.linalg.norm(ref["x"]), (kind, n, s, basis, resident)
        true_res = np.linalg.norm(b - oracle_mod.spmv(rp, ci, v, x)) / np.linalg.norm(b)
        assert true_res <= 2 * rtol
