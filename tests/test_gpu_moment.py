"""GPU parity of the moment form (option form = 1): the 2s moments accumulated in the SpMV
epilogues (Alg. 5 reduced to nothing) and the scalar work Alg. 6 in one warp, against the oracle's `cvm_fused`,
`sw` and `sstep(form="moment_fused")`.  Tolerances as in test_gpu_parity.py."""
import numpy as np
import pytest

import sstep_inputs as gen

pytestmark = pytest.mark.gpu

TOL_GRAM = 1e-12


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


def solver(cg, torch, c, s, **opts):
    h = cg.SStepCG(0, form=1, **opts)
    h.setup(dev(torch, c["rowptr"]), dev(torch, c["colidx"]), dev(torch, c["vals"]), s)
    return h


MATS = {
    "p7_21": (lambda: gen.make_config(1, N=21), 4, {}),                   # bulk-staged SpMV, ragged last tile
    "p27_13": (lambda: gen.make_config(3, N=13), 3, {}),                  # 4 lanes per row, generic kernel
    "p27_13_bulk": (lambda: gen.make_config(3, N=13), 4, {"spmv_variant": 2}),
    "vc_perm_12": (lambda: gen.make_config(5, N=12), 8, {}),              # variable diagonal, random gather
    "p7_9_generic": (lambda: gen.make_config(1, N=9), 2, {"spmv_variant": 1}),
}


@pytest.mark.parametrize("name", list(MATS))
def test_mpk_moments_parity(oracle_mod, cg_mod, torch_mod, name):
    build, s, opts = MATS[name]
    c = build()
    rp, ci, v = c["rowptr"], c["colidx"], c["vals"]
    r = np.random.default_rng(51).uniform(-1, 1, c["n"])
    dinv = oracle_mod.dinv(rp, ci, v)
    R_ref, AR_ref = oracle_mod.mpk(rp, ci, v, dinv, r, s)
    vm_ref = oracle_mod.cvm_fused(R_ref, AR_ref, r)
    with solver(cg_mod, torch_mod, c, s, **opts) as h:
        R, AR, vm = h.test_mpk_moments(dev(torch_mod, r))
    vm = vm.cpu().numpy()
    nR, nAR = np.linalg.norm(R_ref, axis=1), np.linalg.norm(AR_ref, axis=1)
    # the GPU's columns differ from the oracle's by rounding (<= 1e-13 per row, test_mpk_parity): allow for it
    tol = TOL_GRAM + 2e-13 * s
    assert abs(vm[0] - vm_ref[0]) <= tol * nR[0] * np.linalg.norm(r)
    for j in range(1, s + 1):
        assert abs(vm[2 * j - 1] - vm_ref[2 * j - 1]) <= tol * nR[j - 1] * nAR[j - 1], (name, j)
        if j < s:
            assert abs(vm[2 * j] - vm_ref[2 * j]) <= tol * nR[j] * nAR[j - 1], (name, j)
    assert np.allclose(R.cpu().numpy(), R_ref, rtol=0, atol=1e-12 * np.abs(R_ref).max())


@pytest.mark.parametrize("s", list(range(1, 9)) + [12, 16])
def test_sw_bit_exact(oracle_mod, cg_mod, torch_mod, s):
    """Alg. 6 on the device = the oracle's orc_sw bit for bit, on moments of a real trajectory (first and later
    outer iterations)."""
    c = gen.make_config(2, N=10)
    rp, ci, v, b = c["rowptr"], c["colidx"], c["vals"], c["b"]
    n = c["n"]
    dinv = oracle_mod.dinv(rp, ci, v)
    x = np.zeros(n); r = b.copy(); P = np.zeros((s, n)); AP = np.zeros((s, n))
    t = lambda a: dev(torch_mod, a)
    with solver(cg_mod, torch_mod, c, s) as h:
        alpha = W = None
        for k in range(3):
            R, AR = oracle_mod.mpk(rp, ci, v, dinv, r, s)
            vm = oracle_mod.cvm_fused(R, AR, r)
            if k == 0:
                M = np.array([[vm[i + j + 1] for j in range(s)] for i in range(s)])
                st_r, L = oracle_mod.chol(M)
                beta_r = np.zeros((s, s)); W_r = M
                alpha_r = oracle_mod.chol_solve(L, vm[:s]) if st_r == 0 else np.zeros(s)
                st, beta_g, alpha_g, W_g = h.test_sw(t(vm))
            else:
                st_r, beta_r, alpha_r, W_r = oracle_mod.sw(vm, alpha, W)
                st, beta_g, alpha_g, W_g = h.test_sw(t(vm), t(alpha), t(W))
            assert st == st_r
            if st_r != 0:          # monomial basis at large s: breakdown is a legitimate, identical outcome
                break
            assert np.array_equal(beta_g.cpu().numpy(), beta_r)
            assert np.array_equal(alpha_g.cpu().numpy(), alpha_r)
            assert np.array_equal(W_g.cpu().numpy(), W_r)
            alpha, W = alpha_r, W_r
            P, AP, x, r = oracle_mod.update(R, AR, P, AP, x, r, beta_r, alpha_r)
        assert k >= 1 or s > 8


def test_sw_reports_breakdown(oracle_mod, cg_mod, torch_mod):
    c = gen.make_config(1, N=6)
    with solver(cg_mod, torch_mod, c, 3) as h:
        vm = np.array([1.0, 1.0, 1.0, 1.0, 1.0, 1.0])            # rank-1 Hankel matrix: not positive definite
        st, *_ = h.test_sw(dev(torch_mod, vm))
        assert st == 2
        st_r, _ = oracle_mod.chol(np.ones((3, 3)))
        assert st_r != 0
        good = np.array([3.0, 1.0, 2.0, 0.5, 1.5, 0.2])
        st, beta, alpha, W = h.test_sw(dev(torch_mod, good), dev(torch_mod, np.array([1.0, 1.0, 0.0])),
                                       dev(torch_mod, np.eye(3)))
        assert st == 2                                            # alpha_prev(s) = 0: Alg. 6 divides by it


CASES = [(1, 32, None), (1, 32, 1), (1, 32, 3), (1, 32, 4), (2, 48, None), (3, 24, None), (4, 40, 2), (5, 20, 4)]


@pytest.mark.parametrize("cfg,N,s", CASES)
def test_solve_moment_form_matches_oracle(oracle_mod, cg_mod, torch_mod, cfg, N, s):
    c = gen.make_config(cfg, N=N, s=s)
    s = c["s"]
    rp, ci, v, b = c["rowptr"], c["colidx"], c["vals"], c["b"]
    ref = oracle_mod.sstep(rp, ci, v, b, s, rtol=c["rtol"], maxit=c["maxit"], form="moment_fused")
    assert ref["status"] == 0
    with solver(cg_mod, torch_mod, c, s) as h:
        assert h.get_info("form") == 1
        x, res = h.solve(dev(torch_mod, b), rtol=c["rtol"], maxit=c["maxit"])
        assert res["status"] == 0 and abs(res["outer_iters"] - ref["iters"]) <= 1
        assert res["kernel_launches"] >= res["outer_iters"] * (s + 2)
        if res["outer_iters"] != ref["iters"]:        # compare at the oracle's stopping iteration
            x, res2 = h.solve(dev(torch_mod, b), rtol=0.0, maxit=ref["iters"])
            assert res2["outer_iters"] == ref["iters"]
    x = x.cpu().numpy()
    assert np.linalg.norm(x - ref["x"]) <= 1e-8 * np.linalg.norm(ref["x"])
    true_res = np.linalg.norm(b - oracle_mod.spmv(rp, ci, v, x)) / np.linalg.norm(b)
    assert true_res <= 2 * c["rtol"]
    # and the two forms agree with each other (same Krylov iterates)
    gram = oracle_mod.sstep(rp, ci, v, b, s, rtol=c["rtol"], maxit=c["maxit"])
    assert abs(gram["iters"] - ref["iters"]) <= 1


def test_moment_form_needs_monomial_basis(cg_mod, torch_mod):
    c = gen.make_config(1, N=6)
    with cg_mod.SStepCG(0, form=1, basis=1) as h:
        with pytest.raises(cg_mod.SStepCGError):
            h.setup(dev(torch_mod, c["rowptr"]), dev(torch_mod, c["colidx"]), dev(torch_mod, c["vals"]), 2)
