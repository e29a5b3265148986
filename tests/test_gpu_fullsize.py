"""Parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (config 4: 7-point 320^3,
n = 32 768 000, nnz = 228 761 600, s = 4, persistent grids, bulk-staged SpMV, graph replay).

The C oracle finishes one full-size outer iteration in a few seconds, so every output element is compared (not a
sample): the s Jacobi-fused SpMVs of the MPK, the Gram blocks, the on-device solves, the block update, and the
iterates of the graph-replayed solve loop after 3 outer iterations.  Tolerances as in test_gpu_parity.py
(DESIGN.md "Tolerances").
"""
import numpy as np
import pytest

import sstep_inputs as gen

pytestmark = pytest.mark.gpu

TOL_ROW = 1e-13
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


@pytest.fixture(scope="module")
def full(oracle_mod):
    """Config 4 at full size and the oracle's state after 2 outer iterations (inputs of iteration 3)."""
    c = gen.make_config(4)
    assert c["n"] == 320 ** 3 and c["nnz"] == 7 * 320 ** 3 - 6 * 320 ** 2
    s = 4
    rp, ci, v, b = c["rowptr"], c["colidx"], c["vals"], c["b"]
    n = c["n"]
    dinv = oracle_mod.dinv(rp, ci, v)
    x = np.zeros(n); r = b.copy(); P = np.zeros((s, n)); AP = np.zeros((s, n)); W = np.eye(s)
    xs = []
    for k in range(3):
        R, AR = oracle_mod.mpk(rp, ci, v, dinv, r, s)
        if k == 2:
            state = dict(R=R, AR=AR, P=P, AP=AP, x=x, r=r, W=W)
        M, C, m = oracle_mod.gram(R, AR, AP if k else None, r)
        st, beta, alpha, W = oracle_mod.small_solve(M, C, m, W, first=(k == 0))
        assert st == 0
        P, AP, x, r = oracle_mod.update(R, AR, P, AP, x, r, beta, alpha)
        xs.append(x)
    state.update(M=M, C=C, m=m, beta=beta, alpha=alpha, Wn=W, Pn=P, APn=AP, xn=x, rn=r)
    return dict(c=c, s=s, dinv=dinv, st=state, xs=xs)


def dev(torch, a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def test_fullsize_per_kernel_parity(oracle_mod, cg_mod, torch_mod, full):
    c, s, S, dinv = full["c"], full["s"], full["st"], full["dinv"]
    t = lambda a: dev(torch_mod, a)
    with cg_mod.SStepCG(0) as h:
        h.setup(t(c["rowptr"]), t(c["colidx"]), t(c["vals"]), s)
        assert h.get_info("spmv_bulk") == 1 and h.get_info("lanes") == 1      # the configuration bench.py times
        assert h.get_info("spmv_grid") % h.get_info("num_sms") == 0
        assert h.get_info("gram_staged") == 1 and h.get_info("block_staged") == 0   # s = 4 at 32.8 M rows: TMA-staged Gram, register update
        # a1: the MPK on the oracle's residual of iteration 3 (every element of every column)
        R, AR = h.test_mpk(t(S["r"]))
        R, AR = R.cpu().numpy(), AR.cpu().numpy()
        # row scale of column j: sum |a_ik| |R_j[k]| ; 7-point stencil: 6|x_i| + sum of the neighbours' |x|
        for j in range(s):
            scale = 12.0 * np.abs(S["R"][j]) - gen.apply_poisson7(320, np.abs(S["R"][j]))   # = |A| |x|
            # the j-th column's input differs from the oracle's by the accumulated error of the previous ones
            tol = TOL_ROW * (j + 1)
            assert np.all(np.abs(AR[j] - S["AR"][j]) <= tol * scale), j
            assert np.all(np.abs(R[j] - S["R"][j]) <= tol * np.maximum(np.abs(S["R"][j]), dinv * scale)), j
        del R, AR
        # a2: Gram on identical inputs
        M, C, m = (a.cpu().numpy() for a in h.test_gram(t(S["R"]), t(S["AR"]), t(S["AP"]), t(S["r"])))
        nR, nAR, nAP = (np.linalg.norm(S[k], axis=1) for k in ("R", "AR", "AP"))
        assert np.all(np.abs(M - S["M"]) <= TOL_GRAM * np.outer(nR, nAR))
        assert np.all(np.abs(C - S["C"]) <= TOL_GRAM * np.outer(nAP, nR))
        assert np.all(np.abs(m - S["m"]) <= TOL_GRAM * nR * np.linalg.norm(S["r"]))
        # a3: bit-exact
        st, beta, alpha, W = h.test_small_solve(t(S["M"]), t(S["C"]), t(S["m"]), t(S["W"]))
        assert st == 0
        assert np.array_equal(beta.cpu().numpy(), S["beta"]) and np.array_equal(alpha.cpu().numpy(), S["alpha"])
        assert np.array_equal(W.cpu().numpy(), S["Wn"])
        # a4: update on identical inputs
        Pn, APn, xn, rn, R1, rho = h.test_update(t(S["R"]), t(S["AR"]), t(S["P"]), t(S["AP"]), t(S["x"]), t(S["r"]),
                                                 t(S["beta"]), t(S["alpha"]))
    aB = np.abs(S["beta"])
    sP = np.abs(S["R"]) + aB.T @ np.abs(S["P"])
    sAP = np.abs(S["AR"]) + aB.T @ np.abs(S["AP"])
    assert np.all(np.abs(Pn.cpu().numpy() - S["Pn"]) <= TOL_ROW * sP)
    assert np.all(np.abs(APn.cpu().numpy() - S["APn"]) <= TOL_ROW * sAP)
    sx = np.abs(S["x"]) + np.abs(S["alpha"]) @ sP
    sr = np.abs(S["r"]) + np.abs(S["alpha"]) @ sAP
    assert np.all(np.abs(xn.cpu().numpy() - S["xn"]) <= TOL_ROW * sx)
    assert np.all(np.abs(rn.cpu().numpy() - S["rn"]) <= TOL_ROW * sr)
    assert np.all(np.abs(R1.cpu().numpy() - dinv * S["rn"]) <= TOL_ROW * dinv * sr)
    rr = S["rn"] @ S["rn"]
    assert abs(rho - rr) <= 1e-12 * rr + 2 * np.sqrt(rr) * np.linalg.norm(TOL_ROW * sr)


def test_fullsize_graph_replay_matches_oracle_iterates(cg_mod, torch_mod, full):
    """solve_begin / iterate(k) / solve_end on the bench path: iterate k equals the oracle's iterate k (k = 1, 2, 3)."""
    c, s = full["c"], full["s"]
    t = lambda a: dev(torch_mod, a)
    with cg_mod.SStepCG(0) as h:
        h.setup(t(c["rowptr"]), t(c["colidx"]), t(c["vals"]), s)
        b = t(c["b"])
        for k in (1, 2, 3):
            h.solve_begin(b, None, 0.0)
            h.iterate(k)
            x, res = h.solve_end()
            assert res["outer_iters"] == k and res["status"] == 1
            xr = full["xs"][k - 1]
            assert np.linalg.norm(x.cpu().numpy() - xr) <= 1e-10 * np.linalg.norm(xr), k


def test_config3_full_size(oracle_mod, cg_mod, torch_mod):
    """BASELINE.json config 3 at full size (27-point 160^3, n = 4 096 000, nnz = 109 215 352, s = 4) in the launch
    configuration bench.py times (bulk-staged SpMV, two lanes per row, 512-entry tiles): every row of one SpMV, the
    first three iterates of the graph-replayed loop, and the full solve (x within 1e-8, outer iterations within +-1)."""
    c = gen.make_config(3)
    rp, ci, v, b = c["rowptr"], c["colidx"], c["vals"], c["b"]
    n = c["n"]
    assert n == 160 ** 3 and c["nnz"] == (3 * 160 - 2) ** 3
    t = lambda a: dev(torch_mod, a)
    ref = oracle_mod.sstep(rp, ci, v, b, 4, rtol=1e-8, maxit=2000, xhist_cap=3)
    with cg_mod.SStepCG(0) as h:
        h.setup(t(rp), t(ci), t(v), 4)
        assert h.get_info("spmv_bulk") == 1 and h.get_info("lanes") == 2 and h.get_info("reordered") == 0
        x = np.random.default_rng(13).uniform(-1, 1, n)
        y, yj = h.test_spmv(t(x))
        yo = oracle_mod.spmv(rp, ci, v, x)
        scale = oracle_mod.spmv(rp, ci, np.abs(v), np.abs(x))
        assert np.all(np.abs(y.cpu().numpy() - yo) <= TOL_ROW * scale)
        assert np.all(np.abs(yj.cpu().numpy() - yo / 26.0) <= TOL_ROW * scale / 26.0)
        del y, yj, yo, scale
        bd = t(b)
        for k in (1, 2, 3):
            h.solve_begin(bd, None, 0.0)
            h.iterate(k)
            xk, res = h.solve_end()
            assert res["outer_iters"] == k
            assert np.linalg.norm(xk.cpu().numpy() - ref["xhist"][k - 1]) <= 1e-10 * np.linalg.norm(ref["xhist"][k - 1]), k
        xg, res = h.solve(bd, rtol=1e-8, maxit=2000)
        assert ref["status"] == 0 and res["status"] == 0 and abs(res["outer_iters"] - ref["iters"]) <= 1
        if res["outer_iters"] != ref["iters"]:
            xg, _ = h.solve(bd, rtol=0.0, maxit=ref["iters"])
        assert np.linalg.norm(xg.cpu().numpy() - ref["x"]) <= 1e-8 * np.linalg.norm(ref["x"])


@pytest.mark.parametrize("N,s", [(512, 2), (512, 8), (670, 1)])
def test_large_index_range(cg_mod, torch_mod, N, s):
    """Beyond every BASELINE.json config, up to the library's limit (nnz < 2^31): 7-point 512^3 (n = 134 217 728,
    nnz = 937 951 232: byte offsets of colidx / vals beyond 2^32 and 2^33) and 670^3 (n = 300 763 000,
    nnz = 2 102 647 600 = 0.98 * 2^31: the largest element offsets an int32 CSR can hold; 25 GB of CSR).
    Checked against what the mathematics fixes at any size:
    the closed-form eigenpair of the stencil (A v = lambda v, v = sin x sin x sin) through the SpMV hook
    on every row, and after 3 outer iterations the recurrence residual the solver reports against the true residual
    b - A x evaluated with the same hook."""
    rp, ci, v = gen.poisson7(N)
    n = N ** 3
    assert rp.size - 1 == n and ci.size == 7 * N ** 3 - 6 * N ** 2 < 2 ** 31
    t = lambda a: dev(torch_mod, a)
    torch = torch_mod
    g = torch.arange(1, N + 1, dtype=torch.float64, device="cuda")
    sx = torch.sin(3 * np.pi * g / (N + 1)); sy = torch.sin(5 * np.pi * g / (N + 1)); sz = torch.sin(2 * np.pi * g / (N + 1))
    vec = (sz[:, None, None] * sy[None, :, None] * sx[None, None, :]).reshape(-1).contiguous()     # x fastest
    lam = 6.0 - 2.0 * (np.cos(3 * np.pi / (N + 1)) + np.cos(5 * np.pi / (N + 1)) + np.cos(2 * np.pi / (N + 1)))
    with cg_mod.SStepCG(0) as h:
        h.setup(t(rp), t(ci), t(v), s)
        del rp, ci, v
        assert h.get_info("spmv_bulk") == 1 and h.get_info("reordered") == 0 and h.get_info("resident") == 0
        y, yj = h.test_spmv(vec)
        assert float((y - lam * vec).abs().max()) <= 1e-13 * 12.0
        assert float((yj - (lam / 6.0) * vec).abs().max()) <= 1e-13 * 2.0
        del y, yj
        b = torch.rand(n, dtype=torch.float64, device="cuda", generator=torch.Generator(device="cuda").manual_seed(5)) * 2 - 1
        h.solve_begin(b, None, 0.0)
        h.iterate(3)
        x, res = h.solve_end()
        assert res["outer_iters"] == 3 and res["status"] == 1 and 0 < res["relres"] < 1
        ax, _ = h.test_spmv(x, jacobi=False)
        true = float(torch.linalg.norm(b - ax) / torch.linalg.norm(b))
        assert abs(true - res["relres"]) <= (1e-10 if s <= 4 else 1e-7) * true     # (s = 8: TMA-staged Gram / update kernels)
