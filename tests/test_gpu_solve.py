"""End-to-end GPU parity: sstep_cg_solve (graph-captured loop, device-side stop test; option resident = 1 keeps these
small systems on the graph path -- the resident path has its own file, test_gpu_resident.py) against the oracle's
Alg. 3 (Gram form) on the BASELINE.json configs, at sizes the oracle finishes in seconds, plus the edge and
degenerate cases.  Bars (north_star): final solution relative difference <= 1e-8, outer iterations within +-1.
s = 8 with the paper's monomial basis is "parity unpinned" end to end: there the test enforces
convergence, the true residual and a looser solution bar, and the Chebyshev basis restores the tight bar."""
import numpy as np
import pytest

import sstep_inputs as gen

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch_mod():
    import torch
    assert torch.cuda.is_available()
    return torch


@pytest.fixture(scope="module")
def cg_mod():
    import paper_2501_03743_b200 as cg
    cg.load_library()
    return cg


def dev(torch, a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def gpu_solve(cg, torch, c, s, rtol, maxit, x0=None, **opts):
    opts.setdefault("resident", 1)
    with cg.SStepCG(0, **opts) as h:
        h.setup(dev(torch, c["rowptr"]), dev(torch, c["colidx"]), dev(torch, c["vals"]), s)
        x, res = h.solve(dev(torch, c["b"]), None if x0 is None else dev(torch, x0), rtol=rtol, maxit=maxit)
        return x.cpu().numpy(), res


def rel(a, b):
    return np.linalg.norm(a - b) / np.linalg.norm(b)


CASES = [  # cfg, N, s (None = the config's own)
    (1, 32, None),      # config 1 at full size: 32^3, s=2, rtol 1e-6
    (1, 32, 1), (1, 32, 3), (1, 32, 4), (1, 32, 5),
    (2, 48, None),      # config 2 recipe (s=4, 1e-8) at 48^3
    (3, 24, None),      # config 3 recipe (27-point, s=4) at 24^3
    (4, 40, 2),         # config 4 recipe at 40^3
    (5, 20, 4),         # config 5 recipe (variable coefficient, permuted) with s=4
]


@pytest.mark.parametrize("cfg,N,s", CASES)
def test_solve_matches_oracle(oracle_mod, cg_mod, torch_mod, cfg, N, s):
    c = gen.make_config(cfg, N=N, s=s)
    s = c["s"]
    ref = oracle_mod.sstep(c["rowptr"], c["colidx"], c["vals"], c["b"], s, rtol=c["rtol"], maxit=c["maxit"])
    x, res = gpu_solve(cg_mod, torch_mod, c, s, c["rtol"], c["maxit"])
    assert ref["status"] == 0 and res["status"] == 0
    assert abs(res["outer_iters"] - ref["iters"]) <= 1
    assert res["cg_equiv_iters"] == s * res["outer_iters"]
    assert res["relres"] < c["rtol"]
    if res["outer_iters"] != ref["iters"]:     # compare at the oracle's stopping iteration
        x, res2 = gpu_solve(cg_mod, torch_mod, c, s, 0.0, ref["iters"])
        assert res2["outer_iters"] == ref["iters"]
    assert rel(x, ref["x"]) <= 1e-8
    # and it really solves the system (true residual through the oracle's SpMV)
    true_res = np.linalg.norm(c["b"] - oracle_mod.spmv(c["rowptr"], c["colidx"], c["vals"], x)) / np.linalg.norm(c["b"])
    assert true_res <= 2 * c["rtol"]


def test_config2_full_size(oracle_mod, cg_mod, torch_mod):
    """BASELINE.json config 2 at its full size (128^3, n = 2.1M, nnz = 14.6M, s = 4, rtol 1e-8)."""
    c = gen.make_config(2)
    ref = oracle_mod.sstep(c["rowptr"], c["colidx"], c["vals"], c["b"], 4, rtol=1e-8, maxit=2000)
    x, res = gpu_solve(cg_mod, torch_mod, c, 4, 1e-8, 2000)
    assert ref["status"] == 0 and res["status"] == 0 and abs(res["outer_iters"] - ref["iters"]) <= 1
    if res["outer_iters"] != ref["iters"]:
        x, _ = gpu_solve(cg_mod, torch_mod, c, 4, 0.0, ref["iters"])
    assert rel(x, ref["x"]) <= 1e-8
    assert rel(x, c["xstar"]) <= 1e-5


@pytest.mark.parametrize("cfg,N", [(5, 20), (4, 32)])
def test_s8_monomial_unpinned_and_chebyshev(oracle_mod, cg_mod, torch_mod, cfg, N):
    c = gen.make_config(cfg, N=N, s=8)
    rtol = c["rtol"]
    x, res = gpu_solve(cg_mod, torch_mod, c, 8, rtol, 2000)
    assert res["status"] == 0
    true_res = np.linalg.norm(c["b"] - oracle_mod.spmv(c["rowptr"], c["colidx"], c["vals"], x)) / np.linalg.norm(c["b"])
    assert true_res <= 2 * rtol
    ref = oracle_mod.sstep(c["rowptr"], c["colidx"], c["vals"], c["b"], 8, rtol=rtol, maxit=2000)
    assert ref["status"] == 0 and rel(x, ref["x"]) <= 1e-4
    # Chebyshev basis: the tight bars hold again
    refc = oracle_mod.sstep(c["rowptr"], c["colidx"], c["vals"], c["b"], 8, rtol=rtol, maxit=2000, basis=1)
    xc, resc = gpu_solve(cg_mod, torch_mod, c, 8, rtol, 2000, basis=1)
    assert refc["status"] == 0 and resc["status"] == 0 and abs(resc["outer_iters"] - refc["iters"]) <= 1
    if resc["outer_iters"] != refc["iters"]:
        xc, _ = gpu_solve(cg_mod, torch_mod, c, 8, 0.0, refc["iters"], basis=1)
    assert rel(xc, refc["x"]) <= 1e-8


def test_iterate_trajectory_matches_oracle(oracle_mod, cg_mod, torch_mod):
    """solve_begin / iterate(k) / solve_end: iterate i equals the oracle's iterate i (early iterations, s = 3)."""
    c = gen.make_config(2, N=20)
    ref = oracle_mod.sstep(c["rowptr"], c["colidx"], c["vals"], c["b"], 3, rtol=0.0, maxit=6, xhist_cap=6, history=True)
    with cg_mod.SStepCG(0, resident=1) as h:
        h.setup(dev(torch_mod, c["rowptr"]), dev(torch_mod, c["colidx"]), dev(torch_mod, c["vals"]), 3)
        b = dev(torch_mod, c["b"])
        for k in range(1, 7):
            h.solve_begin(b, None, 0.0)
            h.iterate(k)
            x, res = h.solve_end()
            assert res["outer_iters"] == k and res["status"] == 1
            assert rel(x.cpu().numpy(), ref["xhist"][k - 1]) <= 1e-11
            assert abs(res["relres"] - ref["hist"][k - 1]) <= 1e-9 * ref["hist"][k - 1]
            assert res["kernel_launches"] == 1 + k * h.get_info("kernels_per_outer")


@pytest.mark.parametrize("form", [0, 1])
def test_s1_pipeline_is_the_papers_fcg_comparator(oracle_mod, cg_mod, torch_mod, form):
    """At s = 1 the pipeline is Alg. 2 PFCG-NN step by step (u = B^-1 r, w = A u, the three coupled dots
    alpha = u.r, beta = u.w, gamma = u.s_prev in one reduction, rho = beta - gamma^2/rho_prev, the two axpy pairs;
    PAPER.md:87-126) -- the paper's baseline "fcg".  Its iterates equal the oracle's Alg. 2 (and Alg. 1) iterates, and a
    full solve takes the same number of iterations (reading A15)."""
    c = gen.make_config(4, N=24)
    rp, ci, v, b = c["rowptr"], c["colidx"], c["vals"], c["b"]
    ref2 = oracle_mod.pfcg(rp, ci, v, b, rtol=0.0, maxit=8, xhist_cap=8)
    ref1 = oracle_mod.pcg(rp, ci, v, b, rtol=0.0, maxit=8, xhist_cap=8)
    with cg_mod.SStepCG(0, form=form, resident=1) as h:
        h.setup(dev(torch_mod, rp), dev(torch_mod, ci), dev(torch_mod, v), 1)
        bd = dev(torch_mod, b)
        for k in (1, 2, 5, 8):
            h.solve_begin(bd, None, 0.0)
            h.iterate(k)
            x, res = h.solve_end()
            assert rel(x.cpu().numpy(), ref2["xhist"][k - 1]) <= 1e-12
            assert rel(x.cpu().numpy(), ref1["xhist"][k - 1]) <= 1e-12
        full2 = oracle_mod.pfcg(rp, ci, v, b, rtol=1e-8, maxit=2000)
        x, res = h.solve(bd, rtol=1e-8, maxit=2000)
        assert res["status"] == 0 and abs(res["outer_iters"] - full2["iters"]) <= 1
        assert rel(x.cpu().numpy(), full2["x"]) <= 1e-8


def test_graph_and_direct_launch_agree_bitwise(cg_mod, torch_mod):
    c = gen.make_config(1, N=24)
    xs = []
    for use_graph in (1, 0, 1):
        x, res = gpu_solve(cg_mod, torch_mod, c, 4, 1e-9, 500, use_graph=use_graph)
        assert res["status"] == 0
        xs.append((x, res["outer_iters"]))
    assert xs[0][1] == xs[1][1] == xs[2][1]
    assert np.array_equal(xs[0][0], xs[1][0]) and np.array_equal(xs[0][0], xs[2][0])   # deterministic reductions


def test_edge_cases(oracle_mod, cg_mod, torch_mod):
    c = gen.make_config(1, N=10)
    # x0 != 0 (r0 = b - A x0 through the production SpMV) and x aliasing
    x0 = np.random.default_rng(9).uniform(-1, 1, c["n"])
    ref = oracle_mod.sstep(c["rowptr"], c["colidx"], c["vals"], c["b"], 2, x0=x0, rtol=1e-9, maxit=500)
    x, res = gpu_solve(cg_mod, torch_mod, c, 2, 1e-9, 500, x0=x0)
    assert res["status"] == 0 and abs(res["outer_iters"] - ref["iters"]) <= 1 and rel(x, c["xstar"]) <= 1e-7
    assert abs(res["r0_norm"] - np.linalg.norm(c["b"] - oracle_mod.spmv(c["rowptr"], c["colidx"], c["vals"], x0))) <= 1e-10
    # b = 0: converged at once, x = 0, zero iterations
    cz = dict(c); cz["b"] = np.zeros(c["n"])
    x, res = gpu_solve(cg_mod, torch_mod, cz, 2, 1e-8, 100)
    assert res["status"] == 0 and res["outer_iters"] == 0 and np.all(x == 0)
    # maxit reached -> status 1, x is the last iterate (equals the oracle's)
    ref = oracle_mod.sstep(c["rowptr"], c["colidx"], c["vals"], c["b"], 2, rtol=1e-14, maxit=3)
    x, res = gpu_solve(cg_mod, torch_mod, c, 2, 1e-14, 3)
    assert res["status"] == 1 == ref["status"] and res["outer_iters"] == 3 and rel(x, ref["x"]) <= 1e-12
    # maxit = 0
    x, res = gpu_solve(cg_mod, torch_mod, c, 2, 1e-8, 0)
    assert res["status"] == 1 and res["outer_iters"] == 0 and np.all(x == 0)
    # s = 16 (SMAX) runs and converges on a well-conditioned system with the Chebyshev basis
    rp, ci, v, A = gen.random_spd_csr(400, 0.02, 77)
    cw = dict(rowptr=rp, colidx=ci, vals=v, b=np.random.default_rng(1).uniform(-1, 1, 400), n=400)
    x, res = gpu_solve(cg_mod, torch_mod, cw, 16, 1e-8, 50, basis=1)
    assert res["status"] == 0 and rel(x, np.linalg.solve(A, cw["b"])) <= 1e-7
    # one-row system
    c1 = dict(rowptr=np.array([0, 1], np.int32), colidx=np.array([0], np.int32), vals=np.array([4.0]), b=np.array([2.0]), n=1)
    x, res = gpu_solve(cg_mod, torch_mod, c1, 1, 1e-12, 5)
    assert res["status"] == 0 and abs(x[0] - 0.5) <= 1e-15


def test_x_may_alias_x0_and_peek_reports_history(oracle_mod, cg_mod, torch_mod):
    """include/sstep_cg.h: "`x` ... may alias x0" -- sstep_cg_solve called with the SAME device buffer for x0 and x, on
    the graph path and on the resident path; and sstep_cg_solve_peek after every outer iteration gives the oracle's
    relative-residual history (Alg. 3 l.31-33)."""
    c = gen.make_config(1, N=12)
    x0 = np.random.default_rng(19).uniform(-1, 1, c["n"])
    ref = oracle_mod.sstep(c["rowptr"], c["colidx"], c["vals"], c["b"], 2, x0=x0, rtol=1e-9, maxit=500, history=True)
    t = lambda a: torch_mod.from_numpy(np.ascontiguousarray(a)).cuda()
    for resident in (1, 0):
        with cg_mod.SStepCG(0, resident=resident) as h:
            h.setup(t(c["rowptr"]), t(c["colidx"]), t(c["vals"]), 2)
            buf = t(x0)
            x, res = h.solve(t(c["b"]), x0=buf, rtol=1e-9, maxit=500, out=buf)
            assert x.data_ptr() == buf.data_ptr()
            assert res["status"] == 0 and abs(res["outer_iters"] - ref["iters"]) <= 1
            assert rel(buf.cpu().numpy(), ref["x"]) <= 1e-8 or res["outer_iters"] != ref["iters"]
            assert rel(buf.cpu().numpy(), c["xstar"]) <= 1e-7
            h.solve_begin(t(c["b"]), t(x0), 1e-9)
            hist = []
            for _ in range(500):
                h.iterate(1)
                p = h.solve_peek()
                hist.append(p["relres"])
                if p["status"] != -1:
                    break
            _, res2 = h.solve_end()
            assert res2["outer_iters"] == len(hist) == res["outer_iters"]
            k = min(len(hist), ref["iters"]) // 2
            assert np.allclose(hist[:k], ref["hist"][:k], rtol=1e-6, atol=0)


def test_measure_bandwidth_runs(cg_mod, torch_mod):
    """The measurement aid of bench.py's read-side peak: every variant returns a positive, plausible figure."""
    with cg_mod.SStepCG(0) as h:
        for variant in (0, 1, 2, 3, 4, 5):
            best, mean = h.measure_bandwidth(variant, 256 << 20, passes=1, reps=3)
            assert 100.0 < mean <= best < 20000.0, (variant, best, mean)
        best, _ = h.measure_bandwidth(0, 32 << 20, passes=20, reps=3)      # L2-resident sweep
        assert best > 100.0


def test_rank_deficient_block_reports_breakdown(oracle_mod, cg_mod, torch_mod):
    """Degenerate case of the method (see test_oracle_solvers.test_rank_deficient_last_block)."""
    rp, ci, v = gen.poisson1d(64)
    b = np.random.default_rng(22).uniform(-1, 1, 64)
    c = dict(rowptr=rp, colidx=ci, vals=v, b=b, n=64)
    ref = oracle_mod.sstep(rp, ci, v, b, 3, rtol=1e-11, maxit=30)
    x, res = gpu_solve(cg_mod, torch_mod, c, 3, 1e-11, 30)
    assert ref["status"] == 2 and res["status"] == 2
    assert abs(res["outer_iters"] - ref["iters"]) <= 1 and np.all(np.isfinite(x))


def test_breakdown_contract_x_is_the_last_good_iterate(cg_mod, torch_mod):
    """include/sstep_cg.h, SSTEP_CG_BREAKDOWN: a bad Cholesky pivot / non-finite Gram block is detected BEFORE the block
    update, which is then skipped -- x comes back as the last good iterate.  Here the right-hand side is so large that
    R_1 = D^-1 r overflows in the very first matrix-powers kernel: the first Gram block is non-finite, status 2 after
    zero completed iterations, and x is exactly x0 (graph path and resident path)."""
    c = gen.make_config(1, N=10)
    t = lambda a: torch_mod.from_numpy(np.ascontiguousarray(a)).cuda()
    x0 = np.random.default_rng(2).uniform(-1, 1, c["n"])
    v = c["vals"] * 1e-170                                   # a_ii = 6e-170: dinv = 1.7e169; b ~ 1e150 -> R_1 overflows
    b = np.sign(c["b"]) * 1e150
    for resident in (1, 0):
        with cg_mod.SStepCG(0, resident=resident) as h:
            h.setup(t(c["rowptr"]), t(c["colidx"]), t(v), 2)
            x, res = h.solve(t(b), x0=t(x0), rtol=1e-8, maxit=50)
        assert res["status"] == 2 and res["status_name"] == "breakdown" and res["outer_iters"] == 0, res
        assert np.array_equal(x.cpu().numpy(), x0)


def test_invalid_arguments(cg_mod, torch_mod):
    rp, ci, v = gen.poisson1d(10)
    t = lambda a: dev(torch_mod, a)
    with cg_mod.SStepCG(0) as h:
        with pytest.raises(cg_mod.SStepCGError):
            h.setup(t(rp), t(ci), t(v), 0)
        with pytest.raises(cg_mod.SStepCGError):
            h.setup(t(rp), t(ci), t(v), 17)
        bad = v.copy(); bad[0] = -2.0                       # non-positive diagonal
        with pytest.raises(cg_mod.SStepCGError, match="diagonal"):
            h.setup(t(rp), t(ci), t(bad), 2)
        badc = ci.copy(); badc[3] = 99                       # column out of range
        with pytest.raises(cg_mod.SStepCGError):
            h.setup(t(rp), t(badc), t(v), 2)
        with pytest.raises(cg_mod.SStepCGError):             # solve before a successful setup
            h.solve(t(np.ones(10)))
        with pytest.raises(cg_mod.SStepCGError):
            h.set_option("no_such_option", 1)
        h.setup(t(rp), t(ci), t(v), 1)                       # handle still usable
        x, res = h.solve(t(np.random.default_rng(3).uniform(-1, 1, 10)), rtol=1e-10, maxit=12)
        assert res["status"] == 0


def test_solve_host_end_to_end(oracle_mod, cg_mod, torch_mod):
    c = gen.make_config(1, N=16)
    ref = oracle_mod.sstep(c["rowptr"], c["colidx"], c["vals"], c["b"], 2, rtol=1e-8, maxit=500)
    th = lambda a: torch_mod.from_numpy(np.ascontiguousarray(a)).pin_memory()
    with cg_mod.SStepCG(0) as h:
        x, res = h.solve_host(th(c["rowptr"]), th(c["colidx"]), th(c["vals"]), th(c["b"]), 2, rtol=1e-8, maxit=500)
    assert res["status"] == 0 and abs(res["outer_iters"] - ref["iters"]) <= 1
    assert rel(x.numpy(), ref["x"]) <= 1e-8


def test_solve_host_repeated_calls_on_one_handle(oracle_mod, cg_mod, torch_mod):
    """sstep_cg_solve_host keeps the storage of its device copies for the next call when the sizes are the same (what a
    serving loop and bench.py's e2e leg do): a second system of the SAME sizes but other values and another right-hand side,
    then a system of other sizes, then the first again -- each against the oracle, nothing left over from the call before."""
    th = lambda a: torch_mod.from_numpy(np.ascontiguousarray(a)).pin_memory()
    c1 = gen.make_config(1, N=16)
    k = gen.varcoef_cells(16, 9)
    rp2, ci2, v2 = gen.varcoef7(16, k)                              # same n and nnz as the 16^3 Poisson matrix, other values
    assert rp2.size == c1["rowptr"].size and ci2.size == c1["colidx"].size
    b2 = np.random.default_rng(12).uniform(-1, 1, rp2.size - 1)
    c3 = gen.make_config(3, N=9)
    systems = [(c1["rowptr"], c1["colidx"], c1["vals"], c1["b"], 2), (rp2, ci2, v2, b2, 3),
               (c3["rowptr"], c3["colidx"], c3["vals"], c3["b"], 4), (c1["rowptr"], c1["colidx"], c1["vals"], c1["b"], 2)]
    with cg_mod.SStepCG(0) as h:
        for rp, ci, v, b, s in systems:
            ref = oracle_mod.sstep(rp, ci, v, b, s, rtol=1e-8, maxit=500)
            x, res = h.solve_host(th(rp), th(ci), th(v), th(b), s, rtol=1e-8, maxit=500)
            assert ref["status"] == 0 and res["status"] == 0 and abs(res["outer_iters"] - ref["iters"]) <= 1
            assert rel(x.numpy(), ref["x"]) <= 1e-8


@pytest.mark.parametrize("cfg,N,s,R", [(2, 20, 3, 2), (1, 24, 2, 1), (5, 16, 4, 3), (3, 12, 4, 2)])
def test_residual_replacement_matches_oracle(oracle_mod, cg_mod, torch_mod, cfg, N, s, R):
    """Option replace_every (reading A22) against the oracle's orc_sstep_rr: iterates, reported residuals
    (the replaced, i.e. true, residual on every R-th iteration) and the full solve."""
    c = gen.make_config(cfg, N=N, s=s)
    rp, ci, v, b = c["rowptr"], c["colidx"], c["vals"], c["b"]
    K = 6
    norm_inf_A = np.add.reduceat(np.abs(v), rp[:-1]).max()
    ref = oracle_mod.sstep(rp, ci, v, b, s, rtol=0.0, maxit=K, xhist_cap=K, history=True, replace_every=R)
    full = oracle_mod.sstep(rp, ci, v, b, s, rtol=c["rtol"], maxit=c["maxit"], replace_every=R)
    with cg_mod.SStepCG(0, replace_every=R) as h:
        h.setup(dev(torch_mod, rp), dev(torch_mod, ci), dev(torch_mod, v), s)
        assert h.get_info("resident") == 0 and h.get_info("replace_every") == R
        bd = dev(torch_mod, b)
        for k in range(1, K + 1):
            h.solve_begin(bd, None, 0.0)
            h.iterate(k)
            x, res = h.solve_end()
            assert res["outer_iters"] == k and res["status"] == 1
            assert res["kernel_launches"] == 1 + k * (s + 2) + 2 * (k // R)
            xk = x.cpu().numpy()
            assert rel(xk, ref["xhist"][k - 1]) <= 1e-11
            # an iterate difference dx moves a residual norm by at most ||A dx|| <= ||A||_inf ||dx||_2 (A symmetric): that, not a
            # fixed number, is the floor under the 1e-9 relative bar (27-point: ||A||_inf = 52)
            floor = norm_inf_A * np.linalg.norm(xk - ref["xhist"][k - 1]) / np.linalg.norm(b) + 1e-14
            assert abs(res["relres"] - ref["hist"][k - 1]) <= 1e-9 * ref["hist"][k - 1] + floor
            if k % R == 0:     # the reported residual is the true one (oracle's SpMV of the GPU's iterate)
                true = np.linalg.norm(b - oracle_mod.spmv(rp, ci, v, x.cpu().numpy())) / np.linalg.norm(b)
                # (b - A x cancels: its rounding error is ~1e-16 (||b|| + ||A|| ||x||), an absolute floor on the residual norm)
                assert abs(res["relres"] - true) <= 1e-12 * true + 1e-14
        x, res = h.solve(bd, rtol=c["rtol"], maxit=c["maxit"])
        assert full["status"] == 0 and res["status"] == 0 and abs(res["outer_iters"] - full["iters"]) <= 1
        if res["outer_iters"] == full["iters"]:
            assert rel(x.cpu().numpy(), full["x"]) <= 1e-8
    with cg_mod.SStepCG(0, replace_every=2, form=1) as h:          # Alg. 6 assumes r = r_prev - AP alpha
        with pytest.raises(cg_mod.SStepCGError, match="Gram form"):
            h.setup(dev(torch_mod, rp), dev(torch_mod, ci), dev(torch_mod, v), s)


@pytest.mark.parametrize("cfg,N", [(1, 24), (2, 20), (3, 12), (5, 14)])
def test_pcg_method_matches_oracle_alg1(oracle_mod, cg_mod, torch_mod, cfg, N):
    """Option method = 1: the textbook PCG (Alg. 1) as its own kernel sequence against the oracle's
    orc_pcg: iterates, residual history, iteration count, final solution; graph and direct launches agree bitwise."""
    c = gen.make_config(cfg, N=N)
    rp, ci, v, b = c["rowptr"], c["colidx"], c["vals"], c["b"]
    K = 8
    ref = oracle_mod.pcg(rp, ci, v, b, rtol=0.0, maxit=K, xhist_cap=K, history=True)
    full = oracle_mod.pcg(rp, ci, v, b, rtol=c["rtol"], maxit=5000)
    xs = []
    for use_graph in (1, 0):
        with cg_mod.SStepCG(0, method=1, use_graph=use_graph) as h:
            h.setup(dev(torch_mod, rp), dev(torch_mod, ci), dev(torch_mod, v), 1)
            assert h.get_info("kernels_per_outer") == 3 and h.get_info("resident") == 0
            bd = dev(torch_mod, b)
            for k in (1, 2, 5, K):
                h.solve_begin(bd, None, 0.0)
                h.iterate(k)
                x, res = h.solve_end()
                assert res["outer_iters"] == k and res["status"] == 1 and res["kernel_launches"] == 1 + 3 * k
                assert rel(x.cpu().numpy(), ref["xhist"][k - 1]) <= 1e-12
                assert abs(res["relres"] - ref["hist"][k - 1]) <= 1e-10 * ref["hist"][k - 1]
            x, res = h.solve(bd, rtol=c["rtol"], maxit=5000)
            assert full["status"] == 0 and res["status"] == 0 and abs(res["outer_iters"] - full["iters"]) <= 1
            if res["outer_iters"] == full["iters"]:
                assert rel(x.cpu().numpy(), full["x"]) <= 1e-8
            xs.append(x.cpu().numpy())
            # x0 != 0 and per-kernel times through profile_outer
            x0 = np.random.default_rng(3).uniform(-1, 1, c["n"])
            r0 = oracle_mod.pcg(rp, ci, v, b, x0=x0, rtol=c["rtol"], maxit=5000)
            x, res = h.solve(bd, dev(torch_mod, x0), rtol=c["rtol"], maxit=5000)
            assert res["status"] == 0 and abs(res["outer_iters"] - r0["iters"]) <= 1
            h.solve_begin(bd, None, 0.0)
            t = h.profile_outer(2)
            _, res = h.solve_end(want_x=False)
            assert res["outer_iters"] == 2 and all(ms > 0 for ms in t)
    assert np.array_equal(xs[0], xs[1])
    with cg_mod.SStepCG(0, method=1) as h:
        with pytest.raises(cg_mod.SStepCGError, match="s = 1"):
            h.setup(dev(torch_mod, rp), dev(torch_mod, ci), dev(torch_mod, v), 2)
