"""Pins for the oracle's solvers (Alg. 1, 2, 3 of PAPER.md) against what the
mathematics fixes (north_star (a)-(d); SURVEY.md §8c "Whole solver"):
 (a) tiny spd systems converge in <= n iterations to the dense-LU solution;
 (b) s-step iterate i equals CG iterate i*s;
 (c) conjugacy -- see test_oracle_kernels.test_one_step_invariants;
 (d) the closed-form spectrum of the Poisson stencil bounds the A-norm error
     and the iteration count;
 (e) Alg. 3 at s=1 == Alg. 2 == Alg. 1 iterates;  (f) Gram form == moment form;
 (g) the paper's own 514 iterations;  (h) scipy's CG.
"""
import os

import numpy as np
import pytest
import scipy.sparse as sp
import scipy.sparse.linalg as spla

import sstep_inputs as gen

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def csr_of(c):
    return sp.csr_matrix((c["vals"], c["colidx"], c["rowptr"]), shape=(c["n"], c["n"]))


def tiny_systems():
    out = []
    rp, ci, v, A = gen.random_spd_csr(48, 0.15, 21)
    out.append(("rand48", rp, ci, v, A))
    rp, ci, v = gen.poisson1d(64)
    out.append(("lap1d64", rp, ci, v, sp.csr_matrix((v, ci, rp)).toarray()))
    rp, ci, v = gen.poisson7(4)
    out.append(("p7_4", rp, ci, v, sp.csr_matrix((v, ci, rp)).toarray()))
    return out


# (a) ------------------------------------------------------------------------
@pytest.mark.parametrize("name,rp,ci,v,A", tiny_systems(), ids=lambda t: t if isinstance(t, str) else "")
def test_tiny_spd_converges_to_lu(oracle_mod, name, rp, ci, v, A):
    n = A.shape[0]
    b = np.random.default_rng(22).uniform(-1, 1, n)
    xlu = np.linalg.solve(A, b)
    runs = [("pcg", oracle_mod.pcg(rp, ci, v, b, rtol=1e-11, maxit=n), 1),
            ("pfcg", oracle_mod.pfcg(rp, ci, v, b, rtol=1e-11, maxit=n), 1)]
    # s-step: when s does not divide the grade of b the last block [R_1..R_s] is rank deficient and W is
    # singular (exact breakdown, see test_rank_deficient_last_block); take s | 64 there.
    for s in ((1, 2, 3, 4) if name == "rand48" else (1, 2, 4)):
        for form in ("gram", "moment", "moment_fused"):
            runs.append((f"s{s}{form}", oracle_mod.sstep(rp, ci, v, b, s, rtol=1e-9, maxit=-(-n // s) + 2, form=form), s))
    for tag, res, s in runs:
        assert res["status"] == 0, (tag, res["relres"])
        assert res["iters"] * s <= n + 2 * s, tag                         # CG terminates in <= n steps (+ fp64 slack)
        assert np.linalg.norm(res["x"] - xlu) <= 1e-8 * np.linalg.norm(xlu), tag


def test_rank_deficient_last_block(oracle_mod):
    """Degenerate case of the method: 1-D Laplacian n=64 has grade 64 = 21*3 + 1, so at s=3 the 22nd block
    spans one new dimension only, W = P^T A P is singular and the Cholesky solve must report breakdown
    (status 2) instead of returning garbage; x stays the last good iterate."""
    rp, ci, v = gen.poisson1d(64)
    b = np.random.default_rng(22).uniform(-1, 1, 64)
    res = oracle_mod.sstep(rp, ci, v, b, 3, rtol=1e-11, maxit=30)
    assert res["status"] == 2 and res["iters"] == 21 and np.all(np.isfinite(res["x"]))
    A = sp.csr_matrix((v, ci, rp)).toarray()
    assert np.linalg.norm(b - A @ res["x"]) <= 1e-2 * np.linalg.norm(b)


def test_lap1d_takes_exactly_n_steps(oracle_mod):
    """1-D Laplacian, n distinct eigenvalues, generic b: CG needs all n steps."""
    rp, ci, v = gen.poisson1d(32)
    b = np.random.default_rng(23).uniform(-1, 1, 32)
    assert oracle_mod.pcg(rp, ci, v, b, rtol=1e-9, maxit=100)["iters"] == 32


# (b), (e), (f) ---------------------------------------------------------------
def _problems_b():
    c7 = gen.make_config(1, N=8)
    c27 = gen.make_config(3, N=6)
    c5 = gen.make_config(5, N=6)
    return [c7, c27, c5]


@pytest.mark.parametrize("c", _problems_b(), ids=lambda c: c["name"])
@pytest.mark.parametrize("s", [1, 2, 3, 4])
def test_sstep_iterates_equal_cg_every_s_steps(oracle_mod, c, s):
    nouter = 5
    ref = oracle_mod.pcg(c["rowptr"], c["colidx"], c["vals"], c["b"], rtol=0.0, maxit=nouter * s, xhist_cap=nouter * s)
    ref2 = oracle_mod.pfcg(c["rowptr"], c["colidx"], c["vals"], c["b"], rtol=0.0, maxit=nouter * s, xhist_cap=nouter * s)
    scale = np.linalg.norm(ref["xhist"][-1])
    assert np.abs(ref["xhist"] - ref2["xhist"]).max() <= 1e-13 * scale          # Alg. 1 == Alg. 2
    for form in ("gram", "moment", "moment_fused"):
        res = oracle_mod.sstep(c["rowptr"], c["colidx"], c["vals"], c["b"], s, rtol=0.0, maxit=nouter, form=form,
                               xhist_cap=nouter)
        assert res["status"] == 1 and res["iters"] == nouter
        for i in range(nouter):
            err = np.linalg.norm(res["xhist"][i] - ref["xhist"][(i + 1) * s - 1])
            assert err <= 5e-11 * scale, (form, s, i, err / scale)
        if s == 1:
            assert np.abs(res["xhist"] - ref["xhist"]).max() <= 1e-13 * scale    # (e)


@pytest.mark.parametrize("s", [2, 4, 8])
def test_chebyshev_basis_same_krylov_iterates(oracle_mod, s):
    """The Gram form is basis-agnostic: the Chebyshev MPK spans the same Krylov
    space, so iterates still equal CG's every s steps (DESIGN.md NEXT-1)."""
    c = gen.make_config(1, N=8)
    nouter = 3
    ref = oracle_mod.pcg(c["rowptr"], c["colidx"], c["vals"], c["b"], rtol=0.0, maxit=nouter * s, xhist_cap=nouter * s)
    res = oracle_mod.sstep(c["rowptr"], c["colidx"], c["vals"], c["b"], s, rtol=0.0, maxit=nouter, basis=1,
                           xhist_cap=nouter)
    scale = np.linalg.norm(ref["xhist"][-1])
    for i in range(nouter):
        assert np.linalg.norm(res["xhist"][i] - ref["xhist"][(i + 1) * s - 1]) <= 1e-9 * scale


def test_composed_steps_equal_driver(oracle_mod):
    """The C driver orc_sstep is exactly the composition of the per-step functions the parity tests use."""
    c = gen.make_config(2, N=7)
    s, nouter = 3, 4
    rp, ci, v, b = c["rowptr"], c["colidx"], c["vals"], c["b"]
    dinv = oracle_mod.dinv(rp, ci, v)
    n = c["n"]
    x = np.zeros(n); r = b.copy(); P = np.zeros((s, n)); AP = np.zeros((s, n)); W = np.eye(s)
    for k in range(nouter):
        R, AR = oracle_mod.mpk(rp, ci, v, dinv, r, s)
        M, C, m = oracle_mod.gram(R, AR, AP if k else None, r)
        st, beta, alpha, W = oracle_mod.small_solve(M, C, m, W, first=(k == 0))
        P, AP, x, r = oracle_mod.update(R, AR, P, AP, x, r, beta, alpha)
    res = oracle_mod.sstep(rp, ci, v, b, s, rtol=0.0, maxit=nouter)
    assert np.array_equal(res["x"], x)
    assert np.isclose(res["relres"], np.linalg.norm(r) / np.linalg.norm(b), rtol=1e-14)


# (d) -------------------------------------------------------------------------
@pytest.mark.parametrize("N", [8, 14])
def test_cg_error_bound_from_closed_form_spectrum(oracle_mod, N):
    """||x_k - x*||_A <= 2 ((sqrt(kappa)-1)/(sqrt(kappa)+1))^k ||x_0 - x*||_A with
    kappa = cot^2(pi / (2(N+1))) for the 7-point stencil (constant diagonal, so
    Jacobi does not change kappa); and the residual-based iteration count bound."""
    c = gen.make_config(1, N=N)
    A = csr_of(c)
    xs = c["xstar"]
    kappa = 1.0 / np.tan(np.pi / (2 * (N + 1))) ** 2
    q = (np.sqrt(kappa) - 1) / (np.sqrt(kappa) + 1)
    e0 = np.sqrt(xs @ (A @ xs))
    rtol = 1e-8
    res = oracle_mod.pcg(c["rowptr"], c["colidx"], c["vals"], c["b"], rtol=rtol, maxit=500, xhist_cap=500, history=True)
    assert res["status"] == 0
    for k, xk in enumerate(res["xhist"]):
        e = xk - xs
        assert np.sqrt(e @ (A @ e)) <= 2 * q ** (k + 1) * e0 * (1 + 1e-10)
    # ||r_k||_2 <= sqrt(lmax) ||e_k||_A <= sqrt(kappa) 2 q^k ||r_0||_2  =>  k_stop <= first k with 2 sqrt(kappa) q^k < rtol
    kbound = int(np.ceil(np.log(rtol / (2 * np.sqrt(kappa))) / np.log(q)))
    assert res["iters"] <= kbound
    for s in (2, 4):
        rs = oracle_mod.sstep(c["rowptr"], c["colidx"], c["vals"], c["b"], s, rtol=rtol, maxit=500, xhist_cap=500)
        assert rs["status"] == 0 and rs["iters"] == -(-res["iters"] // s)        # ceil(PCG / s)
        for i, xi in enumerate(rs["xhist"]):
            e = xi - xs
            assert np.sqrt(e @ (A @ e)) <= 2 * q ** ((i + 1) * s) * e0 * (1 + 1e-8)


# (h) -------------------------------------------------------------------------
@pytest.mark.parametrize("cfg,N", [(1, 10), (3, 7), (5, 7)])
def test_pcg_matches_scipy_cg(oracle_mod, cfg, N):
    c = gen.make_config(cfg, N=N)
    A = csr_of(c)
    dinv = 1.0 / A.diagonal()
    its = []
    xs, info = spla.cg(A, c["b"], rtol=1e-8, atol=0.0, M=sp.diags(dinv), callback=lambda xk: its.append(xk.copy()))
    assert info == 0
    res = oracle_mod.pcg(c["rowptr"], c["colidx"], c["vals"], c["b"], rtol=1e-8, maxit=1000, xhist_cap=len(its) + 5)
    assert abs(res["iters"] - len(its)) <= 1          # scipy stops on <=, the paper on <
    k = min(10, len(its), res["iters"])
    scale = np.linalg.norm(its[k - 1])
    for i in range(k):
        assert np.linalg.norm(res["xhist"][i] - its[i]) <= 1e-12 * scale
    assert np.linalg.norm(res["x"] - xs) <= 1e-7 * np.linalg.norm(xs)


def test_status_codes(oracle_mod):
    c = gen.make_config(1, N=6)
    args = (c["rowptr"], c["colidx"], c["vals"], c["b"])
    assert oracle_mod.sstep(*args, 2, rtol=1e-12, maxit=2)["status"] == 1          # maxit
    r = oracle_mod.sstep(*args, 2, rtol=1e-8, maxit=200, x0=c["xstar"])
    # x0 already the solution up to rounding: r0 is rounding noise, the relative test still terminates, x stays put
    assert r["status"] == 0 and np.linalg.norm(r["x"] - c["xstar"]) <= 1e-13 * np.linalg.norm(c["xstar"])
    z = oracle_mod.sstep(c["rowptr"], c["colidx"], c["vals"], np.zeros(c["n"]), 2)
    assert z["status"] == 0 and z["iters"] == 0 and np.all(z["x"] == 0)
    # x0 != 0 path: same answer as x0 = 0
    x0 = np.random.default_rng(5).uniform(-1, 1, c["n"])
    a = oracle_mod.sstep(*args, 3, rtol=1e-10, x0=x0)
    assert a["status"] == 0 and np.linalg.norm(a["x"] - c["xstar"]) <= 1e-8 * np.linalg.norm(c["xstar"])


# residual replacement (reading A22) -----------------------
@pytest.mark.parametrize("s,R", [(1, 3), (2, 1), (3, 2), (4, 5)])
def test_residual_replacement_pins(oracle_mod, s, R):
    """What fixes orc_sstep_rr without an implementation to compare with: (i) R beyond the iteration count changes
    nothing, bit for bit; (ii) on a replacement iteration the reported residual IS the true residual of that iterate
    (recomputed here with scipy's CSR product); on the others it is the recurrence residual, which drifts from the
    true one; (iii) replacing r by b - A x changes r only at rounding level, so the early iterates agree with the
    unreplaced ones; (iv) it still converges to the dense-LU solution."""
    c = gen.make_config(2, N=10)
    rp, ci, v, b = c["rowptr"], c["colidx"], c["vals"], c["b"]
    A = csr_of(c)
    nb = np.linalg.norm(b)
    plain = oracle_mod.sstep(rp, ci, v, b, s, rtol=1e-10, maxit=200, history=True, xhist_cap=200)
    never = oracle_mod.sstep(rp, ci, v, b, s, rtol=1e-10, maxit=200, history=True, xhist_cap=200, replace_every=10 ** 6)
    assert never["iters"] == plain["iters"] and np.array_equal(never["x"], plain["x"]) and np.array_equal(never["hist"], plain["hist"])
    rr = oracle_mod.sstep(rp, ci, v, b, s, rtol=1e-10, maxit=200, history=True, xhist_cap=200, replace_every=R)
    assert rr["status"] == 0 and abs(rr["iters"] - plain["iters"]) <= 1
    for k in range(rr["iters"]):
        true = np.linalg.norm(b - A @ rr["xhist"][k]) / nb
        if (k + 1) % R == 0:
            assert abs(rr["hist"][k] - true) <= 1e-13 * max(true, 1e-16 / nb) + 1e-15, k
    for k in range(min(4, plain["iters"], rr["iters"])):
        assert np.linalg.norm(rr["xhist"][k] - plain["xhist"][k]) <= 1e-12 * np.linalg.norm(plain["xhist"][k])
    xs = np.linalg.solve(A.toarray(), b)
    assert np.linalg.norm(rr["x"] - xs) <= 1e-8 * np.linalg.norm(xs)


def test_residual_replacement_reports_the_true_residual_at_the_accuracy_limit(oracle_mod):
    """Run past the attainable accuracy (rtol = 0) with replacement every iteration: the reported residual stays the
    true residual of the iterate (it cannot drift below what fp64 allows -- the reason the technique exists,
    PAPER.md:251) and the iterate stays at the accuracy limit instead of wandering off."""
    c = gen.make_config(2, N=8)
    rp, ci, v, b = c["rowptr"], c["colidx"], c["vals"], c["b"]
    A = csr_of(c)
    nb = np.linalg.norm(b)
    rr = oracle_mod.sstep(rp, ci, v, b, 2, rtol=0.0, maxit=40, history=True, replace_every=1)
    n_rr = rr["iters"]
    assert n_rr >= 20
    true = np.linalg.norm(b - A @ rr["x"]) / nb
    assert abs(rr["hist"][n_rr - 1] - true) <= 1e-12 * true + 1e-17 and true <= 1e-13


# (g) -------------------------------------------------------------------------
@pytest.mark.slow
def test_paper_514_iterations(oracle_mod):
    """250^3 Poisson, rhs = 1, no preconditioner (== Jacobi on a
    constant diagonal), rtol = 1e-6: PFCG and PCGs(s=1) take 514 iterations on one GPU."""
    with open(os.path.join(GOLDEN, "paper_iterations.txt")) as f:
        gold = {k: int(v) for k, v in (ln.split("#")[0].split() for ln in f if ln.strip() and not ln.startswith("#"))}
    c = gen.make_config(6)
    assert c["n"] == 250 ** 3 and c["nnz"] == 109_000_000
    res = oracle_mod.pfcg(c["rowptr"], c["colidx"], c["vals"], c["b"], rtol=1e-6, maxit=2000)
    assert res["status"] == 0 and res["iters"] == gold["pfcg_250cubed_1gpu"]


# ------------------------------------------------------------------------------------------------ timing legs, fixtures
def test_openmp_build_is_the_same_program_up_to_summation_order(oracle_mod):
    """bench.py's all-core cpu_baseline leg: the same sstep_oracle.c built with -fopenmp.  Its row loops are the serial
    ones (bitwise the same SpMV), its inner products are summed per thread (another order): after a few outer iterations
    the iterate agrees with the serial build to rounding.  The in-loop clock excludes the start-up and reports a time."""
    import sstep_inputs as gen
    c = gen.make_config(2, N=20)
    args = (c["rowptr"], c["colidx"], c["vals"], c["b"], 4, 5)
    per1, start1, o1 = oracle_mod.sstep_timed(*args, omp=False)
    per2, start2, o2 = oracle_mod.sstep_timed(*args, omp=True)
    ref = oracle_mod.sstep(c["rowptr"], c["colidx"], c["vals"], c["b"], 4, rtol=0.0, maxit=5)
    assert np.array_equal(o1["x"], ref["x"])                    # the time log does not touch the arithmetic
    assert np.linalg.norm(o2["x"] - ref["x"]) <= 1e-10 * np.linalg.norm(ref["x"])
    assert per1 > 0 and per2 > 0 and start1 >= 0 and start2 >= 0 and oracle_mod.omp_threads() >= 1
    lib1, lib2 = oracle_mod.lib(False), oracle_mod.lib(True)
    x = np.random.default_rng(3).uniform(-1, 1, c["n"])
    y1 = np.empty(c["n"]); y2 = np.empty(c["n"])
    import ctypes as C
    for L, y in ((lib1, y1), (lib2, y2)):
        L.orc_spmv(C.c_int64(c["n"]), c["rowptr"].ctypes.data_as(C.POINTER(C.c_int32)), c["colidx"].ctypes.data_as(C.POINTER(C.c_int32)),
                   c["vals"].ctypes.data_as(C.POINTER(C.c_double)), x.ctypes.data_as(C.POINTER(C.c_double)), y.ctypes.data_as(C.POINTER(C.c_double)))
    assert np.array_equal(y1, y2)


def test_golden_fixtures_are_consistent_and_reproducible(oracle_mod, tmp_path):
    """tests/golden/config*.txt (written by make_golden.py from the oracle alone): every fixture parses, is a converged
    solve whose history ends below rtol at exactly `iters`, the paper's problem gives the paper's 514 at s = 1 and for
    Alg. 1 and ceil(514 / s) for s = 2..5, and the writer reproduces itself on a small
    grid (the format round-trips, the sample indices are the seeded ones)."""
    import importlib.util, math, os
    gdir = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
    spec = importlib.util.spec_from_file_location("make_golden_cpu", os.path.join(gdir, "make_golden.py"))
    mg = importlib.util.module_from_spec(spec); spec.loader.exec_module(mg)
    paper = int([ln.split()[1] for ln in open(os.path.join(gdir, "paper_iterations.txt")) if ln.startswith("pfcg_250cubed_1gpu")][0])
    for name, (cfg, s, basis, method) in mg.CASES.items():
        g = mg.load(os.path.join(gdir, name + ".txt"))
        assert g["config"] == cfg and g["s"] == s and g["basis"] == basis and g["method"] == method
        assert g["status"] == 0 and g["iters"] == g["hist"].size and g["hist"][-1] < g["rtol"] <= g["hist"][-2]
        assert g["xi"].size == mg.NS == g["nsample"] and np.array_equal(g["xi"], mg.sample_indices(g["n"]))
        assert np.abs(g["xv"]).max() <= g["xmaxabs"] <= g["xnorm2"]
        if cfg == 6:
            assert g["iters"] == math.ceil(paper / s), (name, g["iters"])
    assert mg.load(os.path.join(gdir, "config6_s1.txt"))["iters"] == paper == mg.load(os.path.join(gdir, "config6_pcg.txt"))["iters"]
    # s-step iterates are CG iterates every s steps: the three config-4 solves end at the same point
    g1, g2, g4 = (mg.load(os.path.join(gdir, f"config4_s{s}.txt")) for s in (1, 2, 4))
    assert g2["iters"] == math.ceil(g1["iters"] / 2) and g4["iters"] == math.ceil(g1["iters"] / 4)
    assert np.abs(g2["xv"] - g1["xv"]).max() <= 1e-9 and abs(g4["hist"][0] - g1["hist"][3]) <= 1e-9 * g1["hist"][3]
    # the one fixture the oracle rewrites in under a second at FULL size: every data line of the committed file, to the last digit
    strip = lambda path: [ln for ln in open(path) if not ln.startswith("#")]
    committed = strip(os.path.join(gdir, "config1_s2.txt"))
    mg.HERE = str(tmp_path)
    assert strip(mg.run_case("config1_s2")) == committed
    # writer -> reader on a grid the oracle finishes at once
    mg.HERE = str(tmp_path)
    out = mg.run_case("config4_s4", N=16)
    g = mg.load(out)
    import sstep_inputs as gen
    c = gen.make_config(4, N=16)
    ref = oracle_mod.sstep(c["rowptr"], c["colidx"], c["vals"], c["b"], 4, rtol=c["rtol"], maxit=c["maxit"], history=True)
    assert g["iters"] == ref["iters"] and np.array_equal(g["hist"], ref["hist"]) and np.array_equal(g["xv"], ref["x"][g["xi"]])
