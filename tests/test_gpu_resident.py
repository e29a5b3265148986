"""GPU parity of the resident path (csrc/resident.cuh): the whole loop of Alg. 3 in one
cooperative launch, every CTA's rows kept in shared memory.  Checked the same way as the graph path:
  * stage by stage on identical inputs: the state before an outer iteration is read back through the
    `sstep_cg_test_read_state` hook, the oracle recomputes Alg. 4 (MPK), the Gram blocks, the s x s solves and the
    block updates from THAT state, and every array the iteration leaves is compared at the per-kernel bars
    (SpMV / update 1e-13 per row, Gram 1e-12 at the Cauchy-Schwarz scale, solves bit-exact on the GPU's own M, C, m);
  * end to end against the oracle's Alg. 3 (x within 1e-8, outer iterations within +-1), status codes, edge cases;
  * the same stage test also runs on the graph path (resident = 1), so both loops are held to the same bars.
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
    assert torch.cuda.is_available()
    return torch


@pytest.fixture(scope="module")
def cg_mod():
    import paper_2501_03743_b200 as cg
    cg.load_library()
    return cg


def dev(torch, a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def rel(a, b):
    return np.linalg.norm(a - b) / np.linalg.norm(b)


def abs_csr(rp, ci, v):
    import scipy.sparse as sp
    n = rp.size - 1
    return sp.csr_matrix((np.abs(v), ci, rp), shape=(n, n))


def read(h, name):
    return h.test_read_state(name).cpu().numpy()


STAGE_CASES = [  # name, matrix factory, s, basis
    ("p7_21_s2", lambda: gen.poisson7(21), 2, 0),            # 9261 rows: 148 CTAs x 64 rows, ragged last CTA
    ("p7_32_s4", lambda: gen.poisson7(32), 4, 0),            # config 1's matrix
    ("p7_16_s1", lambda: gen.poisson7(16), 1, 0),
    ("p7_20_s3", lambda: gen.poisson7(20), 3, 0),
    ("p27_13_s5", lambda: gen.poisson27(13), 5, 0),          # 27 entries per row: remainder loop beyond 8
    ("vc_perm_16_s8", lambda: tuple(gen.make_config(5, N=16)[k] for k in ("rowptr", "colidx", "vals")), 8, 0),
    ("p7_24_s6_cheb", lambda: gen.poisson7(24), 6, 1),
    ("tiny_5_s2", lambda: gen.poisson1d(5), 2, 0),           # one CTA, fewer rows than a warp
]


@pytest.mark.parametrize("resident", [2, 1])
@pytest.mark.parametrize("name,make,s,basis", STAGE_CASES, ids=[c[0] for c in STAGE_CASES])
def test_outer_iteration_stage_by_stage(oracle_mod, cg_mod, torch_mod, name, make, s, basis, resident):
    rp, ci, v = make()[:3]
    n = rp.size - 1
    b = np.random.default_rng(5).uniform(-1, 1, n)
    dinv = oracle_mod.dinv(rp, ci, v)
    absA = abs_csr(rp, ci, v)
    with cg_mod.SStepCG(0, resident=resident, basis=basis) as h:
        h.setup(dev(torch_mod, rp), dev(torch_mod, ci), dev(torch_mod, v), s)
        assert h.get_info("resident") == (1 if resident == 2 else 0)
        h.solve_begin(dev(torch_mod, b), None, 0.0)
        iters = 2 if n > 8 else 1
        for k in range(iters):                           # k = 0 (beta = 0, C = 0) and k = 1 (full recurrences)
            x0, r0, P0, AP0, W0 = (read(h, a) for a in ("x", "r", "P", "AP", "W"))
            h.iterate(1)
            R, AR = read(h, "R"), read(h, "AR")
            # a1, Alg. 4 column by column on the GPU's own previous column (identical inputs).  R(:,1) was overwritten by
            # the update with D^-1 r_new; before the iteration it was dinv * r0 (one rounding: checked below for r_new).
            Rg = R.copy(); Rg[0] = dinv * r0
            for j in range(s):
                y = oracle_mod.spmv(rp, ci, v, Rg[j])
                scale = absA @ np.abs(Rg[j]) + 1e-300
                assert np.max(np.abs(AR[j] - y) / scale) <= TOL_ROW, (name, "AR", j)
                if j + 1 < s:
                    if basis == 0:
                        assert np.array_equal(Rg[j + 1], dinv * AR[j]), (name, "R", j + 1)     # one rounded product
                    else:
                        z = dinv * AR[j] - Rg[j]
                        zs = dinv * np.abs(AR[j]) + np.abs(Rg[j])
                        if j >= 1:
                            z, zs = 2.0 * z - Rg[j - 1], 2.0 * zs + np.abs(Rg[j - 1])
                        assert np.max(np.abs(Rg[j + 1] - z) / (zs + 1e-300)) <= TOL_ROW, (name, "R cheb", j + 1)
            # a2: Gram blocks on the GPU's own basis
            M, Cm, m = (read(h, a) for a in ("M", "C", "m"))
            Mo, Co, mo = oracle_mod.gram(Rg, AR, AP0, r0)
            nR, nAR, nAP = (np.linalg.norm(Z, axis=1) for Z in (Rg, AR, AP0))
            assert np.max(np.abs(M - Mo) / (np.outer(nR, nAR) + 1e-300)) <= TOL_GRAM
            assert np.max(np.abs(Cm - Co) / (np.outer(nAP, nR) + 1e-300)) <= TOL_GRAM
            assert np.max(np.abs(m - mo) / (nR * np.linalg.norm(r0) + 1e-300)) <= TOL_GRAM
            # a3: the s x s solves on the GPU's M, C, m and the previous W -- bit-exact
            beta, alpha, W = (read(h, a) for a in ("beta", "alpha", "W"))
            st, bo, ao, Wo = oracle_mod.small_solve(M, Cm, m, W0)
            assert st == 0 and np.array_equal(beta, bo) and np.array_equal(alpha, ao) and np.array_equal(W, Wo), name
            # a4: block updates with the GPU's beta, alpha
            Pn, APn, xn, rn = oracle_mod.update(Rg, AR, P0, AP0, x0, r0, beta, alpha)
            P1, AP1, x1, r1 = (read(h, a) for a in ("P", "AP", "x", "r"))
            sP = np.abs(Rg) + np.abs(beta).T @ np.abs(P0) + 1e-300
            sAP = np.abs(AR) + np.abs(beta).T @ np.abs(AP0) + 1e-300
            assert np.max(np.abs(P1 - Pn) / sP) <= TOL_ROW * s and np.max(np.abs(AP1 - APn) / sAP) <= TOL_ROW * s
            assert np.max(np.abs(x1 - xn) / (np.abs(x0) + np.abs(alpha) @ sP)) <= TOL_ROW * s
            assert np.max(np.abs(r1 - rn) / (np.abs(r0) + np.abs(alpha) @ sAP)) <= TOL_ROW * s
            assert np.array_equal(R[0], dinv * r1)                                   # R_1 of the next iteration
        _, res = h.solve_end(want_x=False)
        assert res["outer_iters"] == iters
        assert abs(res["relres"] - np.linalg.norm(r1) / np.linalg.norm(b)) <= 1e-12 * res["relres"]


CASES = [(1, 32, None), (1, 32, 1), (1, 32, 4), (1, 32, 5), (2, 40, None), (3, 20, None), (4, 36, 2), (5, 20, 4)]


@pytest.mark.parametrize("cfg,N,s", CASES)
def test_resident_solve_matches_oracle(oracle_mod, cg_mod, torch_mod, cfg, N, s):
    c = gen.make_config(cfg, N=N, s=s)
    s = c["s"]
    ref = oracle_mod.sstep(c["rowptr"], c["colidx"], c["vals"], c["b"], s, rtol=c["rtol"], maxit=c["maxit"])
    with cg_mod.SStepCG(0, resident=2) as h:
        h.setup(dev(torch_mod, c["rowptr"]), dev(torch_mod, c["colidx"]), dev(torch_mod, c["vals"]), s)
        assert h.get_info("resident") == 1
        x, res = h.solve(dev(torch_mod, c["b"]), rtol=c["rtol"], maxit=c["maxit"])
        assert res["kernel_launches"] == 2            # init + ONE cooperative launch for the whole loop
        assert ref["status"] == 0 and res["status"] == 0
        assert abs(res["outer_iters"] - ref["iters"]) <= 1 and res["relres"] < c["rtol"]
        if res["outer_iters"] != ref["iters"]:
            x, res2 = h.solve(dev(torch_mod, c["b"]), rtol=0.0, maxit=ref["iters"])
            assert res2["outer_iters"] == ref["iters"]
    x = x.cpu().numpy()
    assert rel(x, ref["x"]) <= 1e-8
    true_res = np.linalg.norm(c["b"] - oracle_mod.spmv(c["rowptr"], c["colidx"], c["vals"], x)) / np.linalg.norm(c["b"])
    assert true_res <= 2 * c["rtol"]


def test_resident_trajectory_and_chunked_iterate(oracle_mod, cg_mod, torch_mod):
    """iterate(k) in one launch, and the same k iterations as k separate launches (state through global memory),
    give the oracle's iterates; the two ways agree bit for bit (fixed-order reductions)."""
    c = gen.make_config(2, N=20)
    ref = oracle_mod.sstep(c["rowptr"], c["colidx"], c["vals"], c["b"], 3, rtol=0.0, maxit=6, xhist_cap=6, history=True)
    with cg_mod.SStepCG(0, resident=2) as h:
        h.setup(dev(torch_mod, c["rowptr"]), dev(torch_mod, c["colidx"]), dev(torch_mod, c["vals"]), 3)
        b = dev(torch_mod, c["b"])
        for k in range(1, 7):
            h.solve_begin(b, None, 0.0)
            h.iterate(k)
            x, res = h.solve_end()
            assert res["outer_iters"] == k and res["status"] == 1
            assert rel(x.cpu().numpy(), ref["xhist"][k - 1]) <= 1e-11
            assert abs(res["relres"] - ref["hist"][k - 1]) <= 1e-9 * ref["hist"][k - 1]
            h.solve_begin(b, None, 0.0)
            for _ in range(k):
                h.iterate(1)
            x2, res2 = h.solve_end()
            assert res2["outer_iters"] == k and np.array_equal(x2.cpu().numpy(), x.cpu().numpy())


def test_resident_and_graph_paths_agree(cg_mod, torch_mod):
    c = gen.make_config(1)
    out = {}
    for resident in (1, 2):
        with cg_mod.SStepCG(0, resident=resident) as h:
            h.setup(dev(torch_mod, c["rowptr"]), dev(torch_mod, c["colidx"]), dev(torch_mod, c["vals"]), c["s"])
            x, res = h.solve(dev(torch_mod, c["b"]), rtol=c["rtol"], maxit=c["maxit"])
            out[resident] = (x.cpu().numpy(), res)
    assert out[1][1]["status"] == 0 == out[2][1]["status"]
    assert out[1][1]["outer_iters"] == out[2][1]["outer_iters"]
    assert rel(out[2][0], out[1][0]) <= 1e-10
    # run to run the resident path is bitwise reproducible
    with cg_mod.SStepCG(0, resident=2) as h:
        h.setup(dev(torch_mod, c["rowptr"]), dev(torch_mod, c["colidx"]), dev(torch_mod, c["vals"]), c["s"])
        x, _ = h.solve(dev(torch_mod, c["b"]), rtol=c["rtol"], maxit=c["maxit"])
    assert np.array_equal(x.cpu().numpy(), out[2][0])


@pytest.mark.parametrize("cfg,N,s", [(1, 32, 2), (1, 24, 1), (2, 36, 4), (4, 30, 3)])
def test_resident_exchange_modes_agree_bitwise(cg_mod, torch_mod, cfg, N, s):
    """resident_sync = 0 (default: tagged-word exchange between the CTAs, no grid barrier, stop test one matrix-powers kernel
    late) and resident_sync = 1 (round 1's grid barriers) run the same arithmetic in the same order: same iteration count,
    same x bit for bit, for a converged solve and for a fixed number of iterations in several launches."""
    c = gen.make_config(cfg, N=N, s=s)
    out = {}
    for sync in (0, 1):
        with cg_mod.SStepCG(0, resident=2, resident_sync=sync) as h:
            h.setup(dev(torch_mod, c["rowptr"]), dev(torch_mod, c["colidx"]), dev(torch_mod, c["vals"]), s)
            assert h.get_info("resident") == 1 and h.get_info("resident_sync") == sync
            b = dev(torch_mod, c["b"])
            x, res = h.solve(b, rtol=c["rtol"], maxit=c["maxit"])
            h.solve_begin(b, None, 0.0)
            for k in (1, 2, 3):              # 6 iterations in three launches: state and tags carry over
                h.iterate(k)
            x6, res6 = h.solve_end()
            out[sync] = (x.cpu().numpy(), res, x6.cpu().numpy(), res6)
    assert out[0][1]["status"] == 0 == out[1][1]["status"]
    assert out[0][1]["outer_iters"] == out[1][1]["outer_iters"] and out[0][1]["relres"] == out[1][1]["relres"]
    assert np.array_equal(out[0][0], out[1][0])
    assert out[0][3]["outer_iters"] == 6 == out[1][3]["outer_iters"] and out[0][3]["relres"] == out[1][3]["relres"]
    assert np.array_equal(out[0][2], out[1][2])


def test_resident_auto_selection_and_limits(cg_mod, torch_mod):
    t = lambda a: dev(torch_mod, a)
    rp, ci, v = gen.poisson7(32)
    with cg_mod.SStepCG(0) as h:                              # auto: config 1's size fits shared memory
        h.setup(t(rp), t(ci), t(v), 2)
        assert h.get_info("resident") == 1 and h.get_info("resident_grid") <= h.get_info("num_sms")
        assert h.get_info("resident_smem_bytes") <= 200 * 1024
    with cg_mod.SStepCG(0, form=1) as h:                      # the moment form stays on the graph path
        h.setup(t(rp), t(ci), t(v), 2)
        assert h.get_info("resident") == 0
    rp, ci, v = gen.poisson7(96)                              # 885k rows: far beyond shared memory
    with cg_mod.SStepCG(0) as h:
        h.setup(t(rp), t(ci), t(v), 2)
        assert h.get_info("resident") == 0
    with cg_mod.SStepCG(0, resident=2) as h:
        with pytest.raises(cg_mod.SStepCGError, match="resident"):
            h.setup(t(rp), t(ci), t(v), 2)


def test_resident_edge_cases(oracle_mod, cg_mod, torch_mod):
    c = gen.make_config(1, N=10)
    t = lambda a: dev(torch_mod, a)

    def solve(cc, s, rtol, maxit, x0=None, **opts):
        with cg_mod.SStepCG(0, resident=2, **opts) as h:
            h.setup(t(cc["rowptr"]), t(cc["colidx"]), t(cc["vals"]), s)
            x, res = h.solve(t(cc["b"]), None if x0 is None else t(x0), rtol=rtol, maxit=maxit)
            return x.cpu().numpy(), res
    x0 = np.random.default_rng(9).uniform(-1, 1, c["n"])
    ref = oracle_mod.sstep(c["rowptr"], c["colidx"], c["vals"], c["b"], 2, x0=x0, rtol=1e-9, maxit=500)
    x, res = solve(c, 2, 1e-9, 500, x0=x0)
    assert res["status"] == 0 and abs(res["outer_iters"] - ref["iters"]) <= 1 and rel(x, c["xstar"]) <= 1e-7
    cz = dict(c); cz["b"] = np.zeros(c["n"])
    x, res = solve(cz, 2, 1e-8, 100)
    assert res["status"] == 0 and res["outer_iters"] == 0 and np.all(x == 0)
    ref = oracle_mod.sstep(c["rowptr"], c["colidx"], c["vals"], c["b"], 2, rtol=1e-14, maxit=3)
    x, res = solve(c, 2, 1e-14, 3)
    assert res["status"] == 1 == ref["status"] and res["outer_iters"] == 3 and rel(x, ref["x"]) <= 1e-12
    x, res = solve(c, 2, 1e-8, 0)
    assert res["status"] == 1 and res["outer_iters"] == 0 and np.all(x == 0)
    rp, ci, v, A = gen.random_spd_csr(400, 0.02, 77)
    cw = dict(rowptr=rp, colidx=ci, vals=v, b=np.random.default_rng(1).uniform(-1, 1, 400), n=400)
    x, res = solve(cw, 16, 1e-7, 50, basis=1)     # (at 1e-8 this system sits on the rounding edge of a second iteration)
    assert res["status"] == 0 and rel(x, np.linalg.solve(A, cw["b"])) <= 1e-6
    c1 = dict(rowptr=np.array([0, 1], np.int32), colidx=np.array([0], np.int32), vals=np.array([4.0]), b=np.array([2.0]), n=1)
    x, res = solve(c1, 1, 1e-12, 5)
    assert res["status"] == 0 and abs(x[0] - 0.5) <= 1e-15
    # degenerate case of the method: rank-deficient last block -> breakdown, x stays finite (the last good iterate)
    rp, ci, v = gen.poisson1d(64)
    cb = dict(rowptr=rp, colidx=ci, vals=v, b=np.random.default_rng(22).uniform(-1, 1, 64), n=64)
    ref = oracle_mod.sstep(rp, ci, v, cb["b"], 3, rtol=1e-11, maxit=30)
    x, res = solve(cb, 3, 1e-11, 30)
    assert ref["status"] == 2 and res["status"] == 2
    assert abs(res["outer_iters"] - ref["iters"]) <= 1 and np.all(np.isfinite(x))
