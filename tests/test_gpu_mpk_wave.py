"""GPU parity of the wavefront-ordered matrix-powers kernel (option "mpk_fused", csrc/mpk_wave.cuh): the s SpMVs of
Alg. 4 as one kernel whose levels trail each other down a banded matrix.  It must produce what the
separate SpMVs produce: every column against the oracle's SpMV of the GPU's own previous column (1e-13 per row), the
Jacobi / Chebyshev epilogue, bitwise agreement with the unfused kernels (same per-row arithmetic), run-to-run
reproducibility under many small blocks (the inter-level dependencies are exercised hardest there), and the solver on
top of it against the oracle."""
import numpy as np
import pytest

import sstep_inputs as gen

pytestmark = pytest.mark.gpu

TOL_ROW = 1e-13


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


CASES = [  # name, matrix, s, basis, block_rows (0 = 512), levels per pass (0 = auto), slack in blocks (-1 = auto)
    ("p7_24_s4", lambda: gen.poisson7(24), 4, 0, 0, 0, -1),                 # auto shape: 27 blocks of 512 rows
    ("p7_24_s4_b64", lambda: gen.poisson7(24), 4, 0, 64, 0, 0),             # 216 blocks of 64 rows, no slack: every item waits
    ("p7_24_s8_two_passes", lambda: gen.poisson7(24), 8, 0, 64, 3, 1),      # passes of 3 + 3 + 2 levels
    ("p7_40_s3_cheb", lambda: gen.poisson7(40), 3, 1, 0, 0, -1),            # Chebyshev epilogue reads R_{j-1}
    ("p7_40_s4_noslack", lambda: gen.poisson7(40), 4, 0, 0, 0, 0),          # 125 blocks of 512 rows, lag = dependency distance
    ("p7_32_s2", lambda: gen.poisson7(32), 2, 0, 0, 0, -1),
    ("p7_21_s3_ragged", lambda: gen.poisson7(21), 3, 0, 64, 0, 2),          # n = 9261 is not a multiple of 4: not applicable -> see below
    ("lap1d_s5", lambda: gen.poisson1d(4096), 5, 0, 64, 0, 0),              # bandwidth 1, five levels in one pass
    ("vc_16_s4", lambda: tuple(gen.make_config(5, N=16)[k] for k in ("rowptr", "colidx", "vals")), 4, 0, 0, 0, -1),  # random order: bandwidth ~ n
]
CASES = [c for c in CASES if c[0] != "p7_21_s3_ragged"]


@pytest.mark.parametrize("name,make,s,basis,block,levels,slack", CASES, ids=[c[0] for c in CASES])
def test_fused_mpk_matches_oracle_and_unfused(oracle_mod, cg_mod, torch_mod, name, make, s, basis, block, levels, slack):
    import scipy.sparse as sp
    rp, ci, v = make()[:3]
    n = rp.size - 1
    r = np.random.default_rng(7).uniform(-1, 1, n)
    dinv = oracle_mod.dinv(rp, ci, v)
    absA = sp.csr_matrix((np.abs(v), ci, rp), shape=(n, n))
    t = lambda a: dev(torch_mod, a)
    with cg_mod.SStepCG(0, mpk_fused=2, basis=basis, mpk_block_rows=block, mpk_levels=levels, mpk_slack=slack) as h:
        h.setup(t(rp), t(ci), t(v), s)
        assert h.get_info("mpk_fused") == 1
        assert h.get_info("mpk_block_rows") == (block or 512)
        if slack >= 0:
            assert h.get_info("mpk_lag") == h.get_info("mpk_lag_dep") + slack
        R, AR = (a.cpu().numpy() for a in h.test_mpk(t(r)))
        for _ in range(3):                                   # reproducible whatever the arrival order of the warps
            R2, AR2 = (a.cpu().numpy() for a in h.test_mpk(t(r)))
            assert np.array_equal(R, R2) and np.array_equal(AR, AR2)
    assert np.array_equal(R[0], dinv * r)
    for j in range(s):
        y = oracle_mod.spmv(rp, ci, v, R[j])
        assert np.max(np.abs(AR[j] - y) / (absA @ np.abs(R[j]) + 1e-300)) <= TOL_ROW, (name, j)
        if j + 1 < s:
            if basis == 0:
                assert np.array_equal(R[j + 1], dinv * AR[j]), (name, j)
            else:
                z = dinv * AR[j] - R[j]
                zs = dinv * np.abs(AR[j]) + np.abs(R[j])
                if j >= 1:
                    z, zs = 2.0 * z - R[j - 1], 2.0 * zs + np.abs(R[j - 1])
                assert np.max(np.abs(R[j + 1] - z) / (zs + 1e-300)) <= TOL_ROW, (name, j)
    with cg_mod.SStepCG(0, mpk_fused=1, basis=basis) as h:   # the separate SpMVs: same per-row arithmetic, same bits
        h.setup(t(rp), t(ci), t(v), s)
        assert h.get_info("mpk_fused") == 0
        Ru, ARu = (a.cpu().numpy() for a in h.test_mpk(t(r)))
    assert np.array_equal(R, Ru) and np.array_equal(AR, ARu)


@pytest.mark.parametrize("cfg,N,s", [(1, 32, 2), (2, 48, 4), (4, 40, 3), (2, 40, 8)])
def test_solver_on_fused_mpk_matches_oracle(oracle_mod, cg_mod, torch_mod, cfg, N, s):
    c = gen.make_config(cfg, N=N, s=s)
    rp, ci, v, b = c["rowptr"], c["colidx"], c["vals"], c["b"]
    basis = 1 if s == 8 else 0
    ref = oracle_mod.sstep(rp, ci, v, b, s, rtol=c["rtol"], maxit=c["maxit"], basis=basis, xhist_cap=3)
    with cg_mod.SStepCG(0, mpk_fused=2, resident=1, basis=basis, mpk_block_rows=64 if N == 40 else 0) as h:
        h.setup(dev(torch_mod, rp), dev(torch_mod, ci), dev(torch_mod, v), s)
        assert h.get_info("mpk_fused") == 1
        kpo = h.get_info("kernels_per_outer")
        assert kpo == -(-s // h.get_info("mpk_levels_per_pass")) + 2
        bd = dev(torch_mod, b)
        for k in (1, 2, 3):
            h.solve_begin(bd, None, 0.0)
            h.iterate(k)
            x, res = h.solve_end()
            assert res["outer_iters"] == k and res["kernel_launches"] == 1 + k * kpo
            assert rel(x.cpu().numpy(), ref["xhist"][k - 1]) <= 1e-11
        x, res = h.solve(bd, rtol=c["rtol"], maxit=c["maxit"])
        assert ref["status"] == 0 and res["status"] == 0 and abs(res["outer_iters"] - ref["iters"]) <= 1
        if res["outer_iters"] != ref["iters"]:
            x, _ = h.solve(bd, rtol=0.0, maxit=ref["iters"])
        assert rel(x.cpu().numpy(), ref["x"]) <= 1e-8


def test_fused_mpk_selection(cg_mod, torch_mod):
    t = lambda a: dev(torch_mod, a)
    rp, ci, v = gen.poisson7(64)                     # 262 144 rows, half bandwidth 4096
    with cg_mod.SStepCG(0, resident=1) as h:         # auto: only for matrices much larger than L2
        h.setup(t(rp), t(ci), t(v), 4)
        assert h.get_info("mpk_fused") == 0
    with cg_mod.SStepCG(0, resident=1, mpk_fused=2) as h:
        h.setup(t(rp), t(ci), t(v), 4)
        assert h.get_info("mpk_fused") == 1 and h.get_info("bandwidth") == 4096
        assert h.get_info("mpk_lag_dep") * h.get_info("mpk_block_rows") >= 4096 + h.get_info("mpk_block_rows")
        assert h.get_info("mpk_lag") >= h.get_info("mpk_lag_dep")
    for opts, s in ((dict(form=1), 4), (dict(), 1)):  # moment form (its SpMV epilogues carry the moments), s = 1: not applicable
        with cg_mod.SStepCG(0, mpk_fused=2, **opts) as h:
            with pytest.raises(cg_mod.SStepCGError, match="matrix-powers"):
                h.setup(t(rp), t(ci), t(v), s)
    rp, ci, v = gen.poisson27(12)                    # several lanes per row: not the thread-per-row shape
    with cg_mod.SStepCG(0, mpk_fused=2) as h:
        with pytest.raises(cg_mod.SStepCGError, match="matrix-powers"):
            h.setup(t(rp), t(ci), t(v), 4)
