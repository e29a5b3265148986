"""sstep_cg_gram_noalloc (include/sstep_cg.h): the allocation-free entry point of step a2 (M = R^T AR, C = AP^T R,
m = R^T r; Eq. 3-4) for callers that cannot call cudaMalloc.  It runs the production Gram kernel on a
static device array of the library image instead of cudaMalloc'ed scratch; its output must equal the existing path's
(sstep_cg_test_gram after sstep_cg_setup) within the Gram tolerance of tests/test_gpu_parity.py, on two calls in a row
(the second one on other data and another size: the shared scratch keeps the first call's contents), and the calls must
not change the device's free memory.  Collected last on purpose (the file name): a failure here hides no other test.
"""
import numpy as np
import pytest

import sstep_inputs as gen

pytestmark = pytest.mark.gpu

TOL_GRAM = 1e-12      # |M - M_ref|(i, j) <= TOL_GRAM * ||a_i||_2 ||b_j||_2, as in tests/test_gpu_parity.py


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


def gram_close(M, Mr, A, B):
    scale = np.outer(np.linalg.norm(A, axis=1), np.linalg.norm(B, axis=1))
    return np.all(np.abs(M - Mr) <= TOL_GRAM * scale)


@pytest.mark.parametrize("s", [1, 3, 4, 8])
def test_gram_noalloc_matches_existing_path_twice_in_a_row(oracle_mod, cg_mod, torch_mod, s):
    torch = torch_mod
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    rng = np.random.default_rng(900 + s)
    with cg_mod.SStepCG(0) as h_static:                     # create only: no setup, no matrix, no workspaces
        M = torch.empty((s, s), dtype=torch.float64, device="cuda")
        C = torch.empty_like(M)
        m = torch.empty(s, dtype=torch.float64, device="cuda")
        for call, n in enumerate((300_001, 70_003)):        # two calls in a row on the shared static scratch
            R, AR, AP = (rng.uniform(-1, 1, (s, n)) for _ in range(3))
            r = rng.uniform(-1, 1, n)
            dR, dAR, dr = dev(R), dev(AR), dev(r)
            dAP_il = dev(AP).t().contiguous()               # interleaved (n, s), as the kernels take it
            M.fill_(float("nan")); C.fill_(float("nan")); m.fill_(float("nan"))
            torch.cuda.synchronize()
            free_before = torch.cuda.mem_get_info()[0]
            h_static.gram_noalloc(dR, dAR, dAP_il, dr, M, C, m)
            torch.cuda.synchronize()
            if call > 0:                                    # (the first launch of a kernel may load its module)
                assert torch.cuda.mem_get_info()[0] == free_before, "the call changed the device's free memory"
            # the existing path: sstep_cg_setup (cudaMalloc'ed scratch) + sstep_cg_test_gram
            rp, ci, v = gen.poisson1d(n)
            with cg_mod.SStepCG(0) as h_ref:
                h_ref.setup(dev(rp), dev(ci), dev(v), s)
                M_ref, C_ref, m_ref = (t.cpu().numpy() for t in h_ref.test_gram(dR, dAR, dev(AP), dr))
            Mg, Cg, mg = M.cpu().numpy(), C.cpu().numpy(), m.cpu().numpy()
            assert np.all(np.isfinite(Mg)) and np.all(np.isfinite(Cg)) and np.all(np.isfinite(mg))
            assert gram_close(Mg, M_ref, R, AR) and gram_close(Cg, C_ref, AP, R), (s, call)
            assert np.all(np.abs(mg - m_ref) <= TOL_GRAM * np.linalg.norm(R, axis=1) * np.linalg.norm(r)), (s, call)
            # and against the oracle's definition (orc_gram), same bar
            Mo, Co, mo = oracle_mod.gram(R, AR, AP, r)
            assert gram_close(Mg, Mo, R, AR) and gram_close(Cg, Co, AP, R)
            assert np.all(np.abs(mg - mo) <= TOL_GRAM * np.linalg.norm(R, axis=1) * np.linalg.norm(r))


def test_gram_noalloc_rejects_sizes_beyond_the_static_scratch(cg_mod, torch_mod):
    torch = torch_mod
    s, n = 9, 1000                                          # the static array holds 2 s^2 + s entries for s <= 8 only
    z = lambda *shape: torch.zeros(shape, dtype=torch.float64, device="cuda")
    with cg_mod.SStepCG(0) as h:
        with pytest.raises(cg_mod.SStepCGError, match=r"1\.\.8"):
            h.gram_noalloc(z(s, n), z(s, n), z(n, s), z(n), z(s, s), z(s, s), z(s))
        # the handle stays usable, and the largest supported block size goes through
        s = 8
        M = z(s, s)
        h.gram_noalloc(torch.ones((s, n), dtype=torch.float64, device="cuda"), torch.ones((s, n), dtype=torch.float64, device="cuda"),
                       z(n, s), z(n), M, z(s, s), z(s))
        torch.cuda.synchronize()
        assert torch.all(M == float(n))
