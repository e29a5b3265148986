"""Programmatic dependent launch (option pdl, include/sstep_cg.h): the kernels of one outer iteration are chained with
programmatic edges so that the next kernel's blocks become resident while the current one drains.  Every kernel touches
solver data only behind `griddepcontrol.wait`, so the results must be BITWISE those of the plainly serialised graph
(pdl = 0) -- for every kernel family on the path: bulk-staged and vector-per-row SpMV, register and TMA-staged Gram /
update kernels, the moment form's scalar-work kernel, the Chebyshev epilogue, the Alg. 1 sequence.  The parity of the
pdl = 1 path against the oracle is what every other GPU test file checks (pdl = 1 is the default)."""
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


def run(cg, torch, c, s, maxit, **opts):
    opts.setdefault("resident", 1)  # graph path: the resident path is one cooperative launch, no chain to overlap
    with cg.SStepCG(0, **opts) as h:
        h.setup(dev(torch, c["rowptr"]), dev(torch, c["colidx"]), dev(torch, c["vals"]), s)
        pdl = h.get_info("pdl")
        x, res = h.solve(dev(torch, c["b"]), None, rtol=c["rtol"], maxit=maxit)
        return x.cpu().numpy(), res, pdl


CASES = [  # cfg, N, s, maxit, options
    (1, 32, 2, 2000, {}),                          # bulk SpMV, register Gram / update, full solve
    (2, 48, 4, 2000, {}),
    (4, 64, 8, 12, {}),                            # TMA-staged Gram / update (s >= 5), fixed number of iterations
    (3, 24, 4, 2000, {"spmv_variant": 1}),         # vector-per-row SpMV (27-point)
    (3, 32, 4, 2000, {}),                          # 27-point on the 512-entry bulk tiles
    (2, 40, 4, 2000, {"form": 1}),                 # moment form: SpMV with moment partials + sw_kernel
    (4, 48, 8, 2000, {"basis": 1}),                # Chebyshev epilogue
    (2, 40, 1, 2000, {"method": 1}),               # Alg. 1 sequence: PDL SpMV between plain kernels
    (5, 24, 4, 2000, {"reorder": 2}),              # reordered copy of the CSR arrays
]


@pytest.mark.parametrize("cfg,N,s,maxit,opts", CASES)
def test_pdl_is_bitwise_the_serialised_graph(cg_mod, torch_mod, cfg, N, s, maxit, opts):
    c = gen.make_config(cfg, N=N, s=s)
    x1, r1, pdl1 = run(cg_mod, torch_mod, c, s, maxit, pdl=1, **opts)
    x0, r0, pdl0 = run(cg_mod, torch_mod, c, s, maxit, pdl=0, **opts)
    assert pdl0 == 0
    assert pdl1 == 1, "the driver refused to capture programmatic edges: the pdl = 1 path was not exercised"
    assert r1["outer_iters"] == r0["outer_iters"] and r1["status"] == r0["status"]
    assert r1["relres"] == r0["relres"]
    assert np.array_equal(x1, x0)


def test_pdl_without_graph_is_bitwise_too(cg_mod, torch_mod):
    """use_graph = 0: the same attribute on plain stream launches (programmatic stream serialisation)."""
    c = gen.make_config(2, N=40, s=4)
    x1, r1, _ = run(cg_mod, torch_mod, c, 4, 2000, pdl=1, use_graph=0)
    x0, r0, _ = run(cg_mod, torch_mod, c, 4, 2000, pdl=0, use_graph=0)
    assert r1["outer_iters"] == r0["outer_iters"] and r1["relres"] == r0["relres"]
    assert np.array_equal(x1, x0)


def test_stopped_solver_with_copies_in_flight(cg_mod, torch_mod):
    """After convergence the remaining graph replays of a chunk find status != running: the bulk SpMV has then already
    staged its first CSR tiles (ahead of griddepcontrol.wait) and must let them land before it exits.  Many such
    replays in a row, then a second solve on the same handle, must leave x and the next solve untouched."""
    c = gen.make_config(1, N=32, s=2)
    with cg_mod.SStepCG(0, resident=1, pdl=1) as h:
        h.setup(dev(torch_mod, c["rowptr"]), dev(torch_mod, c["colidx"]), dev(torch_mod, c["vals"]), 2)
        b = dev(torch_mod, c["b"])
        xa, ra = h.solve(b, None, rtol=c["rtol"], maxit=2000)
        h.solve_begin(b, None, c["rtol"])
        h.iterate(ra["outer_iters"] + 200)  # 200 replays past the stop
        xb, rb = h.solve_end()
        xc, rc = h.solve(b, None, rtol=c["rtol"], maxit=2000)
    assert ra["status"] == 0 and rb["status"] == 0 and rc["status"] == 0
    assert rb["outer_iters"] == ra["outer_iters"] == rc["outer_iters"]
    assert torch_mod.equal(xa, xb) and torch_mod.equal(xa, xc)
