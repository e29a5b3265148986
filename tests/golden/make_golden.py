#!/usr/bin/env python
"""Writes the full-size end-to-end fixtures tests/golden/<case>.txt -- calls ONLY oracle/ (and the seeded input
generators of sstep_inputs/, which hold none of the method's arithmetic).  Nothing here touches the CUDA path.

  python tests/golden/make_golden.py --case config4_s4        (one case; several can run side by side)
  python tests/golden/make_golden.py --list

Each fixture records what the oracle's Alg. 3 (Gram form O2 of DESIGN.md section 2) does on one
BASELINE.json config at FULL size, with the config's own rtol and the stop test of reading A7
(||r||_2 < rtol ||r_0||_2): the outer-iteration count, the status, the relative-residual history
(Alg. 3 l.31-33), ||x||_2 and max|x| at the stopping iteration and NS seeded sample entries of x there.
The GPU tests (tests/test_gpu_golden.py) compare: count within +-1, history, sampled x within 1e-8 (north_star),
true residual.  Cost: under a second (config 1) to 5-15 CPU-minutes (configs 4-6) per case on one thread, run once; the files are committed.
"""
from __future__ import annotations

import argparse
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import oracle  # noqa: E402
import sstep_inputs as gen  # noqa: E402

NS = 2048            # sampled entries of x per fixture
SAMPLE_SEED = 777    # numpy.random.default_rng(SAMPLE_SEED).choice(n, NS, replace=False), sorted

# case -> (config, s, basis, method); method "sstep" = Alg. 3 (Gram form), "sstep_moment" = Alg. 3 with Alg. 5 + 6, "pcg" = Alg. 1
CASES = {
    "config1_s2": (1, 2, 0, "sstep"), "config2_s4": (2, 4, 0, "sstep"), "config3_s4": (3, 4, 0, "sstep"),
    "config4_s1": (4, 1, 0, "sstep"), "config4_s2": (4, 2, 0, "sstep"), "config4_s4": (4, 4, 0, "sstep"),
    "config5_s8_cheb": (5, 8, 1, "sstep"), "config5_s8_mono": (5, 8, 0, "sstep"),
    "config6_s1": (6, 1, 0, "sstep"), "config6_s2": (6, 2, 0, "sstep"), "config6_s3": (6, 3, 0, "sstep"),
    "config6_s4": (6, 4, 0, "sstep"), "config6_s5": (6, 5, 0, "sstep"), "config6_pcg": (6, 1, 0, "pcg"),
    # the paper-literal moment form (Alg. 5 + Alg. 6 with the moments taken in the SpMV epilogues: oracle form "moment_fused")
    "config4_s4_moment": (4, 4, 0, "sstep_moment"), "config6_s4_moment": (6, 4, 0, "sstep_moment"),
}


def sample_indices(n: int) -> np.ndarray:
    return np.sort(np.random.default_rng(SAMPLE_SEED).choice(n, NS, replace=False))


def run_case(name: str, N: int | None = None) -> str:
    cfg, s, basis, method = CASES[name]
    c = gen.make_config(cfg, N=N, s=s)
    t0 = time.time()
    if method == "pcg":
        ref = oracle.pcg(c["rowptr"], c["colidx"], c["vals"], c["b"], rtol=c["rtol"], maxit=c["maxit"], history=True)
    else:
        ref = oracle.sstep(c["rowptr"], c["colidx"], c["vals"], c["b"], s, rtol=c["rtol"], maxit=c["maxit"], basis=basis,
                           history=True, form="moment_fused" if method == "sstep_moment" else "gram")
    dt = time.time() - t0
    x = ref["x"]
    idx = sample_indices(c["n"])
    lines = [
        f"# tests/golden/{name}.txt -- written by `python tests/golden/make_golden.py --case {name}" + (f" --grid {N}`" if N else "`"),
        "# from oracle/ only (oracle.pcg = Alg. 1, PAPER.md:48-73; oracle.sstep = Alg. 3, PAPER.md:158, Gram or moment form; stop test",
        "# ||r||_2 < rtol ||r_0||_2, PAPER.md:259).  Never edited by hand, never written from the CUDA path.",
        f"# workload: sstep_inputs.make_config({cfg}" + (f", N={N}" if N else "") + f") = {c['name']}, n = {c['n']}, nnz = {c['nnz']}, rtol = {c['rtol']:g}",
        f"# oracle wall time {dt:.0f} s (one thread)",
        f"config {cfg}", f"grid {c['N']}", f"n {c['n']}", f"s {s}", f"basis {basis}", f"method {method}", f"rtol {c['rtol']!r}",
        f"status {ref['status']}", f"iters {ref['iters']}", f"relres {ref['relres']!r}",
        f"xnorm2 {float(np.linalg.norm(x))!r}", f"xmaxabs {float(np.abs(x).max())!r}",
        f"sample_seed {SAMPLE_SEED}", f"nsample {NS}",
    ]
    lines += [f"hist {k} {v!r}" for k, v in enumerate(ref["hist"].tolist())]
    lines += [f"x {int(i)} {float(x[i])!r}" for i in idx]
    out = os.path.join(HERE, name + (f"_grid{N}" if N else "") + ".txt")
    with open(out, "w") as f:
        f.write("\n".join(lines) + "\n")
    return out


def load(path: str) -> dict:
    """Parse a fixture (used by the tests; here so that writer and reader of the format sit together)."""
    d: dict = {"hist": [], "xi": [], "xv": []}
    for ln in open(path):
        if ln.startswith("#") or not ln.strip():
            continue
        t = ln.split()
        if t[0] == "hist":
            d["hist"].append(float(t[2]))
        elif t[0] == "x":
            d["xi"].append(int(t[1])); d["xv"].append(float(t[2]))
        elif t[0] in ("method",):
            d[t[0]] = t[1]
        elif t[0] in ("rtol", "relres", "xnorm2", "xmaxabs"):
            d[t[0]] = float(t[1])
        else:
            d[t[0]] = int(t[1])
    d["hist"] = np.array(d["hist"]); d["xi"] = np.array(d["xi"], dtype=np.int64); d["xv"] = np.array(d["xv"])
    return d


if __name__ == "__main__":
    ap = argparse.ArgumentParser()
    ap.add_argument("--case", action="append", default=[])
    ap.add_argument("--grid", type=int, default=0, help="override the grid edge (for trying the script out; full size = 0)")
    ap.add_argument("--list", action="store_true")
    a = ap.parse_args()
    if a.list:
        print("\n".join(CASES))
    for nm in a.case:
        print(run_case(nm, a.grid or None), flush=True)
