"""The headline call -- lm_sqrt_mdot_w at config 3 (N = 131072, phi = 5 %, tol 1e-3, default rule "estimate"), the call
bench.py times -- against the ORACLE's run of the same problem.

The oracle needs ~75 fp64 O(N^2) applies for it (about half an hour of CPU), so its run is stored:
tests/golden/c3_lanczos_tol1e-3.json, written by tests/golden/make_c3_lanczos.py, which imports only oracle/ and the
seeded input generator.  Gates (S4):
  * alpha_k, beta_k for k <= 15 -- before the recurrences separate (plain Lanczos amplifies rounding differences
    geometrically once the top Ritz values have converged) -- to 1e-4 relative in fp32, 1e-9 in fp64;
  * the stop step within the S4(ii) window of the oracle's;
  * the final iterate on the 64 stored rows within 2 tol of the oracle's (both are within the rule's error of the root);
  * sqrt(M) sqrt(M) z = M z on the stored oracle rows of M z (exact for those rows): two applications, each within
    ~2 tol of the root -> 5 tol.
"""
import json
import os

import numpy as np
import pytest

from paper_2510_02135_b200 import workloads

pytestmark = pytest.mark.gpu

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "c3_lanczos_tol1e-3.json")


def rel(a, b):
    a = np.asarray(a, dtype=np.float64).reshape(-1)
    b = np.asarray(b, dtype=np.float64).reshape(-1)
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


@pytest.fixture(scope="module")
def golden():
    with open(GOLDEN) as f:
        g = json.load(f)
    assert g["config"] == 3 and g["rule"] == "estimate" and g["converged"]
    return g


@pytest.fixture(scope="module")
def problem(golden):
    d = workloads.generate(3)
    assert d["N"] == golden["N"] and d["cfg"].tol == golden["tol"] and d["cfg"].seed == golden["seed"]
    return d


def dev(x):
    import torch
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


@pytest.mark.parametrize("prec", ["f32", "f64"])
def test_config3_lanczos_matches_the_oracles_run(golden, problem, prec):
    import torch

    import paper_2510_02135_b200 as lm
    N, tol, ko = golden["N"], golden["tol"], golden["iterations"]
    dt = workloads.np_dtype(prec)
    s = lm.Solver(prec, N, golden["eta"], golden["a"], False)
    s.set_max_iter(200)
    s.set_positions(dev(problem["pos"].astype(dt)))
    y = torch.empty(3 * N, dtype=s.torch_dtype, device="cuda")
    it = s.sqrt_mdot_w(dev(problem["noise"].astype(dt)), tol, y)
    torch.cuda.synchronize()
    assert s.pair_launch_config(1)["kernel"] == "rpy_pair_kernel"
    hist = s.lanczos_history()
    k_cmp = 15
    rtol = 1e-4 if prec == "f32" else 1e-9
    np.testing.assert_allclose(hist["alpha"][:k_cmp], golden["alphas"][:k_cmp], rtol=rtol)
    np.testing.assert_allclose(hist["beta"][:k_cmp], golden["betas"][:k_cmp], rtol=rtol)
    assert abs(it - ko) <= max(2, ko // 3), (prec, it, ko)
    rows = np.asarray(golden["rows"])
    got = y.cpu().numpy().reshape(N, 3)[rows]
    e = rel(got, golden["y_rows"])
    assert e <= 2 * tol, (prec, it, ko, e)
    s.close()


def test_config3_square_root_twice_is_m_on_oracle_rows(golden, problem):
    import torch

    import paper_2510_02135_b200 as lm
    N, tol = golden["N"], golden["tol"]
    s = lm.Solver("f32", N, golden["eta"], golden["a"], False)
    s.set_max_iter(200)
    s.set_positions(dev(problem["pos"]))
    z = dev(problem["noise"])
    y1, y2 = torch.empty_like(z), torch.empty_like(z)
    it1 = s.sqrt_mdot_w(z, tol, y1)
    it2 = s.sqrt_mdot_w(y1, tol, y2)
    torch.cuda.synchronize()
    rows = np.asarray(golden["rows"])
    e = rel(y2.cpu().numpy().reshape(N, 3)[rows], golden["mz_rows"])
    assert e <= 5 * tol, (it1, it2, e)
    s.close()
