"""CPU-only checks of the boundary: liblm.so builds, loads without a GPU, exports every symbol
that include/lm.h declares, fails loudly without a device, and its host-side Lanczos logic
(tridiagonal eigensolve, stopping test; through tests/hooks) matches the oracle and closed forms."""
import math
import os
import re

import numpy as np
import pytest

import paper_2510_02135_b200 as lm
from paper_2510_02135_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "lm.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(lm_[a-z0-9_]+)\s*\(", text)))


def test_header_and_binding_agree():
    names = declared_symbols()
    assert len(names) >= 20
    assert sorted(binding.SIGNATURES) == names


def test_library_exports_every_declared_symbol():
    cdll = lm.lib()
    for name in declared_symbols():
        assert hasattr(cdll, name), name
    assert "sm_100a" in lm.lm_version()


def test_sass_is_blackwell_native():
    """The built library carries sm_100a SASS with the packed fp32 FMA (FFMA2) and the TMA bulk
    copy (UBLKCP) -- not PTX to be JIT-compiled for something else."""
    import subprocess
    lib = os.path.join(ROOT, "paper_2510_02135_b200", "liblm.so")
    lm.lib()
    out = subprocess.run(["cuobjdump", "-sass", lib], capture_output=True, text=True)
    if out.returncode != 0:
        pytest.skip("cuobjdump unavailable")
    assert "sm_100a" in out.stdout
    for mnemonic in ("FFMA2", "UBLKCP", "MUFU.RSQ", "MUFU.RSQ64H", "DFMA", "SYNCS"):
        assert mnemonic in out.stdout, mnemonic


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(lm.LmError) as ei:
        lm.Solver("f32", 128)
    assert ei.value.code == lm.LM_E_CUDA
    from paper_2510_02135_b200 import probe
    with pytest.raises(RuntimeError):
        probe.fma_peak(lm.LM_F32, 0.01)


def host_tridiag(alpha, beta):
    """c = T^{1/2} e_1 from csrc/tridiag_host.h, through the test hooks (tests/hooks)."""
    from tests import hooks
    alpha = np.ascontiguousarray(alpha, dtype=np.float64)
    beta = np.ascontiguousarray(beta, dtype=np.float64)
    out = np.zeros(alpha.size)
    dp = binding.POINTER(binding.c_double)
    rc = hooks.lib().hook_tridiag_sqrt_e1(alpha.size, alpha.ctypes.data_as(dp), beta.ctypes.data_as(dp) if alpha.size > 1 else None, out.ctypes.data_as(dp))
    assert rc == 0, rc
    return out


def test_host_tridiag_sqrt_e1_closed_forms():
    assert host_tridiag([2.25], []) == pytest.approx([1.5])
    al, be = [3.0, 2.0], [1.2]
    det = al[0] * al[1] - be[0] ** 2
    den = math.sqrt(al[0] + al[1] + 2 * math.sqrt(det))
    np.testing.assert_allclose(host_tridiag(al, be), [(al[0] + math.sqrt(det)) / den, be[0] / den], rtol=1e-14)


@pytest.mark.parametrize("k", [1, 2, 3, 8, 33, 100, 400])
def test_host_tridiag_sqrt_e1_vs_oracle(k):
    from oracle import rpy
    rng = np.random.default_rng(k)
    al = 0.05 + rng.random(k)
    be = 0.3 * rng.random(max(k - 1, 0))
    c = host_tridiag(al, be)
    np.testing.assert_allclose(c, rpy.tridiag_sqrt_e1(al, be), rtol=1e-10, atol=1e-13)
    # indefinite T: negative eigenvalues are clamped, not NaN
    al2 = al - 0.6
    c2 = host_tridiag(al2, be)
    assert np.isfinite(c2).all()
    np.testing.assert_allclose(c2, rpy.tridiag_sqrt_e1(al2, be), rtol=1e-9, atol=1e-12)


def test_host_tridiag_bad_args():
    from tests import hooks
    assert hooks.lib().hook_tridiag_sqrt_e1(0, None, None, None) == lm.LM_E_INVALID
    assert hooks.lib().hook_tridiag_sqrt_e1(2, None, None, None) == lm.LM_E_NULL


def test_host_error_estimate_equals_the_oracles_on_random_step_sequences():
    """csrc/lanczos_host.h against oracle/rpy.py (written independently from DESIGN.md reading S3) and the closed
    form for geometric steps: s_k / (1 - rho) for rho >= 1/2."""
    from oracle import rpy
    from tests import hooks
    dp = binding.POINTER(binding.c_double)
    est = lambda s: hooks.lib().hook_error_estimate(np.ascontiguousarray(s, dtype=np.float64).ctypes.data_as(dp), len(s))
    rng = np.random.default_rng(0)
    for n in (2, 3, 4, 5, 9, 19, 20, 21, 22, 60):
        s = np.exp(-0.3 * np.arange(n) + 0.8 * rng.standard_normal(n))
        assert est(s) == pytest.approx(rpy.step_error_estimate(s), rel=1e-13)
    for rho in (0.5, 0.8, 0.97):
        s = 0.2 * rho ** np.arange(2, 30)
        assert est(s) == pytest.approx(s[-1] / (1 - rho), rel=1e-12)
    assert est([1e-3] * 30) == pytest.approx(49e-3, rel=1e-9)
    assert est([0.0, 0.0, 0.0]) == 0.0


@pytest.mark.parametrize("rule", ["estimate", "step"])
def test_host_stopper_stops_where_the_oracle_does(rule):
    """The host stopping test (coefficient space, Gram matrix) fed with the alpha_k, beta_k and Gram columns of an
    exact-arithmetic Lanczos run stops at the oracle's step and yields the oracle's coefficients."""
    from oracle import rpy
    from tests import hooks
    L = hooks.lib()
    dp = binding.POINTER(binding.c_double)
    rng = np.random.default_rng(11)
    N, tol = 150, 1e-3
    pos = rng.random((N, 3)) * 9.0
    M = rpy.dense(pos)
    z = rng.standard_normal(3 * N)
    y, k_or, conv = rpy.lanczos_sqrt_mdot_w(pos, z, tol, apply=lambda v: M @ v, rule=rule)
    assert conv
    # an independent plain recurrence to produce alpha, beta, V
    V = [z / np.linalg.norm(z)]
    st = L.hook_stopper_new(0 if rule == "estimate" else 1, tol, 1e-14, 100)
    col = lambda m: np.ascontiguousarray([V[j] @ V[m] for j in range(m + 1)])
    c0 = col(0)
    L.hook_stopper_gram_column(st, 0, c0.ctypes.data_as(dp))
    beta_prev, k_stop = 0.0, None
    for k in range(1, 101):
        w = M @ V[k - 1] - (beta_prev * V[k - 2] if k > 1 else 0.0)
        alpha = w @ V[k - 1]
        w = w - alpha * V[k - 1]
        beta = np.linalg.norm(w)
        V.append(w / beta)
        verdict = L.hook_stopper_feed(st, k, float(alpha), float(beta))
        if verdict == 1:
            k_stop = k
            break
        assert verdict == 0
        L.hook_stopper_advance(st)
        ck = col(k)
        L.hook_stopper_gram_column(st, k, ck.ctypes.data_as(dp))
        beta_prev = beta
    assert k_stop == k_or
    c = np.zeros(k_stop)
    assert L.hook_stopper_coefficients(st, c.ctypes.data_as(dp), k_stop) == k_stop
    y_host = np.linalg.norm(z) * (np.stack(V[:k_stop], 1) @ c)
    assert np.linalg.norm(y_host - y) <= 1e-10 * np.linalg.norm(y)
    assert L.hook_stopper_last_measure(st) <= tol
    L.hook_stopper_free(st)


def test_workloads_are_seeded_and_shaped():
    from paper_2510_02135_b200 import workloads
    d1, d1b = workloads.generate(1), workloads.generate(1)
    assert d1["pos"].dtype == np.float64 and d1["pos"].shape == (1024, 3)
    assert np.array_equal(d1["pos"], d1b["pos"]) and np.array_equal(d1["forces"], d1b["forces"])
    assert 0 <= d1["pos"].min() and d1["pos"].max() <= 40.0
    d2 = workloads.generate(2)
    assert d2["pos"].dtype == np.float32 and d2["torques"].shape == (16384, 3)
    assert d2["pos"].max() <= workloads.cube_side(16384, 0.10) + 1e-3
    assert workloads.cube_side(16384, 0.10) == pytest.approx(88.207, abs=1e-3)
    assert workloads.cube_side(131072, 0.05) == pytest.approx(222.268, abs=1e-3)
    assert workloads.cube_side(1048576, 0.01) == pytest.approx(760.145, abs=1e-3)
    d3 = workloads.generate(3, N=2048)
    assert d3["noise"].shape == (3 * 2048,) and d3["noise"].dtype == np.float32
    d5 = workloads.generate(5, N=6400)
    assert d5["pos"].dtype == np.float64 and d5["torques"] is not None
    # clusters: contiguous ids, sigma = 3
    c0 = d5["pos"][:100]
    assert np.all(c0.std(0) < 5.0) and np.all(c0.std(0) > 1.5)
    f = workloads.fcc(4, 0.05, 0.1, 0)
    assert f.shape == (256, 3)
