"""CPU-side tests of the C-ABI library: it loads, exports every symbol include/pm.h declares, validates
arguments without a GPU, and its host-side fp64 growth / step factors (Heath quadrature) agree with the
oracle's independent route (the growth ODE of App. A) and with the EdS closed forms."""
import ctypes as C
import os
import re
import subprocess

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def binding():
    from paper_2211_09815_b200 import build
    build.build()
    from paper_2211_09815_b200 import binding
    return binding


def declared_functions():
    src = open(os.path.join(ROOT, "include", "pm.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(pm_[a-z0-9_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol(binding):
    names = declared_functions()
    assert len(names) >= 25
    lib = C.CDLL(binding.LIB_PATH)
    for n in names:
        assert hasattr(lib, n), f"libpm.so does not export {n}"
    assert sorted(binding.EXPORTS) == names, "binding.py and pm.h disagree on the call list"


def test_library_is_built_for_sm_100a(binding):
    out = subprocess.run(["cuobjdump", "-lelf", binding.LIB_PATH], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def test_workspace_query_and_argument_checks(binding):
    a = [0.5, 0.75, 1.0]
    n1 = binding.workspace_bytes((64, 64, 64), (32, 32, 32), 0.3, a)
    n2 = binding.workspace_bytes((64, 64, 64), (32, 32, 32), 0.3, np.linspace(0.1, 1.0, 101))
    assert n1 == n2 > 0, "workspace must not depend on the number of steps (PAPER.md L37, L400-402)"
    big = binding.workspace_bytes((1024,) * 3, (512,) * 3, 0.3, a)
    assert 40e9 < big < 80e9
    for bad in [dict(mesh=(64, 64, 63)), dict(mesh=(1, 64, 64)), dict(lattice=(0, 32, 32)), dict(omega_m=0.0),
                dict(omega_m=1.5), dict(a=[0.5, 0.5]), dict(a=[0.5, -1.0]), dict(mesh=(8192, 64, 64)),
                dict(lattice=(7, 32, 32))]:
        kw = dict(mesh=(64, 64, 64), lattice=(32, 32, 32), omega_m=0.3, a=a)
        kw.update(bad)
        with pytest.raises(binding.PMError) as e:
            binding.workspace_bytes(**kw)
        assert e.value.code == binding.PM_EINVAL
    assert b"PM_ESTATE" in binding._lib.pm_strerror(binding.PM_ESTATE)


def test_no_cpu_fallback(binding):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(RuntimeError):
        binding.PM((16, 16, 16), (8, 8, 8), 1.0, [0.5, 1.0])


def test_host_growth_eds_closed_forms(binding):
    # PAPER.md eq. 14-15, A7 with D1 = a: G_D = a^1.5, G_K = 1.5 a
    for a in (1 / 64, 0.1, 0.5, 1.0):
        D1, D1p, GD, GK = binding.host_growth(1.0, a)
        np.testing.assert_allclose([D1, D1p, GD, GK], [a, a, a ** 1.5, 1.5 * a], rtol=1e-12)
    a0, a1 = 0.25, 0.3125
    ah = 0.5 * (a0 + a1)
    K1, D, K2 = binding.host_step_factors(1.0, a0, a1)
    np.testing.assert_allclose(K1, (ah ** 1.5 - a0 ** 1.5) / (1.5 * a0), rtol=1e-12)
    np.testing.assert_allclose(D, (a1 - a0) / ah ** 1.5, rtol=1e-12)
    np.testing.assert_allclose(K2, (a1 ** 1.5 - ah ** 1.5) / (1.5 * a1), rtol=1e-12)


@pytest.mark.parametrize("om", [0.3, 0.7, 1.0])
def test_host_growth_matches_oracle_ode(binding, orc, om):
    for a in (1 / 64, 0.2, 0.6, 1.0):
        g = binding.host_growth(om, a)
        go, gd = orc.growth(om, a), orc.GD_GK(om, a)
        np.testing.assert_allclose(g, [go[0], go[1], gd[0], gd[1]], rtol=2e-8)
    for a0, a1 in ((1 / 64, 2 / 64), (0.5, 0.515625), (63 / 64, 1.0)):
        ah = 0.5 * (a0 + a1)
        ref = [orc.kick_factor(om, a0, a0, ah), orc.drift_factor(om, ah, a0, a1), orc.kick_factor(om, a1, ah, a1)]
        np.testing.assert_allclose(binding.host_step_factors(om, a0, a1), ref, rtol=2e-8)


def test_own_fft_memory_order_is_the_dif_digit_reversal(binding):
    """pm_host_fft_order against an independent numpy run of the same in-place decimation-in-frequency schedule
    (radix 16 per stage, 8 where a radix-2 stage would otherwise remain, csrc/pm_fft.cu): position p of the staged result must hold numpy.fft.fft's bin out[p]."""
    rng = np.random.default_rng(3)
    for n in (8, 16, 32, 64, 128, 256, 512, 1024):
        order = np.asarray(binding.host_fft_order(n))
        assert sorted(order.tolist()) == list(range(n))                  # a permutation
        x = rng.standard_normal(n) + 1j * rng.standard_normal(n)
        y = x.copy()
        L = n
        while L > 1:
            R = (8 if (L.bit_length() - 1) % 4 == 1 else 16) if L >= 16 else L
            Lr = L // R
            for blk in range(n // L):
                for j in range(Lr):
                    idx = blk * L + j + Lr * np.arange(R)
                    a = y[idx]
                    q = np.arange(R)
                    # R-point DFT over m, then the stage twiddle w_L^(j q), stored at blk L + j + q L/R
                    y[idx] = (np.exp(-2j * np.pi * np.outer(q, np.arange(R)) / R) @ a) * np.exp(-2j * np.pi * j * q / L)
            L = Lr
        ref = np.fft.fft(x)
        assert np.allclose(y, ref[order], rtol=1e-10, atol=1e-10), n
    with pytest.raises(binding.PMError):
        binding.host_fft_order(48)


def test_host_ic_factors_match_the_oracle_by_another_route():
    """pm_host_ic_factors integrates eq. A1 in D (RK4), the oracle eq. A5 in G: D2, D2' agree; EdS closed form (A3)."""
    from oracle import pm_oracle as orc
    from paper_2211_09815_b200 import binding
    for om, a0 in ((1.0, 0.25), (0.3, 1.0 / 64), (0.3, 0.5)):
        np.testing.assert_allclose(binding.host_ic_factors(om, a0), orc.ic_factors(om, a0), rtol=3e-8)
    f = binding.host_ic_factors(1.0, 0.25)
    np.testing.assert_allclose(f, [0.25, 3 / 7 * 0.0625, 0.25 ** 1.5, 6 / 7 * 0.25 ** 2.5], rtol=1e-9)
