"""Host-side checks of libmicsa.so that need no GPU (-m "not gpu"):
the library loads, exports every symbol include/micsa.h declares, its host
logic (thresholds, workspace sizing, argument validation) is right, and it
fails loudly -- no CPU fallback -- when there is no device."""
import ctypes
import re
from pathlib import Path

import numpy as np
import pytest

ROOT = Path(__file__).resolve().parent.parent


def _has_gpu():
    try:
        import torch
        return torch.cuda.is_available()
    except Exception:
        return False


def test_exports_every_declared_symbol(micsa):
    header = (ROOT / "include" / "micsa.h").read_text()
    body = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\b(micsa_[a-z0-9_]+)\s*\(", body))
    assert declared, "no declarations parsed"
    assert declared == set(micsa.EXPORTS)
    lib = ctypes.CDLL(str(micsa.LIB_PATH))
    for name in declared:
        assert hasattr(lib, name), name


def test_no_torch_types_in_abi():
    header = (ROOT / "include" / "micsa.h").read_text()
    assert "torch" not in re.sub(r"/\*.*?\*/", "", header, flags=re.S).lower()
    assert 'extern "C"' in header


@pytest.mark.parametrize("T", [3.0, 2.0, 1.5, 1.1019, 0.9, 0.7, 0.2, 0.05, 1e3,
                               2.9971971971971973, 0.2028028028028028])
def test_thresholds_equal_oracle(micsa, oracle, T):
    """DESIGN.md R7: both sides compute the integer thresholds on the host in
    float64; bit-exact refresh parity rests on their equality."""
    np.testing.assert_array_equal(micsa.debug_thresholds(T), oracle.thresholds(T))


def test_thresholds_equal_oracle_on_config5_ramp(micsa, oracle):
    from micsa_workloads import CONFIGS, schedule_for
    for T, _, _ in schedule_for(CONFIGS[5]):
        np.testing.assert_array_equal(micsa.debug_thresholds(T), oracle.thresholds(T))


@pytest.mark.parametrize("T", [0.0, -1.0, float("nan"), float("inf")])
def test_thresholds_reject_bad_T(micsa, T):
    with pytest.raises(micsa.MicsaError) as ei:
        micsa.debug_thresholds(T)
    assert ei.value.code == micsa.MICSA_ERR_INVALID


def test_workspace_bytes(micsa):
    # config 4: 4.096M sites x (1 spin + 2 daemon + 2 staged daemon words) x 4 B + 3 bond planes x 2 B
    N = 160 ** 3
    packed = N * 4 * 5 + N * 3 * 2
    ws = micsa.workspace_bytes(160, 16, 2)
    assert packed <= ws <= packed + 65536
    assert micsa.workspace_bytes(64, 1024, 1) >= 64 ** 3 * 32 * 4 * 6
    # invalid geometry -> 0 and an error string
    assert micsa.workspace_bytes(7, 1, 1) == 0 and "even" in micsa.last_error()
    assert micsa.workspace_bytes(0, 1, 1) == 0
    assert micsa.workspace_bytes(8, 0, 1) == 0
    assert micsa.workspace_bytes(8, 1, 0) == 0


def test_invalid_create_arguments(micsa):
    for args in [(7, 1, 2, 1), (8, 0, 2, 1), (8, 1, 0, 1), (-2, 1, 1, 1)]:
        with pytest.raises(micsa.MicsaError):
            micsa.MicSA(*args, use_torch=False)
    with pytest.raises(micsa.MicsaError):
        micsa.MicSA(8, 1, 2, 1, sample_offset=3, use_torch=False)


@pytest.mark.skipif(_has_gpu(), reason="checks the no-GPU failure mode")
def test_fails_loudly_without_gpu(micsa):
    with pytest.raises(micsa.MicsaError) as ei:
        micsa.MicSA(8, 1, 2, 1, use_torch=False)
    assert "no CPU fallback" in str(ei.value)
    with pytest.raises(micsa.MicsaError):
        micsa.MicSA(8, 1, 2, 1, use_torch=True)


def test_null_context_is_an_error_not_a_crash(micsa):
    lib = micsa._lib
    assert lib.micsa_sweep(None, 1) == micsa.MICSA_ERR_INVALID
    assert lib.micsa_refresh_demons(None, 1.0, 0) == micsa.MICSA_ERR_INVALID
    assert lib.micsa_measure(None, None, None, None) == micsa.MICSA_ERR_INVALID
    assert lib.micsa_destroy(None) == micsa.MICSA_OK


def test_product_does_not_import_oracle():
    """The product path must not route through the oracle (or any CPU path)."""
    for p in (ROOT / "paper_2506_16240_b200").rglob("*"):
        if p.suffix in (".py", ".cu", ".cuh", ".h"):
            txt = p.read_text()
            assert "oracle" not in txt.lower().replace("no cpu fallback", ""), p


@pytest.mark.parametrize("T", [50.0, 3.0, 2.0, 1.1019, 0.9, 0.7, 0.3, 0.2, 0.05, 1e6])
def test_metropolis_thresholds_equal_oracle(micsa, oracle, T):
    """The Boltzmann factors exp(-4k/T) * 2^32 of the canonical comparator are
    computed on the host on both sides; bit-exact parity rests on their equality."""
    np.testing.assert_array_equal(micsa.debug_metropolis_thresholds(T), oracle.metropolis_thresholds(T))
    with pytest.raises(micsa.MicsaError):
        micsa.debug_metropolis_thresholds(0.0)


@pytest.mark.parametrize("T", [0.3, 0.7, 0.9, 1.1019, 1.4, 2.0, 3.0, 10.0, 100.0])
def test_effective_temperature_inverts_eq12(micsa, T):
    """Eq. (12) as printed, and its inverse."""
    import math
    b = 1.0 / T
    e = 4 * math.exp(-4 * b) / (1 - math.exp(-4 * b)) - 16 * math.exp(-16 * b) / (1 - math.exp(-16 * b))
    assert abs(micsa.effective_temperature(e) - T) < 1e-9 * max(1.0, T * T)
    for bad in (0.0, 6.0, -1.0, float("nan")):
        with pytest.raises(micsa.MicsaError):
            micsa.effective_temperature(bad)


def test_pow2_schedule_is_the_papers_rule():
    from micsa_workloads import pow2_schedule
    sch = pow2_schedule(0.7, 5)
    assert [n for _, n, _ in sch] == [1, 2, 4, 8, 16, 32] and sum(n for _, n, _ in sch) == 63
    assert all(T == 0.7 and every == n for T, n, every in sch)


def test_xi_equals_oracle(micsa, oracle):
    """micsa_xi (host arithmetic of the library) against the oracle's numpy trapezoid (Eq. 17-18, reading R22)."""
    rng = np.random.default_rng(5)
    for n in (2, 5, 41, 81):
        c = np.exp(-np.arange(n) / 7.3) * (1.0 + 0.05 * rng.standard_normal(n))
        c[0] = 1.0
        for c_min in (0.0, 0.01, 0.2):
            try:
                want = oracle.xi(c, c_min)
            except ValueError:
                with pytest.raises(micsa.MicsaError):
                    micsa.xi(c, c_min)
                continue
            np.testing.assert_allclose(micsa.xi(c, c_min), want, rtol=1e-13)
    with pytest.raises(micsa.MicsaError):
        micsa.xi(np.array([1.0]), 0.0)
    with pytest.raises(micsa.MicsaError):
        micsa.xi(np.array([1.0, -0.5, 0.3]), 0.0)
