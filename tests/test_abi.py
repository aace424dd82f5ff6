"""The C-ABI library loads here (no GPU) and exports every symbol include/potts.h declares; the host-side entry
points that need no device (argument checks, workspace sizes, derived observables) behave as documented."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def pb():
    import paper_1101_0876_b200 as pb
    from paper_1101_0876_b200 import build
    build.build()                      # nvcc cross-compiles for sm_100a without a GPU
    pb.load_library()
    return pb


def _declared():
    text = open(os.path.join(ROOT, "include", "potts.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(potts[38]?_[a-z_0-9]+)\s*\(", text)))


def test_every_declared_symbol_is_exported(pb):
    names = _declared()
    assert len(names) >= 20
    lib = ctypes.CDLL(pb.LIB_PATH)
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/potts.h but not exported"
    assert sorted(pb.EXPORTED_SYMBOLS) == names         # the binding wraps exactly the declared set
    assert "sm_100a" in pb.potts_version()


def test_no_fallback_in_product(pb):
    # the product never imports the oracle, and the library has no CPU path to fall back to
    for fn in os.listdir(os.path.join(ROOT, "paper_1101_0876_b200")):
        if fn.endswith(".py"):
            assert "oracle" not in open(os.path.join(ROOT, "paper_1101_0876_b200", fn)).read().replace("the oracle", "")


def test_workspace_bytes_and_shape_errors(pb):
    u8 = pb.potts_workspace_bytes(1024, 6)
    assert u8 >= 1024 * 1024
    assert pb.potts_workspace_bytes(8192, 24, pb.LAYOUT_PACKED) < pb.potts_workspace_bytes(8192, 24, pb.LAYOUT_U8)
    assert pb.potts_workspace_bytes(8192, 9, pb.LAYOUT_PACKED) < pb.potts_workspace_bytes(8192, 24, pb.LAYOUT_PACKED)
    for L, q, layout, code in ((63, 9, 0, pb.ERR_ARG), (64, 1, 0, pb.ERR_ARG), (64, 257, 0, pb.ERR_ARG),
                               (48, 9, 0, pb.ERR_UNSUPPORTED), (64, 9, 7, pb.ERR_ARG),
                               (64, 33, pb.LAYOUT_PACKED, pb.ERR_UNSUPPORTED), (96, 9, pb.LAYOUT_PACKED, pb.ERR_UNSUPPORTED)):
        with pytest.raises(pb.PottsError) as e:
            pb.potts_workspace_bytes(L, q, layout)
        assert e.value.code == code, (L, q, layout)


def test_host_observables_against_exact_arithmetic(pb):
    from fractions import Fraction
    rng = np.random.default_rng(5)
    N, T = 32768 * 32768, 0.7177
    E = (-1_650_000_000 + rng.integers(-40_000, 40_000, size=200)).astype(np.int64)   # 1e9-fold cancellation in the variance
    me, cv, bl = pb.potts_observables(E, N, T)
    n = len(E)
    s1 = sum(int(x) for x in E); s2 = sum(int(x) ** 2 for x in E); s4 = sum(int(x) ** 4 for x in E)
    want_me = Fraction(s1, n * N)
    want_cv = Fraction(n * s2 - s1 * s1, n * n) / (Fraction(N) * Fraction(T) ** 2)
    want_bl = 1 - Fraction(s4, n) / (3 * Fraction(s2, n) ** 2)
    for got, want in ((me, want_me), (cv, want_cv), (bl, want_bl)):
        assert abs(Fraction(got) - want) <= Fraction(1, 10 ** 12) * abs(want)
    assert pb.potts_magnetisation(np.array([10, 70, 20], dtype=np.int64), 3) == pytest.approx((3 * 0.7 - 1) / 2, rel=1e-15)
    with pytest.raises(pb.PottsError):
        pb.potts_observables(np.zeros(0, dtype=np.int64), 16, 1.0)


def test_host_susceptibility_against_exact_arithmetic(pb):
    """potts_susceptibility (Eq. 11) against exact rationals formed here, and closed cases."""
    from fractions import Fraction
    rng = np.random.default_rng(11)
    q, N, T, n = 9, 32768 * 32768, 0.7177, 300
    H = np.zeros((n, q), dtype=np.int64)
    for k in range(n):                                   # near-ordered histograms: m ~ 0.9 with tiny fluctuations
        minor = rng.integers(10_000_000, 10_100_000, size=q - 1)
        H[k, 1:] = minor
        H[k, 0] = N - minor.sum()
    m1, m2, chi = pb.potts_susceptibility(H, q, T)
    ms = [(Fraction(q * int(H[k].max()), N) - 1) / (q - 1) for k in range(n)]
    w1 = sum(ms) / n
    w2 = sum(m * m for m in ms) / n
    wchi = N * (w2 - w1 * w1) / Fraction(T)
    for got, want in ((m1, w1), (m2, w2), (chi, wchi)):
        assert abs(Fraction(got) - want) <= Fraction(1, 10 ** 12) * abs(want)
    # closed cases: ordered -> m = 1, chi = 0; {ordered, uniform} -> <m> = <m^2> = 1/2, chi = N/(4T)
    assert pb.potts_susceptibility([[400, 0, 0, 0]] * 3, 4, 0.7) == (1.0, 1.0, 0.0)
    assert pb.potts_susceptibility([[400, 0, 0, 0], [100, 100, 100, 100]], 4, 2.0) == (0.5, 0.5, 400 / 2.0 * 0.25)
    for bad in ([[1, 2], [2, 2]], [[0, 0]], [[-1, 5]]):
        with pytest.raises(pb.PottsError):
            pb.potts_susceptibility(bad, 2, 1.0)


def test_product_fails_loudly_without_a_gpu(pb):
    """No CPU fallback: on a box without a CUDA device every constructor refuses (on a GPU box this test is moot)."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(pb.PottsError) as e:
        pb.Potts(64, 4, 1)
    assert e.value.code == pb.ERR_CUDA
    with pytest.raises(pb.PottsError):
        pb.PottsBatch(64, 4, [1, 2])
    lib = pb.load_library()
    h = ctypes.c_void_p()
    rc = lib.potts_create(ctypes.byref(h), 64, 4, 1, 0)            # the C entry point itself, no Python in between
    assert rc == pb.ERR_CUDA and not h.value
    assert b"CUDA" in lib.potts_last_error() or b"device" in lib.potts_last_error()
