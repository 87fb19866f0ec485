"""The branch-free fp64 division helpers of csrc/smaug_device.cuh against the compiler's IEEE-754 `/`, on the GPU,
through the C ABI (smaug_selftest_division).  Bit-identity of every stage kernel with the oracle rests on them
("Division"): 0 mismatches are required on every range the kernels feed them, and the guarded
form (`kappa_ratio`: zero guard + 2^200 rescue) must be exact on tiny and denormal M1 as well -- that is the form every
hyperviscosity ratio goes through (the unguarded fast path is taken only after a warp vote that every M1 >= 2^-923).
The last test shows the check has teeth: raw `ddiv` IS wrong below ~2^-960, which is why callers never reach there."""
import pytest

pytestmark = pytest.mark.gpu
DRAWS = 1 << 27          # per range and helper (1184 x 256 threads x 442 draws)


@pytest.fixture(scope="module")
def pkg():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the gpu-marked tests need a B200")
    import paper_1710_06423_b200 as p
    p.lib()
    return p


@pytest.mark.parametrize("lo,hi", [(-5, 5), (-40, 40), (-300, 300), (-700, -600), (-900, -700), (600, 900)])
def test_division_helpers_exact_on_ordinary_numbers(pkg, lo, hi):
    r = pkg.selftest_division(lo, hi, seed=1710 + lo, draws=DRAWS)
    assert r["draws"] >= DRAWS // 2
    assert (r["ddiv"], r["drcp"], r["ratio_div"], r["kappa_ratio"]) == (0, 0, 0, 0), r


@pytest.mark.parametrize("lo,hi", [(-923, -880), (-990, -920), (-1022, -960), (-1074, -1000)])
def test_guarded_ratio_exact_on_tiny_and_denormal_m1(pkg, lo, hi):
    """ratio_div / kappa_ratio rescale both operands by 2^200 when M1 < 2^-923 (exact), so the quotient of the
    hyperviscosity ratio is correctly rounded down to denormal M1; M1 = 0 gives 0."""
    r = pkg.selftest_division(lo, hi, seed=7 - lo, draws=DRAWS)
    assert (r["ratio_div"], r["kappa_ratio"]) == (0, 0), r


def test_unguarded_division_is_wrong_below_2_to_minus_960(pkg):
    """The reason for the guard: the remainder of the unguarded fast path underflows for tiny operands."""
    r = pkg.selftest_division(-1020, -900, seed=3, draws=DRAWS)
    assert r["ddiv"] > 0, r
    assert (r["ratio_div"], r["kappa_ratio"]) == (0, 0), r
