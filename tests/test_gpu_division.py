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


def test_fp64_pipe_throughput_and_latency(pkg, capsys):
    """The micro-benchmark behind DESIGN.md section 5 (smaug_selftest_fp64_pipe): a dependent DFMA costs ~9 cycles, the
    fp64 pipe of an SM sub-partition takes one warp instruction per two cycles (64 lanes per SM), and three warps per
    scheduler -- what the hot kernel has -- need two independent chains each to fill it."""
    rows = {}
    for ilp in (1, 2, 4, 8):
        for warps in (1, 2, 3, 4):
            rows[(ilp, warps)] = pkg.selftest_fp64_pipe(ilp, warps)
    with capsys.disabled():
        print("\nfp64 pipe: cycles per warp instruction and sub-partition (cycles per trip)")
        for ilp in (1, 2, 4, 8):
            print(f"  ILP {ilp}: " + "  ".join(f"{w} warps {rows[(ilp, w)][0]:.2f} ({rows[(ilp, w)][1]:.1f})" for w in (1, 2, 3, 4)))
    lat = rows[(1, 1)][1]
    assert 7.0 <= lat <= 11.0, lat                               # dependent-issue latency of DFMA
    assert 1.9 <= rows[(8, 4)][0] <= 2.2, rows[(8, 4)]           # saturated: one per two cycles
    assert rows[(1, 3)][0] >= 2.7 and rows[(2, 3)][0] <= 2.4     # three warps: one chain each is not enough, two are
