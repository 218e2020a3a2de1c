"""The branch-free reciprocal and square root of the CUDA path (csrc/marut_common.cuh) against IEEE division and square
root (numpy on the host: correctly rounded) over the operand ranges the kernels feed them (densities, pressures,
squared sound speeds) and over the whole normal range: rcp_pos / sqrt_pos bit for bit, rcp_pos_2ulp / sqrt_pos_2ulp
(the line kernel's, without the final correction step) within 2 ulp."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _eval(x, variant=0):
    import torch

    from paper_2605_26388_b200 import binding as mb

    xd = torch.from_numpy(x).cuda()
    r, s = torch.empty_like(xd), torch.empty_like(xd)
    mb.marut_debug_rcp_sqrt(xd, r, s, variant)
    torch.cuda.synchronize()
    return r.cpu().numpy(), s.cpu().numpy()


def _check(x):
    r, s = _eval(x)
    assert np.array_equal(r.view(np.uint64), (1.0 / x).view(np.uint64))
    assert np.array_equal(s.view(np.uint64), np.sqrt(x).view(np.uint64))


def test_rcp_sqrt_bit_exact_physical_ranges():
    rng = np.random.default_rng(20260526)
    n = 4_000_000
    _check(rng.uniform(0.1, 10.0, n))                     # densities
    _check(rng.uniform(1e-3, 1e6, n))                     # pressures, a^2 (SI and non-dimensional)
    _check(np.exp(rng.uniform(np.log(1e-12), np.log(1e12), n)))


def test_rcp_sqrt_bit_exact_whole_normal_range_and_edges():
    rng = np.random.default_rng(7)
    n = 4_000_000
    # random mantissas with exponents over (almost) the whole normal range: 1/x must stay normal as well
    expo = rng.integers(-1000, 1000, n)
    _check(np.ldexp(rng.uniform(1.0, 2.0, n), expo))
    # mantissa edge cases: powers of two, values next to them and next to perfect squares
    base = np.array([1.0, 2.0, 4.0, 0.5, 3.0, 9.0, 16.0, 1e10, 1e-10])
    _check(np.ascontiguousarray(np.concatenate([base, np.nextafter(base, np.inf)])))
    # the one operand class where the Newton sequence without the slow path is only faithfully rounded: an all-ones
    # mantissa, x = 2^k (1 - 2^-53), whose reciprocal lies 2^-106 above a rounding midpoint: one ulp low, never more
    below = np.ascontiguousarray(np.nextafter(base, 0.0))
    r, s = _eval(below)
    ulp = np.abs(r.view(np.int64) - (1.0 / below).view(np.int64))
    assert ulp.max() <= 1
    assert np.array_equal(s.view(np.uint64), np.sqrt(below).view(np.uint64))


def test_the_line_kernels_variants_stay_within_two_ulp():
    rng = np.random.default_rng(99)
    n = 4_000_000
    base = np.array([1.0, 2.0, 4.0, 0.5, 3.0, 9.0, 16.0, 1e10, 1e-10])
    edges = np.concatenate([base, np.nextafter(base, np.inf), np.nextafter(base, 0.0)])
    for x in (rng.uniform(0.1, 10.0, n), rng.uniform(1e-3, 1e6, n), np.ldexp(rng.uniform(1.0, 2.0, n), rng.integers(-1000, 1000, n)),
              np.ascontiguousarray(edges)):
        r, s = _eval(x, variant=1)
        assert np.abs(r.view(np.int64) - (1.0 / x).view(np.int64)).max() <= 2
        assert np.abs(s.view(np.int64) - np.sqrt(x).view(np.int64)).max() <= 2
