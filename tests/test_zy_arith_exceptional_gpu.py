"""The one exceptional case of the branch-free IEEE division: divisors whose mantissa is all ones, where the
last Newton correction lands on the correctly rounded quotient only for a good enough reciprocal seed
(tests/test_device_math_on_host.py shows it with perturbed seeds).  This checks it with the hardware's actual seed.  In a file
of its own that is collected after the parity tests: it probes a property of the hardware, not of the kernels' logic."""
import pytest

pytestmark = pytest.mark.gpu


def test_division_by_all_ones_mantissa_divisors_is_correctly_rounded_on_this_gpu():
    import paper_1204_6192_b200 as hsg
    assert hsg.hsg_selftest_arith(50_000_000, seed=777, exceptional=True) == 0
