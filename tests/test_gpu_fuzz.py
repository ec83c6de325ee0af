"""Bounded, fixed-seed runs of the two fuzz campaign drivers (tests/fuzz_attention.py, tests/fuzz_random_ops.py), so that
every GPU test run covers a slice of what the campaigns in profiles/r02_sanitizer.md covered at length."""
import pytest

pytestmark = pytest.mark.gpu


def test_attention_fuzz_bounded():
    import fuzz_attention
    assert fuzz_attention.main(20261, 120) == 0


def test_random_operation_fuzz_bounded():
    import fuzz_random_ops
    assert fuzz_random_ops.main(20262, 12) == 0
