"""The last word on child tests that timed out.  conftest.isolated() runs a few GPU tests in a child process and
kills a child whose launch never completes; so that `-x` does not stop there and hide every later test, that test is
reported as xfail -- and its node id is recorded.  This test, collected after every test that uses isolated() (and
before tests/test_zz_no_alloc.py, which must stay last), turns any such record into a failure of the run: a hang can
be skipped over, it cannot pass."""
import pytest

from conftest import TIMEOUT_LOG, timed_out_children

pytestmark = pytest.mark.gpu


def test_no_child_test_timed_out():
    hung = timed_out_children()
    assert not hung, f"child tests that never finished (launch hung), from {TIMEOUT_LOG}: {hung}"
