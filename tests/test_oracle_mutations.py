"""Opt-in (SW_RUN_MUTATIONS=1, a few minutes of CPU): every single-line mutation of the oracle listed in
tests/oracle_mutations.py must be caught by the oracle's pin tests."""
import os

import pytest

import oracle_mutations


def test_mutation_patterns_still_match_the_source():
    text = open(oracle_mutations.SRC).read()
    for name, find, _ in oracle_mutations.MUTATIONS:
        assert text.count(find) == 1, name


@pytest.mark.skipif(os.environ.get("SW_RUN_MUTATIONS") != "1", reason="runs the oracle test files once per mutation; set SW_RUN_MUTATIONS=1")
def test_every_mutation_is_caught():
    assert oracle_mutations.main() == 0
