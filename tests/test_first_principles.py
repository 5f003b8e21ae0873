"""P1: the oracle against a second-quantised evaluation that uses no index formula."""
import numpy as np
import pytest

from bqc_inputs import make_inputs, worked_example
from oracle import t_oracle as orc
from fock_space import first_principles_t


@pytest.mark.parametrize("case", ["worked234", "rand225", "rand322"])
def test_oracle_matches_first_principles(case):
    if case == "worked234":
        inp = worked_example(2, 3, 4)
    elif case == "rand225":
        inp = make_inputs(2, 2, 5, seed=7, t1_std=0.05, t2_std=0.05)
    else:
        inp = make_inputs(3, 2, 4, seed=11, t1_std=0.05, t2_std=0.05)
    e4_fp, e5_fp = first_principles_t(inp)
    e4 = orc.t_energy(inp, with_t1=False)
    et = orc.t_energy(inp, with_t1=True)
    assert abs(e4_fp) > 0
    assert e4 == pytest.approx(e4_fp, rel=1e-11, abs=1e-18)
    assert (et - e4) == pytest.approx(e5_fp, rel=1e-10, abs=1e-18)


def test_first_principles_reproduces_survey_value():
    # SURVEY.md §8(c) P2, (2,3,4): E[4], E[5] — ties the in-repo P1 to the stored fixture
    e4, e5 = first_principles_t(worked_example(2, 3, 4))
    assert e4 == pytest.approx(-1.986490875488184e-06, rel=1e-11)
    assert e5 == pytest.approx(+1.045821059563959e-06, rel=1e-11)
