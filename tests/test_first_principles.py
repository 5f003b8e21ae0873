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


@pytest.mark.parametrize("shape,seed", [((2, 2, 5), 7), ((3, 2, 4), 11), ((2, 3, 4), 5)])
def test_fock_term_matches_first_principles(shape, seed):
    """SURVEY.md §8(f) NEXT-3 / PAPER.md:298-303 Eqs. (5),(7): with an occupied-virtual Fock block the
    oracle's extra V terms must reproduce <0|T2+ F_ov R3 W_N T2|0>, evaluated without any index formula."""
    import copy
    inp = make_inputs(*shape, seed=seed, t1_std=0.05, t2_std=0.05, f_std=0.1)
    e4_fp, e5_fp, ef_fp = first_principles_t(inp, with_fock=True)
    canon = copy.copy(inp)
    canon.f_ov = None
    e_canon = orc.t_energy(canon)
    e_fock = orc.t_energy(inp)
    assert abs(ef_fp) > 1e-7
    assert e_canon == pytest.approx(e4_fp + e5_fp, rel=1e-11)
    assert (e_fock - e_canon) == pytest.approx(ef_fp, rel=1e-10, abs=1e-18)
