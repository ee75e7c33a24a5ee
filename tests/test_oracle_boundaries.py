"""Pins of the oracle's exact-boundary behaviour through the whole path (raw banks -> decode -> Compass): the
hand-built cases of tests/adversarial_cases.py place a residual exactly ON a cut and one ulp either side; the oracle
must accept / reject as SURVEY.md 8(c) steps 2-7 say (<= is inside).  tests/test_gpu_adversarial.py runs the same
cases through the CUDA path."""
import pytest

import adversarial_cases as AC
import oracle


def run(geom, b, p):
    return oracle.run_batch(b, geom, p)


@pytest.mark.parametrize("layer", [0, 1, 2, 3])
def test_window_edge_exact(geom, layer):
    AC.case_window_edge_exact(run, geom, layer)


@pytest.mark.parametrize("layer", [0, 1, 2, 3])
def test_y_edge_exact(geom, layer):
    AC.case_y_edge_exact(run, geom, layer)


def test_seed_cut_edges(geom):
    AC.case_seed_cut_edges(run, geom)


def test_chi2_cut_edge(geom):
    AC.case_chi2_cut_edge(run, geom)


def test_abs_d_ties_at_the_cap(geom):
    AC.case_abs_d_ties_at_the_cap(run, geom)


def test_exact_chi2_ties_across_lanes(geom):
    AC.case_exact_chi2_ties_across_lanes(run, geom)
