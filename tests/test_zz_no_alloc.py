"""nanobte_get_boundary_heat_noalloc (csrc/noalloc.cu): the per-tag boundary heat through the library's static device
scratch, against the existing path nanobte_get_boundary_heat (`-m gpu`).  Collected last on purpose (the file name): the
suite runs with pytest -x.  The two paths add the same face terms in different orders, so they agree to rounding of the
sums: 1e-12 of the largest per-tag heat, three orders inside the 1e-9 the parity tests allow this quantity.
"""
import copy

import numpy as np
import pytest

from paper_2607_03226_b200 import workloads as wl

pytestmark = pytest.mark.gpu

TOL = 1e-12
MAX_TAGS = 256  # NANOBTE_NOALLOC_MAX_TAGS


def close(a, b):
    return np.abs(a - b).max() <= TOL * max(np.abs(b).max(), 1e-300)


def test_two_calls_in_a_row_match_the_existing_path():
    from paper_2607_03226_b200.binding import Solver
    pr = wl.config_finfet(nx=32, ny=16, nz=16, B=3, n_polar=2, n_azim=8)
    g = Solver(pr)
    seen = []
    for step in range(2):  # two different states, the second call finds the first call's contents in the scratch
        g.sweep()
        g.update_temperature()
        want = g.get_boundary_heat()
        assert np.abs(want).max() > 0
        got_host = g.get_boundary_heat_noalloc()
        got_dev = g.get_boundary_heat_noalloc(device=True).cpu().numpy()
        assert close(got_host, want), (step, got_host, want)
        assert np.array_equal(got_dev, got_host)  # fixed summation order: bitwise the same, whatever the destination
        assert np.array_equal(g.get_boundary_heat(), want)  # the existing path is untouched by the new one
        seen.append(got_host)
    assert not np.array_equal(seen[0], seen[1])
    g.close()


def test_solvers_share_the_scratch_one_after_the_other():
    """A second solver with another tag count (2-D, unstructured) uses the same static array right after the first."""
    from paper_2607_03226_b200.binding import Solver
    a = Solver(wl.config_cube(n=20, B=3, n_polar=2, n_azim=8, mode="synthetic"))
    b = Solver(wl.config_triangles(n=24, side=1e-7, B=3, D=8, hole_radius=1.5e-8))
    for g in (a, b):
        g.sweep()
        g.update_temperature()
    for _ in range(2):
        for g in (a, b):
            assert close(g.get_boundary_heat_noalloc(), g.get_boundary_heat())
    a.close()
    b.close()


def test_more_tags_than_the_scratch_holds_is_refused():
    from paper_2607_03226_b200.binding import Solver
    pr = copy.deepcopy(wl.config_nongray_square(n=24, B=3, D=8))
    tags = list(pr["mesh"]["tags"])
    pr["mesh"]["tags"] = tags + [tags[-1]] * (MAX_TAGS + 1 - len(tags))  # unused entries: no face carries them
    g = Solver(pr)
    g.sweep()
    g.update_temperature()
    want = g.get_boundary_heat()
    assert want.shape == (MAX_TAGS + 1,) and not want[len(tags):].any()
    with pytest.raises(Exception, match="static scratch holds at most 256"):
        g.get_boundary_heat_noalloc()
    g.close()
    pr["mesh"]["tags"] = pr["mesh"]["tags"][:MAX_TAGS]  # exactly the maximum is accepted
    g = Solver(pr)
    g.sweep()
    g.update_temperature()
    assert close(g.get_boundary_heat_noalloc(), g.get_boundary_heat())
    g.close()
