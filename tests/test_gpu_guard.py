"""Memory-safety check the library carries itself (compute-sanitizer is closed on this GPU pool).

With MHD_GUARD=1 at mhd_init every array of the context lies between guard bands of a NaN pattern and
itself starts as that pattern (include/mhd.h, mhd_debug_guard_errors).  For every kernel path and
reconstruction, on ragged and degenerate grids, with periodic and outflow boundaries:
  * no guard word is damaged after several steps          -> no write outside an array;
  * the state is finite and BIT-IDENTICAL to that of an unguarded context (zero-initialised, arrays
    back to back) -> no result depends on anything read outside an array or never written
    (the update kernels do read such operands unconditionally and discard them: that is the design).
"""
import numpy as np
import pytest

from paper_2402_05240_b200 import inputs
from helpers import FIELDS

pytestmark = pytest.mark.gpu

PATHS = {"default": {}, "three-kernel predictor": {"MHD_STAGE_TY": "0"}, "fused corrector tail": {"MHD_CT_FUSED": "1"},
         "cooperative kernel": {"MHD_SMALL": "1"}}


@pytest.fixture(scope="module")
def mhd():
    from paper_2402_05240_b200 import mhd as m
    return m


def run(mhd, p, n, bc):
    sh = inputs.field_shapes(*n)
    st = {f: np.ascontiguousarray(p.state[f][:sh[f][0], :sh[f][1], :sh[f][2]]) for f in FIELDS}
    g = mhd.Mhd(*n, p.gamma, p.recon, bc)
    g.set_state(st)
    for _ in range(2):
        g.step(0.5 * g.compute_dt(0.4))
    g.advance(3, 0.2)
    out = (g.get_state(), g.get_half_state(), g.guard_errors())
    g.close()
    return out


@pytest.mark.parametrize("path", list(PATHS))
@pytest.mark.parametrize("recon", [0, 1, 2, 3, 4])
def test_no_access_outside_the_arrays(mhd, monkeypatch, path, recon):
    for k, v in PATHS[path].items():
        monkeypatch.setenv(k, v)
    p = inputs.random_smooth(n=(70, 40, 36), seed=60 + recon, recon=recon)
    for n, bc in (((37, 21, 19), (0, 0, 0)), ((66, 9, 34), (1, 0, 1)), ((5, 3, 2), (0, 1, 0)), ((1, 1, 1), (0, 0, 0)),
                  ((16, 38, 5), (1, 1, 1))):
        monkeypatch.delenv("MHD_GUARD", raising=False)
        ref_state, ref_half, ref_err = run(mhd, p, n, bc)
        assert ref_err == -1
        monkeypatch.setenv("MHD_GUARD", "1")
        state, half, err = run(mhd, p, n, bc)
        assert err == 0, (path, recon, n, bc, err)
        for f in FIELDS:
            assert np.all(np.isfinite(state[f])), (path, recon, n, f)
            assert np.array_equal(state[f], ref_state[f]), (path, recon, n, bc, f)
            assert np.array_equal(half[f], ref_half[f]), (path, recon, n, bc, "half", f)
