"""GPU parity of the launch-bound-grid path (csrc/mhd_small.cuh): the whole of mhd_advance as ONE
cooperative kernel with grid-wide barriers between the stages of a step.  It is used by mhd_advance on
grids of at most 64^3 cells; MHD_SMALL=1 at mhd_init routes mhd_step through it as well (any size), so
that every one-step parity case can be run against it; MHD_SMALL=0 switches it off."""
import numpy as np
import pytest

import oracle as orc
from paper_2402_05240_b200 import inputs
from helpers import divb_normalised, rel_diff, FIELDS

pytestmark = pytest.mark.gpu
TOL_STEP = 1e-12


@pytest.fixture(scope="module")
def mhd():
    from paper_2402_05240_b200 import mhd as m
    return m


def close(a, b, tol, what):
    rd = rel_diff(a, b)
    assert max(rd.values()) <= tol, "%s: %s" % (what, rd)


@pytest.mark.parametrize("recon", [0, 1, 2, 3, 4])
@pytest.mark.parametrize("n", [(37, 21, 19), (16, 70, 5), (4, 4, 4), (2, 1, 3)])
def test_one_step_through_the_cooperative_kernel(mhd, monkeypatch, recon, n):
    monkeypatch.setenv("MHD_SMALL", "1")
    p = inputs.random_smooth(n=(40, 72, 20), seed=41 + recon, recon=recon)
    sh = inputs.field_shapes(*n)
    st = {f: np.ascontiguousarray(p.state[f][:sh[f][0], :sh[f][1], :sh[f][2]]) for f in FIELDS}
    st["bx"][:, :, -1] = st["bx"][:, :, 0]; st["by"][:, -1, :] = st["by"][:, 0, :]; st["bz"][-1, :, :] = st["bz"][0, :, :]
    o = orc.Oracle(*n, p.gamma, recon)
    o.set_state(st)
    g = mhd.Mhd(*n, p.gamma, recon)
    g.set_state(st)
    dt = o.compute_dt(0.4)
    assert abs(g.compute_dt(0.4) - dt) <= 1e-13 * dt
    n0 = g.launch_count()
    o.step(dt); g.step(dt)
    assert g.launch_count() - n0 == 1                      # one launch: it IS the cooperative kernel
    close(g.get_half_state(), o.get_half_state(), TOL_STEP, "half state")
    out = g.get_state()
    close(out, o.get_state(), TOL_STEP, "full state")
    dt2 = o.compute_dt(0.4)
    assert abs(g.compute_dt(0.4) - dt2) <= 1e-13 * dt2     # the rate of U^{n+1} reduced inside the kernel
    o.close(); g.close()


def test_brio_wu_outflow_steps_through_the_cooperative_kernel(mhd, monkeypatch):
    monkeypatch.setenv("MHD_SMALL", "1")
    p = inputs.riemann("brio_wu", 64, 4, axis=0, recon=1)
    o = orc.Oracle(*p.n, p.gamma, p.recon, p.bc)
    o.set_state(p.state)
    g = mhd.Mhd(*p.n, p.gamma, p.recon, p.bc)
    state = p.state
    for s in range(10):
        g.set_state(state)
        dt = o.compute_dt(p.cfl)
        o.step(dt); g.step(dt)
        state = o.get_state()
        close(g.get_state(), state, TOL_STEP, "brio-wu step %d" % (s + 1))
    o.close(); g.close()


@pytest.mark.parametrize("recon,nsteps", [(1, 9), (2, 6)])
def test_advance_on_a_launch_bound_grid(mhd, monkeypatch, recon, nsteps):
    """mhd_advance on 32^3 (config c1's size) takes the cooperative kernel by itself: n steps in one
    launch, dt formed on the device every step.  Against the kernel-by-kernel path (MHD_SMALL=0) and
    against the oracle."""
    p = inputs.random_smooth(n=(32, 32, 32), seed=8, recon=recon)
    out = {}
    for mode in ("0", "auto"):
        if mode == "0":
            monkeypatch.setenv("MHD_SMALL", "0")
        else:
            monkeypatch.delenv("MHD_SMALL", raising=False)
        g = mhd.Mhd(*p.n, p.gamma, p.recon)
        g.set_state(p.state)
        n0 = g.launch_count()
        t = g.advance(nsteps, 0.4, want_time=True)
        nl = g.launch_count() - n0
        out[mode] = (g.get_state(), t, nl)
        g.close()
    assert out["auto"][2] <= 3 and out["0"][2] >= 7 * nsteps     # (+ the first CFL reduction's two launches)
    assert abs(out["auto"][1] - out["0"][1]) <= 1e-13 * out["0"][1]
    close(out["auto"][0], out["0"][0], 1e-13 * nsteps, "cooperative vs kernel-by-kernel")
    o = orc.Oracle(*p.n, p.gamma, p.recon)
    o.set_state(p.state)
    tsum = 0.0
    for _ in range(nsteps):
        dt = o.compute_dt(0.4)
        o.step(dt); tsum += dt
    assert abs(out["auto"][1] - tsum) <= 1e-12 * tsum
    close(out["auto"][0], o.get_state(), 10 * nsteps * TOL_STEP, "cooperative advance vs oracle")
    o.close()
