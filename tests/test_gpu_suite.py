"""GPU parity on the rest of the paper's test suite: the kernels against the
oracle on the circularly polarised Alfven wave, the advecting field loop, the Riemann problems of
Table 2, the blast in the paper's box and the Orszag-Tang vortex, including the
non-cubic boxes (mhd_set_domain).  Smooth problems: free-running to the end time at 1e-9; problems
with discontinuities: every step a one-step case from the oracle's state at 1e-12."""
import numpy as np
import pytest

import oracle as orc
from paper_2402_05240_b200 import inputs
from helpers import run_to_time, divb_normalised, rel_diff, FIELDS, totals

pytestmark = pytest.mark.gpu

TOL_STEP, TOL_RUN, TOL_DIVB = 1e-12, 1e-9, 1e-12


@pytest.fixture(scope="module")
def mhd():
    from paper_2402_05240_b200 import mhd as m
    return m


def pair(mhd, p):
    o = orc.Oracle(*p.n, p.gamma, p.recon, p.bc, p.domain)
    o.set_state(p.state)
    g = mhd.Mhd(*p.n, p.gamma, p.recon, p.bc, domain=p.domain)
    g.set_state(p.state)
    return o, g


def stepwise(mhd, p, n_steps, what, alfven_units=False, switch_steps=0, switch_cells=0):
    """n_steps one-step parity cases, each from the oracle's own state.  alfven_units: the field is a
    passive tracer (|B| << sqrt(rho)|v|, field loop): the round-off of the O(1) velocities enters the
    induction equation at 1e-16 ABSOLUTE, so B is compared in units of max(|B|, |m|/sqrt(rho)).
    switch_steps / switch_cells: at most that many steps may miss the tolerance, each in at most that
    many cells per field (a discontinuous limiter switch taken on the other side, R11);
    every other step and every other cell is held to TOL_STEP."""
    o, g = pair(mhd, p)
    state = p.state
    worst = 0.0
    off_steps = []
    for s in range(n_steps):
        g.set_state(state)
        dt = o.compute_dt(p.cfl)
        assert abs(g.compute_dt(p.cfl) - dt) <= 1e-13 * dt
        o.step(dt); g.step(dt)
        state = o.get_state()
        out = g.get_state()
        rd = rel_diff(out, state)
        if alfven_units:
            vs = max(np.abs(state[m]).max() for m in ("mx", "my", "mz")) / np.sqrt(state["rho"].max())
            for f in ("bx", "by", "bz"):
                rd[f] = np.abs(out[f] - state[f]).max() / max(np.abs(state[f]).max(), vs)
        assert divb_normalised(out, p.n, p.domain) <= TOL_DIVB
        if max(rd.values()) > TOL_STEP and switch_steps:
            cells = max(int((np.abs(out[f] - state[f]) > TOL_STEP * max(np.abs(state[f]).max(), 1e-300)).sum())
                        for f in FIELDS)
            assert cells <= switch_cells, "%s step %d: %d cells off, %s" % (what, s + 1, cells, rd)
            off_steps.append(s + 1)
            assert len(off_steps) <= switch_steps, "%s: steps off %s" % (what, off_steps)
            continue
        assert max(rd.values()) <= TOL_STEP, "%s step %d: %s" % (what, s + 1, rd)
        worst = max(worst, max(rd.values()))
    o.close(); g.close()
    return worst


@pytest.mark.parametrize("recon", [1, 2])
def test_cpaw_full_period(mhd, recon):
    """PAPER.md:358-370 at 32 x 16 x 16 in the 3 x 1.5 x 1.5 box: one period, free-running, and the
    GPU's own error against the exact solution equals the oracle's."""
    p = inputs.cpaw(16, recon=recon)
    o, g = pair(mhd, p)
    n_o = run_to_time(o, p)
    n_g = run_to_time(g, p)
    assert n_o == n_g
    out, ref = g.get_state(), o.get_state()
    rd = rel_diff(out, ref)
    assert max(rd.values()) <= TOL_RUN, rd
    assert divb_normalised(out, p.n, p.domain) <= TOL_DIVB
    e_g, e_o = inputs.wave_error(p.state, out), inputs.wave_error(p.state, ref)
    assert e_g == pytest.approx(e_o, rel=1e-6) and e_g < 0.03
    o.close(); g.close()


def test_field_loop_quarter_period(mhd):
    """PAPER.md:378-391 at 16 x 16 x 32 in the 1 x 1 x 2 box: stepwise parity over the first 20 steps
    (PLMC: on a uniform background perturbed at 1e-6 the PPM flush of R7 switches at the 1e-12 level,
    DESIGN.md R10), then PPMC free-running to t = 0.25: div B at round-off, field energy only decays."""
    stepwise(mhd, inputs.field_loop(16, recon=1), 20, "field loop", alfven_units=True)
    p = inputs.field_loop(16, recon=2)
    p.t_end = 0.25
    g = mhd.Mhd(*p.n, p.gamma, p.recon, p.bc, domain=p.domain)
    g.set_state(p.state)
    run_to_time(g, p)
    out = g.get_state()
    assert divb_normalised(out, p.n, p.domain) <= TOL_DIVB
    b0, b1 = inputs.cell_centred_b(p.state), inputs.cell_centred_b(out)
    e0, e1 = sum(x ** 2 for x in b0).mean(), sum(x ** 2 for x in b1).mean()
    assert 0.6 < e1 / e0 < 1.0
    t0, t1 = totals(p.state), totals(out)
    for f in ("rho", "E", "mx", "my", "mz"):
        assert abs(t1[f] - t0[f]) <= 1e-12 * abs(t0[f])
    g.close()


@pytest.mark.parametrize("name,axis,flip", [("dai_woodward", 0, False), ("ryu_jones_1a", 1, False),
                                            ("ryu_jones_4d", 2, True), ("einfeldt", 0, False)])
@pytest.mark.parametrize("recon", [1, 2])
def test_riemann_problems_of_table_2(mhd, name, axis, flip, recon):
    """96 x 4 x 4 along x, y or z (one of them flipped), outflow along the tube:
    30 one-step parity cases, then a free run to t_max that must stay positive and planar."""
    p = inputs.riemann(name, n_long=96, n_trans=4, axis=axis, recon=recon, flip=flip)
    hot = (name == "ryu_jones_1a" and recon == 2)
    stepwise(mhd, p, 4 if hot else 30, "%s recon %d" % (name, recon))
    g = mhd.Mhd(*p.n, p.gamma, p.recon, p.bc)
    g.set_state(p.state)
    if hot:
        # Kinetic energy is 50x the thermal one here and the scheme has no floors (G18): at 96 cells
        # (the paper uses 512) PPMC drives the pressure of the collision cell negative from the fifth
        # step on -- in the oracle too (min P = -0.79, then -2.1).  Four steps are compared; after
        # that the library must say so instead of returning garbage.
        with pytest.raises(mhd.MhdError, match="non-physical"):
            run_to_time(g, p)
        g.close()
        return
    run_to_time(g, p)
    out = g.get_state()
    assert out["rho"].min() > 0 and np.all(np.isfinite(out["E"]))
    rho = np.moveaxis(out["rho"], 2 - axis, 0)          # tube axis first
    assert np.all(rho == rho[:, :1, :1])               # every transverse column identical
    g.close()


@pytest.mark.parametrize("recon", [1, 2])
def test_blast_in_the_papers_box(mhd, recon):
    """PAPER.md:455-465 at 24 x 36 x 24 in the 1 x 1.5 x 1 box: 10 one-step parity cases; free run of
    the PLMC case keeps the z-mirror and point symmetries at round-off (R11 for PPMC)."""
    p = inputs.blast_paper(24, recon=recon)
    # PPMC: the mirror-symmetric flat tops of this problem sit on the PPM extremum switch (R11),
    # where a difference in the last bit of an amplitude selects another parabola: seen in one of the ten
    # steps (the fourth: 66 of 20,736 cells per field, up to 3e-5).  At most one such step and at most
    # 132 such cells are let through; the other nine steps agree to 1e-13.
    if recon == 1:
        stepwise(mhd, p, 10, "paper blast recon 1")
    else:
        stepwise(mhd, p, 10, "paper blast recon 2", switch_steps=1, switch_cells=132)
    g = mhd.Mhd(*p.n, p.gamma, p.recon, p.bc, domain=p.domain)
    g.set_state(p.state)
    for _ in range(12):
        g.step(g.compute_dt(p.cfl))
    rho = g.get_state()["rho"]
    assert rho.min() > 0
    if recon == 1:
        assert np.abs(rho - rho[::-1]).max() < 1e-13 and np.abs(rho - rho[::-1, ::-1, ::-1]).max() < 1e-13
    g.close()


def test_orszag_tang(mhd):
    """PAPER.md:475 at 48 x 48 x 6, PPMC: 15 one-step parity cases; free run to t = 0.2 keeps every
    z-plane bit-identical, B_z = m_z = 0 exactly, conserves mass and energy, div B at round-off."""
    p = inputs.orszag_tang(48, nz=6, recon=2)
    stepwise(mhd, p, 15, "Orszag-Tang")
    p.t_end = 0.2
    g = mhd.Mhd(*p.n, p.gamma, p.recon, p.bc)
    g.set_state(p.state)
    run_to_time(g, p)
    out = g.get_state()
    for f in FIELDS[:5] + ("bx", "by"):
        assert np.all(out[f] == out[f][:1]), f
    # (the oracle keeps B_z = m_z = 0 exactly; the kernels' closed-form R.(L.W) leaves round-off)
    assert np.abs(out["bz"]).max() <= 1e-14 and np.abs(out["mz"]).max() <= 1e-14
    assert divb_normalised(out, p.n, p.domain) <= TOL_DIVB
    t0, t1 = totals(p.state), totals(out)
    assert abs(t1["rho"] - t0["rho"]) <= 1e-13 * t0["rho"] and abs(t1["E"] - t0["E"]) <= 1e-13 * t0["E"]
    g.close()
