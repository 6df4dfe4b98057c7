"""Pins for the two round-off guards the oracle carries (readings R6 and R7).

Both were added after the first kernel existed (commit 50b58a2), so they need pins of their own:
  * R6 (Eq. 16 "otherwise" branch): between mirror-image states the contact is
    at rest analytically; HLLD then returns a mass flux of exactly zero, so that the CT upwinding
    takes the "otherwise" (average) branch instead of the sign of a 1e-16 residue.
  * R7 (extremum test of the PPM limiter, O10 step 3): differences that are zero to round-off
    count as zero.
What fixes them: (i) the mirror symmetry PAPER.md:465 asserts for the blast ("symmetric
contours") -- with the guards the oracle keeps it to round-off, without them it does not;
(ii) they touch round-off ties only: every pin that does not sit on such a tie (linear-wave
errors T8, HLLD identities T2-T5, the Sod run T14, a generic random field) gives the same numbers
with the guards switched off.
"""
import numpy as np
import pytest

import oracle as orc
from paper_2402_05240_b200 import inputs
from helpers import run_to_time, FIELDS

G = 5.0 / 3.0


@pytest.fixture
def guards():
    yield orc.set_guards
    orc.set_guards(True, True)


def mirror_pair(rng):
    rho, P = rng.uniform(0.2, 3.0), rng.uniform(0.1, 3.0)
    u, v, w = rng.normal(size=3)
    by, bz = rng.normal(size=2)
    # mirror image across the face: normal velocity flips, tangential components and the field
    # (an axial vector with the normal component continuous) are as M&K's symmetry T3 maps them
    WL = np.array([rho, u, v, w, P, by, bz])
    WR = np.array([rho, -u, v, w, P, by, bz])
    return WL, WR


def test_R6_mass_flux_between_mirror_states_is_exactly_zero(guards):
    rng = np.random.default_rng(5)
    seen_residue = 0
    for _ in range(400):
        WL, WR = mirror_pair(rng)
        bx = 0.0   # with B_n = 0 the two states are exact mirror images (B_n would flip otherwise)
        F = orc.hlld(G, WL, WR, bx)
        assert F[0] == 0.0
        guards(False, True)
        Fraw = orc.hlld(G, WL, WR, bx)
        guards(True, True)
        cf = max(orc.fast_speed(G, WL[0], WL[4], bx, WL[5], WL[6]), orc.fast_speed(G, WR[0], WR[4], bx, WR[5], WR[6]))
        assert abs(Fraw[0]) <= 1e-14 * 2 * WL[0] * cf          # the residue is round-off ...
        seen_residue += Fraw[0] != 0.0
        np.testing.assert_array_equal(F[1:], Fraw[1:])         # ... and nothing else is touched
    assert seen_residue > 20                                   # ... of either sign: noise, not physics


def test_R6_leaves_generic_fluxes_alone(guards):
    rng = np.random.default_rng(6)
    for _ in range(500):
        WL = np.array([rng.uniform(0.2, 3), *rng.normal(size=3), rng.uniform(0.1, 3), *rng.normal(size=2)])
        WR = np.array([rng.uniform(0.2, 3), *rng.normal(size=3), rng.uniform(0.1, 3), *rng.normal(size=2)])
        bx = rng.normal()
        F = orc.hlld(G, WL, WR, bx)
        guards(False, True)
        Fraw = orc.hlld(G, WL, WR, bx)
        guards(True, True)
        np.testing.assert_array_equal(F, Fraw)


def _wave_err(N, recon):
    p = inputs.linear_wave(N, 4, 4, "fast", recon=recon)
    o = orc.Oracle(*p.n, p.gamma, p.recon)
    o.set_state(p.state)
    run_to_time(o, p)
    e = inputs.wave_error(p.state, o.get_state())
    o.close()
    return e


def _sod_rho(N=64):
    g = 1.4
    x = (np.arange(N) + 0.5) / N
    one = np.ones((2, 2, N))
    sh = inputs.field_shapes(N, 2, 2)
    st = inputs.from_primitives(np.where(x < 0.5, 1.0, 0.125) * one, 0 * one, 0 * one, 0 * one,
                                np.where(x < 0.5, 1.0, 0.1) * one, np.zeros(sh["bx"]), np.zeros(sh["by"]),
                                np.zeros(sh["bz"]), g)
    p = inputs.Problem("sod", (N, 2, 2), g, st, bc=(1, 0, 0), recon=2, t_end=0.1)
    o = orc.Oracle(*p.n, p.gamma, p.recon, p.bc)
    o.set_state(p.state)
    run_to_time(o, p)
    rho = o.get_state()["rho"][0, 0].copy()
    o.close()
    return rho


def test_guards_do_not_move_the_pins_that_are_not_round_off_ties(guards):
    """T8 (linear-wave errors, PLMC and PPMC), a PPMC Sod run and one step of a generic random field
    give the same numbers with R6 and R7 switched off."""
    p = inputs.random_smooth(n=(12, 10, 8), seed=4, recon=2)

    def one_step():   # (the oracle holds ONE grid: every run re-creates it)
        o = orc.Oracle(*p.n, p.gamma, 2)
        o.set_state(p.state)
        o.step(0.9 * o.compute_dt(0.4))
        out = o.get_state()
        o.close()
        return out
    ref = {"w1": _wave_err(32, 1), "w2": _wave_err(32, 2), "sod": _sod_rho(), "rs": one_step()}
    guards(False, False)
    assert _wave_err(32, 1) == pytest.approx(ref["w1"], rel=1e-9)
    # (the wave is a 1e-6 perturbation of a uniform state: its characteristic differences DO come
    # within 1e-12 of zero at the crests, so R7 acts there; the error norm moves in the 4th digit)
    assert _wave_err(32, 2) == pytest.approx(ref["w2"], rel=2e-3)
    # at the numerical foot of the rarefaction the differences pass through 1e-12 |q| and R7 flushes
    # them: the effect is bounded by the size of what is flushed
    np.testing.assert_allclose(_sod_rho(), ref["sod"], rtol=0, atol=5e-12)
    got = one_step()
    for f in FIELDS:
        np.testing.assert_array_equal(got[f], ref["rs"][f])


@pytest.mark.parametrize("recon", [1, 2])
def test_guards_are_what_keeps_the_blast_mirror_symmetric(guards, recon):
    """the blast keeps its symmetry.  In the paper's box (B in the x-y plane) the
    z-mirror image of the state must be the state; with the guards the oracle keeps this to
    round-off for PLMC over 6 steps (PPMC over 3: reading R11, the extremum switch of PPM itself),
    without R6 it is lost in the first steps."""
    def z_asym(n_steps):
        p = inputs.blast_paper(nx=16, recon=recon)
        o = orc.Oracle(*p.n, p.gamma, p.recon, p.bc, p.domain)
        o.set_state(p.state)
        worst = 0.0
        for _ in range(n_steps):
            o.step(o.compute_dt(p.cfl))
            st = o.get_state()
            worst = max(worst, float(np.max(np.abs(st["rho"] - st["rho"][::-1]))))
        o.close()
        return worst
    steps = 6 if recon == 1 else 3
    assert z_asym(steps) < 1e-13
    guards(False, True)
    assert z_asym(steps) > 1e-9
