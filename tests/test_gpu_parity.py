"""GPU parity: libmhd.so (through the C ABI binding) against the CPU oracle, element by element
on the same seeded inputs.  Tolerances are BASELINE.json's: max relative difference per field
<= 1e-12 after one step, <= 1e-9 after a full run, normalised |div B| dx / |B| <= 1e-12 every step.
"""
import numpy as np
import pytest

import oracle as orc
from paper_2402_05240_b200 import inputs
from helpers import run_to_time, divb_normalised, rel_diff, FIELDS, totals, roundoff_floor, max_excess

pytestmark = pytest.mark.gpu

TOL_STEP = 1e-12
TOL_RUN = 1e-9
TOL_DIVB = 1e-12


@pytest.fixture(scope="module")
def mhd():
    from paper_2402_05240_b200 import mhd as m
    return m


def make_pair(mhd, p, **kw):
    o = orc.Oracle(*p.n, p.gamma, p.recon, p.bc, p.domain)
    o.set_state(p.state)
    g = mhd.Mhd(*p.n, p.gamma, p.recon, p.bc, domain=p.domain, **kw)
    g.set_state(p.state)
    return o, g


def assert_close(a, b, tol, what, floor=None):
    """max|a-b| <= tol * max|b| per field (companion norm for identically-zero fields); with `floor`
    (helpers.roundoff_floor) the absolute fp64 round-off floor of the update is added to the bound."""
    if floor is not None:
        ex = max_excess(a, b, tol, floor)
        assert max(ex.values()) <= 0.0, "%s: excess over tol*|f|+floor %s; rel diffs %s" % (what, ex, rel_diff(a, b))
        return
    rd = rel_diff(a, b)
    worst = max(rd.values())
    assert worst <= tol, "%s: per-field max relative difference %s" % (what, rd)
    return worst


def test_roundtrip_set_get(mhd):
    p = inputs.random_smooth(n=(37, 21, 19), seed=3)
    g = mhd.Mhd(*p.n, p.gamma, p.recon)
    g.set_state(p.state)
    out = g.get_state()
    for f in FIELDS:
        if f in ("bx", "by", "bz"):
            a = inputs._active(out[f], f)
            b = inputs._active(p.state[f], f)
            assert np.array_equal(a, b), f
        else:
            assert np.array_equal(out[f], p.state[f]), f
    g.close()


@pytest.mark.parametrize("recon", [0, 1, 2, 3, 4])
@pytest.mark.parametrize("n", [(37, 21, 19), (130, 9, 34), (16, 70, 5)])
def test_one_step_random_smooth(mhd, recon, n):
    """Ragged sizes spanning several x-pencil blocks (127 faces) and march chunks."""
    p = inputs.random_smooth(n=n, seed=11 + recon, recon=recon)
    o, g = make_pair(mhd, p)
    dt_o = o.compute_dt(p.cfl)
    dt_g = g.compute_dt(p.cfl)
    assert abs(dt_g - dt_o) <= 1e-13 * dt_o
    o.step(dt_o)
    g.step(dt_o)
    assert_close(g.get_half_state(), o.get_half_state(), TOL_STEP, "half state")
    out = g.get_state()
    assert_close(out, o.get_state(), TOL_STEP, "full state")
    assert divb_normalised(out, p.n) <= TOL_DIVB
    o.close(); g.close()


@pytest.mark.parametrize("recon,n", [(1, (67, 45, 23)), (2, (31, 12, 40))])
def test_fused_predictor_stage_agrees_with_the_three_kernel_path(mhd, recon, n, monkeypatch):
    """The predictor stage runs as one kernel (csrc/mhd_stage.cuh: tiles of 30 x 10 columns with a
    halo, marching in z-chunks); MHD_STAGE_TY=0 at mhd_init selects the earlier formulation (fluxes,
    edge fields and half update as three kernels through HBM).  Same arithmetic, different summation
    order in the z difference and the face updates only: the half state agrees to rounding, over
    several tiles and chunks with ragged edges."""
    p = inputs.random_smooth(n=n, seed=77, recon=recon)
    out = {}
    for ty in ("0", "12"):
        monkeypatch.setenv("MHD_STAGE_TY", ty)
        g = mhd.Mhd(*p.n, p.gamma, p.recon, p.bc)
        g.set_state(p.state)
        n0 = g.launch_count()
        g.step(g.compute_dt(p.cfl))
        out[ty] = (g.get_half_state(), g.get_state(), g.launch_count() - n0)
        g.close()
    assert out["0"][2] - out["12"][2] == 3               # ghost fill + three launches became one
    assert_close(out["12"][0], out["0"][0], 1e-13, "half state, fused vs three kernels")
    assert_close(out["12"][1], out["0"][1], 1e-13, "full state, fused vs three kernels")


@pytest.mark.parametrize("recon", [1, 2, 3, 4])
def test_uniform_state_bit_for_bit(mhd, recon):
    p = inputs.uniform(n=(8, 6, 5), recon=recon)
    g = mhd.Mhd(*p.n, p.gamma, p.recon)
    g.set_state(p.state)
    dt = g.compute_dt(0.4)
    for _ in range(3):
        g.step(dt)
    out = g.get_state()
    for f in FIELDS:
        assert np.array_equal(out[f], p.state[f]), f
    g.close()


@pytest.mark.parametrize("n", [(1, 1, 1), (2, 1, 3), (5, 3, 2), (4, 4, 4)])
@pytest.mark.parametrize("recon", [1, 2, 3, 4])
def test_tiny_grids(mhd, n, recon):
    """Grids thinner than the ghost depth: periodic images wrap more than once."""
    p = inputs.random_smooth(n=(8, 8, 8), seed=5, recon=recon)
    st = {}
    sh = inputs.field_shapes(*n)
    for f in FIELDS:
        st[f] = np.ascontiguousarray(p.state[f][:sh[f][0], :sh[f][1], :sh[f][2]])
    # periodic closure of the staggered field: face n equals face 0
    st["bx"][:, :, -1] = st["bx"][:, :, 0]
    st["by"][:, -1, :] = st["by"][:, 0, :]
    st["bz"][-1, :, :] = st["bz"][0, :, :]
    q = inputs.Problem(name="tiny", n=n, gamma=p.gamma, state=st, recon=recon)
    o, g = make_pair(mhd, q)
    dt = o.compute_dt(0.4)
    assert abs(g.compute_dt(0.4) - dt) <= 1e-13 * dt
    o.step(dt); g.step(dt)
    assert_close(g.get_state(), o.get_state(), TOL_STEP, "tiny %s" % (n,))
    o.close(); g.close()


def test_c1_linear_wave_full_run(mhd):
    """BASELINE.json configs[0]: 32^3 fast wave, one period, vs the oracle and the closed form."""
    p = inputs.linear_wave(32, 32, 32, "fast", recon=1)
    o, g = make_pair(mhd, p)
    n_o = run_to_time(o, p)
    n_g = run_to_time(g, p)
    assert n_o == n_g
    out = g.get_state()
    # momenta are 1e-6 perturbations updated by differences of O(1) fluxes: round-off floor applies
    assert_close(out, o.get_state(), TOL_RUN, "C1 final state", floor=roundoff_floor(p.state, p.gamma, n_o))
    # closed form: the wave returns to its initial state; same error as the oracle's run
    err = inputs.wave_error(p.state, out)
    assert err == pytest.approx(inputs.wave_error(p.state, o.get_state()), rel=1e-6)
    assert 5e-8 < err < 8e-8
    assert divb_normalised(out, p.n) <= TOL_DIVB
    o.close(); g.close()


@pytest.mark.parametrize("axis", [1, 2])
def test_linear_wave_other_axes_ppmc(mhd, axis):
    p = inputs.linear_wave(16, 16, 16, "fast", axis=axis, recon=2)
    o, g = make_pair(mhd, p)
    run_to_time(o, p); run_to_time(g, p)
    out = g.get_state()
    assert_close(out, o.get_state(), TOL_RUN, "PPMC wave axis %d" % axis,
                 floor=roundoff_floor(p.state, p.gamma, 100))
    assert inputs.wave_error(p.state, out) == pytest.approx(inputs.wave_error(p.state, o.get_state()), rel=1e-6)
    o.close(); g.close()


@pytest.mark.parametrize("recon,gold", [(1, 6.5165e-8), (2, 2.832e-8)])
def test_linear_wave_golden_value(mhd, recon, gold):
    """tests/golden/linear_wave_errors.txt (N = 32, transverse 4x4 so that dt is set by x): the CUDA
    path reproduces the recorded L2-of-L1 error of the closed-form test."""
    p = inputs.linear_wave(32, 4, 4, "fast", recon=recon)
    g = mhd.Mhd(*p.n, p.gamma, p.recon)
    g.set_state(p.state)
    run_to_time(g, p)
    assert inputs.wave_error(p.state, g.get_state()) == pytest.approx(gold, rel=2e-3)
    g.close()


def test_c2_brio_wu_outflow(mhd):
    """BASELINE.json configs[1]: 256x16x16, outflow in x, to t = 0.1."""
    p = inputs.riemann("brio_wu", 256, 16, axis=0, recon=1)
    o, g = make_pair(mhd, p)
    dt = o.compute_dt(p.cfl)
    o.step(dt); g.step(dt)
    assert_close(g.get_state(), o.get_state(), TOL_STEP, "C2 one step")
    # the full run, from the initial state again: each side takes its own dt (both from Eq. 11) and clips the
    # last step; same number of steps (243), final states within north_star's full-run tolerance (seen: 3e-14).
    # (Until round 2 the oracle's run started from its state after the first step, so the step counts
    # differed by one and the comparison of the final states was skipped.)
    o.set_state(p.state); g.set_state(p.state)
    n_o = run_to_time(o, p)
    n_g = run_to_time(g, p)
    out, ref = g.get_state(), o.get_state()
    assert n_g == n_o
    assert_close(out, ref, TOL_RUN, "C2 final state")
    # planar invariants (pin T12)
    assert np.all(out["bx"] == 0.75)
    assert np.max(np.abs(out["mz"])) <= 1e-14 and np.max(np.abs(out["bz"])) <= 1e-14
    assert np.array_equal(out["rho"], np.broadcast_to(out["rho"][0:1, 0:1, :], out["rho"].shape))
    o.close(); g.close()


@pytest.mark.parametrize("axis", [1, 2])
def test_riemann_other_axes_outflow(mhd, axis):
    p = inputs.riemann("dai_woodward", 64, 8, axis=axis, recon=2, flip=(axis == 2))
    o, g = make_pair(mhd, p)
    for _ in range(5):
        dt = o.compute_dt(p.cfl)
        o.step(dt); g.step(dt)
    assert_close(g.get_state(), o.get_state(), 5 * TOL_STEP, "riemann axis %d" % axis)
    o.close(); g.close()


def test_c4_blast_small(mhd):
    """Shape of BASELINE.json configs[3] at 32^3: PPMC, strong shock, 20 steps.  Every step is a
    one-step parity case from the oracle's own state (the limiters are discontinuous switches, so a
    free-running pair may legitimately part ways at a tie; BASELINE.json asks 1e-12 per step and
    1e-9 only for the smooth-wave run).  The free-running GPU state is checked for what is unique:
    positivity, div B, point symmetry about the centre, and closeness to the oracle run."""
    p = inputs.blast(32, recon=2, n_steps=20)
    o, g = make_pair(mhd, p)
    state = p.state
    worst = 0.0
    for s in range(p.n_steps):
        g.set_state(state)
        dt = o.compute_dt(p.cfl)
        assert abs(g.compute_dt(p.cfl) - dt) <= 1e-13 * dt
        o.step(dt); g.step(dt)
        state = o.get_state()
        worst = max(worst, assert_close(g.get_state(), state, TOL_STEP, "blast step %d" % (s + 1)))
    ref = state
    # free-running GPU
    g.set_state(p.state)
    for s in range(p.n_steps):
        g.step(g.compute_dt(p.cfl))
    out = g.get_state()
    assert np.min(out["rho"]) > 0.0 and np.all(np.isfinite(out["E"]))
    assert divb_normalised(out, p.n) <= TOL_DIVB
    for f in ("rho", "E"):   # point symmetry about the box centre (T13)
        assert np.max(np.abs(out[f] - out[f][::-1, ::-1, ::-1])) <= 1e-11 * np.max(np.abs(out[f]))
    rd = rel_diff(out, ref)
    assert max(rd.values()) <= 1e-9, "blast 20 steps free-running: %s" % rd
    o.close(); g.close()


@pytest.mark.parametrize("recon", [3, 4])
def test_primitive_limiting_brio_wu_and_blast_steps(mhd, recon):
    """PLMP / PPMP on the discontinuous problems: 12 steps of Brio-Wu (outflow x) and
    8 of the 24^3 blast, every step a one-step parity case from the oracle's own state."""
    for p, nsteps in ((inputs.riemann("brio_wu", 64, 4, axis=0, recon=recon), 12), (inputs.blast(24, recon=recon), 8)):
        o, g = make_pair(mhd, p)
        state = p.state
        for s in range(nsteps):
            g.set_state(state)
            dt = o.compute_dt(p.cfl)
            o.step(dt); g.step(dt)
            state = o.get_state()
            out = g.get_state()
            what = "%s recon %d step %d" % (p.name, recon, s + 1)
            # (Round 1 counted up to 48 PPMP blast cells between 1e-12 and 5e-12 here: the flush of reading R7 is a
            # switch of size tau and the two implementations took different sides of it ahead of the blast wave.
            # With the branch-free limiter of round 2 the eight steps agree to 8e-16; a flip of the switch still shows,
            # as 1.5e-13 in step 9, under the tolerance.)
            assert_close(out, state, TOL_STEP, what)
            assert divb_normalised(out, p.n) <= TOL_DIVB
        o.close(); g.close()


def test_c3_turbulence_small_multi_step(mhd):
    """Shape of BASELINE.json configs[2]/[4] at 48^3: Mach-1 turbulence, beta = 1, PLMC, 5 steps."""
    p = inputs.turbulence(48, n_steps=5)
    o, g = make_pair(mhd, p)
    t0 = totals(p.state)
    for s in range(p.n_steps):
        dt = o.compute_dt(p.cfl)
        assert abs(g.compute_dt(p.cfl) - dt) <= 1e-12 * dt
        o.step(dt); g.step(dt)
        out = g.get_state()
        assert divb_normalised(out, p.n) <= TOL_DIVB
        assert_close(out, o.get_state(), (s + 1) * 10 * TOL_STEP if s else TOL_STEP, "turbulence step %d" % s)
    t1 = totals(out)
    for f in ("rho", "E"):
        assert abs(t1[f] - t0[f]) <= 1e-13 * abs(t0[f])
    o.close(); g.close()


def test_advance_matches_stepwise_and_device_io(mhd, monkeypatch):
    """mhd_advance (dt kept on the device) == {compute_dt; step} loop; device set/get == host set/get."""
    import torch
    monkeypatch.setenv("MHD_SMALL", "0")                # the kernel-by-kernel path (bitwise comparison below)
    p = inputs.random_smooth(n=(40, 24, 18), seed=8, recon=1)
    g = mhd.Mhd(*p.n, p.gamma, p.recon)
    g.set_state(p.state)
    tsum = 0.0
    for _ in range(3):
        dt = g.compute_dt(0.4)
        g.step(dt); tsum += dt
    ref = g.get_state()
    dev_in = {f: torch.from_numpy(np.ascontiguousarray(p.state[f])).cuda() for f in FIELDS}
    g.set_state_device(dev_in)
    t = g.advance(3, 0.4, want_time=True)
    assert abs(t - tsum) <= 1e-14 * tsum
    dev_out = {f: torch.empty_like(dev_in[f]) for f in FIELDS}
    g.get_state_device(dev_out)
    torch.cuda.synchronize()
    for f in FIELDS:
        assert np.array_equal(dev_out[f].cpu().numpy(), ref[f]), f
    g.close()


@pytest.mark.parametrize("n", [(600, 3, 600), (600, 600, 3), (3, 700, 520)])
def test_thin_slabs_with_many_blocks(mhd, n):
    """Grids with a handful of cells along one sweep axis and thousands of blocks across it (the marching
    sweeps then take one chunk per column; a chunk count of zero once divided by zero here): one PLMC
    step against the oracle."""
    p = inputs.random_smooth(n=n, seed=9, recon=1)
    o, g = make_pair(mhd, p)
    dt = o.compute_dt(p.cfl)
    assert abs(g.compute_dt(p.cfl) - dt) <= 1e-13 * dt
    o.step(dt); g.step(dt)
    out = g.get_state()
    assert_close(out, o.get_state(), TOL_STEP, "thin slab %s" % (n,))
    assert divb_normalised(out, p.n) <= TOL_DIVB
    o.close(); g.close()


def test_advance_profile_is_bitwise_advance_and_names_its_kernels(mhd, monkeypatch):
    """mhd_advance_profile (bench.py's per-kernel times) runs the steps of mhd_advance with an event after
    every launch: the state after K profiled steps is bit for bit that of K plain steps, a step is the dt
    kernel plus six stage kernels, every duration is positive, and a following plain call carries on."""
    monkeypatch.setenv("MHD_SMALL", "0")
    p = inputs.random_smooth(n=(45, 33, 21), seed=5, recon=1)
    ref = mhd.Mhd(*p.n, p.gamma, p.recon, p.bc)
    ref.set_state(p.state)
    for _ in range(5):
        ref.step(ref.compute_dt(0.4))
    want = ref.get_state()
    ref.close()
    g = mhd.Mhd(*p.n, p.gamma, p.recon, p.bc)
    g.set_state(p.state)
    prof = g.advance_profile(3, 0.4)
    assert [name for name, _ in prof] == ["k_finish_dt", "k_predictor_stage", "k_flux_x", "k_flux_march<1>",
                                          "k_flux_march<2>+update", "k_ct(corrector)", "k_update(B)+cfl"]
    assert all(t > 0.0 for _, t in prof)
    g.advance(2, 0.4)
    got = g.get_state()
    for f in FIELDS:
        assert np.array_equal(got[f], want[f]), f
    one = g.step_profile(g.compute_dt(0.4))              # the one-step variant still returns the six stage kernels
    assert [name for name, _ in one] == [name for name, _ in prof][1:]
    with pytest.raises(mhd.MhdError):
        g.advance_profile(0, 0.4)
    g.close()


@pytest.mark.parametrize("recon,bc", [(1, (0, 0, 0)), (2, (1, 0, 0))])
def test_advance_graph_path_is_bitwise_the_stepwise_path(mhd, recon, bc, monkeypatch):
    """On a non-default stream and a small grid mhd_advance replays a CUDA graph of two steps; an odd
    step count, a second call (other orientation of the B ping-pong) and a boundary change in between
    must all give exactly what the kernel-by-kernel path gives."""
    import torch
    monkeypatch.setenv("MHD_SMALL", "0")                # (a grid this small would take the cooperative kernel)
    p = inputs.random_smooth(n=(33, 20, 17), seed=12, recon=recon)
    ref = mhd.Mhd(*p.n, p.gamma, p.recon, bc)           # default stream: no graph
    ref.set_state(p.state)
    for _ in range(7 + 6):
        ref.step(ref.compute_dt(0.4))
    want = ref.get_state()
    ref.close()
    stream = torch.cuda.Stream()
    g = mhd.Mhd(*p.n, p.gamma, p.recon, bc, stream=stream)
    g.set_state(p.state)
    n0 = g.launch_count()
    g.advance(7, 0.4)                                    # 3 graph launches + 1 plain step
    n7 = g.launch_count() - n0
    g.advance(6, 0.4)                                    # graph for the other parity
    got = g.get_state()
    for f in FIELDS:
        assert np.array_equal(got[f], want[f]), f
    assert n7 >= 7 * 7                                    # launch_count() counts replayed kernels too
    g.close()


def test_internal_cudamalloc_and_stream(mhd):
    import torch
    p = inputs.random_smooth(n=(20, 12, 10), seed=9, recon=2)
    o = orc.Oracle(*p.n, p.gamma, p.recon)
    o.set_state(p.state)
    s = torch.cuda.Stream()
    g = mhd.Mhd(*p.n, p.gamma, p.recon, use_torch_workspace=False, stream=s)
    g.set_state(p.state)
    dt = o.compute_dt(0.4)
    o.step(dt); g.step(dt)
    assert_close(g.get_state(), o.get_state(), TOL_STEP, "cudaMalloc + stream")
    g.close(); o.close()
    mhd.lib().mhd_set_stream(None)


def test_error_codes(mhd):
    L = mhd.lib()
    L.mhd_finalize()
    assert L.mhd_step(0.1) == -2
    assert L.mhd_init(0, 4, 4, 1.4, 1) == -1
    assert L.mhd_init(4, 4, 4, 1.0, 1) == -1
    assert L.mhd_init(4, 4, 4, 1.4, 7) == -1
    assert L.mhd_init(4, 4, 4, 1.4, 1) == 0
    assert L.mhd_step(-1.0) == -1
    assert L.mhd_set_boundary(3, 0) == -1
    # a state with negative pressure is reported by the CFL kernel, not silently floored (G18)
    p = inputs.uniform(n=(4, 4, 4))
    st = {k: v.copy() for k, v in p.state.items()}
    st["E"][1, 2, 3] = 0.0
    g = mhd.Mhd(4, 4, 4, p.gamma, 1)
    g.set_state(st)
    with pytest.raises(mhd.MhdError):
        g.compute_dt(0.4)
    g.close()


@pytest.mark.parametrize("recon", [1, 2])
def test_corrector_fluxes_against_oracle(mhd, recon):
    """mhd_get_flux: the corrector (Step 7) flux components that the library keeps in
    memory -- all seven of the x and y sweeps, mass and the two induction components of the z sweep (its
    momentum / energy fluxes are consumed in the sweep) -- against the oracle's, face by face; the call
    is made after mhd_get_state, which must not disturb them (host I/O is staged elsewhere)."""
    p = inputs.random_smooth(n=(37, 21, 19), seed=31, recon=recon)
    o, g = make_pair(mhd, p)
    dt = o.compute_dt(p.cfl)
    o.step(dt); g.step(dt)
    g.get_state()
    for axis in range(3):
        ref = {c: o.get_flux(axis, c) for c in range(7)}
        scale = max(np.abs(r).max() for r in ref.values())
        for c in range(7):
            if axis == 2 and 1 <= c <= 4:
                with pytest.raises(mhd.MhdError):
                    g.get_flux(axis, c)
                continue
            got = g.get_flux(axis, c)
            assert np.abs(got - ref[c]).max() <= TOL_STEP * scale, (axis, c)
    o.close(); g.close()


def test_unphysical_flag_belongs_to_the_state_it_was_computed_on(mhd):
    """MHD_ERR_UNPHYSICAL is not sticky: after a bad state, mhd_set_state(good) + mhd_compute_dt
    succeeds (PAPER.md:523 on error reporting; SURVEY.md 8(b) error convention)."""
    p = inputs.random_smooth(n=(12, 10, 8), seed=21)
    bad = {k: v.copy() for k, v in p.state.items()}
    bad["E"][3, 2, 1] = 0.0
    g = mhd.Mhd(*p.n, p.gamma, 1)
    g.set_state(bad)
    with pytest.raises(mhd.MhdError):
        g.compute_dt(0.4)
    g.set_state(p.state)
    o = orc.Oracle(*p.n, p.gamma, 1)
    o.set_state(p.state)
    dt = g.compute_dt(0.4)
    assert abs(dt - o.compute_dt(0.4)) <= 1e-13 * dt
    g.step(dt)
    assert g.compute_dt(0.4) > 0.0          # the flag of the new state, folded into the full update
    assert g.advance(2, 0.4, want_time=True) > 0.0
    g.close(); o.close()


@pytest.mark.timeout(1800)
def test_full_size_256_cube_ten_steps(mhd):
    """BASELINE.json configs[2] as stated: 256^3, 10 steps.  Every step is a one-step parity case
    from the oracle's own state, every cell (1e-12), and the free-running GPU state after the 10
    steps (mhd_advance, the call bench.py times) is compared with the oracle's at the run bound."""
    p = inputs.turbulence(256, n_steps=10)
    o, g = make_pair(mhd, p)
    state = p.state
    for s in range(p.n_steps):
        if s:
            g.set_state(state)
        dt = o.compute_dt(p.cfl)
        assert abs(g.compute_dt(p.cfl) - dt) <= 1e-13 * dt
        o.step(dt); g.step(dt)
        state = o.get_state()
        out = g.get_state()
        assert_close(out, state, TOL_STEP, "256^3 step %d" % (s + 1))
        assert divb_normalised(out, p.n) <= TOL_DIVB
    g.set_state(p.state)
    g.advance(p.n_steps, p.cfl)
    out = g.get_state()
    assert_close(out, state, TOL_RUN, "256^3 ten free-running steps")
    assert divb_normalised(out, p.n) <= TOL_DIVB
    o.close(); g.close()


def _sub_box(state, org, m):
    """m^3 cells of a full-size state starting at org = (i0, j0, k0), in the ABI layout of an m^3 grid."""
    i0, j0, k0 = org
    s = {f: np.ascontiguousarray(state[f][k0:k0 + m, j0:j0 + m, i0:i0 + m]) for f in FIELDS[:5]}
    s["bx"] = np.ascontiguousarray(state["bx"][k0:k0 + m, j0:j0 + m, i0:i0 + m + 1])
    s["by"] = np.ascontiguousarray(state["by"][k0:k0 + m, j0:j0 + m + 1, i0:i0 + m])
    s["bz"] = np.ascontiguousarray(state["bz"][k0:k0 + m + 1, j0:j0 + m, i0:i0 + m])
    return s


@pytest.mark.timeout(3000)
@pytest.mark.parametrize("workload", ["c4", "c5"])
def test_full_size_sampled_parity(mhd, workload):
    """BASELINE.json configs[3] (512^3 blast, PPMC) and configs[4] (640^3 turbulence, PLMC) at FULL
    size, in the launch configuration bench.py times.  The oracle cannot hold these grids, so it
    recomputes sampled blocks one by one: an m^3 block (m = N/16) of the state before the step is
    advanced by the oracle as a small periodic box with dt scaled by N/m = 16 (ideal MHD has no
    length scale; the factor is a power of two, so dt/Delta is the same number bit for bit); one
    step reaches at most 7 cells, so the block's interior (8 cells from its rim) is exact and must
    match the GPU's full-grid result to 1e-12.  Steps 1, 2, the middle and the last step of the
    config's run (20 for c4, 10 for c5) are checked, each from the GPU's own state before it, plus
    div B and positivity on the whole grid."""
    if workload == "c4":
        p = inputs.blast(512, recon=2)
        N, m = 512, 32
        orgs = [(256 - 16, 256 - 16, 256 - 16), (256 + 51 - 16, 256 - 16, 256 - 10), (256 - 40, 256 + 30, 256 - 45),
                (10, 400, 77)]
    else:
        p = inputs.turbulence(640)
        N, m = 640, 40
        rng = np.random.default_rng(99)
        orgs = [tuple(int(x) for x in rng.integers(0, N - m, 3)) for _ in range(4)] + [(0, 0, 0), (N - m, N - m, N - m)]
    g = mhd.Mhd(*p.n, p.gamma, p.recon, p.bc)
    g.set_state(p.state)
    before = p.state
    worst = 0.0
    # the config's own step count (c4: 20, c5: 10): steps 1, 2, the middle one and the last one are
    # checked, each from the GPU's own state before it; the steps in between run through mhd_advance
    nsteps = 20 if workload == "c4" else 10
    done = 0
    for step in (1, 2, nsteps // 2, nsteps):
        if step - 1 > done:
            g.advance(step - 1 - done, p.cfl)
            done = step - 1
            p.state = None                      # (host memory: at most two full states at a time)
            before = after = None
            before = g.get_state()
        dt = g.compute_dt(p.cfl)
        g.step(dt)
        done += 1
        after = g.get_state()
        assert np.min(after["rho"]) > 0.0 and np.all(np.isfinite(after["E"]))
        for org in orgs:
            o = orc.Oracle(m, m, m, p.gamma, p.recon)
            o.set_state(_sub_box(before, org, m))
            o.step(dt * (N // m))
            ref = o.get_state()
            o.close()
            got = _sub_box(after, org, m)
            c = slice(8, m - 8)
            for f in FIELDS:
                a, b = got[f][c, c, c], ref[f][c, c, c]
                scale = max(np.abs(before[f]).max(), 1e-300) if f not in ("mx", "my", "mz") else \
                    max(np.abs(before["rho"]).max(), 1e-300)
                d = np.abs(a - b).max() / scale
                worst = max(worst, d)
                assert d <= TOL_STEP, "%s step %d block %s field %s: %.3e" % (workload, step, org, f, d)
        before = after
    assert g.max_divb() * (1.0 / N) / np.sqrt(np.mean(before["bx"] ** 2 + 0) * 3) <= TOL_DIVB
    g.close()
