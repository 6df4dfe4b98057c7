"""Shared test helpers: drivers for the oracle grid and the parity metric (no method arithmetic)."""
import numpy as np

from paper_2402_05240_b200 import inputs

FIELDS = inputs.FIELDS


def run_to_time(sim, p, max_steps=100000):
    """{compute_dt; step} until p.t_end, final step clipped. Returns #steps."""
    t, n = 0.0, 0
    while t < p.t_end * (1.0 - 1e-14) and n < max_steps:
        dt = sim.compute_dt(p.cfl)
        if t + dt > p.t_end:
            dt = p.t_end - t
        sim.step(dt)
        t += dt
        n += 1
    return n


def run_steps(sim, p, n_steps):
    dts = []
    for _ in range(n_steps):
        dt = sim.compute_dt(p.cfl)
        sim.step(dt)
        dts.append(dt)
    return dts


def divb_normalised(state, n):
    """max |sum_a dB_a/Delta_a| * min(Delta) / B_rms over active cells (SURVEY.md 8(c) parity metric)."""
    nx, ny, nz = n
    bx, by, bz = state["bx"], state["by"], state["bz"]
    div = ((bx[:, :, 1:] - bx[:, :, :-1]) * nx + (by[:, 1:, :] - by[:, :-1, :]) * ny
           + (bz[1:, :, :] - bz[:-1, :, :]) * nz)
    bcx = 0.5 * (bx[:, :, 1:] + bx[:, :, :-1])
    bcy = 0.5 * (by[:, 1:, :] + by[:, :-1, :])
    bcz = 0.5 * (bz[1:, :, :] + bz[:-1, :, :])
    brms = np.sqrt(np.mean(bcx ** 2 + bcy ** 2 + bcz ** 2))
    return float(np.max(np.abs(div)) / max(nx, ny, nz) / brms)


def rel_diff(a, b):
    """Per-field max|a-b| / max|b| with the companion-norm rule for identically-zero fields
    (SURVEY.md 8(c) "Parity metric"): momenta are normalised by |m|_inf, B by |B|_inf."""
    out = {}
    mnorm = max(np.max(np.abs(b[f])) for f in ("mx", "my", "mz"))
    bnorm = max(np.max(np.abs(b[f])) for f in ("bx", "by", "bz"))
    for f in FIELDS:
        den = np.max(np.abs(b[f]))
        if f in ("mx", "my", "mz"):
            den = max(den, mnorm) if den < 1e-3 * mnorm else den
        if f in ("bx", "by", "bz"):
            den = max(den, bnorm) if den < 1e-3 * bnorm else den
        den = max(den, 1e-300)
        out[f] = float(np.max(np.abs(a[f] - b[f])) / den)
    return out


def totals(state):
    """Sums of the conserved cell quantities over the active grid."""
    return {f: float(np.sum(state[f])) for f in ("rho", "mx", "my", "mz", "E")}
