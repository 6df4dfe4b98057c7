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


def divb_normalised(state, n, domain=(1.0, 1.0, 1.0)):
    """max |sum_a dB_a/Delta_a| * min(Delta) / B_rms over active cells (SURVEY.md 8(c) parity metric)."""
    nx, ny, nz = (n[a] / domain[a] for a in range(3))   # 1 / Delta_a
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


EPS = 2.220446049250313e-16


def roundoff_floor(state, gamma, n_steps, cfl=0.4, c=2.0):
    """Absolute fp64 round-off floor of n_steps conservative updates.

    Every step adds dt/Delta * (F_up - F_lo) to a field; each flux carries a rounding error of a few
    eps * |F| whatever the order of operations (the oracle is built without FMA contraction, the
    kernels with it), and dt/Delta * |F_f| <= CFL * S_f with S_f the field's natural scale
    (flux / fastest speed): rho for mass, rho*(|v|+c_f) for momentum, E + p_T for energy, |B| for
    the induction equation.  A field whose own magnitude is far below S_f (the 1e-6 momenta of the
    linear wave, C1, on a background with rho c_f = 2) therefore differs between two correct
    implementations by ~ eps * S_f in absolute terms, not by eps * |f|.
    Floor = c * eps * n_steps * CFL * S_f.
    """
    rho = state["rho"]
    bx, by, bz = state["bx"], state["by"], state["bz"]
    b2 = float(np.max(bx * bx) + np.max(by * by) + np.max(bz * bz))
    v = np.sqrt(state["mx"] ** 2 + state["my"] ** 2 + state["mz"] ** 2) / rho
    e = state["E"]
    p = np.maximum((gamma - 1.0) * (e - 0.5 * rho * v * v), 0.0)   # >= P (B^2/2 not removed)
    cf = np.sqrt((gamma * p + b2) / rho)
    k = c * EPS * n_steps * cfl
    fl = {"rho": k * float(np.max(rho)), "mx": k * float(np.max(rho * (v + cf))),
          "E": k * float(np.max(e) + np.max(p) + 0.5 * b2), "bx": k * float(np.sqrt(b2))}
    fl["my"] = fl["mz"] = fl["mx"]
    fl["by"] = fl["bz"] = fl["bx"]
    return fl


def max_excess(a, b, tol, floor):
    """Per field: max|a-b| - (tol * max|b| + floor_f); parity holds where this is <= 0."""
    out = {}
    for f in FIELDS:
        out[f] = float(np.max(np.abs(a[f] - b[f])) - (tol * np.max(np.abs(b[f])) + floor[f]))
    return out
