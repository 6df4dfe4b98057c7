"""Run the paper's own test suite (section 3.1) on the GPU at or near the paper's
resolutions and print what each test measures, as markdown.  Everything runs through the C ABI
binding; nothing here touches the oracle.

  python -m paper_2402_05240_b200.suite [--quick]

Linear-wave and circularly-polarised-Alfven-wave convergence (Fig. 2, 3), field-loop dissipation and
div B (Fig. 4), blast-wave symmetry (Fig. 11), Orszag-Tang invariants (Fig. 12), with wall time and
cell updates per second of each run.
"""
import argparse
import time

import numpy as np

from . import inputs, mhd


def run(p, stream=None):
    """{compute_dt; step} to p.t_end with the last step clipped. Returns (state, steps, s)."""
    g = mhd.Mhd(*p.n, p.gamma, p.recon, p.bc, domain=p.domain)
    g.set_state(p.state)
    t, n = 0.0, 0
    t0 = time.perf_counter()
    while t < p.t_end * (1.0 - 1e-14):
        dt = g.compute_dt(p.cfl)
        if t + dt > p.t_end:
            dt = p.t_end - t
        g.step(dt)
        t += dt
        n += 1
    g.synchronize()
    el = time.perf_counter() - t0
    out = g.get_state()
    divb = g.max_divb()
    g.close()
    return out, n, el, divb


def rate(p, n, el):
    return p.n[0] * p.n[1] * p.n[2] * n / el / 1e9


def b2_mean(st):
    b = inputs.cell_centred_b(st)
    return float((b[0] ** 2 + b[1] ** 2 + b[2] ** 2).mean())


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--quick", action="store_true", help="smaller grids (a minute instead of several)")
    a = ap.parse_args()
    q = a.quick
    names = {1: "PLMC", 2: "PPMC"}

    print("## Linear fast wave, N x 16 x 16, one period, error of Eq. 34-35 (PAPER.md:333-356, Fig. 2)\n")
    print("| recon | N | error | order | steps | G cell updates/s |\n|---|---|---|---|---|---|")
    for recon in (1, 2):
        prev = None
        for N in ((16, 32, 64) if q else (16, 32, 64, 128, 256, 512)):
            p = inputs.linear_wave(N, 16, 16, "fast", recon=recon)
            out, n, el, _ = run(p)
            e = inputs.wave_error(p.state, out)
            print("| %s | %d | %.4e | %s | %d | %.3f |" % (names[recon], N, e, "-" if prev is None else "%.2f" % np.log2(prev / e),
                                                       n, rate(p, n, el)))
            prev = e

    print("\n## Circularly polarised Alfven wave, 2N x N x N in 3 x 1.5 x 1.5, one period (PAPER.md:358-376, Fig. 3)\n")
    print("| recon | N | error | order | steps | G cell updates/s |\n|---|---|---|---|---|---|")
    for recon in (1, 2):
        prev = None
        for N in ((8, 16, 32) if q else (8, 16, 32, 64, 128)):
            p = inputs.cpaw(N, recon=recon)
            out, n, el, _ = run(p)
            e = inputs.wave_error(p.state, out)
            print("| %s | %d | %.4e | %s | %d | %.3f |" % (names[recon], N, e, "-" if prev is None else "%.2f" % np.log2(prev / e),
                                                       n, rate(p, n, el)))
            prev = e

    print("\n## Advecting field loop, N x N x 2N in 1 x 1 x 2, PPMC, t = 2 (PAPER.md:378-391, Fig. 4)\n")
    print("| N | mean B^2 / initial | max div B (1/length, |B| = 1e-3) | far-corner |B| | steps | G cell updates/s |\n|---|---|---|---|---|---|")
    for N in ((32,) if q else (32, 64, 128)):
        p = inputs.field_loop(N, recon=2)
        out, n, el, divb = run(p)
        b = inputs.cell_centred_b(out)
        far = float(np.sqrt(b[0][0, 0, 0] ** 2 + b[1][0, 0, 0] ** 2 + b[2][0, 0, 0] ** 2))
        print("| %d | %.4f | %.2e | %.1e | %d | %.3f |" % (N, b2_mean(out) / b2_mean(p.state), divb, far, n, rate(p, n, el)))

    print("\n## MHD blast, beta = 0.2, 1 x 1.5 x 1 box, t = 0.2, PLMC (PAPER.md:455-465, Fig. 11)\n")
    p = inputs.blast_paper(60 if q else 200, recon=1)
    out, n, el, divb = run(p)
    rho = out["rho"]
    print("grid %d x %d x %d, %d steps, %.1f s, %.3f G cell updates/s; rho in [%.4f, %.4f]; z-mirror asymmetry %.1e, "
          "point asymmetry %.1e; max div B %.1e\n" % (p.n + (n, el, rate(p, n, el), rho.min(), rho.max(),
                                                      np.abs(rho - rho[::-1]).max(), np.abs(rho - rho[::-1, ::-1, ::-1]).max(), divb)))

    print("## Orszag-Tang vortex, N^3, t = 0.5, PPMC (PAPER.md:467-475, Fig. 12)\n")
    N = 64 if q else 192
    p = inputs.orszag_tang(N, recon=2)
    m0, e0 = float(p.state["rho"].sum()), float(p.state["E"].sum())
    out, n, el, divb = run(p)
    zinv = all(bool(np.all(out[f] == out[f][:1])) for f in ("rho", "mx", "my", "E", "bx", "by"))
    print("grid %d^3, %d steps, %.1f s, %.3f G cell updates/s; rho in [%.4f, %.4f]; every z-plane bit-identical: %s; "
          "mass drift %.1e, energy drift %.1e; max |B_z| %.1e; max div B %.1e"
          % (N, n, el, rate(p, n, el), out["rho"].min(), out["rho"].max(), zinv, abs(out["rho"].sum() - m0) / m0,
             abs(out["E"].sum() - e0) / e0, np.abs(out["bz"]).max(), divb))


if __name__ == "__main__":
    main()
