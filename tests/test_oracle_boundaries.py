"""Pins for the oracle's boundary fill (O12 / G24) and for its grid driver as a whole.

The paper is silent on how outflow boundaries are applied (PAPER.md:499 mentions only the periodic
halo copy); reading O12: every ghost cell copies the nearest active cell along that axis, every
ghost face of the normal field the nearest of the active faces 0..n.  That rule is what
`numpy.pad(mode="edge")` does, and the periodic rule is `mode="wrap"` -- the ghost layers are built
here with numpy.pad, independently of `fill_ghosts` in oracle/mhd_oracle.c, and one whole VL+CT step
with first-order (PCM) reconstruction is then restated in plain Python loops over a tiny grid: Eq. 14
states, point-wise HLLD fluxes (`orc.hlld`, pinned by T2-T5), Table 1 signs, the CT edge formula
(`orc.ct_edge`, pinned by T7), Eq. 19-22 with dt/2, the same again from the half state, Eq. 29-32.
The index arithmetic, the boundary fill, the flux -> variable map and the update order are typed here
a second time; a mistake in the oracle's version of any of them ("copy cell n-2", "face n-1", a
ghost layer too few, a transposed E component) fails the comparison.
"""
import numpy as np
import pytest

import oracle as orc
from paper_2402_05240_b200 import inputs

FIELDS = inputs.FIELDS
NG = 3   # ghost layers a PCM step needs (one fill per step)


def extend(state, n, bc):
    """Ghost-extended copies of the 8 fields, NG layers on every side, index [k+NG, j+NG, i+NG]."""
    out = {}
    for f in FIELDS:
        a = np.array(state[f], dtype=np.float64)
        for ax_np, axis in ((2, 0), (1, 1), (0, 2)):       # numpy axis <-> coordinate axis
            normal = (f == "b" + "xyz"[axis])
            pad = [(0, 0)] * 3
            if bc[axis] == 0:                                # periodic
                if normal:                                   # n distinct faces; face n is face 0
                    a = np.take(a, range(n[axis]), axis=ax_np)
                    pad[ax_np] = (NG, NG + 1)
                else:
                    pad[ax_np] = (NG, NG)
                a = np.pad(a, pad, mode="wrap")
            else:                                            # outflow: nearest active cell / face
                pad[ax_np] = (NG, NG)
                a = np.pad(a, pad, mode="edge")
        out[f] = a
    return out


class Mini:
    """The VL+CT step with PCM reconstruction on arrays that already carry their ghost layers."""

    def __init__(self, n, gamma):
        self.n, self.g = n, gamma
        self.d = [1.0 / n[a] for a in range(3)]

    @staticmethod
    def at(arr, p):
        return arr[p[2] + NG, p[1] + NG, p[0] + NG]

    def prim(self, U, p):
        """O1: v = m / rho, B_cc = mean of the two faces (Eq. 13), P from E."""
        rho = self.at(U["rho"], p)
        v = [self.at(U[m], p) / rho for m in ("mx", "my", "mz")]
        B = []
        for a, f in enumerate(("bx", "by", "bz")):
            up = list(p); up[a] += 1
            B.append(0.5 * (self.at(U[f], p) + self.at(U[f], up)))
        P = (self.g - 1.0) * (self.at(U["E"], p) - 0.5 * rho * sum(x * x for x in v)
                              - 0.5 * sum(x * x for x in B))
        return rho, v, P, B

    def W(self, U, p, a):
        rho, v, P, B = self.prim(U, p)
        t1, t2 = (a + 1) % 3, (a + 2) % 3
        return np.array([rho, v[a], v[t1], v[t2], P, B[t1], B[t2]])

    def stage(self, Ubase, Ustate, dt, lo, hi):
        """PCM + HLLD + CT + update of cells lo..hi-1 (per axis) and their faces, from the state
        Ustate (fluxes, reference field) applied to Ubase.  Returns a dict of increments keyed by
        (field, i, j, k)."""
        n, d = self.n, self.d
        F = {}     # (a, i, j, k) -> 7 fluxes on the lower a-face of cell (i, j, k)
        for a in range(3):      # a-faces lo..hi along a; one more row / plane below in the other axes
            rng = [range(lo[x], hi[x] + 1) if x == a else range(lo[x] - 1, hi[x] + 1) for x in range(3)]
            for k in rng[2]:
                for j in rng[1]:
                    for i in rng[0]:
                        p = [i, j, k]
                        m = list(p); m[a] -= 1
                        bn = self.at(Ustate["b" + "xyz"[a]], p)
                        F[(a, i, j, k)] = orc.hlld(self.g, self.W(Ustate, m, a), self.W(Ustate, p, a), bn)

        def eref(p, c):                                                   # Eq. 18
            _, v, _, B = self.prim(Ustate, p)
            a, b = (c + 1) % 3, (c + 2) % 3
            return -(v[a] * B[b] - v[b] * B[a])

        E = {}     # (c, i, j, k) -> E_c on the edge at the lower (a, b) corner of cell (i, j, k)
        for c in range(3):
            a, b = (c + 1) % 3, (c + 2) % 3
            for k in range(lo[2], hi[2] + 1):
                for j in range(lo[1], hi[1] + 1):
                    for i in range(lo[0], hi[0] + 1):
                        p = [i, j, k]
                        pa = list(p); pa[a] -= 1
                        pb = list(p); pb[b] -= 1
                        pab = list(pa); pab[b] -= 1
                        fa0, fa1 = F[(a, *p)], F[(a, *pb)]
                        fb0, fb1 = F[(b, *p)], F[(b, *pa)]
                        # Table 1: on an a-face E_c = -F_a[B_t1], on a b-face
                        # E_c = +F_b[B_t2]
                        E[(c, i, j, k)] = orc.ct_edge(-fa0[5], -fa1[5], fb0[6], fb1[6], fa0[0], fa1[0],
                                                      fb0[0], fb1[0], eref(p, c), eref(pa, c), eref(pb, c),
                                                      eref(pab, c))
        new = {}
        names = ("rho", "mx", "my", "mz", "E")
        for k in range(lo[2], hi[2]):
            for j in range(lo[1], hi[1]):
                for i in range(lo[0], hi[0]):
                    p = [i, j, k]
                    u = [self.at(Ubase[f], p) for f in names]
                    for a in range(3):                                    # Eq. 19 / 29: x, y, z
                        up = list(p); up[a] += 1
                        fl, fu = F[(a, *p)], F[(a, *up)]
                        c = dt / d[a]
                        u[0] -= c * (fu[0] - fl[0])
                        u[1 + a] -= c * (fu[1] - fl[1])
                        u[1 + (a + 1) % 3] -= c * (fu[2] - fl[2])
                        u[1 + (a + 2) % 3] -= c * (fu[3] - fl[3])
                        u[4] -= c * (fu[4] - fl[4])
                    for f, val in zip(names, u):
                        new[(f, i, j, k)] = val
        for a in range(3):                                                # Eq. 20-22 / 30-32
            b, c = (a + 1) % 3, (a + 2) % 3
            f = "b" + "xyz"[a]
            hi_f = list(hi); hi_f[a] += 1
            for k in range(lo[2], hi_f[2]):
                for j in range(lo[1], hi_f[1]):
                    for i in range(lo[0], hi_f[0]):
                        p = [i, j, k]
                        pc = list(p); pc[c] += 1
                        pb = list(p); pb[b] += 1
                        new[(f, i, j, k)] = (self.at(Ubase[f], p)
                                             + dt / d[c] * (E[(b, *pc)] - E[(b, *p)])
                                             - dt / d[b] * (E[(c, *pb)] - E[(c, *p)]))
        return new

    def step(self, U, dt):
        """One step from ghost-extended U^n; returns (half state on [-1, n+1), new state on [0, n))."""
        n = self.n
        half = self.stage(U, U, 0.5 * dt, [-1, -1, -1], [n[0] + 1, n[1] + 1, n[2] + 1])
        Uh = {f: np.full_like(U[f], np.nan) for f in FIELDS}
        for (f, i, j, k), v in half.items():
            Uh[f][k + NG, j + NG, i + NG] = v
        full = self.stage(U, Uh, dt, [0, 0, 0], list(n))
        return half, full


def gather(d, state_like, n):
    out = {f: np.empty_like(state_like[f]) for f in FIELDS}
    for f in FIELDS:
        nz, ny, nx = out[f].shape
        for k in range(nz):
            for j in range(ny):
                for i in range(nx):
                    out[f][k, j, i] = d[(f, i, j, k)]
    return out


CASES = [((1, 0, 0), (5, 4, 3)), ((0, 1, 0), (4, 5, 3)), ((0, 0, 1), (3, 4, 5)),
         ((1, 1, 1), (4, 3, 5)), ((0, 0, 0), (4, 3, 4))]


@pytest.mark.parametrize("bc,n", CASES)
def test_pcm_step_restated_in_python_with_numpy_pad_ghosts(bc, n):
    # a generic non-uniform state (values differ in every cell next to every boundary)
    p = inputs.random_smooth(n=n, seed=11, recon=0)
    o = orc.Oracle(*n, p.gamma, 0, bc)
    o.set_state(p.state)
    # the fill leaves every active cell and every active face 0..n of the input as it was
    back = o.get_state()
    if all(b == 1 for b in bc):
        for f in FIELDS:
            assert np.array_equal(back[f], p.state[f]), f
    dt = 0.3 * o.compute_dt(0.4)
    o.step(dt)
    mini = Mini(n, p.gamma)
    half, full = mini.step(extend(p.state, n, bc), dt)
    want_half, want_full = gather(half, p.state, n), gather(full, p.state, n)
    got_half, got_full = o.get_half_state(), o.get_state()
    for f in FIELDS:
        np.testing.assert_allclose(got_half[f], want_half[f], rtol=0, atol=2e-15, err_msg="half " + f)
        np.testing.assert_allclose(got_full[f], want_full[f], rtol=0, atol=4e-15, err_msg="full " + f)
    o.close()


def test_outflow_ghosts_are_nearest_active_cell_and_face_not_a_neighbour_of_it():
    """The comparison above must be able to tell the readings apart: with the ghost layers built by
    the two nearest wrong rules ("copy cell n-2" / "face n-1", i.e. reflect-type padding) the
    restated step moves away from the oracle by far more than round-off in the boundary cells."""
    n, bc = (5, 4, 3), (1, 0, 0)
    p = inputs.random_smooth(n=n, seed=11, recon=0)
    o = orc.Oracle(*n, p.gamma, 0, bc)
    o.set_state(p.state)
    dt = 0.3 * o.compute_dt(0.4)
    o.step(dt)
    got = o.get_state()
    U = extend(p.state, n, bc)
    for f in FIELDS:                        # wrong rule: ghost layer l copies the l-th cell inside
        a = U[f]
        last = a.shape[2] - NG - 1          # last active index along x (cell n-1, or face n for bx)
        for l in range(1, NG + 1):
            a[:, :, NG - l] = a[:, :, NG + l]
            a[:, :, last + l] = a[:, :, last - l]
    _, full = Mini(n, p.gamma).step(U, dt)
    want = gather(full, p.state, n)
    assert np.max(np.abs(got["rho"][:, :, -1] - want["rho"][:, :, -1])) > 1e-6
    assert np.max(np.abs(got["rho"][:, :, 0] - want["rho"][:, :, 0])) > 1e-6
    assert np.max(np.abs(got["bx"][:, :, -1] - want["bx"][:, :, -1])) > 1e-8
    o.close()
