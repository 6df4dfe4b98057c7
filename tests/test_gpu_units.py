"""GPU unit parity: the device functions of csrc/mhd_device.cuh, through the mhd_unit_* entry
points of the C ABI, against the oracle's building blocks on the same seeded inputs.  These reach
branches a whole-grid step only visits by luck: every HLLD branch, B_x = 0, B_perp = 0,
supersonic faces, mirror-image states, plateaus next to jumps.
"""
import numpy as np
import pytest

import oracle as orc

pytestmark = pytest.mark.gpu

G = 5.0 / 3.0


@pytest.fixture(scope="module")
def mhd():
    from paper_2402_05240_b200 import mhd as m
    return m


def ulps(a, b):
    """|a - b| in units of the spacing of b."""
    return np.abs(a - b) / np.spacing(np.abs(b))


def test_math_rcp_rsqrt_sqrt_within_two_ulp(mhd):
    """csrc/mhd_math.cuh (hardware seed + one cubically convergent step) against IEEE division / sqrt."""
    rng = np.random.default_rng(11)
    x = 10.0 ** rng.uniform(-30, 30, size=200000)
    x[:5] = [1.0, 2.0, 0.5, 3.0, 1e-200]
    assert ulps(mhd.unit_math(0, x), 1.0 / x).max() <= 2.0
    assert ulps(mhd.unit_math(1, x), 1.0 / np.sqrt(x)).max() <= 2.5   # the numpy value is itself rounded twice
    assert ulps(mhd.unit_math(2, x), np.sqrt(x)).max() <= 1.0
    assert mhd.unit_math(2, np.array([0.0, 4.0, 9.0])).tolist() == [0.0, 2.0, 3.0]
    neg = -x[:1000]
    assert ulps(mhd.unit_math(0, neg), 1.0 / neg).max() <= 2.0


def rand_states(rng, n, vscale=1.0, bscale=1.0):
    W = np.empty((n, 7))
    W[:, 0] = rng.uniform(0.2, 3.0, n)
    W[:, 1:4] = rng.normal(size=(n, 3)) * vscale
    W[:, 4] = rng.uniform(0.05, 3.0, n)
    W[:, 5:7] = rng.normal(size=(n, 2)) * bscale
    return W


def hlld_cases():
    rng = np.random.default_rng(5)
    WL, WR, bx = [], [], []
    for vs, bs, n in ((1.0, 1.0, 3000), (4.0, 0.3, 1500), (0.1, 2.0, 1500), (1.0, 0.0, 300)):
        WL.append(rand_states(rng, n, vs, bs)); WR.append(rand_states(rng, n, vs, bs))
        bx.append(rng.normal(size=n) * bs)
    # a hot state overrunning a cold one, both moving faster than their own fast speed: the regime in which
    # the two outer-speed estimates of Miyoshi & Kusano differ (reading G15, tests/test_oracle_units.py)
    n = 1000
    hot, cold = rand_states(rng, n, 0.3, 0.5), rand_states(rng, n, 0.3, 0.5)
    hot[:, 4] = rng.uniform(4.0, 20.0, n); cold[:, 4] = rng.uniform(0.05, 0.5, n)
    drift = rng.uniform(1.5, 6.0, n) * rng.choice([-1.0, 1.0], n)
    hot[:, 1] += drift; cold[:, 1] += drift
    swap = rng.uniform(size=n) < 0.5
    WL.append(np.where(swap[:, None], hot, cold)); WR.append(np.where(swap[:, None], cold, hot))
    bx.append(rng.normal(size=n) * 0.5)
    WL, WR, bx = np.concatenate(WL), np.concatenate(WR), np.concatenate(bx)
    bx[::7] = 0.0                       # B_x = 0: no double-star region
    WR[5::11] = WL[5::11]               # identical states: F(U,U) = F(U)
    k = slice(3, None, 13)              # degenerate star states: B_perp = 0 on both sides
    WL[k, 5:7] = 0.0; WR[k, 5:7] = 0.0
    return WL, WR, bx


def test_hlld_all_branches(mhd):
    WL, WR, bx = hlld_cases()
    F = mhd.unit_hlld(G, WL, WR, bx)
    ref = np.array([orc.hlld(G, WL[i], WR[i], bx[i]) for i in range(len(bx))])
    scale = np.maximum(np.abs(ref).max(axis=1, keepdims=True), 1.0)
    assert np.all(np.isfinite(F))
    assert (np.abs(F - ref) / scale).max() <= 1e-12


def test_hlld_exactly_degenerate_rotational_discontinuity(mhd):
    """The state of tests/test_oracle_units.py::test_hlld_degenerate_star_state, (a): gamma = 3/2, every
    intermediate exact, D = 0.0 -- the 0/0 of the star state -- and its neighbours B_perp = 1e-14 ... 1e-3."""
    WL = np.array([[1.0, 0.25, 0.5, -0.25, 0.5, 0.0, 0.0]])
    WR = np.array([[1.0, 0.25, -0.5, 0.75, 0.5, 0.0, 0.0]])
    F = mhd.unit_hlld(1.5, WL, WR, np.array([2.0]))[0]
    ref = orc.hlld(1.5, WL[0], WR[0], 2.0)
    assert np.all(np.isfinite(F)) and np.abs(F - ref).max() <= 1e-15
    deltas = 10.0 ** np.arange(-14.0, -2.5, 0.5)
    L = np.repeat(WL, len(deltas), axis=0); R = np.repeat(WR, len(deltas), axis=0)
    L[:, 5] = deltas; L[:, 6] = -0.5 * deltas; R[:, 5] = 0.3 * deltas; R[:, 6] = deltas
    Fd = mhd.unit_hlld(1.5, L, R, np.full(len(deltas), 2.0))
    refd = np.array([orc.hlld(1.5, L[i], R[i], 2.0) for i in range(len(deltas))])
    assert np.all(np.isfinite(Fd)) and np.abs(Fd - refd).max() <= 1e-12


def test_hlld_mass_flux_is_exactly_zero_between_mirror_states(mhd):
    """Reading R6 (Eq. 16 'otherwise' branch): mirror-image states at rest or colliding give an
    exactly zero mass flux on both sides, whatever the round-off of S_M."""
    rng = np.random.default_rng(6)
    n = 2000
    WL = rand_states(rng, n)
    bx = rng.normal(size=n)
    # reflection in the face: u -> -u, B_t -> -B_t (B is a pseudo-vector), B_x unchanged
    WR1 = WL.copy(); WR1[:, 1] = -WL[:, 1]; WR1[:, 5:7] = -WL[:, 5:7]
    # the blast's diagonal symmetry: u -> -u, (v, w) -> (-w, -v), (B_y, B_z) -> (B_z, B_y)
    WR2 = WL.copy(); WR2[:, 1] = -WL[:, 1]
    WR2[:, 2] = -WL[:, 3]; WR2[:, 3] = -WL[:, 2]; WR2[:, 5] = WL[:, 6]; WR2[:, 6] = WL[:, 5]
    for WR in (WR1, WR2):
        F = mhd.unit_hlld(G, WL, WR, bx)
        ref = np.array([orc.hlld(G, WL[i], WR[i], bx[i]) for i in range(n)])
        assert np.all(ref[:, 0] == 0.0)
        assert np.all(F[:, 0] == 0.0)
    rest = WL * [1, 0, 1, 1, 1, 1, 1]   # identical states with u = 0
    assert np.all(mhd.unit_hlld(G, rest, rest, bx)[:, 0] == 0.0)


def stencils(rng, n, R):
    base = rand_states(rng, n, 0.5, 1.0)
    Ws = np.repeat(base[:, None, :], 2 * R + 1, axis=1)
    Ws += 0.2 * rng.normal(size=Ws.shape) * np.array([0.3, 1, 1, 1, 0.1, 1, 1])
    Ws[:, :, 0] = np.abs(Ws[:, :, 0]) + 0.1
    Ws[:, :, 4] = np.abs(Ws[:, :, 4]) + 0.05
    bn = rng.normal(size=n)
    # special structure
    Ws[0::9, :, :] = Ws[0::9, R:R + 1, :]                  # exactly uniform stencil
    Ws[1::9, R + 1:, :] = Ws[1::9, R:R + 1, :]             # plateau on the upper side, jump below
    Ws[2::9, :R, :] = Ws[2::9, R:R + 1, :]                 # plateau on the lower side
    Ws[3::9, :, 5:7] = 0.0                                 # B_perp = 0 everywhere (G16)
    bn[4::9] = 0.0                                         # B_n = 0
    Ws[5::9, R, 5:7] = 0.0                                 # B_perp = 0 in the middle cell only
    Ws[6::9] = Ws[6::9, ::-1][:, :, :].copy()              # reversed order (other monotonic sense)
    return Ws, bn


@pytest.mark.parametrize("recon", [1, 2, 3, 4])
def test_reconstruction_against_oracle(mhd, recon):
    rng = np.random.default_rng(20 + recon)
    n = 4000
    R = 1 if recon in (1, 3) else 2
    Ws, bn = stencils(rng, n, R)
    lo, hi = mhd.unit_reconstruct(G, recon, Ws, bn)
    rlo, rhi = np.empty((n, 7)), np.empty((n, 7))
    for i in range(n):
        if recon == 1:
            rlo[i], rhi[i] = orc.plmc(G, Ws[i, 0], Ws[i, 1], Ws[i, 2], bn[i])
        elif recon == 2:
            rlo[i], rhi[i] = orc.ppmc(G, Ws[i], bn[i])
        elif recon == 3:
            rlo[i], rhi[i] = orc.plmp(Ws[i, 0], Ws[i, 1], Ws[i, 2])
        else:
            rlo[i], rhi[i] = orc.ppmp(Ws[i])
    scale = np.maximum(np.abs(Ws).max(axis=(1, 2))[:, None], 1.0)
    assert np.all(np.isfinite(lo)) and np.all(np.isfinite(hi))
    err = np.maximum(np.abs(lo - rlo), np.abs(hi - rhi)) / scale
    kind = np.arange(n) % 9
    worst = {int(k): float(err[kind == k].max()) for k in range(9)}
    # kinds 3, 5: B_perp = 0 exactly in the cell whose eigenvectors are used.  alpha_s (or alpha_f) is
    # then the square root of a round-off difference, ~1e-8 instead of 0 ("A.R
    # residual up to ~1e-8 only when B_perp = 0 exactly"), in the oracle as in the kernels, and the
    # per-wave limiter turns that into an O(1e-8) difference between any two implementations.
    for k, w in worst.items():
        assert w <= (1e-7 if (k in (3, 5) and recon <= 2) else 1e-12), worst
    # a uniform stencil is returned bit for bit on both faces up to the round trip R.(L.W)
    u = slice(0, None, 9)
    assert np.abs(lo[u] - Ws[u, R]).max() <= 1e-14 and np.abs(hi[u] - Ws[u, R]).max() <= 1e-14


def test_ct_edge_against_oracle(mhd):
    rng = np.random.default_rng(31)
    n = 5000
    x = rng.normal(size=(n, 12))
    x[::3, 4:8] = np.where(rng.random((len(x[::3]), 4)) < 0.5, 0.0, x[::3, 4:8])   # exactly zero mass fluxes
    out = mhd.unit_ct_edge(x)
    ref = np.array([orc.ct_edge(*x[i]) for i in range(n)])
    assert np.abs(out - ref).max() <= 1e-15 * 8
