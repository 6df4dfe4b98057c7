"""Seeded synthetic input generators (numpy only, host arrays).

This module defines the *problems* (initial conditions), not the method: it holds
none of the VL+CT arithmetic and imports neither the CUDA binding nor the oracle.
Tests and bench.py hand the same arrays to both.

Array convention (the C ABI's, include/mhd.h): a state is a dict of 8 float64 arrays
indexed [k, j, i] (i fastest): rho, mx, my, mz, E of shape (nz, ny, nx); bx of shape
(nz, ny, nx+1), by (nz, ny+1, nx), bz (nz+1, ny, nx); face index f is the lower face of
cell f (Eq. 20).  Unit box, Delta_a = 1/n_a.

Recipes (DESIGN.md section "Inputs"):
  linear_wave  -- PAPER.md:333-339 (Eq. 33), eigenvectors per SURVEY.md G19
  riemann      -- PAPER.md:407-429 (Table 2); 'brio_wu' is BASELINE.json configs[1]
  turbulence   -- BASELINE.json configs[2], [4]; stand-in for the paper's turbulent-box
                  motivation, not a paper test
  blast        -- BASELINE.json configs[3]; variant of PAPER.md:455-459
  random_smooth-- small seeded smooth field for parity tests (div B = 0 by construction)
  cpaw         -- circularly polarised Alfven wave, PAPER.md:358-370
  field_loop   -- advecting field loop, PAPER.md:378-391 (Eq. 36)
  orszag_tang  -- PAPER.md:467-475
  blast_paper  -- MHD blast in the paper's own box, PAPER.md:455-459
"""
from dataclasses import dataclass, field

import numpy as np

FIELDS = ("rho", "mx", "my", "mz", "E", "bx", "by", "bz")


@dataclass
class Problem:
    name: str
    n: tuple            # (nx, ny, nz)
    gamma: float
    state: dict
    bc: tuple = (0, 0, 0)   # per axis: 0 periodic, 1 outflow
    recon: int = 1          # 1 PLMC, 2 PPMC
    cfl: float = 0.4
    t_end: float = None
    n_steps: int = None
    meta: dict = field(default_factory=dict)
    domain: tuple = (1.0, 1.0, 1.0)   # box lengths; Delta_a = L_a / n_a


def field_shapes(nx, ny, nz):
    s = {f: (nz, ny, nx) for f in FIELDS[:5]}
    s["bx"] = (nz, ny, nx + 1)
    s["by"] = (nz, ny + 1, nx)
    s["bz"] = (nz + 1, ny, nx)
    return s


def cell_centred_b(state):
    """Arithmetic mean of the two opposing faces (used only to define E of an input)."""
    bx, by, bz = state["bx"], state["by"], state["bz"]
    return (0.5 * (bx[:, :, :-1] + bx[:, :, 1:]),
            0.5 * (by[:, :-1, :] + by[:, 1:, :]),
            0.5 * (bz[:-1, :, :] + bz[1:, :, :]))


def from_primitives(rho, vx, vy, vz, P, bx, by, bz, gamma):
    """Conserved input state from cell-centred rho, v, P and face-centred B."""
    st = {"bx": np.ascontiguousarray(bx, dtype=np.float64),
          "by": np.ascontiguousarray(by, dtype=np.float64),
          "bz": np.ascontiguousarray(bz, dtype=np.float64)}
    bcx, bcy, bcz = cell_centred_b(st)
    st["rho"] = np.ascontiguousarray(rho, dtype=np.float64)
    st["mx"] = st["rho"] * vx
    st["my"] = st["rho"] * vy
    st["mz"] = st["rho"] * vz
    st["E"] = (P / (gamma - 1.0) + 0.5 * st["rho"] * (vx * vx + vy * vy + vz * vz)
               + 0.5 * (bcx * bcx + bcy * bcy + bcz * bcz))
    return st


def _to_axis(arr_local_kji, axis):
    """A field varying along local x (last numpy axis) re-oriented so that it varies
    along global `axis` (0=x,1=y,2=z).  Cyclic: local (x,y,z) -> global (a,a+1,a+2)."""
    # local numpy axes (z,y,x) hold local coords (2,1,0); global coordinate of local c
    # is (c+axis)%3; numpy axis of global coord g is 2-g.
    src = [2, 1, 0]                       # numpy axis -> local coord
    dst_axes = [2 - ((c + axis) % 3) for c in src]
    return np.ascontiguousarray(np.moveaxis(arr_local_kji, [0, 1, 2], dst_axes))


# ------------------------------------------------------------------------------
# C1: linear waves (Eq. 33)
# ------------------------------------------------------------------------------
_SQ5 = np.sqrt(5.0)
# right-going eigenvectors in conserved variables (rho, m_n, m_t1, m_t2, E, B_n, B_t1, B_t2)
# for rho=1, P=1/gamma, B=(1,1.5,0), gamma=5/3; speed c
_WAVES = {
    "fast": (np.array([2.0, 4.0, -2.0, 0.0, 9.0, 0.0, 4.0, 0.0]) / (2.0 * _SQ5), 2.0),
    "alfven": (np.array([0.0, 0.0, 0.0, -1.0, 0.0, 0.0, 0.0, 1.0]), 1.0),
    "slow": (np.array([4.0, 2.0, 4.0, 0.0, 3.0, 0.0, -2.0, 0.0]) / (2.0 * _SQ5), 0.5),
}


def linear_wave(nx=32, ny=32, nz=32, wave="fast", axis=0, direction=+1,
                amplitude=1e-6, recon=1):
    gamma = 5.0 / 3.0
    R, c = _WAVES[wave]
    R = R.copy()
    if direction < 0:
        R[1:4] *= -1.0
    n = (nx, ny, nz)
    na = n[axis]
    # local frame: wave along local x; local grid sizes are the global ones permuted
    nl = [n[(axis + c_) % 3] for c_ in range(3)]   # local (nx', ny', nz')
    xc = (np.arange(na) + 0.5) / na
    s_c = np.sin(2.0 * np.pi * xc)
    rho0, P0 = 1.0, 1.0 / gamma
    B0 = (1.0, 1.5, 0.0)
    E0 = P0 / (gamma - 1.0) + 0.5 * (B0[0] ** 2 + B0[1] ** 2 + B0[2] ** 2)
    ones_c = np.ones((nl[2], nl[1], nl[0]))
    loc = {}
    loc["rho"] = rho0 + amplitude * R[0] * s_c * ones_c
    loc["mn"] = amplitude * R[1] * s_c * ones_c
    loc["mt1"] = amplitude * R[2] * s_c * ones_c
    loc["mt2"] = amplitude * R[3] * s_c * ones_c
    loc["E"] = E0 + amplitude * R[4] * s_c * ones_c
    # faces: B_n on n-faces (x = f/na) is uniform; B_t1 on t1-faces and B_t2 on t2-faces sit at
    # cell-centre positions along the wave axis
    loc["bn"] = B0[0] * np.ones((nl[2], nl[1], nl[0] + 1))
    loc["bt1"] = (B0[1] + amplitude * R[6] * s_c) * np.ones((nl[2], nl[1] + 1, nl[0]))
    loc["bt2"] = (B0[2] + amplitude * R[7] * s_c) * np.ones((nl[2] + 1, nl[1], nl[0]))
    mom = ["mx", "my", "mz"]
    bb = ["bx", "by", "bz"]
    st = {"rho": _to_axis(loc["rho"], axis), "E": _to_axis(loc["E"], axis)}
    for c_, key in enumerate(["mn", "mt1", "mt2"]):
        st[mom[(axis + c_) % 3]] = _to_axis(loc[key], axis)
    for c_, key in enumerate(["bn", "bt1", "bt2"]):
        st[bb[(axis + c_) % 3]] = _to_axis(loc[key], axis)
    sh = field_shapes(nx, ny, nz)
    for f in FIELDS:
        assert st[f].shape == sh[f], (f, st[f].shape, sh[f])
    return Problem(name="linear_%s" % wave, n=n, gamma=gamma, state=st, recon=recon,
                   cfl=0.4, t_end=1.0 / c,
                   meta={"axis": axis, "direction": direction, "speed": c})


def wave_error(initial, final):
    """Eq. 34-35: L2 norm of the per-field L1 errors."""
    e = [np.mean(np.abs(_active(final[f], f) - _active(initial[f], f))) for f in FIELDS]
    return float(np.sqrt(np.sum(np.square(e))))


def _active(a, f):
    """Drop the duplicated upper face so that every field has nx*ny*nz values."""
    if f == "bx":
        return a[:, :, :-1]
    if f == "by":
        return a[:, :-1, :]
    if f == "bz":
        return a[:-1, :, :]
    return a


# ------------------------------------------------------------------------------
# C2 and Table 2: planar Riemann problems
# ------------------------------------------------------------------------------
_S4PI = np.sqrt(4.0 * np.pi)
# gamma, t_max, Bx, (rho, P, vx, vy, vz, By, Bz)_L, (...)_R  -- PAPER.md:409-423 (Table 2)
RIEMANN = {
    "brio_wu": (2.0, 0.1, 0.75, (1.0, 1.0, 0, 0, 0, 1.0, 0), (0.125, 0.1, 0, 0, 0, -1.0, 0)),
    "dai_woodward": (5.0 / 3.0, 0.2, 2 / _S4PI,
                     (1.08, 0.95, 1.2, 0.01, 0.5, 3.6 / _S4PI, 2 / _S4PI),
                     (1.0, 1.0, 0, 0, 0, 4 / _S4PI, 2 / _S4PI)),
    "ryu_jones_1a": (5.0 / 3.0, 0.08, 5 / _S4PI, (1.0, 20.0, 10.0, 0, 0, 5 / _S4PI, 0),
                     (1.0, 1.0, -10.0, 0, 0, 5 / _S4PI, 0)),
    "ryu_jones_4d": (5.0 / 3.0, 0.16, 0.7, (1.0, 1.0, 0, 0, 0, 0, 0), (0.3, 0.2, 0, 0, 1.0, 1.0, 0)),
    "einfeldt": (1.4, 0.16, 0.0, (1.0, 0.45, -2.0, 0, 0, 0.5, 0), (1.0, 0.45, 2.0, 0, 0, 0.5, 0)),
}


def riemann(name="brio_wu", n_long=256, n_trans=16, axis=0, recon=1, flip=False):
    """Planar Riemann problem split at 0.5 along `axis`; outflow along it, periodic across.
    flip=True mirrors the problem (left<->right, normal velocity and B_n sign reversed)."""
    gamma, t_max, bn, SL, SR = RIEMANN[name]
    if flip:
        SL, SR = SR, SL
        SL = (SL[0], SL[1], -SL[2]) + tuple(SL[3:])
        SR = (SR[0], SR[1], -SR[2]) + tuple(SR[3:])
        bn = -bn
    nl = [n_long, n_trans, n_trans]
    xc = (np.arange(n_long) + 0.5) / n_long
    left = xc < 0.5

    def prof(iq):
        return np.where(left, SL[iq], SR[iq])

    ones_c = np.ones((nl[2], nl[1], nl[0]))
    rho = prof(0) * ones_c
    P = prof(1) * ones_c
    vn, vt1, vt2 = prof(2) * ones_c, prof(3) * ones_c, prof(4) * ones_c
    b_n = bn * np.ones((nl[2], nl[1], nl[0] + 1))
    b_t1 = prof(5) * np.ones((nl[2], nl[1] + 1, nl[0]))
    b_t2 = prof(6) * np.ones((nl[2] + 1, nl[1], nl[0]))
    E = (P / (gamma - 1.0) + 0.5 * rho * (vn ** 2 + vt1 ** 2 + vt2 ** 2)
         + 0.5 * (bn ** 2 + (prof(5) ** 2 + prof(6) ** 2) * ones_c))
    mom = ["mx", "my", "mz"]
    bb = ["bx", "by", "bz"]
    st = {"rho": _to_axis(rho, axis), "E": _to_axis(E, axis)}
    for c_, arr in enumerate([rho * vn, rho * vt1, rho * vt2]):
        st[mom[(axis + c_) % 3]] = _to_axis(arr, axis)
    for c_, arr in enumerate([b_n, b_t1, b_t2]):
        st[bb[(axis + c_) % 3]] = _to_axis(arr, axis)
    n = [0, 0, 0]
    for c_ in range(3):
        n[(axis + c_) % 3] = nl[c_]
    bc = [0, 0, 0]
    bc[axis] = 1
    return Problem(name=name, n=tuple(n), gamma=gamma, state=st, bc=tuple(bc), recon=recon,
                   cfl=0.4, t_end=t_max, meta={"axis": axis, "flip": flip})


# ------------------------------------------------------------------------------
# C3 / C5: seeded turbulent velocity + random vector potential
# ------------------------------------------------------------------------------
def _mode_table(rng, kmax, p):
    """Half-space integer modes 1 <= |k| <= kmax in lexicographic (kx, ky, kz) order with
    g_k ~ N(0,1) |k|^-p and phase ~ U[0, 2pi)."""
    ks, amp, ph = [], [], []
    for kx in range(-kmax, kmax + 1):
        for ky in range(-kmax, kmax + 1):
            for kz in range(-kmax, kmax + 1):
                k2 = kx * kx + ky * ky + kz * kz
                if k2 < 1 or k2 > kmax * kmax:
                    continue
                # half space: first non-zero of (kx, ky, kz) positive
                lead = kx if kx != 0 else (ky if ky != 0 else kz)
                if lead < 0:
                    continue
                g = rng.standard_normal()
                phi = rng.uniform(0.0, 2.0 * np.pi)
                ks.append((kx, ky, kz))
                amp.append(g * k2 ** (-0.5 * p))
                ph.append(phi)
    return np.array(ks), np.array(amp), np.array(ph)


def _synthesise(modes, n, off):
    """f(x) = sum_k A_k cos(2 pi k.x + phi_k) at x_a = (i_a + off_a)/n_a, returned [k,j,i].
    Separable evaluation (exact, no FFT): only |k| <= kmax modes exist."""
    ks, amp, ph = modes
    kmax = int(np.abs(ks).max())
    nk = 2 * kmax + 1
    c = np.zeros((nk, nk, nk), dtype=np.complex128)      # [kz, ky, kx]
    c[ks[:, 2] + kmax, ks[:, 1] + kmax, ks[:, 0] + kmax] = amp * np.exp(1j * ph)
    kk = np.arange(-kmax, kmax + 1)
    ex = np.exp(2j * np.pi * np.outer(kk, (np.arange(n[0]) + off[0]) / n[0]))   # [kx, i]
    ey = np.exp(2j * np.pi * np.outer(kk, (np.arange(n[1]) + off[1]) / n[1]))   # [ky, j]
    ez = np.exp(2j * np.pi * np.outer(kk, (np.arange(n[2]) + off[2]) / n[2]))   # [kz, k]
    t1 = c @ ex                                           # [kz, ky, i]
    t2 = np.einsum("yj,zyi->zji", ey, t1)                 # [kz, j, i]
    t2 = t2.reshape(nk, n[1] * n[0])
    out = ez.real.T @ t2.real - ez.imag.T @ t2.imag       # [k, j*i]
    return out.reshape(n[2], n[1], n[0])


def turbulence(n=256, seed=20240207, gamma=5.0 / 3.0, mach=1.0, beta=1.0, kmax=8, n_steps=10,
               recon=1):
    if np.isscalar(n):
        n = (n, n, n)
    nx, ny, nz = n
    rho0, P0 = 1.0, 1.0
    ss = np.random.SeedSequence(seed)
    streams = [np.random.default_rng(s) for s in ss.spawn(6)]
    v = []
    for c_ in range(3):
        modes = _mode_table(streams[c_], kmax, 2.0)
        v.append(_synthesise(modes, n, (0.5, 0.5, 0.5)))
    vrms = np.sqrt(np.mean(v[0] ** 2 + v[1] ** 2 + v[2] ** 2))
    scale = mach * np.sqrt(gamma * P0 / rho0) / vrms
    v = [a * scale for a in v]
    # vector potential on edges: A_x at (i+1/2, j, k) [x-centre, lower y, lower z] etc.
    offs = [(0.5, 0.0, 0.0), (0.0, 0.5, 0.0), (0.0, 0.0, 0.5)]
    A = [_synthesise(_mode_table(streams[3 + c_], kmax, 3.0), n, offs[c_]) for c_ in range(3)]
    dx, dy, dz = 1.0 / nx, 1.0 / ny, 1.0 / nz

    def d(a, ax, h):  # forward difference along numpy axis ax (periodic)
        return (np.roll(a, -1, axis=ax) - a) / h

    # B = curl A on lower faces: Bx(i-1/2,j,k) = dAz/dy - dAy/dz, ...
    bx = d(A[2], 1, dy) - d(A[1], 0, dz)
    by = d(A[0], 0, dz) - d(A[2], 2, dx)
    bz = d(A[1], 2, dx) - d(A[0], 1, dy)
    del A
    bcx = 0.5 * (bx + np.roll(bx, -1, axis=2))
    bcy = 0.5 * (by + np.roll(by, -1, axis=1))
    bcz = 0.5 * (bz + np.roll(bz, -1, axis=0))
    b2 = np.mean(bcx ** 2 + bcy ** 2 + bcz ** 2)
    del bcx, bcy, bcz
    bs = np.sqrt((2.0 * P0 / beta) / b2)
    bx = np.concatenate([bx, bx[:, :, :1]], axis=2) * bs
    by = np.concatenate([by, by[:, :1, :]], axis=1) * bs
    bz = np.concatenate([bz, bz[:1, :, :]], axis=0) * bs
    rho = np.full((nz, ny, nx), rho0)
    P = np.full((nz, ny, nx), P0)
    st = from_primitives(rho, v[0], v[1], v[2], P, bx, by, bz, gamma)
    return Problem(name="turbulence", n=tuple(n), gamma=gamma, state=st, recon=recon, cfl=0.4,
                   n_steps=n_steps, meta={"seed": seed, "mach": mach, "beta": beta, "kmax": kmax})


# ------------------------------------------------------------------------------
# C4: blast (variant of PAPER.md:455-459)
# ------------------------------------------------------------------------------
def blast(n=512, gamma=5.0 / 3.0, recon=2, n_steps=20, p_in=10.0, p_out=0.1, radius=0.1):
    if np.isscalar(n):
        n = (n, n, n)
    nx, ny, nz = n
    x = (np.arange(nx) + 0.5) / nx - 0.5
    y = (np.arange(ny) + 0.5) / ny - 0.5
    z = (np.arange(nz) + 0.5) / nz - 0.5
    r2 = z[:, None, None] ** 2 + y[None, :, None] ** 2 + x[None, None, :] ** 2
    P = np.where(r2 < radius * radius, p_in, p_out)
    b0 = 1.0 / np.sqrt(3.0)
    sh = field_shapes(nx, ny, nz)
    zero = np.zeros((nz, ny, nx))
    st = from_primitives(np.ones((nz, ny, nx)), zero, zero, zero, P,
                         np.full(sh["bx"], b0), np.full(sh["by"], b0), np.full(sh["bz"], b0), gamma)
    return Problem(name="blast", n=tuple(n), gamma=gamma, state=st, recon=recon, cfl=0.4,
                   n_steps=n_steps, meta={"p_in": p_in, "p_out": p_out, "radius": radius})


# ------------------------------------------------------------------------------
# small generic parity case
# ------------------------------------------------------------------------------
def random_smooth(n=(16, 16, 16), seed=1, gamma=5.0 / 3.0, recon=1, amp=0.3, kmax=2):
    """Order-one smooth random field (positive rho and P, div B = 0 from a vector potential)."""
    if np.isscalar(n):
        n = (n, n, n)
    nx, ny, nz = n
    ss = np.random.SeedSequence(seed)
    st_ = [np.random.default_rng(s) for s in ss.spawn(8)]

    def fld(rng, off, p=1.0):
        f = _synthesise(_mode_table(rng, kmax, p), n, off)
        return f / np.max(np.abs(f))

    cc = (0.5, 0.5, 0.5)
    rho = 1.0 + amp * fld(st_[0], cc)
    P = 1.0 + amp * fld(st_[1], cc)
    v = [0.7 * fld(st_[2 + c_], cc) for c_ in range(3)]
    offs = [(0.5, 0.0, 0.0), (0.0, 0.5, 0.0), (0.0, 0.0, 0.5)]
    A = [0.15 * fld(st_[5 + c_], offs[c_]) for c_ in range(3)]
    dx, dy, dz = 1.0 / nx, 1.0 / ny, 1.0 / nz

    def d(a, ax, h):
        return (np.roll(a, -1, axis=ax) - a) / h

    bx = 0.6 + d(A[2], 1, dy) - d(A[1], 0, dz)
    by = -0.4 + d(A[0], 0, dz) - d(A[2], 2, dx)
    bz = 0.3 + d(A[1], 2, dx) - d(A[0], 1, dy)
    bx = np.concatenate([bx, bx[:, :, :1]], axis=2)
    by = np.concatenate([by, by[:, :1, :]], axis=1)
    bz = np.concatenate([bz, bz[:1, :, :]], axis=0)
    st = from_primitives(rho, v[0], v[1], v[2], P, bx, by, bz, gamma)
    return Problem(name="random_smooth", n=tuple(n), gamma=gamma, state=st, recon=recon, cfl=0.4,
                   n_steps=1, meta={"seed": seed})


def uniform(n=(8, 8, 8), gamma=5.0 / 3.0, rho=1.3, P=0.7, v=(0.3, -0.2, 0.5), B=(0.4, 0.9, -0.6),
            recon=1):
    nx, ny, nz = n
    sh = field_shapes(nx, ny, nz)
    c = np.ones((nz, ny, nx))
    st = from_primitives(rho * c, v[0] * c, v[1] * c, v[2] * c, P * c, np.full(sh["bx"], B[0]),
                         np.full(sh["by"], B[1]), np.full(sh["bz"], B[2]), gamma)
    return Problem(name="uniform", n=tuple(n), gamma=gamma, state=st, recon=recon, n_steps=1)


# ------------------------------------------------------------------------------
# The rest of the paper's test suite.  B always from a vector potential
# sampled on cell edges and differenced onto faces, so that div B = 0 to round-off
# (PAPER.md:370, 382, 475).
# ------------------------------------------------------------------------------
def _edge_coords(n, L, origin):
    """Cell-centre and lower-face coordinates along each axis."""
    c = [origin[a] + (np.arange(n[a]) + 0.5) * L[a] / n[a] for a in range(3)]
    f = [origin[a] + np.arange(n[a] + 1) * L[a] / n[a] for a in range(3)]
    return c, f


def _curl_to_faces(Ax, Ay, Az, n, L):
    """Ax on x-edges [k-1/2, j-1/2, i] shape (nz+1, ny+1, nx); Ay (nz+1, ny, nx+1); Az (nz, ny+1, nx+1).
    Returns face fields bx (nz, ny, nx+1), by (nz, ny+1, nx), bz (nz+1, ny, nx)."""
    dx, dy, dz = (L[a] / n[a] for a in range(3))
    bx = (Az[:, 1:, :] - Az[:, :-1, :]) / dy - (Ay[1:, :, :] - Ay[:-1, :, :]) / dz
    by = (Ax[1:, :, :] - Ax[:-1, :, :]) / dz - (Az[:, :, 1:] - Az[:, :, :-1]) / dx
    bz = (Ay[:, :, 1:] - Ay[:, :, :-1]) / dx - (Ax[:, 1:, :] - Ax[:, :-1, :]) / dy
    return bx, by, bz


def cpaw(N=16, recon=1, standing=False, amplitude=0.1):
    """Circularly polarised Alfven wave: periodic 3 x 1.5 x 1.5 box, 2N x N x N
    cells, rho = 1, P = 0.1, B_1 = 1, transverse v and B of amplitude 0.1 rotating with phase
    2 pi x_1, x_1 along e_1 = (cos a cos b, cos a sin b, sin a); one period = 1 (Alfven speed 1).
    sin a = 2/3; sin b is read as 2/sqrt(5) (G25: the printed 1/sqrt(5) is not periodic in
    this box), so e_1 = (1/3, 2/3, 2/3)."""
    gamma = 5.0 / 3.0
    n = (2 * N, N, N)
    L = (3.0, 1.5, 1.5)
    sa, sb = 2.0 / 3.0, 2.0 / np.sqrt(5.0)
    ca, cb = np.sqrt(1 - sa * sa), np.sqrt(1 - sb * sb)
    e1 = np.array([ca * cb, ca * sb, sa])
    e2 = np.array([-sb, cb, 0.0])
    e3 = np.array([-sa * cb, -sa * sb, ca])
    c, f = _edge_coords(n, L, (0.0, 0.0, 0.0))

    def x1(X, Y, Z):
        return e1[0] * X + e1[1] * Y + e1[2] * Z

    def grid(zs, ys, xs):
        return np.meshgrid(zs, ys, xs, indexing="ij")

    A = amplitude
    k2 = 2.0 * np.pi

    def potential(Z, Y, X):  # wave part of A in the wave frame: (0, A sin/(2 pi), A cos/(2 pi))
        ph = k2 * x1(X, Y, Z)
        a2, a3 = A * np.sin(ph) / k2, A * np.cos(ph) / k2
        return [a2 * e2[i] + a3 * e3[i] for i in range(3)]

    Ax = potential(*grid(f[2], f[1], c[0]))[0]
    Ay = potential(*grid(f[2], c[1], f[0]))[1]
    Az = potential(*grid(c[2], f[1], f[0]))[2]
    bx, by, bz = _curl_to_faces(Ax, Ay, Az, n, L)
    bx += e1[0]; by += e1[1]; bz += e1[2]     # uniform B_1 = 1 along e_1
    Zc, Yc, Xc = grid(c[2], c[1], c[0])
    ph = k2 * x1(Xc, Yc, Zc)
    v1 = -1.0 if standing else 0.0
    v2, v3 = A * np.sin(ph), A * np.cos(ph)
    v = [v1 * e1[i] + v2 * e2[i] + v3 * e3[i] for i in range(3)]
    rho = np.ones_like(ph)
    st = from_primitives(rho, v[0], v[1], v[2], 0.1 * rho, bx, by, bz, gamma)
    return Problem(name="cpaw", n=n, gamma=gamma, state=st, recon=recon, cfl=0.4, t_end=1.0, domain=L,
                   meta={"standing": standing})


def field_loop(N=32, recon=2, amplitude=1e-3, radius=0.3):
    """Advecting field loop (Eq. 36): periodic 1 x 1 x 2 box centred at zero,
    N x N x 2N cells, rho = 1, P = 1, v = (1, 1, 2); A_x = 0, A_y = A_z = A (R - r) inside r < R = 0.3
    (r from the box centre, each component sampled on its own edges), A = 1e-3; two periods, t = 2."""
    gamma = 5.0 / 3.0
    n = (N, N, 2 * N)
    L = (1.0, 1.0, 2.0)
    c, f = _edge_coords(n, L, (-0.5, -0.5, -1.0))

    def pot(zs, ys, xs):
        Z, Y, X = np.meshgrid(zs, ys, xs, indexing="ij")
        r = np.sqrt(X * X + Y * Y + Z * Z)
        return np.where(r < radius, amplitude * (radius - r), 0.0)

    Ax = np.zeros((n[2] + 1, n[1] + 1, n[0]))
    Ay = pot(f[2], c[1], f[0])
    Az = pot(c[2], f[1], f[0])
    bx, by, bz = _curl_to_faces(Ax, Ay, Az, n, L)
    one = np.ones((n[2], n[1], n[0]))
    st = from_primitives(one, 1.0 * one, 1.0 * one, 2.0 * one, one, bx, by, bz, gamma)
    return Problem(name="field_loop", n=n, gamma=gamma, state=st, recon=recon, cfl=0.4, t_end=2.0, domain=L)


def orszag_tang(N=192, nz=None, recon=2):
    """Orszag-Tang vortex: periodic unit box, rho = 25/(36 pi), P = 5/(12 pi),
    v = (sin 2 pi y, -sin 2 pi x, 0) as printed, A_z = (B0 / 4 pi)(cos 4 pi x + 2 cos 2 pi y),
    B0 = 1/sqrt(4 pi); gamma = 5/3 (not stated in the paper; the standard choice); t = 0.5."""
    gamma = 5.0 / 3.0
    nz = N if nz is None else nz
    n = (N, N, nz)
    L = (1.0, 1.0, 1.0)
    c, f = _edge_coords(n, L, (0.0, 0.0, 0.0))
    B0 = 1.0 / np.sqrt(4.0 * np.pi)
    Zc, Yf, Xf = np.meshgrid(c[2], f[1], f[0], indexing="ij")
    Az = B0 / (4.0 * np.pi) * (np.cos(4 * np.pi * Xf) + 2.0 * np.cos(2 * np.pi * Yf))
    Ax = np.zeros((n[2] + 1, n[1] + 1, n[0]))
    Ay = np.zeros((n[2] + 1, n[1], n[0] + 1))
    bx, by, bz = _curl_to_faces(Ax, Ay, Az, n, L)
    Z, Y, X = np.meshgrid(c[2], c[1], c[0], indexing="ij")
    rho = 25.0 / (36.0 * np.pi) * np.ones_like(X)
    st = from_primitives(rho, np.sin(2 * np.pi * Y), -np.sin(2 * np.pi * X), np.zeros_like(X),
                         5.0 / (12.0 * np.pi) * np.ones_like(X), bx, by, bz, gamma)
    return Problem(name="orszag_tang", n=n, gamma=gamma, state=st, recon=recon, cfl=0.4, t_end=0.5)


def blast_paper(nx=200, recon=2, p_in=10.0, p_out=0.1, radius=0.1):
    """MHD blast wave as the paper runs it: periodic 1 x 1.5 x 1 box, nx x 1.5 nx x nx
    cells (200 x 300 x 200), rho = 1, v = 0, B = (1, 1, 0)/sqrt(2) (beta = 0.2), P = 10 inside the
    central sphere of radius 0.1 and 0.1 outside; t = 0.2."""
    gamma = 5.0 / 3.0
    n = (nx, (3 * nx) // 2, nx)
    L = (1.0, 1.5, 1.0)
    c, f = _edge_coords(n, L, (-0.5, -0.75, -0.5))
    Z, Y, X = np.meshgrid(c[2], c[1], c[0], indexing="ij")
    P = np.where(X * X + Y * Y + Z * Z < radius * radius, p_in, p_out)
    b = 1.0 / np.sqrt(2.0)
    one = np.ones_like(X)
    st = from_primitives(one, 0 * one, 0 * one, 0 * one, P, b * np.ones((n[2], n[1], n[0] + 1)),
                         b * np.ones((n[2], n[1] + 1, n[0])), np.zeros((n[2] + 1, n[1], n[0])), gamma)
    return Problem(name="blast_paper", n=n, gamma=gamma, state=st, recon=recon, cfl=0.4, t_end=0.2, domain=L)
