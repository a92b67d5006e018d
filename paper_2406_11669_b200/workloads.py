"""Seeded synthetic inputs for the five BASELINE.json workloads.

This module serves BOTH the CUDA library and the oracle and therefore holds none of the
method's arithmetic: it only builds input fields (metric, primitives, vector potential,
mask) with numpy from `numpy.random.Generator(PCG64(seed))`, seed = 20240611 + config
index.  The only physics in here is what an initial-data recipe needs (the Kerr-Schild
metric, a plasma-beta normalisation of the seed field).

Array conventions (same as include/grmhd.h): g = 3 ghosts, cell-centred arrays of shape
(nz+6, ny+6, nx+6), staggered arrays (nz+7, ny+7, nx+7), x fastest, lower-edge convention.
No public benchmark data is involved: the paper's tests are analytic initial data
 and BASELINE.json's configs are synthetic by construction.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

G = 3
SEED0 = 20240611

METRIC_NAMES = ["alpha", "betax", "betay", "betaz", "gxx", "gxy", "gxz", "gyy", "gyz", "gzz",
                "kxx", "kxy", "kxz", "kyy", "kyz", "kzz"]
PRIM_NAMES = ["rho", "vx", "vy", "vz", "press", "Bx", "By", "Bz"]


@dataclass
class Workload:
    name: str
    nx: int
    ny: int
    nz: int
    dx: tuple
    opts: dict                      # keyword arguments of grmhd_opts
    metric: list                    # 16 cell-centred arrays
    prims: list                     # 8 cell-centred arrays (B entries may be None)
    vecpot: list | None = None      # 3 staggered arrays
    mask: np.ndarray | None = None  # uint8 cell-centred
    cfl: float = 0.25
    steps: int = 1                  # the config's full step count
    t_end: float | None = None      # config 1 runs to a time instead
    notes: dict = field(default_factory=dict)

    @property
    def stages(self) -> int:
        return int(self.opts["rk"])

    @property
    def ncells(self) -> int:
        return self.nx * self.ny * self.nz


def cell_coords(n, lo, hi, stag=False):
    """Padded 1-D coordinates: centres x_i = lo + (i+1/2) dx, or lower faces lo + i dx."""
    dx = (hi - lo) / n
    i = np.arange(-G, n + G + (1 if stag else 0), dtype=np.float64)
    return lo + (i + (0.0 if stag else 0.5)) * dx, dx


def _grid3(nx, ny, nz, lo, hi, stag=(False, False, False)):
    x, dx = cell_coords(nx, lo[0], hi[0], stag[0])
    y, dy = cell_coords(ny, lo[1], hi[1], stag[1])
    z, dz = cell_coords(nz, lo[2], hi[2], stag[2])
    Z, Y, X = np.meshgrid(z, y, x, indexing="ij")
    return X, Y, Z, (dx, dy, dz)


def flat_metric(shape):
    one, zero = np.ones(shape), np.zeros(shape)
    m = [zero.copy() for _ in range(16)]
    m[0] = one.copy()
    m[4] = one.copy()
    m[7] = one.copy()
    m[9] = one.copy()
    return m


def wrap_pad(a, stag=(False, False, False)):
    """Periodic padding of an interior (nz,ny,nx) array to the padded (+1 if staggered) shape."""
    out = a
    for ax, st in zip((2, 1, 0), stag):  # x is the last axis
        n = a.shape[ax]
        idx = np.arange(-G, n + G + (1 if st else 0)) % n
        out = np.take(out, idx, axis=ax)
    return np.ascontiguousarray(out)


def _det3(g):
    gxx, gxy, gxz, gyy, gyz, gzz = g
    return (gxx * (gyy * gzz - gyz * gyz) - gxy * (gxy * gzz - gyz * gxz)
            + gxz * (gxy * gyz - gyy * gxz))


def _lower(g, v):
    gxx, gxy, gxz, gyy, gyz, gzz = g
    return (gxx * v[0] + gxy * v[1] + gxz * v[2],
            gxy * v[0] + gyy * v[1] + gyz * v[2],
            gxz * v[0] + gyz * v[1] + gzz * v[2])


def _dot(g, a, b):
    al = _lower(g, a)
    return al[0] * b[0] + al[1] * b[1] + al[2] * b[2]


# --------------------------------------------------------------------------- config 1
def balsara1(nx=256, ny=4, nz=4):
    """Balsara-1 shock tube (Table 1 test 1; Gamma=2, t=0.4), flat space."""
    lo, hi = (-0.5, -0.5 * ny / nx, -0.5 * nz / nx), (0.5, 0.5 * ny / nx, 0.5 * nz / nx)
    X, _, _, dx = _grid3(nx, ny, nz, lo, hi)
    shape = X.shape
    left = X < 0.0
    rho = np.where(left, 1.0, 0.125)
    p = np.where(left, 1.0, 0.1)
    zero = np.zeros(shape)
    Bx = np.full(shape, 0.5)
    By = np.where(left, 1.0, -1.0)
    opts = dict(gamma_ad=2.0, poly_k=1.0, poly_gamma=2.0, rho_atm=1e-10, p_floor=1e-12,
                w_max=100.0, c2p_tol=1e-12, c2p_maxit=100, recon=0, ppm_flatten=1, riemann=0,
                rk=2, bc=(1, 1, 1))
    return Workload("config1_balsara1_%dx%dx%d" % (nx, ny, nz), nx, ny, nz, dx, opts,
                    flat_metric(shape), [rho, zero.copy(), zero.copy(), zero.copy(), p, Bx, By,
                                         zero.copy()],
                    cfl=0.25, steps=0, t_end=0.4)


# --------------------------------------------------------------------------- config 2
def blast(n=128):
    """3-D cylindrical magnetised blast wave, periodic, flat space (BASELINE config 2; a 3-D
    variant of PAPER.md:440-461)."""
    lo, hi = (-6.0,) * 3, (6.0,) * 3
    X, Y, _, dx = _grid3(n, n, n, lo, hi)
    shape = X.shape
    r = np.sqrt(X * X + Y * Y)
    p = np.where(r < 0.8, 1.0, np.where(r < 1.0, 1.0 + (r - 0.8) / 0.2 * (3e-5 - 1.0), 3e-5))
    rho = np.full(shape, 1e-2)
    zero = np.zeros(shape)
    Bx = np.full(shape, 0.1)
    opts = dict(gamma_ad=4.0 / 3.0, poly_k=1.0, poly_gamma=4.0 / 3.0, rho_atm=1e-9,
                p_floor=1e-12, w_max=100.0, c2p_tol=1e-12, c2p_maxit=100, recon=1,
                ppm_flatten=1, riemann=0, rk=3, bc=(0, 0, 0))
    return Workload("config2_blast_%d" % n, n, n, n, dx, opts, flat_metric(shape),
                    [rho, zero.copy(), zero.copy(), zero.copy(), p, Bx, zero.copy(), zero.copy()],
                    cfl=0.25, steps=200)


# --------------------------------------------------------------------------- config 3
def kerr_schild_adm(X, Y, Z, M=1.0, a=0.9, rmin=1.0):
    """Cartesian Kerr-Schild ADM variables alpha, beta^i, gamma_ij (harness-side analytic
    metric; r is clamped from below so excised cells hold finite numbers)."""
    R2 = X * X + Y * Y + Z * Z
    r2 = 0.5 * (R2 - a * a) + np.sqrt(0.25 * (R2 - a * a) ** 2 + a * a * Z * Z)
    r = np.maximum(np.sqrt(np.maximum(r2, 0.0)), rmin)
    H = M * r ** 3 / (r ** 4 + a * a * Z * Z)
    lx = (r * X + a * Y) / (r * r + a * a)
    ly = (r * Y - a * X) / (r * r + a * a)
    lz = Z / r
    alpha = 1.0 / np.sqrt(1.0 + 2.0 * H)
    f = 2.0 * H / (1.0 + 2.0 * H)
    beta = (f * lx, f * ly, f * lz)
    gam = (1.0 + 2.0 * H * lx * lx, 2.0 * H * lx * ly, 2.0 * H * lx * lz,
           1.0 + 2.0 * H * ly * ly, 2.0 * H * ly * lz, 1.0 + 2.0 * H * lz * lz)
    return alpha, beta, gam


def _stationary_K(X, Y, Z, h, adm):
    """K_ij = (gamma_kj d_i beta^k + gamma_ki d_j beta^k + beta^k d_k gamma_ij)/(2 alpha) for
    a stationary metric, derivatives by 4th-order centred differences of the ANALYTIC
    functions with step h (input recipe, not the method's stencil)."""
    alpha, beta, gam = adm(X, Y, Z)
    db = [[None] * 3 for _ in range(3)]   # db[i][k] = d_i beta^k
    dg = [[None] * 6 for _ in range(3)]   # dg[k][c] = d_k gamma_c
    for ax in range(3):
        def ev(s):
            d = [0.0, 0.0, 0.0]
            d[ax] = s * h
            _, b, g = adm(X + d[0], Y + d[1], Z + d[2])
            return b, g
        bp1, gp1 = ev(1.0)
        bm1, gm1 = ev(-1.0)
        bp2, gp2 = ev(2.0)
        bm2, gm2 = ev(-2.0)
        for k in range(3):
            db[ax][k] = (8.0 * (bp1[k] - bm1[k]) - (bp2[k] - bm2[k])) / (12.0 * h)
        for c in range(6):
            dg[ax][c] = (8.0 * (gp1[c] - gm1[c]) - (gp2[c] - gm2[c])) / (12.0 * h)
    sym = {(0, 0): 0, (0, 1): 1, (0, 2): 2, (1, 1): 3, (1, 2): 4, (2, 2): 5,
           (1, 0): 1, (2, 0): 2, (2, 1): 4}
    K = []
    for (i, j) in [(0, 0), (0, 1), (0, 2), (1, 1), (1, 2), (2, 2)]:
        acc = 0.0
        for k in range(3):
            acc = acc + gam[sym[(k, j)]] * db[i][k] + gam[sym[(k, i)]] * db[j][k] \
                + beta[k] * dg[k][sym[(i, j)]]
        K.append(acc / (2.0 * alpha))
    return K


def kerr_blob(n=256):
    """Kerr-Schild black hole (M=1, a=0.9) with an orbiting magnetised blob (BASELINE config 3)."""
    lo, hi = (-20.0,) * 3, (20.0,) * 3
    X, Y, Z, dx = _grid3(n, n, n, lo, hi)
    adm = lambda x, y, z: kerr_schild_adm(x, y, z, 1.0, 0.9, 1.0)
    alpha, beta, gam = adm(X, Y, Z)
    K = _stationary_K(X, Y, Z, 1e-3, adm)
    metric = [alpha, *beta, *gam, *K]
    R = np.sqrt(X * X + Y * Y + Z * Z)
    mask = (R < 1.5).astype(np.uint8)

    def rho_of(x, y, z):
        return 1e-4 + 0.1 * np.exp(-((x - 8.0) ** 2 + y * y + z * z) / 4.0)
    rho = rho_of(X, Y, Z)
    p = 0.01 * rho ** (4.0 / 3.0)
    varpi = np.maximum(np.sqrt(X * X + Y * Y), 1e-6)
    vphi = 0.3 / np.sqrt(np.maximum(R, 1e-6) / 8.0)
    vx, vy, vz = -vphi * Y / varpi, vphi * X / varpi, np.zeros_like(X)
    v2 = _dot(gam, (vx, vy, vz), (vx, vy, vz))
    sc = np.where(v2 > 0.9, np.sqrt(0.9 / np.maximum(v2, 1e-300)), 1.0)
    vx, vy = vx * sc, vy * sc
    # A_phi = max(rho - 0.02, 0) as the covariant coordinate component:
    # A_x = -y A_phi / varpi^2 on x-edges, A_y = x A_phi / varpi^2 on y-edges.
    Xe, Ye, Ze, _ = _grid3(n, n, n, lo, hi, (False, True, True))
    w2 = np.maximum(Xe * Xe + Ye * Ye, 1e-12)
    Ax = -Ye * np.maximum(rho_of(Xe, Ye, Ze) - 0.02, 0.0) / w2
    Xe, Ye, Ze, _ = _grid3(n, n, n, lo, hi, (True, False, True))
    w2 = np.maximum(Xe * Xe + Ye * Ye, 1e-12)
    Ay = Xe * np.maximum(rho_of(Xe, Ye, Ze) - 0.02, 0.0) / w2
    Az = np.zeros_like(Ax)
    # pad cell-centred-shape edge grids to the staggered shape (the extra last index is unused)
    Ax = _to_stag_shape(Ax, (False, True, True))
    Ay = _to_stag_shape(Ay, (True, False, True))
    Az = np.zeros_like(Ax)
    # normalise so that max p / max(b^2/2) = 100
    b2 = _b2_from_vecpot((Ax, Ay, Az), dx, gam, (vx, vy, vz))
    scale = np.sqrt(p.max() / (100.0 * 0.5 * b2.max()))
    Ax, Ay = Ax * scale, Ay * scale
    opts = dict(gamma_ad=4.0 / 3.0, poly_k=0.01, poly_gamma=4.0 / 3.0, rho_atm=1e-11,
                p_floor=1e-18, w_max=100.0, c2p_tol=1e-12, c2p_maxit=100, recon=1,
                ppm_flatten=1, riemann=0, rk=3, bc=(1, 1, 1))
    return Workload("config3_kerrschild_%d" % n, n, n, n, dx, opts, metric,
                    [rho, vx, vy, vz, p, None, None, None], vecpot=[Ax, Ay, Az], mask=mask,
                    cfl=0.25, steps=100)


def _to_stag_shape(a, stag):
    """Arrays built on _grid3(..., stag) have +1 only along staggered axes: pad the rest."""
    pads = []
    for ax, st in zip((0, 1, 2), (stag[2], stag[1], stag[0])):
        pads.append((0, 0 if st else 1))
    return np.ascontiguousarray(np.pad(a, pads, mode="edge"))


def _b2_from_vecpot(A, dx, gam, v):
    """b^2 = B^2/W^2 + (B.v)^2 (eq. 13) of the cell-centred field of a staggered potential;
    used only to NORMALISE seed fields to a target plasma beta."""
    Ax, Ay, Az = A
    Bfx = (Az[:, 1:, :] - Az[:, :-1, :])[:-1, :, :] / dx[1] - (Ay[1:, :, :] - Ay[:-1, :, :])[:, :-1, :] / dx[2]
    Bfy = (Ax[1:, :, :] - Ax[:-1, :, :])[:, :, :-1] / dx[2] - (Az[:, :, 1:] - Az[:, :, :-1])[:-1, :, :] / dx[0]
    Bfz = (Ay[:, :, 1:] - Ay[:, :, :-1])[:, :-1, :] / dx[0] - (Ax[:, 1:, :] - Ax[:, :-1, :])[:, :, :-1] / dx[1]
    # Bfx: (nz+6, ny+6, nx+7) ... centre by averaging the two faces along the own axis
    sg = np.sqrt(_det3(gam))
    Bx = 0.5 * (Bfx[:, :, :-1] + Bfx[:, :, 1:]) / sg
    By = 0.5 * (Bfy[:, :-1, :] + Bfy[:, 1:, :]) / sg
    Bz = 0.5 * (Bfz[:-1, :, :] + Bfz[1:, :, :]) / sg
    B2 = _dot(gam, (Bx, By, Bz), (Bx, By, Bz))
    Bv = _dot(gam, (Bx, By, Bz), v)
    v2 = _dot(gam, v, v)
    return B2 * (1.0 - v2) + Bv * Bv


# --------------------------------------------------------------------------- config 4
def _modes_field(rng, n3, nmodes, kmax, amp):
    """sum_m a_m cos(2 pi k_m.x + phi_m) on the periodic unit box, interior (nz,ny,nx) cells,
    integer k with 1 <= |k| <= kmax, evaluated through separable complex exponentials."""
    nz, ny, nx = n3
    xs = [(-0.5 + (np.arange(n) + 0.5) / n) for n in (nx, ny, nz)]
    out = np.zeros((nz, ny, nx))
    m = 0
    while m < nmodes:
        k = rng.integers(-kmax, kmax + 1, size=3)
        kk = float(np.sqrt((k * k).sum()))
        if kk < 1.0 or kk > kmax:
            continue
        a = amp(rng)
        phi = rng.uniform(0.0, 2.0 * np.pi)
        ex = np.exp(2j * np.pi * k[0] * xs[0])
        ey = np.exp(2j * np.pi * k[1] * xs[1])
        ez = np.exp(2j * np.pi * k[2] * xs[2]) * np.exp(1j * phi)
        out += a * (ez[:, None, None] * ey[None, :, None] * ex[None, None, :]).real
        m += 1
    return out


def c2p_stress(n=256, seed=SEED0 + 3):
    """Perturbed generic metric + smooth random primitives with the stated marginals
    (BASELINE config 4, 'config 4a' of DESIGN.md)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    n3 = (n, n, n)
    flat = [1.0, 0, 0, 0, 1.0, 0, 0, 1.0, 0, 1.0, 0, 0, 0, 0, 0, 0]
    metric = []
    for f in range(16):
        pert = _modes_field(rng, n3, 8, 4, lambda r: r.uniform(-1.0, 1.0) * 0.05 / 8.0)
        metric.append(wrap_pad(flat[f] + pert))
    gam = metric[4:10]

    def unit_field():
        th = _modes_field(rng, n3, 8, 2, lambda r: 0.5)
        return np.arccos(np.cos(th)) / np.pi
    u1, u2, u3, u4 = unit_field(), unit_field(), unit_field(), unit_field()
    rho = wrap_pad(10.0 ** (-8.0 + 8.0 * u1))
    W = wrap_pad(1.0 + 9.0 * u2)
    sigma = wrap_pad(10.0 ** (-3.0 + 4.0 * u3))
    p = rho * wrap_pad(10.0 ** (-2.0 + 2.0 * u4))
    nvec = [wrap_pad(_modes_field(rng, n3, 8, 2, lambda r: r.normal())) for _ in range(3)]
    mvec = [wrap_pad(_modes_field(rng, n3, 8, 2, lambda r: r.normal())) for _ in range(3)]
    nn = np.sqrt(np.maximum(_dot(gam, nvec, nvec), 1e-30))
    vmag = np.sqrt(1.0 - 1.0 / (W * W))
    v = [vmag * c / nn for c in nvec]
    mm = np.sqrt(np.maximum(_dot(gam, mvec, mvec), 1e-30))
    mhat = [c / mm for c in mvec]
    mv = _dot(gam, mhat, v)
    s = np.sqrt(sigma * rho / (1.0 / (W * W) + mv * mv))
    B = [s * c for c in mhat]
    d = 1.0 / n
    opts = dict(gamma_ad=5.0 / 3.0, poly_k=1.0, poly_gamma=5.0 / 3.0, rho_atm=1e-10,
                p_floor=1e-10, w_max=100.0, c2p_tol=1e-12, c2p_maxit=100, recon=1,
                ppm_flatten=1, riemann=0, rk=3, bc=(0, 0, 0))
    return Workload("config4_c2p_stress_%d" % n, n, n, n, (d, d, d), opts, metric,
                    [rho, v[0], v[1], v[2], p, B[0], B[1], B[2]], cfl=0.25, steps=20)


def c2p_states(nstates, seed=SEED0 + 13):
    """'config 4b': iid random states with the config-4 marginals on random perturbed
    metrics, structure-of-arrays (prim 8 x n, metric 10 x n)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    n = int(nstates)
    flat = np.array([1.0, 0, 0, 0, 1.0, 0, 0, 1.0, 0, 1.0])
    met = flat[:, None] + rng.uniform(-0.05, 0.05, size=(10, n))
    gam = [met[4 + c] for c in range(6)]
    rho = 10.0 ** rng.uniform(-8.0, 0.0, n)
    W = rng.uniform(1.0, 10.0, n)
    sigma = 10.0 ** rng.uniform(-3.0, 1.0, n)
    p = rho * 10.0 ** rng.uniform(-2.0, 0.0, n)
    nv = [rng.normal(size=n) for _ in range(3)]
    mvv = [rng.normal(size=n) for _ in range(3)]
    nn = np.sqrt(_dot(gam, nv, nv))
    vmag = np.sqrt(1.0 - 1.0 / (W * W))
    v = [vmag * c / nn for c in nv]
    mm = np.sqrt(_dot(gam, mvv, mvv))
    mhat = [c / mm for c in mvv]
    mv = _dot(gam, mhat, v)
    s = np.sqrt(sigma * rho / (1.0 / (W * W) + mv * mv))
    B = [s * c for c in mhat]
    prim = np.ascontiguousarray(np.stack([rho, v[0], v[1], v[2], p, B[0], B[1], B[2]]))
    return prim, np.ascontiguousarray(met)


# --------------------------------------------------------------------------- config 5
def _random_spectrum_field(rng, n, slope, kmax, shift=(0.0, 0.0, 0.0)):
    """Real periodic Gaussian random field on n^3 with |f_k| ~ k^slope for 1 <= k <= kmax;
    `shift` (in cells) moves the sample points (staggering)."""
    k1 = np.fft.fftfreq(n, 1.0 / n)
    KZ, KY, KX = np.meshgrid(k1, k1, k1[: n // 2 + 1], indexing="ij")
    kk = np.sqrt(KX * KX + KY * KY + KZ * KZ)
    amp = np.where((kk >= 1.0) & (kk <= kmax), np.maximum(kk, 1.0) ** slope, 0.0)
    spec = (rng.normal(size=kk.shape) + 1j * rng.normal(size=kk.shape)) * amp
    ph = np.exp(2j * np.pi * (KX * shift[0] + KY * shift[1] + KZ * shift[2]) / n)
    return spec * ph, (KX, KY, KZ, kk)


def bns_like(n=512, seed=SEED0 + 4):
    """BNS-merger-like block: two Gaussian stars, conformally flat static metric, seeded
    magnetised turbulence (BASELINE config 5; rho_c, Gamma from PAPER.md:532)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    lo, hi = -16.0, 16.0
    d = (hi - lo) / n
    x = lo + (np.arange(n) + 0.5) * d
    Z, Y, X = np.meshgrid(x, x, x, indexing="ij")
    U = np.exp(-((X - 3.0) ** 2 + Y * Y + Z * Z) / 9.0) + np.exp(-((X + 3.0) ** 2 + Y * Y + Z * Z) / 9.0)
    del X, Y, Z
    alpha = 1.0 - 0.2 * U
    psi4 = (1.0 + 0.1 * U) ** 4
    rho = 1.28e-3 * (1e-3 + U)
    p = 100.0 * rho * rho
    cs = np.sqrt(2.0 * p / (rho + 2.0 * p))   # c_s of the Gamma=2 ideal gas, for the Mach scaling
    kmax = min(64, n // 4)
    # solenoidal velocity: project a random vector spectrum
    specs = []
    for _ in range(3):
        s, (KX, KY, KZ, kk) = _random_spectrum_field(rng, n, -11.0 / 6.0, kmax)
        specs.append(s)
    k2 = np.maximum(kk * kk, 1.0)
    div = (KX * specs[0] + KY * specs[1] + KZ * specs[2]) / k2
    specs = [specs[0] - KX * div, specs[1] - KY * div, specs[2] - KZ * div]
    u = [np.fft.irfftn(s, s=(n, n, n), axes=(0, 1, 2)) for s in specs]
    rms = np.sqrt(np.mean(u[0] ** 2 + u[1] ** 2 + u[2] ** 2))
    v = [0.5 * cs * c / rms for c in u]
    v2 = psi4 * (v[0] ** 2 + v[1] ** 2 + v[2] ** 2)
    sc = np.where(v2 > 0.8, np.sqrt(0.8 / np.maximum(v2, 1e-300)), 1.0)
    v = [c * sc for c in v]
    # Kolmogorov vector potential on edges (sample points shifted by half a cell)
    shifts = [(0.0, -0.5, -0.5), (-0.5, 0.0, -0.5), (-0.5, -0.5, 0.0)]
    A = []
    for sh in shifts:
        s, _ = _random_spectrum_field(rng, n, -17.0 / 6.0, kmax, sh)
        A.append(np.fft.irfftn(s, s=(n, n, n), axes=(0, 1, 2)))
    zero = np.zeros_like(U)
    metric_int = [alpha, zero, zero, zero, psi4, zero, zero, psi4, zero, psi4,
                  zero, zero, zero, zero, zero, zero]
    metric = [wrap_pad(m) for m in metric_int]
    Apad = [wrap_pad(A[0], (False, True, True)), wrap_pad(A[1], (True, False, True)),
            wrap_pad(A[2], (True, True, False))]
    Apad = [_to_stag_shape(a, st) for a, st in zip(Apad, [(False, True, True), (True, False, True),
                                                           (True, True, False)])]
    prim = [wrap_pad(rho), wrap_pad(v[0]), wrap_pad(v[1]), wrap_pad(v[2]), wrap_pad(p)]
    gam = metric[4:10]
    b2 = _b2_from_vecpot(Apad, (d, d, d), gam, prim[1:4])
    I = (slice(G, G + n),) * 3
    scale = np.sqrt(prim[4][I].sum() / (10.0 * 0.5 * b2[I].sum()))
    Apad = [a * scale for a in Apad]
    opts = dict(gamma_ad=2.0, poly_k=100.0, poly_gamma=2.0, rho_atm=1e-10, p_floor=1e-18,
                w_max=100.0, c2p_tol=1e-12, c2p_maxit=100, recon=1, ppm_flatten=1, riemann=0,
                rk=4, bc=(0, 0, 0))
    return Workload("config5_bns_%d" % n, n, n, n, (d, d, d), opts, metric,
                    prim + [None, None, None], vecpot=Apad, cfl=0.25, steps=50)


# ------------------------------------------------------------------ smooth-wave test data
def alfven_wave(nx, ny=1, nz=1, axis=0):
    """Circularly polarised Alfven wave (eqs 49-50): A0=1, rho=1, p=0.5,
    v_A=0.5, B^x=1, k=2 pi, Gamma=5/3, periodic, flat space; `axis` = propagation axis."""
    n = [nx, ny, nz]
    L = [1.0, 1.0, 1.0]
    dxs = 1.0 / n[axis]
    lo = [-0.5 * n[a] * dxs for a in range(3)]
    hi = [0.5 * n[a] * dxs for a in range(3)]
    X, Y, Z, dx = _grid3(nx, ny, nz, lo, hi)
    s = (X, Y, Z)[axis]
    shape = X.shape
    kx = 2.0 * np.pi
    a1, a2 = (axis + 1) % 3, (axis + 2) % 3
    v = [np.zeros(shape) for _ in range(3)]
    B = [np.zeros(shape) for _ in range(3)]
    v[a1] = -0.5 * np.cos(kx * s)
    v[a2] = -0.5 * np.sin(kx * s)
    B[axis] = np.ones(shape)
    B[a1] = np.cos(kx * s)
    B[a2] = np.sin(kx * s)
    opts = dict(gamma_ad=5.0 / 3.0, poly_k=1.0, poly_gamma=5.0 / 3.0, rho_atm=1e-10,
                p_floor=1e-12, w_max=100.0, c2p_tol=1e-12, c2p_maxit=100, recon=0,
                ppm_flatten=1, riemann=0, rk=2, bc=(0, 0, 0))
    return Workload("alfven_%d" % n[axis], nx, ny, nz, dx, opts, flat_metric(shape),
                    [np.ones(shape), v[0], v[1], v[2], np.full(shape, 0.5), B[0], B[1], B[2]],
                    cfl=0.2, steps=0, t_end=2.0, notes={"L": L})


def make(config: int, n: int | None = None) -> Workload:
    """BASELINE.json configs[config] at full size (n=None) or reduced linear size n."""
    if config == 0:
        return balsara1(256 if n is None else n)
    if config == 1:
        return blast(128 if n is None else n)
    if config == 2:
        return kerr_blob(256 if n is None else n)
    if config == 3:
        return c2p_stress(256 if n is None else n)
    if config == 4:
        return bns_like(512 if n is None else n)
    raise ValueError("config must be 0..4")
