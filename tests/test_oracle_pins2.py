"""Pins of the oracle steps that GPU-vs-oracle parity cannot check (both sides implement the
same reading): the CFL time step R16, the RK weights R12, the outflow extrapolation of A_i R15,
the face floors of R5, the static face field B~0 of G16 and the PPM flattening coefficient of
G8(c).  Every expected value here is formed in numpy from the paper's formulas or from a closed
form -- never from the oracle's own point functions.  CPU only; nothing calls the CUDA path.

Each test names the mistake in oracle/grmhd_ref.cpp it exists to catch (each was injected by
hand once and turned exactly that test red).
"""
import numpy as np
import pytest

from oracle import ref
from paper_2406_11669_b200 import workloads as wl
from tests.util import G, I3, interior, make_ref
from tests.test_oracle_block import const_fields, smooth_periodic_workload

G53 = 5.0 / 3.0
OPTS = dict(gamma_ad=G53, poly_k=1.0, poly_gamma=G53, rho_atm=1e-10, p_floor=1e-12, w_max=100.0,
            c2p_tol=1e-13, c2p_maxit=100, recon=1, ppm_flatten=1, riemann=0, rk=3, bc=(1, 1, 1))


# ------------------------------------------------------------------------- R16: dt
def _sr_speeds_x(v, cs):
    """Textbook special-relativistic acoustic speeds along the flow (PAPER.md:199 reduces to
    them for B = 0, flat 3-metric): (v -+ cs)/(1 -+ v cs)."""
    return (v - cs) / (1.0 - v * cs), (v + cs) / (1.0 + v * cs)


def _sr_speed_transverse(v, cs):
    """... and across a flow of speed v: +- cs sqrt((1 - v^2)/(1 - v^2 cs^2))."""
    return cs * np.sqrt((1.0 - v * v) / (1.0 - v * v * cs * cs))


def _two_state_block():
    nx, ny, nz = 8, 4, 6
    dx = (0.1, 0.2, 0.05)
    shape = (nz + 6, ny + 6, nx + 6)
    alpha, beta = 0.9, (0.2, -0.1, 0.05)
    met = const_fields(shape, [alpha, *beta, 1, 0, 0, 1, 0, 1, 0, 0, 0, 0, 0, 0])
    # the caller supplies the metric's ghost cells: a lapse 5x larger there would show up in the
    # max if ghost cells entered it
    met[0][:] = 5.0 * alpha
    met[0][I3] = alpha
    states = [(1.0, 0.3, 1.0), (0.5, -0.6, 2.0)]          # (rho, v^x, p): x < mid, x >= mid
    prim = const_fields(shape, [0, 0, 0, 0, 0, 0, 0, 0])
    half = G + nx // 2
    for sl, (rho, v, p) in ((np.s_[:, :, :half], states[0]), (np.s_[:, :, half:], states[1])):
        prim[0][sl], prim[1][sl], prim[4][sl] = rho, v, p
    w = wl.Workload("two_state", nx, ny, nz, dx, dict(OPTS), met, prim, cfl=0.25)
    want = np.zeros(3)
    for rho, v, p in states:
        cs = np.sqrt(G53 * p / (rho + G53 / (G53 - 1.0) * p))
        lm, lp = _sr_speeds_x(v, cs)
        lt = _sr_speed_transverse(v, cs)
        want[0] = max(want[0], abs(alpha * lm - beta[0]), abs(alpha * lp - beta[0]))
        for d in (1, 2):
            want[d] = max(want[d], abs(alpha * lt - beta[d]), abs(-alpha * lt - beta[d]))
    return w, want


def test_R16_maxspeed_and_dt_by_hand():
    """Catches: max over the padded range (ghost lapse is 5x), `max` for `min` over the directions,
    dx/m inverted, a direction's speed built with the wrong shift component."""
    w, want = _two_state_block()
    s = make_ref(w)
    got = np.array(s.stats()["maxspeed"])
    np.testing.assert_allclose(got, want, rtol=1e-14)
    # the limiting direction is z (smallest dx), not x (largest speed)
    ratios = np.array(w.dx) / want
    assert np.argmin(ratios) == 2 and np.argmax(want) == 0
    s.step(1, 0.25)
    st = s.stats()
    np.testing.assert_allclose(st["dt"], 0.25 * ratios.min(), rtol=1e-14)
    np.testing.assert_allclose(st["t"], st["dt"], rtol=0)


def test_R16_step_until_clips_the_last_step():
    """A uniform state on a constant metric does not change (P2), so every CFL step is dt0;
    t_end = 3.4 dt0 must take 4 steps, the last one 0.4 dt0, and land on t_end."""
    shape = (4 + 6,) * 3
    met = const_fields(shape, [0.9, 0.2, -0.1, 0.05, 1, 0, 0, 1, 0, 1, 0, 0, 0, 0, 0, 0])
    prim = const_fields(shape, [1.0, 0.3, 0.0, 0.0, 1.0, 0.0, 0.0, 0.0])
    w = wl.Workload("uniform", 4, 4, 4, (0.1, 0.2, 0.05), dict(OPTS), met, prim, cfl=0.25)
    s = make_ref(w)
    s.step(1, 0.25)
    dt0 = s.stats()["dt"]
    s = make_ref(w)
    t_end = 3.4 * dt0
    n = s.step_until(t_end, 0.25)
    st = s.stats()
    assert n == 4 and st["steps"] == 4
    assert abs(st["t"] - t_end) <= 2e-16 * t_end
    np.testing.assert_allclose(st["dt"], t_end - 3.0 * dt0, rtol=1e-12)
    assert s.step_until(t_end, 0.25) == 0        # already there: no further step


# ------------------------------------------------------------------ R12: RK weights
@pytest.mark.parametrize("rk,order", [(2, 2), (3, 3), (4, 4)])
def test_R12_temporal_order(rk, order):
    """The stage weights (SSP-RK2, SSP-RK3, classic RK4, reading G15) are
    fixed by the observed order in time on a problem whose right-hand side is SMOOTH: a uniform
    fluid on a spatially constant metric with K_ij != 0.  All flux differences and metric
    derivatives vanish identically (P2), no limiter or HLLE switch ever acts, and every cell
    obeys the same ODE d tau~/dt = alpha sqrt(gamma) S_tau(P(U~)) with S_tau = T^{00} beta^i
    beta^j K_ij + 2 T^{0i} beta^j K_ij + T^{ij} K_ij (eq. 19 in 3+1 form, R9).  (With PPM on
    non-uniform data the limiter switches cap the observed order at 2, whatever the tableau.)
    fixed_dt halved three times against a 512-step RK4 run.  Catches 0.75/0.25 swapped, 2/3 for
    1/3, a missing factor 2 on k2 or k3, dt/6 for dt/3, a half step taken as a full one."""
    from tests.test_oracle_block import GENERIC_METRIC
    n, T = 4, 2.0
    shape = (n + 6,) * 3
    met = const_fields(shape, GENERIC_METRIC[:10] + [0.30, -0.10, 0.20, 0.25, 0.05, -0.15])
    prim = const_fields(shape, [0.7, 0.2, -0.1, 0.15, 0.4, 0.3, -0.2, 0.5])
    o = dict(OPTS)
    o.update(bc=(0, 0, 0), c2p_tol=1e-15, rk=rk)
    w = wl.Workload("uniform_K", n, n, n, (0.1, 0.2, 0.15), o, met, prim, cfl=0.25)

    def run(nsteps, rk_):
        s = make_ref(w, rk=rk_)
        s.set_option("fixed_dt", T / nsteps)
        s.step(nsteps, 0.25)
        U = s.get_cons()
        assert np.ptp(interior(U[4])) <= 1e-14 * abs(interior(U[4])).max()   # stays uniform
        return np.array([interior(u)[0, 0, 0] for u in U[:5]])

    start = np.array([interior(u)[0, 0, 0] for u in make_ref(w).get_cons()[:5]])
    exact = run(512, 4)
    assert abs(exact[4] - start[4]) > 0.05 * abs(start[4])       # tau really evolves
    assert np.abs(exact[:4] - start[:4]).max() < 1e-13           # D, S_j have no source here
    errs = [abs(run(m, rk)[4] - exact[4]) for m in (4, 8, 16, 32)]
    rates = [np.log2(errs[q] / errs[q + 1]) for q in range(3)]
    assert min(rates) > order - 0.25 and max(rates) < order + 0.35, (errs, rates)


# ------------------------------------------------------- R15: outflow extrapolation of A_i
def test_R15_linear_vector_potential_is_continued_exactly():
    """PAPER.md:350 'linear extrapolation': a vector potential linear in x, y, z given on the
    edges that bound interior faces must come back linear on ALL padded edges (3 layers, edges
    and corners of the block included), and B~ = curl A uniform up to the last face.  Catches a
    copy instead of 2 A_1 - A_2, a wrong source layer, and a pass that skips corners."""
    nx, ny, nz = 5, 4, 6
    dx = (0.1, 0.2, 0.05)
    shape = (nz + 6, ny + 6, nx + 6)
    met = wl.flat_metric(shape)
    prim = const_fields(shape, [1.0, 0, 0, 0, 1.0, 0, 0, 0])
    sshape = (nz + 7, ny + 7, nx + 7)
    k, j, i = np.meshgrid(*[np.arange(n) - G for n in sshape], indexing="ij")
    # lower convention: A_x at (i, j-1/2, k-1/2), A_y at (i-1/2, j, k-1/2), A_z at (i-1/2, j-1/2, k)
    pos = lambda oi, oj, ok: ((i + oi) * dx[0], (j + oj) * dx[1], (k + ok) * dx[2])
    lin = lambda c, x, y, z: c[0] + c[1] * x + c[2] * y + c[3] * z
    cA = [(0.3, 0.7, -1.1, 0.4), (-0.2, 0.5, 0.9, -1.3), (0.1, -0.6, 0.8, 1.2)]
    full = [lin(cA[0], *pos(0.5, 0, 0)), lin(cA[1], *pos(0, 0.5, 0)), lin(cA[2], *pos(0, 0, 0.5))]
    given = []
    for d, a in enumerate(full):          # only the valid range is handed over; the rest is junk
        g_ = np.full(sshape, 1e30)
        n = [nz, ny, nx]
        sl = tuple(slice(G, G + n[ax] + (0 if (2 - ax) == d else 1)) for ax in range(3))
        g_[sl] = a[sl]
        given.append(g_)
    w = wl.Workload("linA", nx, ny, nz, dx, dict(OPTS), met, prim, vecpot=given, cfl=0.25)
    s = make_ref(w)
    A = s.get_vecpot()
    for d in range(3):
        n = [nz, ny, nx]
        # every edge index that exists: staggered axes run to n + G, the edge's own axis to n + G - 1
        sl = tuple(slice(0, n[ax] + 2 * G + (0 if (2 - ax) == d else 1)) for ax in range(3))
        np.testing.assert_allclose(A[d][sl], full[d][sl], rtol=0, atol=2e-13)
    # B~^x = d_y A_z - d_z A_y etc. (eq. 24 with the permutation symbol): constants
    want = (cA[2][2] - cA[1][3], cA[0][3] - cA[2][1], cA[1][1] - cA[0][2])
    Bf = s.get_bface()
    for d in range(3):
        n = [nz, ny, nx]
        # faces whose four edges all exist
        sl = tuple(slice(0, n[ax] + 2 * G + (1 if (2 - ax) == d else 0)) for ax in range(3))
        np.testing.assert_allclose(Bf[d][sl], want[d], rtol=0, atol=1e-11)


# ------------------------------------------------------------------ R5: face floors
def test_R5_face_floors_by_hand():
    """The Riemann flux of a raw face state equals the flux of the state floored and capped BY
    HAND in numpy (rho, p raised to their floors; v^i scaled so that gamma_ij v^i v^j =
    1 - 1/w_max^2 with the non-diagonal face metric, direction kept).  Catches a missing cap, a
    cap in the flat norm, a cap on W instead of v^2, floors on the wrong slots."""
    o = ref.make_opts(gamma_ad=G53, rho_atm=1e-3, p_floor=1e-2, w_max=2.0)
    m = np.array([0.8, 0.1, -0.05, 0.02, 1.3, 0.2, -0.1, 0.9, 0.15, 1.1])
    g = np.array([[m[4], m[5], m[6]], [m[5], m[7], m[8]], [m[6], m[8], m[9]]])
    PL = np.array([1e-4, 0.9, -0.5, 0.4, 1e-3, 0.3, -0.2, 0.1])     # superluminal in this metric
    PR = np.array([0.7, 0.1, 0.2, -0.1, 0.5, 0.3, 0.4, -0.3])
    v = PL[1:4]
    v2 = v @ g @ v
    assert v2 > 1.0
    hand = PL.copy()
    hand[0], hand[4] = 1e-3, 1e-2
    hand[1:4] = v * np.sqrt((1.0 - 1.0 / 2.0 ** 2) / v2)
    vh = hand[1:4]
    assert abs(1.0 / np.sqrt(1.0 - vh @ g @ vh) - 2.0) < 1e-13        # W = w_max exactly
    for d in range(3):
        Fraw = ref.riemann_pt(d, PL, PR, m, o)
        Fhand = ref.riemann_pt(d, hand, PR, m, o)
        assert np.all(np.isfinite(Fraw))
        np.testing.assert_allclose(Fraw, Fhand, rtol=1e-13, atol=1e-15)
        Fraw = ref.riemann_pt(d, PR, PL, m, o)                        # ... and as the right state
        Fhand = ref.riemann_pt(d, PR, hand, m, o)
        np.testing.assert_allclose(Fraw, Fhand, rtol=1e-13, atol=1e-15)
    # a state inside the limits is left alone: changing w_max does not change its flux
    o2 = ref.make_opts(gamma_ad=G53, rho_atm=1e-3, p_floor=1e-2, w_max=50.0)
    np.testing.assert_array_equal(ref.riemann_pt(0, PR, PR, m, o), ref.riemann_pt(0, PR, PR, m, o2))


# --------------------------------------------------------------- G16: static face field
def test_G16_static_face_field_on_a_varying_metric():
    """B~0 on the face between cells i-1 and i is the mean of sqrt(gamma_c) B^d_c of those two
    cells, and the cell-centred B returned by get_prims is the [1/4, 1/2, 1/4] filter of
    sqrt(gamma) B^d along d divided by the cell's own sqrt(gamma).  Catches a
    dropped sqrt(gamma), the mean taken along the wrong axis, sqrt(gamma) of the wrong cell."""
    n = 6
    rng = np.random.default_rng(16)
    x = (np.arange(n) + 0.5) / n
    Z, Y, X = np.meshgrid(x, x, x, indexing="ij")
    wave = lambda: 0.1 * np.sin(2 * np.pi * (X * rng.integers(1, 3) + Y * rng.integers(1, 3) +
                                             Z * rng.integers(1, 3)) + rng.uniform(0, 6))
    flat = [1.0, 0, 0, 0, 1.0, 0, 0, 1.0, 0, 1.0, 0, 0, 0, 0, 0, 0]
    met = [wl.wrap_pad(flat[q] + (wave() if q < 10 else 0.0 * X)) for q in range(16)]
    prim = [wl.wrap_pad(f) for f in (1.0 + wave(), wave(), wave(), wave(), 1.0 + wave(),
                                     0.5 + wave(), 0.3 + wave(), -0.4 + wave())]
    o = dict(OPTS)
    o["bc"] = (0, 0, 0)
    w = wl.Workload("g16", n, n, n, (1.0 / n,) * 3, o, met, prim, cfl=0.25)
    s = make_ref(w)
    gxx, gxy, gxz, gyy, gyz, gzz = met[4:10]
    sg = np.sqrt(gxx * (gyy * gzz - gyz ** 2) - gxy * (gxy * gzz - gyz * gxz) +
                 gxz * (gxy * gyz - gyy * gxz))
    Bf = s.get_bface()
    Pc = s.get_prims()
    for d in range(3):
        ax = 2 - d                                   # numpy axis of direction d
        sB = sg * prim[5 + d]
        face = 0.5 * (np.roll(sB, 1, axis=ax) + sB)  # face i-1/2 at index i
        np.testing.assert_allclose(Bf[d][:-1, :-1, :-1][I3], face[I3], rtol=1e-14)
        filt = (0.25 * np.roll(sB, 1, axis=ax) + 0.5 * sB + 0.25 * np.roll(sB, -1, axis=ax)) / sg
        np.testing.assert_allclose(Pc[5 + d][I3], filt[I3], rtol=1e-13)
        assert np.abs(Pc[5 + d][I3] - prim[5 + d][I3]).max() > 1e-4   # it IS a filter here


# ------------------------------------------------------------ G8(c): flattening coefficient
def _flat_line(ratio, dv, level=0.0):
    """12 cells, linear q (slope 0.5); a pressure profile with
    (p_{c+1} - p_{c-1})/(p_{c+2} - p_{c-2}) = ratio at cell c = 5 (p_3 = 1, p_7 = 3, p_6 = 2.5,
    p_4 = 2.5 - 2 ratio; `level` is added everywhere) and a converging (dv > 0) or diverging
    normal velocity across that cell."""
    q = 2.0 + 0.5 * np.arange(12.0)
    p = np.array([1.0, 1.0, 1.0, 1.0, 2.5 - 2.0 * ratio, 1.7, 2.5, 3.0, 3.0, 3.0, 3.0, 3.0]) + level
    v = np.zeros(12)
    v[4], v[6] = 0.5 * dv, -0.5 * dv
    return q, p, v


def test_G8c_flattening_coefficient_between_its_ends():
    """f = clamp(10 ((p_{c+1}-p_{c-1})/(p_{c+2}-p_{c-2}) - 0.75), 0, 1) where the shock switch
    |p_{c+1}-p_{c-1}| > 0.33 min(p_{c+1}, p_{c-1}) and v_{c-1} > v_{c+1} is on (reading G8(c)).
    For linear q the unflattened PPM face values of cell c are q_c -+ slope/2 and survive the
    monotonisation, so the flattened ones are q_c -+ (1-f) slope/2: f can be read off.  Catches a
    changed 10 / 0.75 / 0.33, a flipped velocity test, f applied as (1-f)."""
    for ratio, want in ((0.80, 0.5), (0.775, 0.25), (0.76, 0.1), (0.70, 0.0), (0.95, 1.0)):
        q, p, v = _flat_line(ratio, dv=0.2)
        qL, qR = ref.recon_line(1, 1, q, press=p, vnorm=v)
        # cell 5: q^+ = qL[6] (left state of face 6), q^- = qR[5]
        f_plus = 1.0 - (qL[6] - q[5]) / 0.25
        f_minus = 1.0 - (q[5] - qR[5]) / 0.25
        assert abs(f_plus - want) < 1e-12 and abs(f_minus - want) < 1e-12, (ratio, f_plus, f_minus)
    # the switch, part 1: a diverging flow leaves f = 0
    q, p, v = _flat_line(0.8, dv=-0.2)
    qL, qR = ref.recon_line(1, 1, q, press=p, vnorm=v)
    assert abs(qL[6] - (q[5] + 0.25)) < 1e-14
    # part 2: the same pressure differences (dp1 = 1.6) on a level just below / just above
    # dp1 / 0.33 = min(p_4, p_6): on (f = 0.5) / off (f = 0)
    for fac, on in ((0.99, True), (1.01, False)):
        level = 1.6 / 0.33 * fac - 0.9
        q, p, v = _flat_line(0.8, dv=0.2, level=level)
        qL, qR = ref.recon_line(1, 1, q, press=p, vnorm=v)
        want = q[5] + (0.125 if on else 0.25)
        assert abs(qL[6] - want) < 1e-12, (fac, qL[6], want)


# --------------------------------------------------------------- R7: HLLE, a worked number
def test_R7_hlle_worked_number():
    """eq. (29) on a flat-space, B = 0 hydrodynamic Riemann problem, every ingredient from the
    textbook special-relativistic formulas in numpy (D = rho W, S = rho h W^2 v, tau = rho h W^2
    - p - D; F = (D v, S v + p, S - D v); speeds (v -+ cs)/(1 -+ v cs)): no oracle point function
    enters the expected value."""
    Gam = 1.4
    o = ref.make_opts(gamma_ad=Gam, rho_atm=1e-12, p_floor=1e-30)
    flat = np.array([1.0, 0, 0, 0, 1.0, 0, 0, 1.0, 0, 1.0])

    def side(rho, v, p):
        W = 1.0 / np.sqrt(1.0 - v * v)
        h = 1.0 + Gam / (Gam - 1.0) * p / rho
        D, S = rho * W, rho * h * W * W * v
        tau = rho * h * W * W - p - D
        cs = np.sqrt(Gam * p / (rho * h))
        U = np.array([D, S, tau])
        F = np.array([D * v, S * v + p, S - D * v])
        return U, F, (v - cs) / (1.0 - v * cs), (v + cs) / (1.0 + v * cs)

    UL, FL, lmL, lpL = side(1.0, 0.4, 1.0)
    UR, FR, lmR, lpR = side(0.3, -0.2, 0.2)
    cmax, cmin = max(0.0, lpL, lpR), -min(0.0, lmL, lmR)
    want = (cmin * FR + cmax * FL - cmax * cmin * (UR - UL)) / (cmax + cmin)
    PL = np.array([1.0, 0.4, 0, 0, 1.0, 0, 0, 0])
    PR = np.array([0.3, -0.2, 0, 0, 0.2, 0, 0, 0])
    got = ref.riemann_pt(0, PL, PR, flat, o)
    np.testing.assert_allclose(got[[0, 1, 4]], want, rtol=1e-14)
    assert np.all(got[[2, 3, 5, 6, 7]] == 0.0)
    # supersonic to the right: the flux is the left flux (P7), here with its worked value
    UL, FL, lmL, lpL = side(1.0, 0.9, 0.01)
    assert lmL > 0
    got = ref.riemann_pt(0, np.array([1.0, 0.9, 0, 0, 0.01, 0, 0, 0]),
                         np.array([1.0, 0.9, 0, 0, 0.01, 0, 0, 0]), flat, o)
    np.testing.assert_allclose(got[[0, 1, 4]], FL, rtol=1e-14)


# ------------------------------------------------------------ F2: Lax-Friedrichs, eq. (30)
def test_F2_lxf_worked_number():
    """eq. (30): F = [F_r + F_l - c_wave (U_r - U_l)] / 2 with c_wave =
    max(c_max, c_min), on flat-space B = 0 Riemann problems with every ingredient from the textbook
    special-relativistic formulas in numpy (as test_R7_hlle_worked_number): no oracle point
    function enters the expected value.  The mistakes it exists to catch: the sign of the
    dissipation term, c_wave = min or c_max alone, a missing 1/2, U and F swapped."""
    Gam = 1.4
    o = ref.make_opts(gamma_ad=Gam, rho_atm=1e-12, p_floor=1e-30, riemann=1)
    flat = np.array([1.0, 0, 0, 0, 1.0, 0, 0, 1.0, 0, 1.0])

    def side(rho, v, p):
        W = 1.0 / np.sqrt(1.0 - v * v)
        h = 1.0 + Gam / (Gam - 1.0) * p / rho
        D, S = rho * W, rho * h * W * W * v
        tau = rho * h * W * W - p - D
        cs = np.sqrt(Gam * p / (rho * h))
        return (np.array([D, S, tau]), np.array([D * v, S * v + p, S - D * v]),
                (v - cs) / (1.0 - v * cs), (v + cs) / (1.0 + v * cs))

    # (left state, right state): in the first c_max > c_min, in the second (both flows to the
    # left) c_min > c_max, so that max(c_max, c_min) is told apart from either of its arguments
    for (rl, vl, pl), (rr, vr, pr) in (((1.0, 0.4, 1.0), (0.3, -0.2, 0.2)),
                                       ((0.5, -0.6, 0.3), (1.2, -0.3, 0.8))):
        UL, FL, lmL, lpL = side(rl, vl, pl)
        UR, FR, lmR, lpR = side(rr, vr, pr)
        cmax, cmin = max(0.0, lpL, lpR), -min(0.0, lmL, lmR)
        assert abs(cmax - cmin) > 0.05
        want = 0.5 * (FR + FL - max(cmax, cmin) * (UR - UL))
        got = ref.riemann_pt(0, np.array([rl, vl, 0, 0, pl, 0, 0, 0]),
                             np.array([rr, vr, 0, 0, pr, 0, 0, 0]), flat, o)
        np.testing.assert_allclose(got[[0, 1, 4]], want, rtol=1e-14)
        assert np.all(got[[2, 3, 5, 6, 7]] == 0.0)
        # and it is NOT the HLLE flux of the same states (the option is honoured)
        hlle = ref.riemann_pt(0, np.array([rl, vl, 0, 0, pl, 0, 0, 0]),
                              np.array([rr, vr, 0, 0, pr, 0, 0, 0]), flat,
                              ref.make_opts(gamma_ad=Gam, rho_atm=1e-12, p_floor=1e-30, riemann=0))
        assert np.abs(hlle[[0, 1, 4]] - want).max() > 1e-3
    # consistency: equal states give the physical flux, whatever c_wave is
    UL, FL, _, _ = side(0.7, 0.25, 0.4)
    P = np.array([0.7, 0.25, 0, 0, 0.4, 0, 0, 0])
    np.testing.assert_allclose(ref.riemann_pt(0, P, P, flat, o)[[0, 1, 4]], FL, rtol=1e-14)


def test_F2_lxf_is_more_dissipative_than_hlle_on_a_block():
    """PAPER.md:206 ("more dissipative than HLLE"): an entropy wave (uniform v and p, sinusoidal
    rho) advected on a periodic flat block keeps its amplitude exactly; both schemes lose some,
    the LxF run more; both conserve the total rest mass to round-off (eq. 30 is a conservative
    flux)."""
    n = 16
    x = (np.arange(n) + 0.5) / n
    Z, Y, X = np.meshgrid(x, x, x, indexing="ij")
    one = np.ones_like(X)
    prim = [1.0 + 0.2 * np.sin(2 * np.pi * X), 0.3 * one, 0 * one, 0 * one, one, 0 * one, 0 * one,
            0 * one]
    prim = [wl.wrap_pad(q) for q in prim]
    metric = wl.flat_metric(prim[0].shape)
    amps, mass = {}, {}
    for riemann in (0, 1):
        o = dict(OPTS); o.update(riemann=riemann, recon=0, rk=2, bc=(0, 0, 0))
        s_ = ref.RefSolver(n, n, n, (1.0 / n,) * 3, ref.make_opts(**o))
        s_.set_metric(metric); s_.set_prims(prim)
        D0 = interior(s_.get_cons()[0]).copy()
        s_.step(20, 0.25)
        D1 = interior(s_.get_cons()[0])
        amps[riemann] = (D1.max() - D1.min()) / (D0.max() - D0.min())
        mass[riemann] = abs(D1.sum() - D0.sum()) / D0.sum()
    assert amps[1] < amps[0] < 1.0, amps
    assert amps[0] - amps[1] > 1e-3, amps
    assert mass[0] < 1e-13 and mass[1] < 1e-13, mass


# ------------------------------------------------ mask: the right cells, on every substep
def test_mask_marks_the_right_cells_on_every_substep():
    """`set_mask` (excised region, config 3): the cells given as mask[k+G, j+G, i+G] != 0 -- and
    only those -- are reset to the atmosphere on EVERY substep (G20), on a non-cubic block with an
    asymmetric mask, so that a transposed or shifted index, a mask applied once per step only, or
    one that also eats its neighbours cannot pass (config 3's own mask is a sphere on a cubic
    grid: symmetric under every index permutation)."""
    nx, ny, nz = 9, 7, 5
    shape = (nz + 2 * G, ny + 2 * G, nx + 2 * G)
    o = dict(OPTS); o.update(rk=3, bc=(1, 1, 1), rho_atm=1e-7)
    met = const_fields(shape, [1.0, 0, 0, 0, 1, 0, 0, 1, 0, 1, 0, 0, 0, 0, 0, 0])
    prim = const_fields(shape, [1.0, 0.1, -0.05, 0.02, 0.5, 0.01, 0.02, -0.01])
    marked = [(1, 2, 3), (7, 0, 4), (4, 6, 0)]            # (i, j, k), all different in every index
    mask = np.zeros(shape, dtype=np.uint8)
    for i, j, k in marked:
        mask[k + G, j + G, i + G] = 1
    mask[0, 0, 0] = 1                                      # a ghost cell: must be ignored
    s = ref.RefSolver(nx, ny, nz, (0.1, 0.1, 0.1), ref.make_opts(**o))
    s.set_metric(met); s.set_prims(prim); s.set_mask(mask)
    nsteps = 2
    s.step(nsteps, 0.2)
    P = s.get_prims()
    rho = interior(P[0])
    is_atmo = np.zeros((nz, ny, nx), dtype=bool)
    for i, j, k in marked:
        is_atmo[k, j, i] = True
    assert np.all(rho[is_atmo] == 1e-7)
    assert np.all(interior(P[1])[is_atmo] == 0.0) and np.all(interior(P[3])[is_atmo] == 0.0)
    assert np.all(rho[~is_atmo] > 0.5), "only the marked cells are reset"
    st = s.stats()
    assert st["atmo"] == len(marked) * 3 * nsteps, st["atmo"]   # every substep of every step
    # without the mask nothing is reset
    s2 = ref.RefSolver(nx, ny, nz, (0.1, 0.1, 0.1), ref.make_opts(**o))
    s2.set_metric(met); s2.set_prims(prim)
    s2.step(nsteps, 0.2)
    assert s2.stats()["atmo"] == 0 and np.all(interior(s2.get_prims()[0]) > 0.5)


# -------------------------------------------- R15 / A1: ghost fill of the primitives
@pytest.mark.parametrize("bc", [(1, 1, 1), (0, 0, 0), (0, 1, 0), (1, 0, 1)])
def test_R15_ghost_fill_of_the_primitives(bc):
    """Row A1: after set_prims the three ghost layers of rho, v^i, p hold, on a
    periodic axis, the wrapped interior value (period n) and, on an outflow axis, the value of the
    nearest interior cell -- faces, edges and corners alike (x, then y, then z pass).  Expected
    values by a numpy index map (wrap / clamp per axis), the caller's ghost values being junk.
    Catches: a mirror instead of a copy, a wrap with period n + 1, a pass that leaves the corners
    unfilled, periodic and outflow confused."""
    nx, ny, nz = 7, 5, 4
    rng = np.random.default_rng(3)
    shape = (nz + 2 * G, ny + 2 * G, nx + 2 * G)
    met = const_fields(shape, [1.0, 0, 0, 0, 1, 0, 0, 1, 0, 1, 0, 0, 0, 0, 0, 0])
    inner = [rng.uniform(0.5, 1.5, (nz, ny, nx)), rng.uniform(-0.2, 0.2, (nz, ny, nx)),
             rng.uniform(-0.2, 0.2, (nz, ny, nx)), rng.uniform(-0.2, 0.2, (nz, ny, nx)),
             rng.uniform(0.5, 1.5, (nz, ny, nx))]
    prim = []
    for q in inner:
        a = np.full(shape, 123.456)            # junk in the caller's ghost cells
        a[I3] = q
        prim.append(a)
    prim += [np.zeros(shape)] * 3
    o = dict(OPTS); o.update(bc=bc)
    s = ref.RefSolver(nx, ny, nz, (0.1, 0.1, 0.1), ref.make_opts(**o))
    s.set_metric(met); s.set_prims(prim)
    P = s.get_prims()

    def index_map(n, periodic):
        i = np.arange(-G, n + G)
        return i % n if periodic else np.clip(i, 0, n - 1)
    ix, iy, iz = (index_map(n, b == 0) for n, b in zip((nx, ny, nz), bc))
    for f in range(5):
        want = inner[f][np.ix_(iz, iy, ix)]
        assert np.array_equal(P[f], want), (bc, f)


# ------------------------------------------------ eq. (17): densitised inside, plain outside
def test_get_cons_is_undensitised_and_the_state_is_densitised():
    """eq. (17): the evolved variables are sqrt(gamma) U, the ABI's get_cons
    returns U itself (include/grmhd.h: 'UNdensitised D, S_x, S_y, S_z, tau').  On a constant
    metric with sqrt(gamma) = 2 (gamma = diag(4, 1, 1), alpha = 0.9) and a fluid at rest the
    closed forms are D = rho, S_j = 0, tau = rho eps + B_i B^i / 2 -- not twice that -- while the
    conserved total the block carries, sum sqrt(gamma) D, is twice sum rho."""
    nx, ny, nz = 6, 5, 4
    shape = (nz + 2 * G, ny + 2 * G, nx + 2 * G)
    met = const_fields(shape, [0.9, 0, 0, 0, 4.0, 0, 0, 1.0, 0, 1.0, 0, 0, 0, 0, 0, 0])
    rho, p, B = 1.3, 0.7, (0.2, -0.3, 0.1)
    prim = const_fields(shape, [rho, 0, 0, 0, p, *B])
    o = dict(OPTS); o.update(bc=(0, 0, 0))
    s = ref.RefSolver(nx, ny, nz, (0.1, 0.1, 0.1), ref.make_opts(**o))
    s.set_metric(met); s.set_prims(prim)
    U = s.get_cons()
    B2 = 4.0 * B[0] ** 2 + B[1] ** 2 + B[2] ** 2            # B_i B^i with gamma_xx = 4
    np.testing.assert_allclose(interior(U[0]), rho, rtol=1e-14)
    for r in (1, 2, 3):
        assert np.abs(interior(U[r])).max() < 1e-15
    np.testing.assert_allclose(interior(U[4]), p / (G53 - 1.0) + 0.5 * B2, rtol=1e-13)
    for d in range(3):
        np.testing.assert_allclose(interior(U[5 + d]), B[d], rtol=1e-13)
