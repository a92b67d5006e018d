"""Pins of the oracle's 1-D backup con2prim (Palenzuela et al. scheme, eqs
42-45; DESIGN.md pin P15, readings G23-G25).  CPU only; nothing here calls the CUDA path."""
import numpy as np

from oracle import ref
from paper_2406_11669_b200 import workloads as wl

G53 = 5.0 / 3.0


def gam_mat(m):
    return np.array([[m[4], m[5], m[6]], [m[5], m[7], m[8]], [m[6], m[8], m[9]]])


def _opts(**kw):
    d = dict(gamma_ad=G53, rho_atm=1e-12, p_floor=1e-30, w_max=100.0)
    d.update(kw)
    return ref.make_opts(**d)


def _true_x(P, M, Gamma):
    """x = h W of a primitive state (independent numpy)."""
    g = gam_mat(M)
    v = P[1:4]
    W = 1.0 / np.sqrt(1.0 - v @ g @ v)
    eps = P[4] / ((Gamma - 1.0) * P[0])
    return (1.0 + Gamma * eps) * W, W, eps


def test_P15_relations_44_45_hold_at_the_true_state():
    """At x = hW of a known state, eq. (44) gives its W, eq. (45) (with t^2/x^2, G23) its eps,
    and eq. (43) f(x) = 0.  A t^2/x in eq. (45) as printed fails this for B.S != 0."""
    prim, met = wl.c2p_states(400)
    o = _opts()
    worst = np.zeros(3)
    for n in range(prim.shape[1]):
        P, M = prim[:, n], met[:, n]
        U = ref.prim2con_pt(P, M, G53)
        x, W, eps = _true_x(P, M, G53)
        Wh, eh, f = ref.c2p1d_relations_pt(U, M, o, x)
        h = 1.0 + G53 * eps
        worst = np.maximum(worst, [abs(Wh - W) / W, abs(eh - eps) / h, abs(f) / x])
    assert worst[0] < 1e-10 and worst[1] < 1e-9 and worst[2] < 1e-9, worst


def test_P15_bracket_of_the_paper_contains_the_root():
    """1 + q - s < hW < 2 + 2q - s on the seeded physical states."""
    prim, met = wl.c2p_states(2000)
    for n in range(prim.shape[1]):
        P, M = prim[:, n], met[:, n]
        U = ref.prim2con_pt(P, M, G53)
        g = gam_mat(M)
        B = P[5:8]
        q, s = U[4] / U[0], (B @ g @ B) / U[0]
        x, _, _ = _true_x(P, M, G53)
        assert 1.0 + q - s < x < 2.0 + 2.0 * q - s, (n, 1 + q - s, x, 2 + 2 * q - s)


def test_P15_roundtrip_and_agreement_with_the_2d_scheme():
    """prim -> cons -> prim through the 1-D scheme: 1e-11 in the P1 norm (the bracketing
    iteration stops at a relative bracket width of 1e-14, amplified like P1); the 2-D and the
    1-D scheme return the same primitives."""
    prim, met = wl.c2p_states(1500)
    o = _opts()
    worst = np.zeros(3)
    agree = np.zeros(3)
    maxit = 0
    for n in range(prim.shape[1]):
        P, M = prim[:, n], met[:, n]
        U = ref.prim2con_pt(P, M, G53)
        p1, st, it = ref.con2prim1d_pt(U, M, o)
        assert st == 0
        maxit = max(maxit, it)
        rhoh = P[0] + 2.5 * P[4]
        worst = np.maximum(worst, [abs(p1[0] - P[0]) / P[0], np.abs(p1[1:4] - P[1:4]).max(),
                                   abs(p1[4] - P[4]) / rhoh])
        p2, _, bits, _ = ref.con2prim_pt(U, M, o)
        assert bits == 0
        agree = np.maximum(agree, [abs(p1[0] - p2[0]) / p2[0], np.abs(p1[1:4] - p2[1:4]).max(),
                                   abs(p1[4] - p2[4]) / rhoh])
    assert worst.max() < 1e-11, worst
    assert agree.max() < 1e-11, agree
    assert maxit <= 60


def test_P15_closed_forms():
    """S_i = 0, B = 0 (fluid at rest): x = h, rho = D, rho eps = tau; flat space."""
    flat = np.array([1.0, 0, 0, 0, 1.0, 0, 0, 1.0, 0, 1.0])
    o = _opts(gamma_ad=1.4)
    rho, p = 0.7, 0.3
    U = ref.prim2con_pt(np.array([rho, 0, 0, 0, p, 0, 0, 0]), flat, 1.4)
    p1, st, _ = ref.con2prim1d_pt(U, flat, o)
    assert st == 0
    assert abs(p1[0] - rho) < 1e-13 and np.abs(p1[1:4]).max() < 1e-14 and abs(p1[4] - p) < 1e-13
    # B = 0, moving fluid: textbook SRHD relation z = tau + D + p, v = S/z
    P = np.array([1.1, 0.5, -0.3, 0.2, 0.4, 0, 0, 0])
    U = ref.prim2con_pt(P, flat, 1.4)
    p1, st, _ = ref.con2prim1d_pt(U, flat, o)
    assert st == 0
    z = U[4] + U[0] + p1[4]
    assert np.allclose(p1[1:4], U[1:4] / z, atol=1e-13)


def test_backup_takes_over_when_the_2d_scheme_fails():
    """With a Newton budget too small to converge the 2-D scheme fails (status 2 ->
    atmosphere); with the backup enabled the state is recovered (status bit 16)
    and equals the original primitives."""
    prim, met = wl.c2p_states(200)
    o_bad = _opts(c2p_maxit=2)
    nback = 0
    for n in range(prim.shape[1]):
        P, M = prim[:, n], met[:, n]
        U = ref.prim2con_pt(P, M, G53)
        _, _, bits, _ = ref.con2prim_pt(U, M, o_bad)
        p, u, bb, _ = ref.con2prim_backup_pt(U, M, o_bad)
        if bits & 2:
            assert bb == 16, (n, bb)
            nback += 1
            rhoh = P[0] + 2.5 * P[4]
            assert abs(p[0] - P[0]) < 1e-11 * P[0] and abs(p[4] - P[4]) < 1e-11 * rhoh
            assert np.abs(p[1:4] - P[1:4]).max() < 1e-11
            assert np.array_equal(u, U[:5])
        else:
            assert bb == bits
    assert nback > 50


def _numpy_cons(P, M, Gamma):
    """Eqs (13), (37), (20)-(22) written out in numpy; does not call
    the oracle."""
    g = gam_mat(M)
    rho, v, p, B = P[0], P[1:4], P[4], P[5:8]
    vl, Bl = g @ v, g @ B
    W = 1.0 / np.sqrt(1.0 - v @ vl)
    ab0 = W * (B @ vl)                               # alpha b^0, eq. (13)
    b2 = (B @ Bl + ab0 ** 2) / W ** 2                # b^2, eq. (13)
    bl = Bl / W + ab0 * vl                           # b_i, eq. (37)
    h = 1.0 + Gamma * p / ((Gamma - 1.0) * rho)      # eq. (46)
    D = rho * W                                      # eq. (20)
    S = (rho * h + b2) * W ** 2 * vl - ab0 * bl      # eq. (21)
    tau = (rho * h + b2) * W ** 2 - (p + 0.5 * b2) - ab0 ** 2 - D   # eq. (22)
    return D, S, tau, W, h


def test_P15_recovered_state_satisfies_eqs_20_22_and_43_45_in_numpy():
    """The pin that does not pass through the oracle's own eq. (44)/(45) code: conserved
    states that come from NO known primitive state (a consistent state with tau and S_j pushed
    away from it) are recovered by the 1-D scheme; the recovered primitives, put through eqs
    (20)-(22) in numpy, must give back the conserved input, and x = hW of the recovered state
    must satisfy eqs (44), (45), (43) evaluated in numpy with the q, r, s, t of eq. (42)."""
    prim, met = wl.c2p_states(600)
    o = _opts()
    rng = np.random.default_rng(4245)
    worst = np.zeros(5)
    for n in range(prim.shape[1]):
        P, M = prim[:, n], met[:, n]
        U = ref.prim2con_pt(P, M, G53)
        U[4] *= 1.0 + 0.2 * rng.random()             # more energy: stays inside the physical region
        U[1:4] *= 1.0 - 0.1 * rng.random()           # less momentum
        p1, st, _ = ref.con2prim1d_pt(U, M, o)
        assert st == 0, n
        Prec = np.concatenate([p1, U[5:8]])
        D, S, tau, W, h = _numpy_cons(Prec, M, G53)
        sc = max(np.abs(U[1:4]).max(), U[4] + U[0])
        worst[0] = max(worst[0], abs(D - U[0]) / U[0])
        worst[1] = max(worst[1], np.abs(S - U[1:4]).max() / sc)
        worst[2] = max(worst[2], abs(tau - U[4]) / (U[4] + U[0]))
        # eqs (42)-(45) in numpy at x = hW of the recovered state
        g = gam_mat(M)
        gu = np.linalg.inv(g)
        B = U[5:8]
        q, r = U[4] / U[0], (U[1:4] @ gu @ U[1:4]) / U[0] ** 2
        s, t = (B @ g @ B) / U[0], (B @ U[1:4]) / U[0] ** 1.5
        x = h * W
        iw2 = 1.0 - (r * x * x + t * t * (2.0 * x + s)) / (x * x * (x + s) ** 2)      # (44)
        eps = -1.0 + x * np.sqrt(iw2) * (1.0 - 1.0 / iw2) + \
            (1.0 + q - s + 0.5 * (t * t / (x * x) + s * iw2)) / np.sqrt(iw2)          # (45), G23
        worst[3] = max(worst[3], abs(iw2 - 1.0 / W ** 2) * W ** 2)
        worst[4] = max(worst[4], abs(x - (1.0 + G53 * eps) / np.sqrt(iw2)) / x)       # (43)
        assert 1.0 + q - s < x < 2.0 + 2.0 * q - s
    assert worst[0] < 1e-11 and worst[1] < 1e-10 and worst[2] < 1e-10, worst
    assert worst[3] < 1e-9 and worst[4] < 1e-9, worst
