"""Pins of the oracle's generalised Lorenz gauge (row F3; eqs 26-28,
31, 32; DESIGN.md pin P17, readings G29-G32).  CPU only; nothing here calls the CUDA path."""
import numpy as np

from oracle import ref
from paper_2406_11669_b200 import workloads as wl
from tests.test_oracle_block import smooth_periodic_workload
from tests.util import G, interior, make_ref


def _with_vecpot(w, seed=3):
    """Add a smooth periodic vector potential on the edges (so that A_j is not small)."""
    n = w.nx
    rng = np.random.default_rng(seed)
    x = np.arange(n) / n
    Z, Y, X = np.meshgrid(x, x, x, indexing="ij")
    stag = (True, True, True)
    A = []
    for c in range(3):
        k = rng.integers(-1, 2, 3)
        a = 0.05 * np.sin(2 * np.pi * (k[0] * X + k[1] * Y + k[2] * Z) + rng.uniform(0, 6))
        A.append(wl._to_stag_shape(wl.wrap_pad(a, stag), stag))
    w.vecpot = A
    return w


def test_P17_B_is_gauge_independent():
    """The gauge term of eq. (31) is a discrete gradient (vertex differences on the edges): its
    discrete curl vanishes, so B, the conserved variables and the primitives of a Lorenz-gauge run
    equal those of the algebraic-gauge run to round-off, while A and Psi differ."""
    w = _with_vecpot(smooth_periodic_workload(8, seed=6, curved=True))
    s0, s1 = make_ref(w), make_ref(w)
    s1.set_option("gauge", 1.0)
    s0.step(4, 0.25)
    s1.step(4, 0.25)
    B0, B1 = s0.get_bface(), s1.get_bface()
    bs = max(np.abs(b).max() for b in B0)
    for d in range(3):
        assert np.abs(B0[d] - B1[d])[G:-G - 1, G:-G - 1, G:-G - 1].max() < 1e-12 * bs
    for a, b in zip(s0.get_cons(), s1.get_cons()):
        assert np.abs(interior(a) - interior(b)).max() < 1e-12 * max(np.abs(interior(a)).max(), 1)
    A0, A1 = s0.get_vecpot(), s1.get_vecpot()
    assert max(np.abs(a - b).max() for a, b in zip(A0, A1)) > 1e-6
    assert np.abs(s1.get_psi()).max() > 1e-6 and np.abs(s0.get_psi()).max() == 0.0


def test_P17_rhs_terms_against_numpy():
    """Flat space with a constant shift, Psi = 0: eq. (31) adds +d_i(beta^j A_j) to d_t A_i and
    eq. (32) gives d_t Psi = -d_j A^j, with A_j averaged to the vertices (G30), the gradient as
    the 2-point vertex difference on the edge (G31) and the divergence as the centred vertex
    difference (G32) -- evaluated here independently with numpy rolls on the periodic block."""
    n = 8
    w = _with_vecpot(smooth_periodic_workload(n, seed=2, curved=False))
    beta = (0.3, -0.2, 0.1)
    for d in range(3):
        w.metric[1 + d] = np.full_like(w.metric[0], beta[d])
    s0, s1 = make_ref(w), make_ref(w)
    s1.set_option("gauge", 1.0)
    _, dA0 = s0.rhs()
    dA1, dPsi = s1.rhs_gauge()
    dx = w.dx[0]
    I = slice(G, G + n)
    A = [a[I, I, I] for a in w.vecpot]          # periodic interior, index (k, j, i)
    # vertex (i-1/2, j-1/2, k-1/2): A_x = mean over i-1, i (axis 2); A_y over j-1, j; A_z over k
    Av = [0.5 * (A[0] + np.roll(A[0], 1, 2)), 0.5 * (A[1] + np.roll(A[1], 1, 1)),
          0.5 * (A[2] + np.roll(A[2], 1, 0))]
    GA = -(beta[0] * Av[0] + beta[1] * Av[1] + beta[2] * Av[2])
    for d, ax in ((0, 2), (1, 1), (2, 0)):
        want = -(np.roll(GA, -1, ax) - GA) / dx
        got = (dA1[d] - dA0[d])[I, I, I]
        assert np.abs(got - want).max() < 1e-12, d
    # eq. (32): F^j = alpha sqrt(gamma) A^j - beta^j Psi = A_j here
    div = sum((np.roll(Av[d], -1, ax) - np.roll(Av[d], 1, ax)) / (2 * dx)
              for d, ax in ((0, 2), (1, 1), (2, 0)))
    assert np.abs(dPsi[I, I, I] + div).max() < 1e-12


def test_P17_damping_of_psi():
    """eq. (28)/(32): with xi = 1.5/dt and nothing else acting on it, Psi decays
    -- compare a run with the damping to one without (xi = 0)."""
    w = _with_vecpot(smooth_periodic_workload(8, seed=6, curved=False))
    s_d, s_u = make_ref(w), make_ref(w)
    for s, xi in ((s_d, 1.5), (s_u, 0.0)):
        s.set_option("gauge", 1.0)
        s.set_option("lorenz_xi", xi)
        s.step(6, 0.25)
    pd, pu = np.abs(s_d.get_psi()).max(), np.abs(s_u.get_psi()).max()
    assert 0 < pd < 0.7 * pu


def test_P17_damping_term_carries_the_lapse():
    """eqs (28), (32): d_t Psi = -d_j F_Psi^j - xi ALPHA Psi.  With a constant
    lapse alpha = 0.8 (flat gamma, no shift) and Psi != 0 after a few steps, the oracle's d_t Psi is
    compared with -d_j(alpha A_j) - (lorenz_xi/dt) alpha Psi formed in numpy from the A_i and Psi it
    returns (vertex means and centred vertex differences as in test_P17_rhs_terms_against_numpy).
    Catches the damping term without its lapse (test_P17_damping_of_psi runs with alpha = 1) and
    the flux without it."""
    n = 8
    alpha = 0.8
    w = _with_vecpot(smooth_periodic_workload(n, seed=4, curved=False))
    w.metric[0] = np.full_like(w.metric[0], alpha)
    s = make_ref(w)
    s.set_option("gauge", 1.0)
    s.set_option("lorenz_xi", 1.5)
    s.step(3, 0.25)
    dt = s.stats()["dt"]
    _, dPsi = s.rhs_gauge()
    I = slice(G, G + n)
    A = [a[I, I, I] for a in s.get_vecpot()]
    Psi = s.get_psi()[I, I, I]
    assert np.abs(Psi).max() > 1e-6
    dx = w.dx[0]
    Av = [0.5 * (A[0] + np.roll(A[0], 1, 2)), 0.5 * (A[1] + np.roll(A[1], 1, 1)),
          0.5 * (A[2] + np.roll(A[2], 1, 0))]
    div = sum((np.roll(alpha * Av[d], -1, ax) - np.roll(alpha * Av[d], 1, ax)) / (2 * dx)
              for d, ax in ((0, 2), (1, 1), (2, 0)))
    want = -div - (1.5 / dt) * alpha * Psi
    scale = np.abs(want).max()
    assert np.abs(dPsi[I, I, I] - want).max() < 1e-12 * max(scale, 1.0)
    # the two terms are told apart: without the lapse on the damping the answer moves by far more
    assert np.abs((1.5 / dt) * (1.0 - alpha) * Psi).max() > 1e-6 * max(scale, 1.0)
