"""Pins of the oracle's upwind constrained transport (row F1; eqs 33-35;
DESIGN.md pin P16, readings G26-G28).  CPU only; nothing here calls the CUDA path."""
import numpy as np

from oracle import ref
from paper_2406_11669_b200 import workloads as wl
from tests.test_oracle_block import div_bface, smooth_periodic_workload
from tests.util import G, I3, interior, make_ref

OPTS = dict(gamma_ad=5.0 / 3.0, poly_k=1.0, poly_gamma=5.0 / 3.0, rho_atm=1e-10, p_floor=1e-12,
            w_max=100.0, c2p_tol=1e-13, c2p_maxit=100, recon=1, ppm_flatten=0, riemann=0, rk=2,
            bc=(0, 0, 0))


def _line_workload(axis, N=16):
    """Smooth data that depend on one coordinate only, flat space, periodic.  Arrays are
    [z][y][x]; `axis` 0/1/2 = x/y/z.  Vector components are rotated with the axis so that the
    three runs are the same problem."""
    n = [2, 2, 2]
    n[axis] = N
    x, dx = wl.cell_coords(N, -0.5, 0.5)
    shape = (n[2] + 6, n[1] + 6, n[0] + 6)
    sh = [1, 1, 1]
    sh[2 - axis] = N + 6
    X = np.broadcast_to(x.reshape(sh), shape)
    s2, c2 = np.sin(2 * np.pi * X), np.cos(2 * np.pi * X)
    vn, v1, v2 = 0.2 + 0.1 * s2, 0.1 * c2, 0.05 * s2        # normal, first, second transverse
    Bn, B1, B2 = np.full(shape, 0.7), 0.5 * s2, 0.3 * c2
    v = [None] * 3
    B = [None] * 3
    for t, (vv, bb) in enumerate(((vn, Bn), (v1, B1), (v2, B2))):
        v[(axis + t) % 3] = vv
        B[(axis + t) % 3] = bb
    prim = [1 + 0.2 * s2, v[0], v[1], v[2], 1 + 0.1 * s2, B[0], B[1], B[2]]
    return wl.Workload("line", n[0], n[1], n[2], (dx, dx, dx), dict(OPTS), wl.flat_metric(shape),
                       prim)


def test_P16_uct_reduces_to_the_hlle_flux_in_1d():
    """For data that depend on one coordinate only (flat space) eqs (33)-(35) give
    E_c = -F^a(B^b) and E_b = +F^a(B^c), the HLLE fluxes of the two transverse field
    components -- where flux-CT gives half HLLE, half central (P6).  All three orientations."""
    for a in range(3):
        b, c = (a + 1) % 3, (a + 2) % 3
        s = make_ref(_line_workload(a))
        s.set_option("emf", 1.0)
        dU, dA = s.rhs()
        F = s.fluxes()
        N = 16
        for m in range(G, G + N):
            ind = [G, G, G]
            ind[2 - a] = m
            ind = tuple(ind)
            Ec, Eb = -dA[c][ind], -dA[b][ind]
            assert np.isclose(Ec, -F[a][5 + b][ind], rtol=1e-12, atol=1e-14), (a, m)
            assert np.isclose(Eb, +F[a][5 + c][ind], rtol=1e-12, atol=1e-14), (a, m)
        # and the three orientations are the same problem
        if a == 0:
            ref0 = [-dA[c][G, G, G:G + N].copy(), -dA[b][G, G, G:G + N].copy()]
        else:
            sl = [G, G, G]
            sl[2 - a] = slice(G, G + N)
            sl = tuple(sl)
            assert np.allclose(-dA[c][sl], ref0[0], rtol=1e-12, atol=1e-14)
            assert np.allclose(-dA[b][sl], ref0[1], rtol=1e-12, atol=1e-14)


def test_P16_uniform_state_and_divB():
    """Uniform state on a constant generic metric: the UCT electric field is uniform, B does not
    change (bitwise); on smooth 3-D data div B~ is preserved to round-off."""
    w = smooth_periodic_workload(8, seed=4, curved=True)
    s = make_ref(w)
    s.set_option("emf", 1.0)
    Bf0 = s.get_bface()
    d0 = div_bface(Bf0, w.dx)[I3]
    bscale = max(np.abs(b).max() for b in Bf0) / min(w.dx)
    s.step(3, 0.25)
    assert s.stats()["c2p_fail"] == 0
    d1 = div_bface(s.get_bface(), w.dx)[I3]
    assert np.abs(d1 - d0).max() < 1e-13 * bscale
    # the two schemes are different discretisations of the same induction equation
    s2 = make_ref(w)
    s2.step(3, 0.25)
    B1, B2 = s.get_prims()[5:], s2.get_prims()[5:]
    diff = max(np.abs(interior(a) - interior(b)).max() for a, b in zip(B1, B2))
    assert 0 < diff < 0.05 * max(np.abs(interior(b)).max() for b in B2)


def _alfven_error(N, emf):
    w = wl.alfven_wave(N)
    s = make_ref(w, recon=1, rk=3)
    s.set_option("emf", float(emf))
    s.set_option("fixed_dt", 0.2 * w.dx[0])
    s.step_until(2.0, 0.2)
    st = s.stats()
    assert st["c2p_fail"] == 0 and st["atmo"] == 0
    By = interior(s.get_prims()[6])
    return float(np.sqrt(np.mean((By - interior(w.prims[6])) ** 2)))


def test_P16_alfven_wave_converges_with_uct():
    """Circularly polarised Alfven wave, PPM + RK3: at least second order
    with UCT (measured orders 2.9, 2.6), errors of the same size as flux-CT's (UCT carries the
    full HLLE dissipation, flux-CT half of it plus a central part, P6)."""
    Ns = [16, 32, 64]
    eu = [_alfven_error(N, 1) for N in Ns]
    ef = [_alfven_error(N, 0) for N in Ns]
    assert eu[0] > eu[1] > eu[2]
    assert np.log2(eu[1] / eu[2]) > 1.6, eu
    assert np.log2(eu[0] / eu[1]) > 1.6, eu
    assert all(u < 3.0 * f for u, f in zip(eu, ef)), (eu, ef)
