"""Block-level pins of the oracle (P2-P6, P12-P14).  CPU only; nothing here
calls the CUDA path.  Golden numbers live in tests/golden/ with their citations."""
import os

import numpy as np
import pytest

from oracle import ref
from paper_2406_11669_b200 import workloads as wl
from tests.util import G, I3, interior, make_ref

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def gold(name):
    rows = {}
    for line in open(os.path.join(GOLD, name)):
        if line.startswith("#") or not line.strip():
            continue
        t = line.split()
        rows[t[0]] = [float(x) for x in t[1:]]
    return rows


def const_fields(shape, vals):
    return [np.full(shape, float(v)) for v in vals]


# Spatially constant, non-trivial alpha, beta^i, gamma_ij.  K_ij = 0: a metric that is constant in
# space AND held fixed in time has K_ij = (D_i beta_j + D_j beta_i)/(2 alpha) = 0 (eq. 4,
# PAPER.md:59); a non-zero K_ij would make the tau source T^{ij} K_ij of eq. (19) non-zero.
GENERIC_METRIC = [0.8, 0.3, -0.1, 0.05, 1.44, 0.1, -0.05, 1.1, 0.07, 0.9,
                  0.0, 0.0, 0.0, 0.0, 0.0, 0.0]


def smooth_periodic_workload(n=8, seed=1, curved=False, opts=None):
    """Smooth random periodic data on the unit box (flat or perturbed metric)."""
    rng = np.random.default_rng(seed)
    x = (np.arange(n) + 0.5) / n
    Z, Y, X = np.meshgrid(x, x, x, indexing="ij")

    def f(amp):
        k = rng.integers(-1, 2, 3)
        return amp * np.sin(2 * np.pi * (k[0] * X + k[1] * Y + k[2] * Z) + rng.uniform(0, 6))
    prim = [1.0 + f(0.2), f(0.2), f(0.2), f(0.2), 1.0 + f(0.3), 0.5 + f(0.2), f(0.3), f(0.3)]
    prim = [wl.wrap_pad(p) for p in prim]
    shape = prim[0].shape
    if curved:
        flat = [1.0, 0, 0, 0, 1.0, 0, 0, 1.0, 0, 1.0, 0, 0, 0, 0, 0, 0]
        metric = [wl.wrap_pad(flat[i] + f(0.05)) for i in range(16)]
    else:
        metric = wl.flat_metric(shape)
    o = dict(gamma_ad=5.0 / 3.0, poly_k=1.0, poly_gamma=5.0 / 3.0, rho_atm=1e-10, p_floor=1e-12,
             w_max=100.0, c2p_tol=1e-13, c2p_maxit=100, recon=1, ppm_flatten=1, riemann=0, rk=3,
             bc=(0, 0, 0))
    if opts:
        o.update(opts)
    return wl.Workload("smooth", n, n, n, (1.0 / n,) * 3, o, metric, prim, cfl=0.25)


# ------------------------------------------------------------------------------ P2
@pytest.mark.parametrize("recon,rk", [(0, 2), (1, 3), (1, 4)])
def test_P2_uniform_state_constant_generic_metric(recon, rk):
    n = 6
    shape = (n + 6,) * 3
    w = wl.Workload("uniform", n, n, n, (0.1, 0.2, 0.15),
                    dict(gamma_ad=5.0 / 3.0, poly_k=1.0, poly_gamma=5.0 / 3.0, rho_atm=1e-10,
                         p_floor=1e-12, w_max=100.0, c2p_tol=1e-12, c2p_maxit=100, recon=recon,
                         ppm_flatten=1, riemann=0, rk=rk, bc=(0, 1, 0)),
                    const_fields(shape, GENERIC_METRIC),
                    const_fields(shape, [0.7, 0.2, -0.1, 0.15, 0.4, 0.3, -0.2, 0.5]))
    s = make_ref(w)
    dU, dA = s.rhs()
    for r in range(5):
        assert np.all(dU[r] == 0.0), r           # RHS identically zero (R8: flux differences
    U0 = s.get_cons()                            # and FD derivatives vanish on constants)
    B0 = s.get_bface()
    s.step(3, 0.25)
    U1 = s.get_cons()
    B1 = s.get_bface()
    for r in range(8):
        assert np.array_equal(interior(U0[r]), interior(U1[r])), r   # bit-identical
    for d in range(3):
        assert np.array_equal(B0[d], B1[d])
    A = s.get_vecpot()
    # E is uniform and non-zero (v x B != 0): A grows uniformly, its curl stays exactly zero
    assert np.abs(A[2][I3]).max() > 0 and np.ptp(A[2][G:-G - 1, G:-G - 1, G:-G - 1]) == 0.0


# ------------------------------------------------------------------------------ P3
@pytest.mark.parametrize("recon,rk", [(0, 2), (1, 3)])
def test_P3_conservation_periodic_flat(recon, rk):
    w = smooth_periodic_workload(8, opts=dict(recon=recon, rk=rk))
    s = make_ref(w)
    sg = 1.0
    U0 = [interior(u).sum() * sg for u in s.get_cons()[:5]]
    scale = [np.abs(interior(u)).sum() for u in s.get_cons()[:5]]
    s.step(2, 0.25)
    st = s.stats()
    assert st["c2p_fail"] == 0 and st["p_fix"] == 0 and st["atmo"] == 0
    U1 = [interior(u).sum() for u in s.get_cons()[:5]]
    for r in range(5):
        assert abs(U1[r] - U0[r]) <= 2e-13 * scale[r], (r, U0[r], U1[r])


# ------------------------------------------------------------------------------ P4
def _shock_1d(axis, n=32, mirror=False):
    """Balsara-1-like 1-D Riemann problem along `axis` with all components non-trivial."""
    dims = [4, 4, 4]
    dims[axis] = n
    nx, ny, nz = dims
    d = 1.0 / n
    lo = [-0.5 * dims[a] * d for a in range(3)]
    hi = [0.5 * dims[a] * d for a in range(3)]
    X, Y, Z, dx = wl._grid3(nx, ny, nz, lo, hi)
    s = (X, Y, Z)[axis]
    if mirror:
        s = -s
    left = s < 0
    a1, a2 = (axis + 1) % 3, (axis + 2) % 3
    v = [None] * 3
    B = [None] * 3
    sgn = -1.0 if mirror else 1.0
    v[axis] = sgn * np.where(left, 0.2, -0.1)
    v[a1] = np.where(left, 0.1, 0.0)
    v[a2] = np.where(left, 0.0, 0.05)
    B[axis] = sgn * np.full(s.shape, 0.5)
    B[a1] = np.where(left, 1.0, -1.0)
    B[a2] = np.where(left, 0.3, 0.1)
    rho = np.where(left, 1.0, 0.125)
    p = np.where(left, 1.0, 0.1)
    o = dict(gamma_ad=2.0, poly_k=1.0, poly_gamma=2.0, rho_atm=1e-10, p_floor=1e-12, w_max=100.0,
             c2p_tol=1e-13, c2p_maxit=100, recon=1, ppm_flatten=1, riemann=0, rk=3, bc=(1, 1, 1))
    return wl.Workload("shock", nx, ny, nz, dx, o, wl.flat_metric(s.shape),
                       [rho, v[0], v[1], v[2], p, B[0], B[1], B[2]], cfl=0.25)


def test_P4_axis_permutation_and_mirror():
    sols = []
    for axis in range(3):
        s = make_ref(_shock_1d(axis))
        s.step(5, 0.25)
        P = [interior(q) for q in s.get_prims()]
        # bring to (line) order: take the pencil along `axis` through the block
        sl = [1, 1, 1]
        line = lambda q: np.moveaxis(q, 2 - axis, 0)[:, 1, 1]
        a1, a2 = (axis + 1) % 3, (axis + 2) % 3
        sols.append(np.array([line(P[0]), line(P[1 + axis]), line(P[1 + a1]), line(P[1 + a2]),
                              line(P[4]), line(P[5 + axis]), line(P[5 + a1]), line(P[5 + a2])]))
    assert np.abs(sols[0]).max() > 0.5
    for k in (1, 2):
        assert np.abs(sols[k] - sols[0]).max() < 1e-12
    # mirror x -> -x (v^x, B^x flip)
    s = make_ref(_shock_1d(0, mirror=True))
    s.step(5, 0.25)
    P = [interior(q)[1, 1, ::-1] for q in s.get_prims()]
    m = np.array([P[0], -P[1], P[2], P[3], P[4], -P[5], P[6], P[7]])
    assert np.abs(m - sols[0]).max() < 1e-12


# ------------------------------------------------------------------------------ P5
def _alfven_error(N, recon=0, rk=2):
    w = wl.alfven_wave(N)
    s = make_ref(w, recon=recon, rk=rk)
    s.set_option("fixed_dt", 0.2 * w.dx[0])      # Courant factor 0.2
    s.step_until(2.0, 0.2)                        # one period: v_A = 0.5, L = 1
    st = s.stats()
    assert st["c2p_fail"] == 0 and st["p_fix"] == 0 and st["atmo"] == 0
    By = interior(s.get_prims()[6])
    return float(np.sqrt(np.mean((By - interior(w.prims[6])) ** 2)))


def test_P5_alfven_wave_second_order():
    """minmod+HLLE+RK2, CFL 0.2, periodic, N = 8..128 => ~2nd order in
    L2(B^y) after one period (Fig. 4).  Golden values: independent prototype (tests/golden)."""
    g = gold("alfven_l2_by.txt")
    Ns = [8, 16, 32, 64, 128]
    errs = [_alfven_error(N) for N in Ns]
    for N, e in zip(Ns, errs):
        assert abs(e - g[str(N)][0]) < 0.1 * g[str(N)][0], (N, e, g[str(N)])
    orders = [np.log2(errs[i] / errs[i + 1]) for i in range(len(errs) - 1)]
    assert all(o > 1.6 for o in orders[1:]), orders
    assert all(errs[i + 1] < errs[i] for i in range(len(errs) - 1))


def test_P5_entropy_wave_advection():
    """rho = 1 + 0.1 sin(2 pi x) advected with uniform v, p: exact solution = translation."""
    errs = {}
    for recon, rk in [(0, 2), (1, 3)]:
        es = []
        for N in (16, 32, 64):
            x, dx = wl.cell_coords(N, -0.5, 0.5)
            shape = (7, 7, N + 6)
            X = np.broadcast_to(x, shape)
            prim = [1.0 + 0.1 * np.sin(2 * np.pi * X), np.full(shape, 0.5), np.zeros(shape),
                    np.zeros(shape), np.ones(shape), np.full(shape, 0.1), np.zeros(shape),
                    np.zeros(shape)]
            o = dict(gamma_ad=5.0 / 3.0, poly_k=1.0, poly_gamma=5.0 / 3.0, rho_atm=1e-10,
                     p_floor=1e-12, w_max=100.0, c2p_tol=1e-13, c2p_maxit=100, recon=recon,
                     ppm_flatten=1, riemann=0, rk=rk, bc=(0, 0, 0))
            w = wl.Workload("entropy", N, 1, 1, (dx, dx, dx), o, wl.flat_metric(shape), prim)
            s = make_ref(w)
            s.set_option("fixed_dt", 0.25 * dx)
            s.step_until(2.0, 0.25)               # one period at v = 0.5
            rho = interior(s.get_prims()[0])
            es.append(float(np.sqrt(np.mean((rho - interior(prim[0])) ** 2))))
        errs[(recon, rk)] = es
    mm, ppm = errs[(0, 2)], errs[(1, 3)]
    assert mm[0] > mm[1] > mm[2] and ppm[0] > ppm[1] > ppm[2]
    assert np.log2(mm[1] / mm[2]) > 1.3
    assert np.log2(ppm[1] / ppm[2]) > 1.8 and ppm[2] < 0.25 * mm[2]


# ------------------------------------------------------------------------------ P6
def div_bface(Bf, dx):
    """face-centred discrete divergence of the densitised field on all cells with 6 faces."""
    return ((Bf[0][:-1, :-1, 1:] - Bf[0][:-1, :-1, :-1]) / dx[0]
            + (Bf[1][:-1, 1:, :-1] - Bf[1][:-1, :-1, :-1]) / dx[1]
            + (Bf[2][1:, :-1, :-1] - Bf[2][:-1, :-1, :-1]) / dx[2])


def test_P6_divB_preserved_and_ct_update():
    w = smooth_periodic_workload(8, seed=4, curved=True)
    s = make_ref(w)
    Bf0 = s.get_bface()
    d0 = div_bface(Bf0, w.dx)[I3]
    bscale = max(np.abs(b).max() for b in Bf0) / min(w.dx)
    # curl(RHS_A) on faces equals minus the CT divergence of the stored B-row fluxes
    dU, dA = s.rhs()
    F = s.fluxes()
    dBx = (dA[2][:, 1:, :] - dA[2][:, :-1, :])[:-1, :, :] / w.dx[1] - (dA[1][1:, :, :] - dA[1][:-1, :, :])[:, :-1, :] / w.dx[2]
    # CT form of  d_t B~^x = -d_y F~^y(B^x) - d_z F~^z(B^x)  with edge-averaged fluxes:
    Ez = -dA[2]
    Ey = -dA[1]
    want = -(Ez[:, 1:, :] - Ez[:, :-1, :])[:-1, :, :] / w.dx[1] + (Ey[1:, :, :] - Ey[:-1, :, :])[:, :-1, :] / w.dx[2]
    assert np.abs(dBx - want)[G:-G, G:-G, G:-G].max() < 1e-13 * bscale
    # and E_z is the 4-point mean with the signs of G14: F~^x(B^y) = -E_z, F~^y(B^x) = +E_z
    i, j, k = 5, 6, 4
    ez = 0.25 * (-F[0][6][k, j - 1, i] - F[0][6][k, j, i] + F[1][5][k, j, i - 1] + F[1][5][k, j, i])
    assert np.isclose(Ez[k, j, i], ez, rtol=1e-14, atol=1e-16)
    s.step(3, 0.25)
    d1 = div_bface(s.get_bface(), w.dx)[I3]
    assert np.abs(d1 - d0).max() < 1e-13 * bscale
    # a field that comes from a potential only has zero divergence to round-off
    shape_st = tuple(n_ + 1 for n_ in w.prims[0].shape)
    rng = np.random.default_rng(0)
    x = (np.arange(8)) / 8.0
    Z, Y, X = np.meshgrid(x, x, x, indexing="ij")
    A = [wl._to_stag_shape(wl.wrap_pad(np.sin(2 * np.pi * (X + 2 * Y - Z) + c), (True, True, True)), (True, True, True))
         for c in (0.3, 1.1, 2.0)]
    w2 = smooth_periodic_workload(8, seed=4, curved=True)
    w2.prims[5:] = [None, None, None]
    w2.vecpot = A
    s2 = make_ref(w2)
    assert np.abs(div_bface(s2.get_bface(), w.dx)).max() < 1e-12 * 2 * np.pi / min(w.dx)
    s2.step(2, 0.25)
    assert np.abs(div_bface(s2.get_bface(), w.dx)[I3]).max() < 1e-12 * 2 * np.pi / min(w.dx)


def test_P6_flux_ct_is_half_hlle_half_central_in_1d():
    """For x-only data E_z(i-1/2) = -1/2 F^x(B^y)_{i-1/2} - 1/4 (f_{i-1} + f_i), f = cell-centre
    x-flux of B^y: the known flux-CT property."""
    N = 16
    x, dx = wl.cell_coords(N, -0.5, 0.5)
    shape = (8, 8, N + 6)
    X = np.broadcast_to(x, shape)
    s2 = np.sin(2 * np.pi * X)
    prim = [1 + 0.2 * s2, 0.2 + 0.1 * s2, 0.1 * np.cos(2 * np.pi * X), np.zeros(shape),
            1 + 0.1 * s2, np.full(shape, 0.7), 0.5 * s2, np.zeros(shape)]
    o = dict(gamma_ad=5.0 / 3.0, poly_k=1.0, poly_gamma=5.0 / 3.0, rho_atm=1e-10, p_floor=1e-12,
             w_max=100.0, c2p_tol=1e-13, c2p_maxit=100, recon=0, ppm_flatten=1, riemann=0, rk=2,
             bc=(0, 0, 0))
    w = wl.Workload("x-only", N, 2, 2, (dx, dx, dx), o, wl.flat_metric(shape), prim)
    s = make_ref(w)
    dU, dA = s.rhs()
    F = s.fluxes()
    P = s.get_prims()
    k = j = G
    for i in range(G, G + N):
        f = lambda ii: ref.flux_pt(0, [q[k, j, ii] for q in P], [1, 0, 0, 0, 1, 0, 0, 1, 0, 1.0], 5.0 / 3.0)[6]
        want = -0.5 * F[0][6][k, j, i] - 0.25 * (f(i - 1) + f(i))
        assert np.isclose(-dA[2][k, j, i], want, rtol=1e-13, atol=1e-15)


# ------------------------------------------------------------------------------ P12
def test_P12_bruteforce_rhs_on_4cubed():
    """A deliberately naive second evaluator of L(Y) (python loops over cells, faces and edges,
    nothing reused, its own index arithmetic and FD stencil) against the oracle's ref_rhs on a
    4^3 periodic block with a curved metric.  Pins the R4-R11 indexing."""
    n = 4
    w = smooth_periodic_workload(n, seed=9, curved=True)
    s = make_ref(w)
    o = ref.make_opts(**w.opts)
    dU, dA = s.rhs()
    P = s.get_prims()          # rho,v,p,Bc incl. ghosts
    Bf = s.get_bface()
    met = w.metric
    dx = w.dx
    Gam = w.opts["gamma_ad"]
    at = lambda q, i, j, k: q[k + G, j + G, i + G]
    E = [(1, 0, 0), (0, 1, 0), (0, 0, 1)]

    def face_flux(d, i, j, k):
        """all 8 densitised flux rows at the lower d-face of cell (i,j,k)"""
        e = E[d]
        cells = [(i + s_ * e[0], j + s_ * e[1], k + s_ * e[2]) for s_ in range(-3, 3)]
        mf = []
        for f in range(10):
            q = [at(met[f], *c) for c in cells[1:5]]
            mf.append((-q[0] + 9 * q[1] + 9 * q[2] - q[3]) / 16)
        g = np.array([[mf[4], mf[5], mf[6]], [mf[5], mf[7], mf[8]], [mf[6], mf[8], mf[9]]])
        sg = np.sqrt(np.linalg.det(g))
        pline = np.array([at(P[4], *c) for c in cells])
        vline = np.array([at(P[1 + d], *c) for c in cells])
        PL, PR = np.zeros(8), np.zeros(8)
        for v in range(8):
            q = np.array([at(P[v], *c) for c in cells])
            qL, qR = ref.recon_line(w.opts["recon"], w.opts["ppm_flatten"], q, pline, vline)
            PL[v], PR[v] = qL[3], qR[3]
        PL[5 + d] = PR[5 + d] = at(Bf[d], i, j, k) / sg
        return sg * ref.riemann_pt(d, PL, PR, mf, o)

    def fd(q, a, i, j, k):
        e = E[a]
        c = lambda s_: at(q, i + s_ * e[0], j + s_ * e[1], k + s_ * e[2])
        return (c(-2) - 8 * c(-1) + 8 * c(1) - c(2)) / (12 * dx[a])

    worst = 0.0
    scaleU = max(np.abs(interior(q)).max() for q in dU)
    for k in range(n):
        for j in range(n):
            for i in range(n):
                div = np.zeros(8)
                for d in range(3):
                    e = E[d]
                    div += (face_flux(d, i + e[0], j + e[1], k + e[2]) - face_flux(d, i, j, k)) / dx[d]
                m = [at(met[f], i, j, k) for f in range(16)]
                g = np.array([[m[4], m[5], m[6]], [m[5], m[7], m[8]], [m[6], m[8], m[9]]])
                sg = np.sqrt(np.linalg.det(g))
                dal = [fd(met[0], a, i, j, k) for a in range(3)]
                dbe = [[fd(met[1 + b], a, i, j, k) for b in range(3)] for a in range(3)]
                dga = [[fd(met[4 + c], a, i, j, k) for c in range(6)] for a in range(3)]
                S = ref.source_pt([at(q, i, j, k) for q in P], m[:10], m[10:], dal,
                                  np.array(dbe).reshape(-1), np.array(dga).reshape(-1), Gam)
                L = -div[:5] + m[0] * sg * S
                got = np.array([at(dU[r], i, j, k) for r in range(5)])
                worst = max(worst, np.abs(L - got).max())
    assert worst < 1e-13 * scaleU, worst
    # edges: E_x(i,j-1/2,k-1/2), E_y(i-1/2,j,k-1/2), E_z(i-1/2,j-1/2,k); d_t A = -E
    worstA = 0.0
    scaleA = max(np.abs(q).max() for q in dA)
    for k in range(n + 1):
        for j in range(n + 1):
            for i in range(n + 1):
                if i < n:
                    ex = 0.25 * (-face_flux(1, i, j, k - 1)[7] - face_flux(1, i, j, k)[7]
                                 + face_flux(2, i, j - 1, k)[6] + face_flux(2, i, j, k)[6])
                    worstA = max(worstA, abs(-ex - at(dA[0], i, j, k)))
                if j < n:
                    ey = 0.25 * (-face_flux(2, i - 1, j, k)[5] - face_flux(2, i, j, k)[5]
                                 + face_flux(0, i, j, k - 1)[7] + face_flux(0, i, j, k)[7])
                    worstA = max(worstA, abs(-ey - at(dA[1], i, j, k)))
                if k < n:
                    ez = 0.25 * (-face_flux(0, i, j - 1, k)[6] - face_flux(0, i, j, k)[6]
                                 + face_flux(1, i - 1, j, k)[5] + face_flux(1, i, j, k)[5])
                    worstA = max(worstA, abs(-ez - at(dA[2], i, j, k)))
    assert worstA < 1e-13 * scaleA, worstA


# ------------------------------------------------------------------------------ P13
def _const_metric_advection(N, beta_x, t_end):
    x, dx = wl.cell_coords(N, -0.5, 0.5)
    shape = (7, 7, N + 6)
    X = np.broadcast_to(x, shape)
    mvals = [0.8, beta_x, 0, 0, 1.44, 0.1, 0, 1.0, 0, 1.0, 0, 0, 0, 0, 0, 0]
    prim = [1.0 + 0.1 * np.sin(2 * np.pi * X), np.full(shape, 0.25), np.zeros(shape), np.zeros(shape),
            np.ones(shape), np.zeros(shape), np.zeros(shape), np.zeros(shape)]
    o = dict(gamma_ad=5.0 / 3.0, poly_k=1.0, poly_gamma=5.0 / 3.0, rho_atm=1e-10, p_floor=1e-12,
             w_max=100.0, c2p_tol=1e-13, c2p_maxit=100, recon=0, ppm_flatten=1, riemann=0, rk=2,
             bc=(0, 0, 0))
    w = wl.Workload("cma", N, 1, 1, (dx, dx, dx), o, const_fields(shape, mvals), prim)
    s = make_ref(w)
    s.set_option("fixed_dt", 0.25 * dx)
    s.step_until(t_end, 0.25)
    rho = interior(s.get_prims()[0])[0, 0]
    return rho, interior(prim[0])[0, 0]


def test_P13_constant_metric_advection():
    """eq. (18) D-row: d_t(sqrt(gamma) D) + d_i(sqrt(gamma) D v~^i) = 0: on a
    spatially constant metric the profile moves rigidly at v~^x = alpha v^x - beta^x = -0.1;
    one coordinate period is t = 10.  beta^x = alpha v^x = 0.2 freezes it."""
    g = gold("const_metric_advection_l2_rho.txt")
    errs = []
    for N in (16, 32, 64):
        rho, rho0 = _const_metric_advection(N, 0.3, 10.0)
        e = float(np.sqrt(np.mean((rho - rho0) ** 2)))
        errs.append(e)
        assert abs(e - g[str(N)][0]) < 0.1 * g[str(N)][0], (N, e)
        # no phase shift: cross-correlation peaks at zero lag
        cc = [np.dot(np.roll(rho - 1, s_), rho0 - 1) for s_ in range(-3, 4)]
        assert int(np.argmax(cc)) == 3
    assert np.log2(errs[0] / errs[1]) > 1.25 and np.log2(errs[1] / errs[2]) > 1.25
    # frozen profile: no translation at all, pure in-place diffusion
    rho, rho0 = _const_metric_advection(32, 0.2, 5.0)
    cc = [np.dot(np.roll(rho - 1, s_), rho0 - 1) for s_ in range(-3, 4)]
    assert int(np.argmax(cc)) == 3
    assert np.sqrt(np.mean((rho - rho0) ** 2)) < 0.02
    # half a period with the moving profile must be a half-box shift (wrong alpha/beta placement
    # gives an O(0.1) mismatch here)
    rho, rho0 = _const_metric_advection(64, 0.3, 5.0)
    assert np.sqrt(np.mean((rho - np.roll(rho0, 32)) ** 2)) < 0.01


# ------------------------------------------------------------------------------ P14
def _rindler(N, recon):
    g_acc, Gam, K = 0.5, 5.0 / 3.0, 1.0
    x, dx = wl.cell_coords(N, 0.0, 1.0)
    shape = (8, 8, N + 6)
    X = np.broadcast_to(x, shape)
    alpha = 1.0 + g_acc * X
    h = 2.5 / alpha                                  # h alpha = const: hydrostatic balance
    rho = ((h - 1.0) * (Gam - 1.0) / (Gam * K)) ** (1.0 / (Gam - 1.0))
    p = K * rho ** Gam
    metric = wl.flat_metric(shape)
    metric[0] = alpha.copy()
    z = np.zeros(shape)
    o = dict(gamma_ad=Gam, poly_k=K, poly_gamma=Gam, rho_atm=1e-10, p_floor=1e-12, w_max=100.0,
             c2p_tol=1e-13, c2p_maxit=100, recon=recon, ppm_flatten=1, riemann=0, rk=2,
             bc=(1, 0, 0))
    return wl.Workload("rindler", N, 2, 2, (dx, dx, dx), o, metric,
                       [rho, z.copy(), z.copy(), z.copy(), p, np.full(shape, 0.05), z.copy(), z.copy()])


def test_P14_rindler_hydrostatic_equilibrium():
    """Flat spacetime in Rindler-type slicing alpha = 1 + g x: an isentropic fluid at rest with
    h alpha = const is in equilibrium, so L(U~) must vanish to truncation error and converge
    (sources of eq. 19 balancing the pressure flux of eq. 18)."""
    gref = gold("rindler_residual.txt")
    res = {}
    for N in (16, 32, 64, 128):
        s = make_ref(_rindler(N, 0))
        dU, _ = s.rhs()
        cut = slice(G + 4, -(G + 4))
        res[N] = [np.abs(dU[r][G, G, cut]).max() for r in (0, 1, 4)]
    for N in (16, 128):
        for a, b in zip(res[N], gref[str(N)]):
            assert 0.3 * b < a < 3.0 * b, (N, res[N], gref[str(N)])
    # the cut is 4 CELLS from each wall, so the sampled region grows with N (towards the dense
    # end): the observed order approaches 2 from below (1.4-1.6, 1.7-1.8, 1.8-1.9)
    for N, omin in ((16, 1.3), (32, 1.6), (64, 1.75)):
        for a, b in zip(res[N], res[2 * N]):
            assert np.log2(a / b) > omin, (N, res)
    # PPM converges at least as fast
    r32 = np.abs(make_ref(_rindler(32, 1)).rhs()[0][1][G, G, G + 4:-(G + 4)]).max()
    r64 = np.abs(make_ref(_rindler(64, 1)).rhs()[0][1][G, G, G + 4:-(G + 4)]).max()
    assert np.log2(r32 / r64) > 1.7
    # drift stays small and shrinks with resolution in cells the walls cannot have reached
    drift = []
    for N in (32, 64):
        w = _rindler(N, 0)
        s = make_ref(w)
        s.set_option("fixed_dt", 0.25 * w.dx[0])
        nst = N // 8
        s.step(nst, 0.25)                 # t = 1/32: signals travel < 1/32 + stencil
        v = s.get_prims()[1][G, G, G:-G]
        m = N // 4
        drift.append(np.abs(v[m:-m]).max())
    assert drift[1] < drift[0] / 3.0 and drift[0] < 1e-3
