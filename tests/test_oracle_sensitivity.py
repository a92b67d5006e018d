"""How far does the ORACLE's own answer move when its inputs change by one ulp?  That distance is
the noise floor of any comparison against it, and it is what justifies the two places where the
GPU parity tests do not assert north_star's 1e-11 on every cell:

  * config 4 (con2prim stress) after one RK3 step: cells driven to the edge of the recovery's
    domain (W -> w_max, failed recoveries, pressure fixes) respond to one ulp with > 1e-11;
  * a SECOND step on data with switches (pressure fixes in the cold medium of config 5).

Measurements on the CPU oracle only; nothing here calls the CUDA path, and nothing here pins the
oracle's arithmetic (the pins are in test_oracle_points/_block/_pins2/...).
"""
import numpy as np

from paper_2406_11669_b200 import workloads as wl
from tests.util import cons_errors, make_ref


def _perturbed(w, seed=7):
    """The same workload with every primitive moved by -1, 0 or +1 ulp (seeded)."""
    rng = np.random.default_rng(seed)
    pr = [None if p is None else p * (1.0 + rng.integers(-1, 2, p.shape) * 2.220446049250313e-16)
          for p in w.prims]
    return wl.Workload(**{**w.__dict__, "prims": pr})


def test_config4_one_ulp_response_exceeds_the_bar():
    """c2p_stress at 64^3, one RK3 step: measured 2.3e-11 (D), 1.8e-11 (S), 1.5e-11 (tau), in cells
    that end the step at the Lorentz-factor cap; the B rows (static face field) stay at 1e-13."""
    w = wl.c2p_stress(64)
    a, b = make_ref(w), make_ref(_perturbed(w))
    a.step(1, w.cfl)
    b.step(1, w.cfl)
    e = cons_errors(b.get_cons(), a.get_cons())
    assert max(e["D"], e["Sx"], e["Sy"], e["Sz"], e["tau"]) > 5e-12, e
    assert max(e["Bx"], e["By"], e["Bz"]) < 1e-11, e
    st = a.stats()
    assert st["w_cap"] > 0 and st["c2p_fail"] > 0     # the step does leave the recovery's domain


def test_second_step_amplifies_one_ulp_on_the_bns_block():
    """bns_like(32), upwind CT, RK4: the one-ulp response is 2e-13 after one step and 10x that
    after two (2.6e-12 measured; 5.6e-11 with flux-CT at 64^3): pressure fixes in the cold medium
    between the stars are switches.  north_star's 1e-11 is a ONE-step statement."""
    w = wl.bns_like(32)
    a, b = make_ref(w), make_ref(_perturbed(w))
    for s in (a, b):
        s.set_option("emf", 1.0)
    errs = []
    for _ in range(2):
        a.step(1, w.cfl)
        b.step(1, w.cfl)
        errs.append(max(cons_errors(b.get_cons(), a.get_cons()).values()))
    assert errs[0] < 1e-12 and errs[1] > 3.0 * errs[0], errs
    assert a.stats()["p_fix"] > 1000


def test_blast_history_is_chaotic_under_one_ulp():
    """The 48^3 cylindrical blast over 50 RK3 steps (PPM + flattening, ~1 % of the cell-substeps
    pressure-fixed): two ORACLE runs whose inputs differ by one ulp end 4e-3 apart in the parity
    norm and with different pressure-fix counts (2e-2 after 200 steps at 64^3).  Every pressure
    fix is a switch; once one flips the two runs follow different, equally valid discrete
    histories.  This is why the full-length GPU run of the blast is compared through its step
    count, counters to a relative 2e-3 and a reported drift -- and why 1e-9 after 100 steps is
    asserted on smooth data only (north_star)."""
    w = wl.blast(48)
    a, b = make_ref(w), make_ref(_perturbed(w))
    a.step(50, w.cfl)
    b.step(50, w.cfl)
    e = max(cons_errors(b.get_cons(), a.get_cons()).values())
    sa, sb = a.stats(), b.stats()
    assert e > 1e-6, e
    assert sa["p_fix"] > 100000 and abs(sa["p_fix"] - sb["p_fix"]) <= 2e-3 * sa["p_fix"]
    assert sa["c2p_fail"] == sb["c2p_fail"] == 0
