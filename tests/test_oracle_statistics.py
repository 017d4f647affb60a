"""Statistical pins of the fp64 oracle (no GPU): thermostat, equation of state, Poiseuille flow.

P:L<n> = /root/reference/PAPER.md line n; R<n> = DESIGN.md reading n.  Boxes are smaller than the
paper's 10^3 so that the whole CPU suite stays within a few minutes; tolerances cover the
statistical error of the shorter averages and, for the EOS, the accuracy of the paper's fitted form.
"""
import math

import numpy as np
import pytest

import mdpd_workloads as wl
from oracle.mdpd_ref import RefSim

from helpers import kinetic_temperature, profile


def eos_paper(rho, A=-40.0, B=25.0, rd=0.75, kT=1.0, alpha=0.101, c=4.16, d=18.0):
    """P:L89 Fig. 3(b): p = rho kT + alpha A rho^2 + 2 alpha B rd^4 (rho^3 - c rho^2 + d)   (R13)."""
    return rho * kT + alpha * A * rho ** 2 + 2 * alpha * B * rd ** 4 * (rho ** 3 - c * rho ** 2 + d)


@pytest.mark.parametrize("dens", [6.5, 7.0, 8.0])
def test_thermostat_and_equation_of_state(dens):
    """sigma^2 = 2 gamma kT => equilibrium kT = 1 within 2 % at dt = 0.01 (BASELINE north_star);
    virial pressure vs the paper's closed-form mDPD EOS: p(6.5) = 22.5, p(7) = 60.2, p(8) = 170.9."""
    L = 6.0
    c = wl.make_liquid(L, density=dens, seed=5)
    s = RefSim(c["params"])
    s.load_particles(c["pos"], c["vel"])
    s.step(600)
    n, V = len(c["pos"]), L ** 3
    kts, ps = [], []
    for _ in range(200):
        s.step(5)
        kt = kinetic_temperature(s.get_state()["vel"])
        kts.append(kt)
        ps.append(n * kt / V + s.counters()["virial_c"] / (3 * V))
    assert abs(np.mean(kts) - 1.0) < 0.02
    p_ref = eos_paper(dens)
    assert abs(p_ref - {6.5: 22.5, 7.0: 60.2, 8.0: 170.9}[dens]) < 0.06   # the paper's formula, evaluated by hand
    assert abs(np.mean(ps) - p_ref) < max(0.05 * p_ref, 2.0), (np.mean(ps), p_ref)


def test_poiseuille_parabola_and_no_slip():
    """Body-force driven flow between flat frozen walls (BASELINE config 2, scaled to 6 x 6 x 12):
    v_x(z) = (rho g / 2 mu)(z - z_a)(z_b - z): quadratic-fit residual small, zeros at the walls (no slip)."""
    c = wl.make_poiseuille(L=12.0, wall=2.0, gx=0.05, seed=7, Lxy=6.0)
    s = RefSim(c["params"])
    s.load_particles(c["pos"], c["vel"], c["type"])
    s.load_wall_mask(c["mask"], c["voxel"])
    fl = c["type"] == 0
    s.step(1500)
    nb = 16
    acc, cnt = np.zeros(nb), np.zeros(nb)
    for _ in range(600):
        s.step(5)
        st = s.get_state()
        ctr, m, k = profile(st["pos"][fl, 2], st["vel"][fl, 0], 2.0, 10.0, nb)
        acc += m * k
        cnt += k
    v = acc / cnt
    co = np.polyfit(ctr, v, 2)
    roots = np.sort(np.roots(co).real)
    resid = np.abs(v - np.polyval(co, ctr)).max() / v.max()
    assert co[0] < 0 and 0.25 < v.max() < 0.8
    assert abs(roots[0] - 2.0) < 0.3 and abs(roots[1] - 10.0) < 0.3, roots
    assert resid < 0.08, resid
    # walls hold: every fluid particle is still in the pore, wall particles did not move
    st = s.get_state()
    assert (st["pos"][fl, 2] >= 2.0).all() and (st["pos"][fl, 2] < 10.0).all()
    assert (st["pos"][~fl] == c["pos"][~fl].astype(np.float64)).all()
    assert s.counters()["bounces"] > 0
    # flat density profile across the channel (no depletion / pile-up beyond 6 %)
    assert np.abs(cnt / cnt.mean() - 1).max() < 0.06
