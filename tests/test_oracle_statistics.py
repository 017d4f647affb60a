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


def test_original_dpd_equation_of_state():
    """Figure 3(a) of the paper: the original DPD model, a_ij = 25 (A = +25, B = 0 in Eq. (1)), kT = 1, gamma = 4.5:
    p = rho kT + 0.1 a rho^2 = 67.5 at rho = 5 (the quadratic form is the high-density limit of the measured EOS: 5 %)."""
    L, dens = 6.0, 5.0
    c = wl.make_liquid(L, density=dens, seed=6, A=25.0, B=0.0)
    s = RefSim(c["params"])
    s.load_particles(c["pos"], c["vel"])
    s.step(400)
    n, V = len(c["pos"]), L ** 3
    ps = []
    for _ in range(120):
        s.step(5)
        ps.append(n * kinetic_temperature(s.get_state()["vel"]) / V + s.counters()["virial_c"] / (3 * V))
    p_ref = dens + 0.1 * 25.0 * dens ** 2
    assert p_ref == 67.5
    assert abs(np.mean(ps) - p_ref) < 0.05 * p_ref, np.mean(ps)


def shear_wave_viscosity():
    """Kinematic viscosity of the periodic mDPD liquid, no walls, no body force: a transverse velocity wave
    v_x = A sin(k z) decays as exp(-nu k^2 t) (linearised Navier-Stokes).  8 x 8 x 12 box, k = 2 pi / 12, A = 1; the
    amplitude is the Fourier projection (2 / N) sum v_x sin(k z), fitted while it is above 0.25 (noise sqrt(2 / N) = 0.02)."""
    box = (8.0, 8.0, 12.0)
    c = wl.make_liquid(box, seed=11)
    n = len(c["pos"])
    s = RefSim(c["params"])
    s.load_particles(c["pos"].astype(np.float64), c["vel"].astype(np.float64), c["type"])
    s.step(300)                                    # equilibrate the random start
    st = s.get_state()
    k = 2.0 * np.pi / box[2]
    v = st["vel"].copy()
    v[:, 0] += np.sin(k * st["pos"][:, 2])
    s2 = RefSim(c["params"])
    s2.load_particles(st["pos"], v, c["type"])
    ts, am = [], []
    for it in range(80):
        s2.step(5)
        q = s2.get_state()
        am.append(2.0 / n * np.sum(q["vel"][:, 0] * np.sin(k * q["pos"][:, 2])))
        ts.append((it + 1) * 5 * c["params"]["dt"])
    ts, am = np.array(ts), np.array(am)
    sel = am > 0.25
    assert sel.sum() > 40
    slope = np.polyfit(ts[sel], np.log(am[sel]), 1)[0]
    resid = np.abs(np.log(am[sel]) - np.polyval(np.polyfit(ts[sel], np.log(am[sel]), 1), ts[sel])).max()
    assert resid < 0.08                             # a clean exponential
    return -slope / k ** 2


def test_poiseuille_parabola_no_slip_and_viscosity():
    """Body-force driven flow between flat frozen walls (BASELINE config 2, scaled to 8 x 8 x 12), SURVEY.md S8c:
    (i)  v_x(z) = (rho g / 2 mu)(z - z_a)(z_b - z): quadratic-fit residual < 3 % of v_max (1-rc bins, 384 particles each,
         900 samples 5 steps apart: ~0.7 % noise per bin);
    (ii) fitted zeros within 0.3 of the wall faces z = 2, 10 (no slip);
    (iii) the viscosity from the curvature, mu = rho g / (2 |a_2|), against the viscosity of the SAME liquid measured
         with no wall and no body force at all (decay of a transverse velocity wave in a periodic box, above): within
         10 % (two independent noisy measurements: ~3 % each; measured 5.56 vs 5.25)."""
    c = wl.make_poiseuille(L=12.0, wall=2.0, gx=0.05, seed=7, Lxy=8.0)
    s = RefSim(c["params"])
    s.load_particles(c["pos"], c["vel"], c["type"])
    s.load_wall_mask(c["mask"], c["voxel"])
    fl = c["type"] == 0
    s.step(1500)
    nb = 8
    acc, cnt = np.zeros(nb), np.zeros(nb)
    for _ in range(900):
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
    assert resid < 0.03, resid
    mu_channel = 6.0 * 0.05 / (2.0 * abs(co[0]))
    mu_wave = 6.0 * shear_wave_viscosity()
    assert abs(mu_channel / mu_wave - 1.0) < 0.10, (mu_channel, mu_wave)
    # walls hold: every fluid particle is still in the pore, wall particles did not move
    st = s.get_state()
    assert (st["pos"][fl, 2] >= 2.0).all() and (st["pos"][fl, 2] < 10.0).all()
    assert (st["pos"][~fl] == c["pos"][~fl].astype(np.float64)).all()
    assert s.counters()["bounces"] > 0
    # flat density profile across the channel (no depletion / pile-up beyond 6 %)
    assert np.abs(cnt / cnt.mean() - 1).max() < 0.06
