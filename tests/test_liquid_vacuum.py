"""Section 4.1 of the paper: liquid-vacuum interface, A = -50, B = 25, rd = 0.75 rc, gamma = 12.4, fcc
start in |x| <= 10 rc, 5 000 steps to equilibrate, 5 000 steps of averaging, density profile in 2 rc bins along x.
The paper PRINTS the density at the centre of the slab: 6.88 ("for both USER-MESO 2.5 and our CPU code, matching the
value reported in Ghoufi and Malfreyt").  The oracle is pinned to it on a reduced slab (CPU), the CUDA path reproduces
the paper's full-size run (100^3 box, 820 000 particles).  Both give 6.81-6.82, 1 % below the printed value, inside the
1.5 % tolerance used here (R20); the closed-form EOS of PAPER.md L89 puts the zero-pressure density at 6.85.
The paper also PRINTS the interfacial tension gamma_WV = 12.4: the oracle gives 12.3 +- 0.3 on the reduced slab, the
CUDA path 12.37 +- 0.02 on the full-size run (conservative virial + kinetic part, R21)."""
import numpy as np
import pytest

import mdpd_workloads as wl

PAPER_CENTRE_DENSITY = 6.88
PAPER_TENSION = 12.4            # gamma_WV "is 12.4 for both USER-MESO 2.5 and its CPU counterpart"
TOL = 0.015


def test_workload_is_the_papers():
    c = wl.make_liquid_vacuum()
    assert len(c["pos"]) == 820_000
    assert c["params"]["A"] == -50.0 and c["params"]["B"] == 25.0 and c["params"]["rd"] == 0.75
    assert abs(c["params"]["sigma"] ** 2 - 2 * 12.4 * 1.0) < 1e-9     # sigma^2 = 2 gamma kT
    x = c["pos"][:, 0]
    assert x.min() == 40.0 and x.max() == 60.0                        # |x - 50| <= 10


def pressure_diag(vel, W, volume):
    """P_aa = (sum_i m v_a^2 + sum_pairs r_a F^C_a) / V, a = x, y, z (mass 1; conservative virial, R21)."""
    v = np.asarray(vel, np.float64)
    return np.array([((v[:, a] ** 2).sum() + W[a]) / volume for a in range(3)])


def test_oracle_slab_centre_density_and_tension_match_the_paper():
    """Reduced slab (24 x 7 x 7 box, 2 450 particles): the bulk density of the slab and the tension of its two flat
    interfaces are intensive.  gamma_WV = (L_x / 2) <P_xx - (P_yy + P_zz) / 2> (the 1/2 is for the two
    interfaces, R21)."""
    from oracle.mdpd_ref import RefSim
    c = wl.make_liquid_vacuum(L=24.0, Lyz=7.0, half_width=6.0)
    Lx, V = 24.0, 24.0 * 7.0 * 7.0
    s = RefSim(c["params"])
    s.load_particles(c["pos"].astype(np.float64), c["vel"].astype(np.float64), c["type"])
    s.step(2000)
    dens, g = [], []
    for k in range(2000):
        s.step(1)
        st = s.get_state()
        P = pressure_diag(st["vel"], s.virial(), V)
        g.append(P[0] - 0.5 * (P[1] + P[2]))
        if k % 50 == 49:
            x = st["pos"][:, 0]
            dens.append((np.abs(x - x.mean()) < 1.5).sum() / (3.0 * 7.0 * 7.0))
    rho = float(np.mean(dens))
    assert abs(rho / PAPER_CENTRE_DENSITY - 1.0) < TOL, rho
    # regression guard on the oracle itself: this seeded, serial run gives 6.817 (0.9 % under the printed 6.88, DESIGN.md
    # R20); the 1.5 % band above is centred on the paper's value and would let the oracle drift to 6.78 or 6.98 unnoticed
    assert abs(rho - 6.82) < 0.05, rho
    gamma = 0.5 * Lx * float(np.mean(g))
    assert abs(gamma - PAPER_TENSION) < 1.0, gamma      # 12.28 +- 0.27 (block averages) on this small slab


@pytest.mark.gpu
def test_gpu_full_size_run_reproduces_the_papers_density_and_tension():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("the -m gpu suite needs a CUDA device (no CPU fallback exists)")
    import paper_1903_10134_b200 as pk
    pk.build()
    c = wl.make_liquid_vacuum()
    c["params"]["headroom"] = 2.0               # the fcc start (density 4) contracts to a liquid of density 6.9
    sim = pk.Simulation(c["params"])
    sim.load_particles(c["pos"], c["vel"], c["type"])
    sim.step(5000)                              # equilibration
    hist = np.zeros(50)
    nsamp = 0
    g = []
    for k in range(250):                        # 5 000 steps of averaging: stress every 20 steps, profile every 100
        sim.step(20)
        st = sim.get_state(pos=(k % 5 == 4), force=False, rho=False)
        P = pressure_diag(st["vel"], sim.compute_virial(), 100.0 ** 3)
        g.append(P[0] - 0.5 * (P[1] + P[2]))
        if k % 5 == 4:
            hist += np.histogram(st["pos"][:, 0], bins=50, range=(0.0, 100.0))[0]   # 2 rc bins along x
            nsamp += 1
    assert sim.counters()["faults"] == 0
    prof = hist / nsamp / (2.0 * 100.0 * 100.0)
    centre = float(prof[24:26].mean())          # the two bins around x = 50 (the paper's x = 0)
    assert abs(centre / PAPER_CENTRE_DENSITY - 1.0) < TOL, (centre, prof[18:32])
    assert prof[:18].sum() == 0.0 and prof[32:].sum() == 0.0        # vacuum outside the slab
    assert abs(prof[23:27] - centre).max() < 0.02                   # flat plateau
    gamma = 0.5 * 100.0 * float(np.mean(g))     # the paper's second printed value: 12.4; measured here 12.37 +- 0.02
    assert abs(gamma - PAPER_TENSION) < 0.25, gamma
