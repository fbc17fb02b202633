"""Pins for the oracle's integrator (O2): velocity Verlet, isokinetic rescale, uniform scaling."""
import math
import os

import numpy as np
import pytest

from paper_1412_8502_b200 import inputs

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _cf(name):
    for line in open(os.path.join(GOLD, "closed_forms.txt")):
        t = line.split("#")[0].split()
        if len(t) == 2 and t[0] == name:
            return float(t[1])
    raise KeyError(name)


def test_p4_two_body_small_oscillation_period(orc):
    """An np pair released near the potential minimum oscillates with period 2 pi / sqrt(V''/mu),
    mu = M/2 (closed_forms.txt) and its centre of mass stays put -- pins force sign, the 1/M in the
    kicks, the half-kick/drift order and dt handling together."""
    p = orc.Params(r_c=20.0)
    r0 = _cf("np_minimum_r0_fm")
    amp = 0.004
    L = 100.0
    x = np.array([[50.0 - (r0 + amp) / 2, 50.0, 50.0], [50.0 + (r0 + amp) / 2, 50.0, 50.0]])
    v = np.zeros((2, 3))
    is_p = [0, 1]
    dt = 0.05
    sep = []
    F = None
    cnt = 0
    for _ in range(1400):
        x, v, L, cnt, F, _ = orc.step(x, v, is_p, L, p, 1.0, 0, 1.0, dt, 1, cnt, F)
        sep.append(x[1, 0] - x[0, 0] - r0)
    sep = np.array(sep)
    # successive downward zero crossings of (r - r0) -> period
    idx = np.where((sep[:-1] > 0) & (sep[1:] <= 0))[0]
    t = (idx + sep[idx] / (sep[idx] - sep[idx + 1]) + 1) * dt
    period = np.diff(t).mean()
    assert period == pytest.approx(_cf("np_small_oscillation_period_fm_c"), rel=2e-3)
    assert x.mean(0) == pytest.approx([50.0, 50.0, 50.0], abs=1e-12)
    assert cnt == 1400


def _total_energy(orc, x, v, is_p, L, p):
    return orc.forces(x, is_p, L, p)[2] + orc.kinetic(v, p.mass)


@pytest.mark.parametrize("Y_P", [0.0])
def test_p8_energy_error_scales_as_dt_squared(orc, Y_P):
    """NVE: the velocity-Verlet energy error is O(dt^2): halving dt cuts it ~4x.  A pure-neutron
    system is used so the potential is smooth at r_c (nuclear terms ~1e-49 there, D1)."""
    p = orc.Params(r_c=11.5)
    N = 512
    x, v, is_p, L = inputs.uniform_state(N, Y_P, 0.04, 1.0, seed=21)
    # relax overlaps a little so that forces are moderate: spread on a jittered lattice
    g = int(round(N ** (1 / 3) + 0.5))
    lat = np.array([[i, j, k] for i in range(g) for j in range(g) for k in range(g)][:N], dtype=float)
    x = orc.wrap((lat + 0.5) * (L / g) + 0.15 * (x / L - 0.5), L)
    assert L / 2 > p.r_c
    E0 = _total_energy(orc, x, v, is_p, L, p)
    errs = []
    for dt in (1.0, 0.5, 0.25):
        n = int(round(40.0 / dt))
        xs, vs, Ls, _, _, _ = orc.step(x, v, is_p, L, p, 1.0, 0, 1.0, dt, n)
        errs.append(abs(_total_energy(orc, xs, vs, is_p, Ls, p) - E0))
    assert errs[0] / errs[1] == pytest.approx(4.0, rel=0.35)
    assert errs[1] / errs[2] == pytest.approx(4.0, rel=0.35)
    assert errs[2] < 1e-3 * abs(E0)


def test_time_reversibility(orc):
    """Velocity Verlet is time reversible: run n steps, flip v, run n steps, recover x."""
    p = orc.Params(r_c=10.0)
    x, v, is_p, L = inputs.uniform_state(100, 0.3, 0.02, 1.0, seed=3)
    x1, v1, L1, _, F1, _ = orc.step(x, v, is_p, L, p, 1.0, 0, 1.0, 0.5, 25)
    x2, v2, _, _, _, _ = orc.step(x1, -v1, is_p, L1, p, 1.0, 0, 1.0, 0.5, 25, 0, F1)
    d = x2 - x
    d -= L * np.round(d / L)
    assert np.abs(d).max() < 1e-9
    assert np.abs(v2 + v).max() < 1e-11


def test_kinetic_energy_hand_values(orc):
    """orc_kinetic = sum 1/2 M |v|^2 against values worked by hand, so that the prefactor is pinned by
    something other than the thermostat that uses it: one nucleon at v = (0.1, 0, 0) c carries 1/2 939 0.01 = 4.695 MeV;
    components add in quadrature; particles add."""
    assert orc.kinetic(np.array([[0.1, 0.0, 0.0]]), 939.0) == pytest.approx(4.695, rel=1e-15)
    assert orc.kinetic(np.array([[0.3, -0.4, 0.0]]), 2.0) == pytest.approx(0.25, rel=1e-15)
    assert orc.kinetic(np.array([[0.1, 0, 0], [0, 0.2, 0], [0, 0, -0.2]]), 100.0) == pytest.approx(0.5 + 2.0 + 2.0, rel=1e-15)
    assert orc.kinetic(np.zeros((5, 3)), 939.0) == 0.0
    # and the thermostat target of PAPER.md:110: mean KE per particle 3/2 T  <=>  KE = 3/2 N T
    v = np.full((1000, 3), math.sqrt(0.75 / 939.0))
    assert orc.kinetic(v, 939.0) == pytest.approx(1.5 * 1000 * 0.75, rel=1e-14)


def test_p9_thermostat(orc):
    """After a rescale step sum 1/2 M v^2 = (3/2) N T exactly; only on steps whose
    1-based count is a multiple of the interval, counter persisting across calls (D7)."""
    p = orc.Params(r_c=10.0)
    N, T = 120, 0.75
    x, v, is_p, L = inputs.uniform_state(N, 0.2, 0.02, 3.0, seed=8)
    xs, vs, Ls, cnt, F, _ = orc.step(x, v, is_p, L, p, T, 10, 1.0, 1.0, 9)
    assert orc.kinetic(vs, p.mass) != pytest.approx(1.5 * N * T, rel=1e-3)
    xs, vs, Ls, cnt, F, _ = orc.step(xs, vs, is_p, Ls, p, T, 10, 1.0, 1.0, 1, cnt, F)
    assert cnt == 10
    assert orc.kinetic(vs, p.mass) == pytest.approx(1.5 * N * T, rel=1e-13)
    xs, vs, Ls, cnt, F, _ = orc.step(xs, vs, is_p, Ls, p, T, 10, 1.0, 1.0, 3, cnt, F)
    assert orc.kinetic(vs, p.mass) != pytest.approx(1.5 * N * T, rel=1e-6)
    # interval 0 = off: equals plain NVE
    a = orc.step(x, v, is_p, L, p, T, 0, 1.0, 1.0, 12)
    b = orc.step(x, v, is_p, L, p, 99.0, 0, 1.0, 1.0, 12)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])


def test_p10_uniform_scaling(orc):
    """pasta_expand(s): every pair distance x s, density / s^3, velocities untouched (D9); 20 000
    fused steps at s = 4^(1/20000) give L/L0 = 4, i.e. n 0.08 -> 0.00125."""
    p = orc.Params(r_c=10.0)
    x, v, is_p, L = inputs.uniform_state(50, 0.4, 0.02, 1.0, seed=9)
    s = 1.37
    xs, Ls = orc.expand(x, L, s)
    assert Ls == L * s

    def pd(x, L):
        d = x[:, None, :] - x[None, :, :]
        d -= L * np.round(d / L)
        return np.sqrt((d ** 2).sum(-1))

    assert np.allclose(pd(xs, Ls), s * pd(x, L), rtol=1e-12, atol=1e-10)
    sps = inputs.CONFIGS[3]["scale_per_step"]
    assert sps == pytest.approx(1.0000693171203765, rel=1e-15)
    Lk = 86.1774
    for _ in range(20000):
        Lk = sps * Lk
    assert Lk / 86.1774 == pytest.approx(4.0, rel=1e-10)
    assert 0.08 / 4.0 ** 3 == pytest.approx(0.00125)


def test_fused_scaling_step_matches_definition(orc):
    """O2 with s != 1: x' = s (x + dt v'), L' = s L, wrapped into [0, L'); with zero forces (single
    particle) the result is checked by hand."""
    p = orc.Params(r_c=5.0)
    x = np.array([[39.0, 1.0, 20.0]])
    v = np.array([[0.9, -0.8, 0.0]])
    L, s, dt = 40.0, 1.01, 2.0
    xs, vs, Ls, cnt, F, PE = orc.step(x, v, [0], L, p, 1.0, 0, s, dt, 1)
    assert Ls == pytest.approx(40.4)
    exp = np.array([[s * (39.0 + 1.8), s * (1.0 - 1.6), s * 20.0]])
    exp -= Ls * np.floor(exp / Ls)
    assert xs == pytest.approx(exp, abs=1e-12)
    assert np.array_equal(vs, v) and PE == 0.0
    assert (xs >= 0).all() and (xs < Ls).all()


def test_wrap_edge_cases(orc):
    L = 10.0
    x = np.array([[0.0, -0.0, 10.0], [-1e-18, 9.999999999999998, 25.0], [-10.0, -3.0, 1e-300]])
    w = orc.wrap(x, L)
    assert (w >= 0).all() and (w < L).all()
    assert w[0, 2] == 0.0 and w[1, 0] == 0.0 and w[1, 2] == 5.0 and w[2, 1] == 7.0


def test_maxwell_boltzmann_inputs():
    """P15 on the shared generator: mean 0, variance T/M per component (reading D15)."""
    x, v, is_p, L = inputs.uniform_state(51200, 0.4, 0.08, 1.0, seed=1)
    assert L == pytest.approx(86.1774, abs=1e-4)
    assert is_p.sum() == 20480 and is_p[:20480].all()
    assert abs(v.mean()) < 4 * math.sqrt(1.0 / 939.0) / math.sqrt(v.size)
    assert v.var() == pytest.approx(1.0 / 939.0, rel=4 * math.sqrt(2.0 / v.size))
    assert (x >= 0).all() and (x < L).all()
    assert inputs.n_protons(2048, 0.30) == 614 and inputs.n_protons(409600, 0.30) == 122880


def test_linear_box_only_expansion_of_the_paper(orc):
    """PAPER.md:100-108, Eq. 3a (reading D25).  Pins: (i) l(t) = l(0)(1 + xi_dot t) exactly as written, after any
    number of steps and across calls; (ii) positions are NOT scaled: with the potential switched off a particle
    that crosses no face moves as x0 + v t to rounding while the box grows by 50 %; (iii) a particle that does
    cross re-enters at x - L of the box it left, with its velocity unchanged; (iv) xi_dot = 0 is
    plain velocity Verlet (identical to orc.step with s = 1)."""
    free = orc.Params(a=0.0, b=0.0, c=0.0, alpha=0.0, r_c=5.0)
    L0, xi, dt = 40.0, 5e-3, 2.0
    x = np.array([[10.0, 20.0, 30.0], [39.5, 5.0, 5.0]])
    v = np.array([[0.01, -0.02, 0.005], [0.1, 0.0, 0.0]])
    is_p = np.array([1, 0], dtype=np.uint8)
    xo, vo, L, ne, cnt, F, pe = orc.step_linear(x, v, is_p, L0, xi, free, 1.0, 0, dt, 50)
    assert L == L0 * (1.0 + xi * (dt * 50.0)) and ne == 50 and cnt == 50
    assert np.allclose(xo[0], x[0] + v[0] * 100.0, rtol=0, atol=1e-12) and np.array_equal(vo, v)
    # particle 1 leaves the box of side L0 (1 + xi dt 2) = 40.8 during step 3 (x = 40.1 after it is drifted in a
    # box that has grown twice) ... track it by hand
    xs, Ls = 39.5, L0
    for n in range(1, 51):
        xs = xs + 0.1 * dt
        if xs >= Ls:
            xs -= Ls
        Ls = L0 * (1.0 + xi * (dt * n))
    assert xo[1, 0] == pytest.approx(xs, abs=1e-12)
    x2, v2, L2, ne2, cnt2, _, _ = orc.step_linear(xo, vo, is_p, L0, xi, free, 1.0, 0, dt, 25, n_exp=ne, step_count=cnt)
    assert L2 == L0 * (1.0 + xi * (dt * 75.0)) and ne2 == 75
    xr, vr, isr, Lr = inputs.uniform_state(64, 0.3, 0.02, 1.0, seed=3)
    prm = orc.Params(r_c=5.0)
    a = orc.step_linear(xr, vr, isr, Lr, 0.0, prm, 1.0, 10, 2.0, 12)
    b = orc.step(xr, vr, isr, Lr, prm, 1.0, 10, 1.0, 2.0, 12)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1]) and a[2] == b[2]
