"""Pins for the oracle's pair potential and the all-pairs force/energy sum (O1).

Each pin is something other than the oracle itself: values another party evaluated from Eq. 1
(golden/two_particle_table.txt), hand-derived closed forms (golden/closed_forms.txt), finite
differences, numerical quadrature by scipy, statistical expectations, symmetries, brute force.
"""
import math
import os

import numpy as np
import pytest
from scipy import integrate

from paper_1412_8502_b200 import inputs

GOLD = os.path.join(os.path.dirname(__file__), "golden")
SPEC = {"np": (0, 1), "nn": (0, 0), "pp": (1, 1)}


def _closed_forms():
    out = {}
    for line in open(os.path.join(GOLD, "closed_forms.txt")):
        line = line.split("#")[0].split()
        if len(line) == 2:
            out[line[0]] = float(line[1])
    return out


def test_p1_two_particle_table(orc):
    """Eq. 1a-c + Table I: V and F of an isolated pair against the stored table."""
    p = orc.Params(r_c=1e9)
    n = 0
    for line in open(os.path.join(GOLD, "two_particle_table.txt")):
        if line.startswith("#") or not line.strip():
            continue
        kind, r, V, F = line.split()
        v, f = orc.pair(p, float(r), *SPEC[kind])
        digits = 1e-4 if kind == "np" and float(r) > 11 else 2e-9
        assert v == pytest.approx(float(V), rel=digits)
        if F != "nan":
            assert f == pytest.approx(float(F), rel=2e-9)
        n += 1
    assert n == 9


def test_p1_table_regenerated_in_long_double():
    """the stored table (the surveyor's evaluation) regenerated here, independently of the oracle, by
    writing Eq. 1a-c with the constants of Table I, alpha hbar c = 1.44 MeV fm and
    lambda = 10 fm in x87 extended precision (numpy.longdouble, 64-bit mantissa) -- V as printed in the
    paper, F = -dV/dr differentiated by hand term by term.  Two independent evaluations of the paper's formula must
    agree to the digits the table prints."""
    ld = np.longdouble
    if np.finfo(ld).nmant < 63:
        pytest.skip("numpy.longdouble is not the x87 extended type on this host")
    a, b, c, Lam, alpha, lam = ld(110), ld(-26), ld(24), ld(5) / ld(4), ld(144) / ld(100), ld(10)
    n = 0
    for line in open(os.path.join(GOLD, "two_particle_table.txt")):
        if line.startswith("#") or not line.strip():
            continue
        kind, r, V, F = line.split()
        r = ld(r)
        B = b - c if kind == "np" else b + c                     # Eq. 1a vs 1b/1c: the sign of c by isospin
        g1, g2 = np.exp(-r * r / Lam), np.exp(-r * r / (2 * Lam))
        v = a * g1 + B * g2                                       # a e^{-r^2/Lambda} + (b -+ c) e^{-r^2/2 Lambda}
        f = (2 * r / Lam) * a * g1 + (r / Lam) * B * g2           # -d/dr of the two Gaussians
        if kind == "pp":
            y = alpha * np.exp(-r / lam) / r                      # Eq. 1c: + alpha e^{-r/lambda} / r
            v, f = v + y, f + y * (1 / r + 1 / lam)
        assert float(v) == pytest.approx(float(V), rel=1e-4 if float(r) > 11 else 2e-9), (kind, r)
        if F != "nan":
            assert float(f) == pytest.approx(float(F), rel=2e-9), (kind, r)
        n += 1
    assert n == 9


def test_p1_pair_in_box_matches_isolated_pair(orc):
    """The N-body sum for N = 2 in a big periodic box reproduces the table: force direction (repulsive
    at 1 fm pushes i away from j), the factor 1/2 in e_i, PE = V."""
    p = orc.Params(r_c=20.0)
    L = 100.0
    for kind, (si, sj) in SPEC.items():
        for r in (1.0, 2.0):
            x = np.array([[10.0, 20.0, 30.0], [10.0 + r, 20.0, 30.0]])
            F, e, PE, diag = orc.forces(x, [si, sj], L, p)
            V, Fr = orc.pair(p, r, si, sj)
            assert PE == pytest.approx(V, rel=1e-14)
            assert e[0] == pytest.approx(0.5 * V, rel=1e-14) and e[1] == pytest.approx(0.5 * V, rel=1e-14)
            # F on particle 0 points along x_0 - x_1 = -r xhat when repulsive
            assert F[0, 0] == pytest.approx(-Fr, rel=1e-13)
            assert F[1, 0] == pytest.approx(+Fr, rel=1e-13)
            assert np.all(F[:, 1:] == 0.0)
            assert diag["ordered_pairs"] == 2


def test_p2_force_is_minus_gradient(orc):
    """F = -dV/dr by central differences, all three species pairs, several r (NORTH STAR pin)."""
    p = orc.Params(r_c=1e9)
    h = 1e-5
    for si, sj in SPEC.values():
        for r in (0.4, 0.9, 1.7, 2.5, 4.0, 7.0):
            vp, _ = orc.pair(p, r + h, si, sj)
            vm, _ = orc.pair(p, r - h, si, sj)
            _, f = orc.pair(p, r, si, sj)
            assert f == pytest.approx(-(vp - vm) / (2 * h), rel=5e-8, abs=1e-10)


def test_p3_np_extremum(orc):
    """The np minimum has a hand-derivable location, depth and curvature (closed_forms.txt)."""
    cf = _closed_forms()
    p = orc.Params(r_c=1e9)
    r0 = math.sqrt(-2 * 1.25 * math.log(5.0 / 22.0))
    assert r0 == pytest.approx(cf["np_minimum_r0_fm"], rel=1e-8)
    V, F = orc.pair(p, r0, 0, 1)
    assert V == pytest.approx(cf["np_minimum_V_MeV"], rel=1e-8)
    assert abs(F) < 1e-12
    h = 1e-4
    curv = -(orc.pair(p, r0 + h, 0, 1)[1] - orc.pair(p, r0 - h, 0, 1)[1]) / (2 * h)
    assert curv == pytest.approx(cf["np_curvature_MeV_fm2"], rel=1e-6)


def test_volume_integrals_by_quadrature(orc):
    """int V d^3r of each Gaussian pair type has a textbook closed form (Gaussian integrals); scipy
    quadrature of the oracle's V(r) must reproduce it -- fails on a swapped Lambda/2Lambda, a wrong
    sign of c, or a/b misplacement.  Screened-Coulomb part: int_0^rc 4 pi r^2 alpha e^{-r/lambda}/r."""
    cf = _closed_forms()
    p = orc.Params(r_c=1e9)

    def vol(si, sj, rmax):
        f = lambda r: 4 * math.pi * r * r * orc.pair(p, r, si, sj)[0]
        return integrate.quad(f, 0, rmax, epsabs=1e-9, epsrel=1e-11, limit=400, points=[1, 2, 4, 8])[0]

    assert vol(0, 0, 30.0) == pytest.approx(cf["I_like_MeV_fm3"], rel=2e-6)
    assert vol(0, 1, 30.0) == pytest.approx(cf["I_np_MeV_fm3"], rel=2e-6)
    for rc, key in ((17.0, "I_c_rc17_MeV_fm3"), (20.0, "I_c_rc20_MeV_fm3")):
        coul = vol(1, 1, rc) - vol(0, 0, rc)
        assert coul == pytest.approx(cf[key], rel=2e-5)


def test_screened_coulomb_is_yukawa(orc):
    """(V_pp - V_nn) r e^{r/lambda} = alpha and F_c r^2 e^{r/lambda}/alpha = 1 + r/lambda
    (Eq. 1c); value at the 20 fm cut-off from closed_forms.txt."""
    cf = _closed_forms()
    p = orc.Params(r_c=1e9)
    for r in (0.5, 3.0, 10.0, 19.99):
        vpp, fpp = orc.pair(p, r, 1, 1)
        vnn, fnn = orc.pair(p, r, 0, 0)
        assert (vpp - vnn) * r * math.exp(r / 10.0) == pytest.approx(1.44, rel=1e-10)
        assert (fpp - fnn) * r * r * math.exp(r / 10.0) / 1.44 == pytest.approx(1 + r / 10.0, rel=1e-10)
    vpp, fpp = orc.pair(p, 20.0, 1, 1)
    assert vpp == pytest.approx(cf["V_c_rc20_MeV"], rel=1e-3)
    assert fpp == pytest.approx(cf["F_c_rc20_MeV_fm"], rel=1e-3)


def test_nuclear_force_negligible_beyond_11p5(orc):
    """"it will rarely register for separations greater than this, even in 64-bit"."""
    p = orc.Params(r_c=1e9)
    V, F = orc.pair(p, 11.5, 0, 1)
    assert 1e-22 < abs(V) < 1e-21 and abs(F) < 1e-20


def test_cutoff_is_strict_and_unshifted(orc):
    """D1/D2: every term is evaluated iff r < r_c; plain truncation, no shift."""
    p = orc.Params(r_c=20.0)
    L = 100.0
    inside = np.array([[1.0, 1.0, 1.0], [1.0 + 19.999999, 1.0, 1.0]])
    outside = np.array([[1.0, 1.0, 1.0], [21.0, 1.0, 1.0]])  # r = 20 exactly
    _, _, PEi, di = orc.forces(inside, [1, 1], L, p)
    _, _, PEo, do = orc.forces(outside, [1, 1], L, p)
    assert PEi == pytest.approx(1.44 * math.exp(-1.9999999) / 19.999999, rel=1e-9)
    assert PEo == 0.0 and do["ordered_pairs"] == 0 and di["ordered_pairs"] == 2


def test_coincident_particles_reading_d2(orc):
    """D2: r = 0 between distinct particles: Gaussian terms as written (V = a + B, zero force),
    Coulomb term skipped."""
    p = orc.Params(r_c=20.0)
    x = np.array([[5.0, 5.0, 5.0], [5.0, 5.0, 5.0]])
    for (si, sj), V0 in (((0, 1), 110 - 50.0), ((0, 0), 110 - 2.0), ((1, 1), 110 - 2.0)):
        F, e, PE, _ = orc.forces(x, [si, sj], 100.0, p)
        assert PE == pytest.approx(V0, rel=1e-15)
        assert np.all(F == 0.0)


def test_nearest_image_across_faces(orc):
    """only the nearest periodic image interacts."""
    p = orc.Params(r_c=17.0)
    L = 40.0
    x = np.array([[0.5, 39.5, 20.0], [39.0, 0.75, 20.0]])  # true separation (1.5, -1.25, 0)
    F, e, PE, _ = orc.forces(x, [0, 1], L, p)
    r = math.hypot(1.5, 1.25)
    V, Fr = orc.pair(p, r, 0, 1)
    assert PE == pytest.approx(V, rel=1e-13)
    assert F[0] == pytest.approx(np.array([1.5, -1.25, 0.0]) / r * Fr, rel=1e-12)


@pytest.mark.parametrize("cfg", [1])
def test_p5_newtons_third_law_and_p6_invariances(orc, cfg):
    c = inputs.CONFIGS[cfg]
    x, v, is_p, L = inputs.uniform_state(512, c["Y_P"], c["density"] * 512 / 512, c["T"], seed=11)
    L = 2.2 * c["r_c"]
    x = x / x.max() * L * 0.999
    p = orc.Params(r_c=c["r_c"])
    F, e, PE, _ = orc.forces(x, is_p, L, p)
    assert np.abs(F.sum(0)).max() <= 1e-12 * np.abs(F).sum()
    assert e.sum() == pytest.approx(PE, rel=1e-14)
    # translation + re-wrap, and a shift by exactly L
    for shift in (np.array([3.7, -11.2, 25.1]), np.array([L, 0.0, -L])):
        F2, _, PE2, _ = orc.forces(orc.wrap(x + shift, L), is_p, L, p)
        assert PE2 == pytest.approx(PE, rel=1e-11)
        assert np.abs(F2 - F).max() <= 1e-9 * np.abs(F).max()
    # permutation within species
    rng = np.random.default_rng(0)
    Np = int(is_p.sum())
    perm = np.concatenate([rng.permutation(Np), Np + rng.permutation(len(is_p) - Np)])
    F3, _, PE3, _ = orc.forces(x[perm], is_p[perm], L, p)
    assert PE3 == pytest.approx(PE, rel=1e-12)
    assert np.abs(F3 - F[perm]).max() <= 1e-10 * np.abs(F).max()
    # reflection x -> L - x flips the force
    F4, _, PE4, _ = orc.forces(orc.wrap(L - x, L), is_p, L, p)
    assert PE4 == pytest.approx(PE, rel=1e-11)
    assert np.abs(F4 + F).max() <= 1e-9 * np.abs(F).max()


@pytest.mark.parametrize("N,ratio", [(64, 3.0), (300, 3.4), (512, 4.2), (400, 5.0)])
def test_p7_all_pairs_vs_cell_list(orc, N, ratio):
    """Brute force vs the independent 27-cell enumeration, incl. particles on cell faces and at 0."""
    p = orc.Params(r_c=6.0)
    L = ratio * p.r_c
    rng = np.random.default_rng(N)
    x = rng.random((N, 3)) * L
    nc = orc.ncell(L, p.r_c, 1)
    w = L / nc
    x[:10] = np.floor(x[:10] / w) * w  # exactly on cell faces
    x[10] = 0.0
    x = orc.wrap(x, L)
    is_p = inputs.species(N, 0.3)
    F, e, PE, d = orc.forces(x, is_p, L, p)
    Fc, ec, PEc, npairs = orc.forces_cells(x, is_p, L, p)
    assert npairs == d["ordered_pairs"]
    assert PEc == pytest.approx(PE, rel=1e-12)
    assert np.abs(Fc - F).max() <= 1e-12 * max(1.0, np.abs(F).max())
    assert np.abs(ec - e).max() <= 1e-12 * max(1.0, np.abs(e).max())


def test_targets_subset_matches_full(orc):
    p = orc.Params(r_c=8.0)
    x, v, is_p, L = inputs.uniform_state(300, 0.3, 0.05, 1.0, seed=4)
    F, e, PE, _ = orc.forces(x, is_p, L, p)
    t = np.array([7, 0, 299, 150])
    Fs, es, PEs, _ = orc.forces(x, is_p, L, p, targets=t)
    assert np.array_equal(Fs, F[t]) and np.array_equal(es, e[t])


def test_p11_ideal_gas_energy_and_p12_neighbour_count(orc):
    """<PE/N> of uniform random positions = (n/2)[(Yp^2+Yn^2) I_like + 2 Yp Yn I_np + Yp^2 I_c]
    and ordered pairs/particle = n (4 pi/3) r_c^3 -- pins the species
    weights, the 1/2, the cut-off and the nearest-image sum statistically."""
    cf = _closed_forms()
    c = inputs.CONFIGS[1]
    N, Y, n = 4096, c["Y_P"], c["density"]
    x, v, is_p, L = inputs.uniform_state(N, Y, n, 1.0, seed=5)
    p = orc.Params(r_c=17.0)
    assert L / 2 > p.r_c
    F, e, PE, d = orc.forces(x, is_p, L, p)
    Yp = is_p.mean()
    Yn = 1 - Yp
    expect = 0.5 * n * ((Yp ** 2 + Yn ** 2) * cf["I_like_MeV_fm3"] + 2 * Yp * Yn * cf["I_np_MeV_fm3"]
                        + Yp ** 2 * cf["I_c_rc17_MeV_fm3"])
    assert expect == pytest.approx(11.27, abs=0.01)  # SURVEY's cfg1 figure
    assert PE / N == pytest.approx(expect, rel=0.06)
    assert d["ordered_pairs"] / N == pytest.approx(n * 4 * math.pi / 3 * 17.0 ** 3, rel=0.01)


def test_range_split_of_the_paper(orc):
    """nuclear terms cut at r_nuc = 11.5 fm, Coulomb not.  Pins of the oracle's r_nuc switch:
    (i) off by default and equal to the single cut-off reading when r_nuc >= r_c; (ii) beyond r_nuc an np/nn pair
    feels nothing and a pp pair exactly the Yukawa term alpha exp(-r/lambda)/r with F = V (1/r + 1/lambda);
    (iii) inside r_nuc nothing changes; (iv) "it will rarely register ... even in 64-bit IEEE arithmetic"
    (PAPER.md:126): on a config-1 system the split changes no force by more than 1e-19 MeV/fm."""
    full, split = orc.Params(r_c=17.0), orc.Params(r_c=17.0, r_nuc=11.5)
    for r in (0.5, 3.0, 11.499):
        for pi, pj in ((0, 0), (0, 1), (1, 1)):
            assert orc.pair(split, r, pi, pj) == orc.pair(full, r, pi, pj)
    for r in (11.5, 12.0, 16.9):
        assert orc.pair(split, r, 0, 0) == (0.0, 0.0) and orc.pair(split, r, 1, 0) == (0.0, 0.0)
        V, F = orc.pair(split, r, 1, 1)
        Vy = 1.44 * math.exp(-r / 10.0) / r
        assert V == pytest.approx(Vy, rel=1e-14) and F == pytest.approx(Vy * (1.0 / r + 0.1), rel=1e-14)
    assert orc.pair(orc.Params(r_c=17.0, r_nuc=17.0), 16.0, 0, 1) == orc.pair(full, 16.0, 0, 1)
    x, v, is_p, L = inputs.config_state(1, seed=4)
    Ff, ef, pef, _ = orc.forces(x, is_p, L, full)
    Fs, es, pes, _ = orc.forces(x, is_p, L, split)
    # F_i and e_i are each summed by one thread in a fixed order: bitwise reproducible, so the split may move them by
    # at most the dropped terms (< 1e-21 each).  The total PE is an OpenMP reduction whose grouping follows the thread
    # count: it is compared to a few ulp of itself (1 ulp of 2.5e4 MeV is 3.6e-12), not to an absolute 1e-16.
    assert np.abs(Ff - Fs).max() < 1e-19 and np.abs(ef - es).max() < 1e-19
    assert abs(pef - pes) <= 4 * np.spacing(abs(pef)) and abs(ef.sum() - es.sum()) < 1e-16


def test_coulomb_without_cutoff_nearest_image_cube(orc):
    """"we do not use a cutoff radius for the Coulomb potential ... each proton interacts with the
    nearest periodic image of every other proton" while the nuclear terms stop at 11.5 fm.  Pins of the oracle's
    coul_nocut switch: (i) a proton pair beyond r_c feels exactly the Yukawa term, repulsive, along the nearest image;
    (ii) past L/2 along an axis the image flips; (iii) the interaction region is the CUBE of side L, not the sphere
    of radius L/2; (iv) np and nn pairs beyond r_nuc feel nothing; (v) on a random system the switch adds exactly the
    proton pairs beyond r_c, summed here independently with numpy; total force stays zero."""
    L = 60.0
    on = orc.Params(r_c=20.0, r_nuc=11.5, coul_nocut=1.0)
    off = orc.Params(r_c=20.0, r_nuc=11.5)
    yuk = lambda r: 1.44 * math.exp(-r / 10.0) / r
    pp = np.array([1, 1], dtype=np.uint8)

    def two(d, is_p, prm):
        x = np.array([[5.0, 5.0, 5.0], [5.0 + d[0], 5.0 + d[1], 5.0 + d[2]]])
        F, e, pe, _ = orc.forces(orc.wrap(x, L), is_p, L, prm)
        return F, pe

    F, pe = two((25.0, 0, 0), pp, on)                       # (i) beyond r_c, inside L/2
    assert pe == pytest.approx(yuk(25.0), rel=1e-14)
    assert F[0] == pytest.approx([-yuk(25.0) * (1 / 25.0 + 0.1), 0, 0], rel=1e-13, abs=1e-18) and np.allclose(F[0], -F[1], rtol=0, atol=1e-18)
    assert two((25.0, 0, 0), pp, off)[1] == 0.0
    F, pe = two((40.0, 0, 0), pp, on)                       # (ii) nearest image is 20 fm away on the other side
    assert pe == pytest.approx(yuk(20.0), rel=1e-14) and F[0, 0] == pytest.approx(+yuk(20.0) * (1 / 20.0 + 0.1), rel=1e-13)
    F, pe = two((25.0, 25.0, 25.0), pp, on)                 # (iii) r = 43.3 fm > L/2 = 30 fm, every component < L/2
    r = 25.0 * math.sqrt(3.0)
    assert pe == pytest.approx(yuk(r), rel=1e-14) and np.allclose(F[0], -yuk(r) * (1 / r + 0.1) / r * 25.0, rtol=1e-13)
    for is_p in (np.array([1, 0], dtype=np.uint8), np.array([0, 0], dtype=np.uint8)):   # (iv)
        F, pe = two((12.0, 0, 0), is_p, on)
        assert pe == 0.0 and not F.any()
    with pytest.raises(ValueError):
        orc.forces(np.zeros((2, 3)), pp, L, orc.Params(r_c=20.0, coul_nocut=1.0))
    # (v) random system: config-1 density, wider box so that L/2 > r_c leaves a shell and corners
    x, v, is_p, Lb = inputs.uniform_state(3000, 0.3, 0.02, 1.0, seed=8)
    Fa, ea, pea, _ = orc.forces(x, is_p, Lb, on)
    Fb, eb, peb, _ = orc.forces(x, is_p, Lb, off)
    xp = x[is_p == 1]
    d = xp[:, None, :] - xp[None, :, :]
    d -= Lb * np.round(d / Lb)
    rr = np.sqrt((d ** 2).sum(-1))
    far = rr >= 20.0
    np.fill_diagonal(far, False)
    extra = 0.5 * (1.44 * np.exp(-rr[far] / 10.0) / rr[far]).sum()
    assert far.sum() > 1e5 and pea - peb == pytest.approx(extra, rel=1e-10)
    gfar = np.where(far, 1.44 * np.exp(-rr / 10.0) / np.where(rr > 0, rr, 1.0) * (1.0 / np.where(rr > 0, rr, 1.0) + 0.1) / np.where(rr > 0, rr, 1.0), 0.0)
    assert np.allclose((Fa - Fb)[is_p == 1], (gfar[:, :, None] * d).sum(1), rtol=1e-9, atol=1e-12)
    assert not (Fa - Fb)[is_p == 0].any()
    assert np.abs(Fa.sum(0)).max() <= 1e-10 * np.abs(Fa).sum()
