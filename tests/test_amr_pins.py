"""CPU pins of the NEXT-3 oracle (oracle/z4c_amr.hpp): restriction and prolongation at a factor-2 refinement
boundary by Lagrange interpolation, PAPER.md:98-118 (Eq. 1 at 104, Eq. 2 at 108, stencil n = N_g + 1 at 112,
"always within the active region" at 114), and the two-level step of PAPER.md:69-88 / the test of PAPER.md:171.
Each pin checks the oracle against something other than itself: exact rational arithmetic, polynomial exactness,
the stated order of convergence, closed-form data."""
from dataclasses import replace
from fractions import Fraction

import numpy as np
import pytest

from paper_2409_10383_b200 import inputs as I


def lagrange_exact(nodes, x):
    """Eq. (1) in exact rational arithmetic (product over m != i, reading Q17)."""
    out = []
    for i, xi in enumerate(nodes):
        l = Fraction(1)
        for m, xm in enumerate(nodes):
            if m != i:
                l *= (Fraction(x) - xm) / (Fraction(xi) - xm)
        out.append(l)
    return out


@pytest.mark.parametrize("ng", [2, 3, 4])
def test_A1_weights_against_exact_rationals(oracle, ng):
    n, nf = ng + 1, 16
    for Il in range(nf // 2):
        s, w = oracle.restrict_weights(Il, ng, nf)
        assert 0 <= s and s + n <= nf                                   # inside the active region
        ex = lagrange_exact(range(s, s + n), Fraction(4 * Il + 1, 2))    # the coarse node sits at 2 Il + 1/2
        assert np.array_equal(w, [float(e) for e in ex])                # exact dyadic rationals (R-I1)
        assert sum(ex) == 1
        # Q21: unless a block face forces a shift, the stencil holds the n nodes nearest to the target
        free = 2 * Il + 1 - (n + 1) // 2
        if 0 <= free <= nf - n:
            assert s == free
            d_in = max(abs(q - (2 * Il + 0.5)) for q in range(s, s + n))
            d_out = min(abs(q - (2 * Il + 0.5)) for q in (s - 1, s + n))
            assert d_in <= d_out
    for i in range(-2 * ng, 2 * ng + 4):
        s, w = oracle.prolong_weights(i, ng)
        X = Fraction(2 * i + 1, 4) - Fraction(1, 2)                     # fine node i in coarse-index units
        ex = lagrange_exact(range(s, s + n), X)
        assert np.array_equal(w, [float(e) for e in ex])                # exact dyadic rationals (R-I1)
        d_in = max(abs(q - float(X)) for q in range(s, s + n))         # Q22: the n nearest coarse nodes
        d_out = min(abs(q - float(X)) for q in (s - 1, s + n))
        assert d_in <= d_out
    if ng == 3:   # the numbers themselves: symmetric interior stencil and the lopsided one next to a face
        assert np.array_equal(oracle.restrict_weights(3, 3, 16)[1], np.array([-1, 9, 9, -1]) / 16.0)
        assert np.array_equal(oracle.restrict_weights(0, 3, 16)[1], np.array([5, 15, -5, 1]) / 16.0)
        assert np.array_equal(oracle.restrict_weights(7, 3, 16)[1], np.array([1, -5, 15, 5]) / 16.0)
        assert np.array_equal(oracle.prolong_weights(-2, 3)[1], np.array([-5, 35, 105, -7]) / 128.0)
        assert np.array_equal(oracle.prolong_weights(-1, 3)[1], np.array([-7, 105, 35, -5]) / 128.0)


def poly3(z, y, x, a, b, c):
    return x ** a * y ** b * z ** c


@pytest.mark.parametrize("ng", [2, 3, 4])
def test_A2_both_operators_exact_on_degree_ng_polynomials(oracle, ng):
    """n = N_g + 1 points per axis reproduce every monomial x^a y^b z^c with a, b, c <= N_g (tensor product)."""
    nf, h = 8 if ng < 4 else 10, 0.1
    Nf = 2 * nf
    xf = (np.arange(Nf) + 0.5) * h
    xc = (np.arange(Nf // 2) + 0.5) * 2 * h
    rng = np.random.default_rng(ng)
    for _ in range(6):
        a, b, c = rng.integers(0, ng + 1, 3)
        fine = poly3(xf[:, None, None], xf[None, :, None], xf[None, None, :], a, b, c)[None]
        want = poly3(xc[:, None, None], xc[None, :, None], xc[None, None, :], a, b, c)
        got = oracle.restrict(fine, ng, nf)[0]
        assert np.abs(got - want).max() <= 2e-13 * max(1.0, np.abs(want).max()), (a, b, c)
    # prolongation: coarse 12^3 (outflow so nothing wraps), fine box at coarse cell (4,4,4), ghost shell of width ng
    Nc, o = 12, (4, 4, 4)
    X = (np.arange(Nc) + 0.5) * 2 * h
    lo, hi = (-ng,) * 3, (8 + ng,) * 3
    xg = (2 * o[0] + np.arange(lo[0], hi[0]) + 0.5) * h
    for _ in range(6):
        a, b, c = rng.integers(0, ng + 1, 3)
        coarse = poly3(X[:, None, None], X[None, :, None], X[None, None, :], a, b, c)[None]
        want = poly3(xg[:, None, None], xg[None, :, None], xg[None, None, :], a, b, c)
        got = oracle.prolong(coarse, ng, 1, o, lo, hi)[0]
        assert np.abs(got - want).max() <= 2e-13 * max(1.0, np.abs(want).max()), (a, b, c)
    # one degree more is NOT reproduced (the stencil is no wider than claimed)
    fine = (xf[None, None, :] ** (ng + 1) * np.ones((Nf, Nf, 1)))[None]
    assert np.abs(oracle.restrict(fine, ng, nf)[0] - xc[None, None, :] ** (ng + 1)).max() > 1e-9


def test_A3_restriction_never_leaves_the_active_region_of_its_block(oracle):
    """PAPER.md:114. Every fine MeshBlock carries its own cubic polynomial (discontinuous across block faces): the
    restricted values are exact block by block only if no stencil reaches into a neighbouring block."""
    ng, nf, nb = 3, 8, 2
    Nf = nf * nb
    h = 0.25
    xf = (np.arange(Nf) + 0.5) * h
    xc = (np.arange(Nf // 2) + 0.5) * 2 * h
    rng = np.random.default_rng(5)
    coef = rng.uniform(-1, 1, (nb, nb, nb, 4))

    def field(z, y, x, bz, by, bx):
        k = coef[bz, by, bx]
        return k[0] + k[1] * x ** 3 + k[2] * y ** 2 * z + k[3] * x * y * z

    fine = np.empty((1, Nf, Nf, Nf))
    want = np.empty((Nf // 2,) * 3)
    for bz in range(nb):
        for by in range(nb):
            for bx in range(nb):
                sf = lambda b: slice(b * nf, (b + 1) * nf)
                sc = lambda b: slice(b * nf // 2, (b + 1) * nf // 2)
                fine[0, sf(bz), sf(by), sf(bx)] = field(xf[sf(bz), None, None], xf[None, sf(by), None],
                                                        xf[None, None, sf(bx)], bz, by, bx)
                want[sc(bz), sc(by), sc(bx)] = field(xc[sc(bz), None, None], xc[None, sc(by), None],
                                                     xc[None, None, sc(bx)], bz, by, bx)
    got = oracle.restrict(fine, ng, nf)[0]
    assert np.abs(got - want).max() <= 1e-12


@pytest.mark.parametrize("ng", [2, 3, 4])
def test_A4_order_of_convergence(oracle, ng):
    """the interpolation error falls at order n = N_g + 1 (3rd for 2 ghosts, 5th for 4 ghosts)."""
    n = ng + 1
    errs_r, errs_p = [], []
    f = lambda z, y, x: np.sin(1.3 * x + 0.2) * np.cos(0.9 * y) * np.sin(1.1 * z + 0.5)
    for Nf in (32, 64):
        h = 2.0 / Nf
        xf = (np.arange(Nf) + 0.5) * h
        xc = (np.arange(Nf // 2) + 0.5) * 2 * h
        fine = f(xf[:, None, None], xf[None, :, None], xf[None, None, :])[None]
        R = oracle.restrict(fine, ng, Nf)[0]             # one block: symmetric stencils except next to the faces
        errs_r.append(np.abs(R - f(xc[:, None, None], xc[None, :, None], xc[None, None, :])).max())
        coarse = f(xc[:, None, None], xc[None, :, None], xc[None, None, :])[None]
        m = Nf // 4                                      # fine box = the middle half of the coarse grid
        o = (m // 2,) * 3
        lo, hi = (-ng,) * 3, (m + ng,) * 3               # the box with its ghost shell (interior values are checked too)
        xg = (2 * o[0] + np.arange(lo[0], hi[0]) + 0.5) * h
        Pv = oracle.prolong(coarse, ng, 1, o, lo, hi)[0]
        errs_p.append(np.abs(Pv - f(xg[:, None, None], xg[None, :, None], xg[None, None, :])).max())
    for e in (errs_r, errs_p):
        order = np.log2(e[0] / e[1])
        assert n - 0.5 < order < n + 0.7, (ng, order, e)


def test_A5_prolongation_of_restriction_residual_and_periodic_wrap(oracle):
    """P(R f) - f is O(h^n) on smooth data, and prolongation past the edge of a periodic coarse mesh reads the
    wrapped coarse nodes (O2)."""
    ng = 3
    res = []
    for Nf in (32, 64):
        h = 1.0 / Nf
        xf = (np.arange(Nf) + 0.5) * h
        f = lambda z, y, x: 1.0 + 0.3 * np.sin(2 * np.pi * x) * np.cos(2 * np.pi * y) * np.cos(4 * np.pi * z)
        fine = f(xf[:, None, None], xf[None, :, None], xf[None, None, :])[None]
        coarse = oracle.restrict(fine, ng, 16)                      # blocks of 16^3: lopsided stencils at every face
        back = oracle.prolong(coarse, ng, 0, (0, 0, 0), (0, 0, 0), (Nf,) * 3)[0]   # periodic: the whole fine grid
        res.append(np.abs(back - fine[0]).max())
        # ghost shell past the periodic edge = the values at the wrapped positions
        shell = oracle.prolong(coarse, ng, 0, (0, 0, 0), (-3, 0, 0), (0, 4, 4))[0]
        assert np.array_equal(shell, back[:4, :4, Nf - 3:])
    assert 3.5 < np.log2(res[0] / res[1]) < 4.7, res


def _two_level_wave(ncoarse, n):
    """E2 of the paper on BASELINE's wave (along x): coarse ncoarse^3 periodic mesh in blocks of n^3,
    the corner coarse block refined once (2x2x2 fine blocks of n^3 at half the spacing), one dt for both levels."""
    pc = replace(I.params_linear_wave(ncoarse, n), cfl=0.125)        # dt = 0.25 * (dx/2)
    pf = replace(pc, nb=(2, 2, 2), dx=pc.dx / 2, cfl=0.25, bc=1)
    return pc, pf


def test_A6_two_level_wave_converges_and_levels_stay_consistent(oracle):
    """'the same linear wave evolution but now with a corner of the Mesh refined at one level higher'.
    With n = N_g + 1 = 4 point interpolation applied at every RK stage the two-level error against the analytic wave
    is set by the interpolation, not by the 4th-order differencing: it must fall by ~2^3..2^4 per
    halving of h on BOTH levels (measured 9.6 / 10.6), stay far below the wave (1e-8), and the two levels must agree
    where they overlap. (The paper's 'consistently lower than without refinement' is a statement about 6th-order runs
    over a full period in the L1 norm of Eq. 3; at these short times the unrefined error is still ~1e-14.)"""
    errs = []
    for N, n, nsteps in ((16, 8, 8), (32, 16, 16)):
        pc, pf = _two_level_wave(N, n)
        uc0, uf0 = I.linear_wave_data(pc), I.linear_wave_data(pf)
        uc, uf, bad = oracle.step_two_level(pc, pf, n, (0, 0, 0), uc0, uf0, nsteps)
        assert bad == 0 and abs(pc.dt - pf.dt) < 1e-15
        t = nsteps * pc.dt
        ec = np.abs(uc[I.GYY] - I.linear_wave_data(pc, t=t)[I.GYY]).max()
        ef = np.abs(uf[I.GYY] - I.linear_wave_data(pf, t=t)[I.GYY]).max()
        errs.append((ec, ef))
        # the covered coarse nodes ARE the restriction of the fine level (step B.1), bit for bit
        assert np.array_equal(uc[:, :n, :n, :n], oracle.restrict(uf, 3, n))
    assert errs[0][0] < 2e-11 and errs[0][1] < 2e-11
    assert 6.0 < errs[0][0] / errs[1][0] < 20.0 and 6.0 < errs[0][1] / errs[1][1] < 20.0, errs
    # Minkowski is a fixed point of the whole two-level protocol (weights sum to one)
    pc, pf = _two_level_wave(32, 16)
    mc, mf = I.minkowski(pc), I.minkowski(pf)
    vc, vf, bad = oracle.step_two_level(pc, pf, 16, (0, 0, 0), mc, mf, 2)
    assert bad == 0 and np.abs(vc - mc).max() < 1e-15 and np.abs(vf - mf).max() < 1e-15


def test_A7_two_level_rejects_mismatched_time_steps(oracle):
    pc, pf = _two_level_wave(32, 16)
    bad = oracle.step_two_level(replace(pc, cfl=0.25), pf, 16, (0, 0, 0), I.minkowski(pc), I.minkowski(pf), 1)[2]
    assert bad == -1


def test_A8_difference_from_reference_form_reproduces_constants_bitwise(oracle):
    """R-I1: Eq. (2) as f_r + sum l_i (f_i - f_r). A constant that is not a dyadic rational comes back bit for bit from
    both operators (a plain weighted sum would round 64 products), and a 1e-8 perturbation of 1 is interpolated with an
    error far below one ulp of 1 before the final rounding."""
    ng, nf = 3, 8
    c = 0.1
    fine = np.full((1, 16, 16, 16), c)
    assert np.all(oracle.restrict(fine, ng, nf) == c)
    coarse = np.full((1, 12, 12, 12), c)
    assert np.all(oracle.prolong(coarse, ng, 0, (2, 2, 2), (-3, -3, -3), (11, 11, 11)) == c)
    h = 1.0 / 16
    xf = (np.arange(16) + 0.5) * h
    xc = (np.arange(8) + 0.5) * 2 * h
    pert = lambda z, y, x: 1e-8 * (x * x * y - z ** 3)
    fine = (1.0 + pert(xf[:, None, None], xf[None, :, None], xf[None, None, :]))[None]
    want = 1.0 + pert(xc[:, None, None], xc[None, :, None], xc[None, None, :])
    assert np.abs(oracle.restrict(fine, ng, nf)[0] - want).max() <= 2.3e-16      # one final rounding of ~1
