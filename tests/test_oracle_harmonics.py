"""Pins for b_lm, B_lm, C_lm (l = 1..8) and the 4- and 5-body invariants (paper App.B, Eq.7-8, B9 P:454)."""
import os

import numpy as np
from scipy.special import eval_legendre

from cases import golden, random_rotation
from oracle import gnep_oracle as orc

L_OF = np.concatenate([[l] * (2 * l + 1) for l in range(1, 9)])
NLM = 80


def _paper_formulas():
    path = os.path.join(os.path.dirname(__file__), "golden", "blm_paper.txt")
    out = []
    for line in open(path):
        if line.startswith("#") or ":" not in line:
            continue
        lm, expr = line.split(":")
        l, m = (int(v) for v in lm.split())
        out.append((l, m, expr.strip()))
    return out


def test_blm_match_printed_formulas():
    rng = np.random.default_rng(1)
    forms = _paper_formulas()
    assert len(forms) == NLM and [f[:2] for f in forms] == [(l, m) for l in range(1, 9) for m in range(2 * l + 1)]
    for _ in range(10):
        x, y, z = rng.normal(size=3)
        b, _ = orc.blm_raw(x, y, z)
        for l, m, expr in forms:
            val = eval(expr, {"x": x, "y": y, "z": z, "r2": x * x + y * y + z * z})
            assert abs(b[l * l - 1 + m] - val) < 1e-12 * max(1, abs(val))


def test_blm_harmonic_and_homogeneous():
    rng = np.random.default_rng(2)
    h = 0.1
    for _ in range(5):
        p = rng.normal(size=3)
        b0, g0 = orc.blm_raw(*p)
        # homogeneity: b(t r) = t^l b(r); Euler: r . grad b = l b
        bt, _ = orc.blm_raw(*(1.7 * p))
        np.testing.assert_allclose(bt, 1.7 ** L_OF * b0, rtol=1e-12, atol=1e-12)
        np.testing.assert_allclose(g0 @ p, L_OF * b0, rtol=1e-12, atol=1e-12)
        # Laplacian = 0: the 8th-order-accurate central stencil of the second derivative is exact for polynomials of
        # degree <= 9 (the b_lm have degree l <= 8)
        w = [-205.0 / 72, 8.0 / 5, -1.0 / 5, 8.0 / 315, -1.0 / 560]
        lap = np.zeros(NLM)
        for ax in range(3):
            e = np.zeros(3); e[ax] = h
            f = lambda q: orc.blm_raw(*q)[0]
            lap += (w[0] * b0 + sum(w[k] * (f(p + k * e) + f(p - k * e)) for k in range(1, 5))) / (h * h)
        assert np.max(np.abs(lap) / (1 + np.abs(b0))) < 1e-7


def test_grad_blm_fd():
    rng = np.random.default_rng(3)
    h = 1e-6
    for _ in range(5):
        p = rng.normal(size=3) * 2.0
        _, gb = orc.blm_raw(*p)
        _, dB = orc.blm(*p)
        for ax in range(3):
            e = np.zeros(3); e[ax] = h
            fd_b = (orc.blm_raw(*(p + e))[0] - orc.blm_raw(*(p - e))[0]) / (2 * h)
            fd_B = (orc.blm(*(p + e))[0] - orc.blm(*(p - e))[0]) / (2 * h)
            np.testing.assert_allclose(gb[:, ax], fd_b, atol=1e-7 * max(1, np.abs(fd_b).max()))
            np.testing.assert_allclose(dB[:, ax], fd_B, atol=2e-8 * max(1, np.abs(fd_B).max()))


def test_addition_theorem_fixes_clm():
    """sum_m C_lm B_lm(r1) B_lm(r2) = (2l+1)/(4 pi) P_l(cos theta12)  (library Legendre as the referee)."""
    rng = np.random.default_rng(4)
    C = orc.clm()
    for _ in range(20):
        r1, r2 = rng.normal(size=3), rng.normal(size=3) * 3
        B1, _ = orc.blm(*r1)
        B2, _ = orc.blm(*r2)
        ct = r1 @ r2 / np.linalg.norm(r1) / np.linalg.norm(r2)
        for l in range(1, 9):
            sl = slice(l * l - 1, l * l + 2 * l)
            lhs = np.sum(C[sl] * B1[sl] * B2[sl])
            assert abs(lhs - (2 * l + 1) / (4 * np.pi) * eval_legendre(l, ct)) < 1e-12


def test_sc_lattice_closed_form():
    """Perfect simple-cubic neighbours (first two shells, unit weights): odd/low moments vanish, l=4 value."""
    sites = [np.array(v, float) for v in
             [(1, 0, 0), (-1, 0, 0), (0, 1, 0), (0, -1, 0), (0, 0, 1), (0, 0, -1)] +
             [(a, b, 0) for a in (1, -1) for b in (1, -1)] + [(a, 0, b) for a in (1, -1) for b in (1, -1)] +
             [(0, a, b) for a in (1, -1) for b in (1, -1)]]
    assert len(sites) == 18
    S = sum(orc.blm(*p)[0] for p in sites)
    assert np.max(np.abs(S[:15])) < 1e-12          # l = 1,2,3 vanish by cubic symmetry
    assert abs(S[15] - golden("sc_l4_S0")[0]) < 1e-12 and abs(S[22] - golden("sc_l4_S7")[0]) < 1e-12
    assert np.max(np.abs(np.delete(S[15:24], [0, 7]))) < 1e-12
    q4l = np.sum(orc.clm()[15:24] * S[15:24] ** 2)
    assert abs(q4l - golden("sc_l4_q")[0]) < 1e-9


def _M_from_s(s):
    s0, s1, s2, s3, s4 = s
    Mzz = s0 / 3; Mxx = (-s0 / 3 + s3) / 2; Myy = (-s0 / 3 - s3) / 2
    return np.array([[Mxx, s4 / 2, s1], [s4 / 2, Myy, s2], [s1, s2, Mzz]])


def test_p4_is_108_det_M_and_invariant():
    rng = np.random.default_rng(5)
    assert abs(orc.kappa4() - golden("kappa4")[0]) < 1e-15
    for _ in range(10):
        r = rng.normal(size=(6, 3)); g = rng.normal(size=6)
        s = sum(gi * orc.blm(*ri)[0][3:8] for gi, ri in zip(g, r))
        M = sum(gi * (np.outer(ri, ri) / (ri @ ri) - np.eye(3) / 3) for gi, ri in zip(g, r))
        np.testing.assert_allclose(_M_from_s(s), M, atol=1e-12)
        P = orc.p4(s)
        assert abs(P - 108 * np.linalg.det(M)) < 1e-10 * max(1, abs(P))
        assert abs(np.trace(M @ M @ M) - 3 * np.linalg.det(M)) < 1e-12
        R = random_rotation(rng)
        s_rot = sum(gi * orc.blm(*(R @ ri))[0][3:8] for gi, ri in zip(g, r))
        assert abs(orc.p4(s_rot) - P) < 1e-10 * max(1, abs(P))
    # single neighbour with weight g: P4 = 8 g^3 for every direction
    for _ in range(3):
        d = rng.normal(size=3)
        assert abs(orc.p4(0.7 * orc.blm(*d)[0][3:8]) - 8 * 0.7 ** 3) < 1e-12


def test_p4_grad_hessian_fd():
    rng = np.random.default_rng(6)
    s = rng.normal(size=5)
    _, g, H = orc.p4(s, True)
    h = 1e-5
    for a in range(5):
        e = np.zeros(5); e[a] = h
        assert abs(g[a] - (orc.p4(s + e) - orc.p4(s - e)) / (2 * h)) < 1e-7
        gp = orc.p4(s + e, True)[1]; gm = orc.p4(s - e, True)[1]
        np.testing.assert_allclose(H[a], (gp - gm) / (2 * h), atol=1e-7)
    np.testing.assert_allclose(H, H.T)


def test_p5_is_the_quartic_invariant_of_the_l1_moments():
    """q5 = kappa5 |v|^4 (R41): rotation invariant, single neighbour of weight g gives kappa5 g^4, equals
    q_{l=1}^2 / 3 with q_{l=1} = 3/(4 pi) |v|^2 (Eq.7 with the C_1m of the addition theorem), kappa5 = 3/(16 pi^2)."""
    rng = np.random.default_rng(6)
    assert abs(orc.kappa5() - 3 / (16 * np.pi ** 2)) < 1e-16
    pts = rng.normal(size=(7, 3)); wts = rng.normal(size=7)
    def moments(P):
        return sum(w * orc.blm(*p)[0][:3] for w, p in zip(wts, P))
    s = moments(pts)
    R = random_rotation(rng)
    assert abs(orc.p5(s) - orc.p5(moments(pts @ R.T))) < 1e-13 * abs(orc.p5(s))
    q1 = np.sum(orc.clm()[:3] * s ** 2)
    assert abs(orc.p5(s) - q1 ** 2 / 3) < 1e-14 * abs(q1 ** 2)
    g = 0.37
    one = g * orc.blm(0.2, -0.4, 0.9)[0][:3]
    assert abs(orc.p5(one) - orc.kappa5() * g ** 4) < 1e-15


def test_p5_grad_hessian_fd():
    rng = np.random.default_rng(8)
    s = rng.normal(size=3)
    v, g, H = orc.p5(s, want_grad=True)
    h = 1e-5
    for a in range(3):
        e = np.zeros(3); e[a] = h
        assert abs((orc.p5(s + e) - orc.p5(s - e)) / (2 * h) - g[a]) < 1e-8
        gp = orc.p5(s + e, want_grad=True)[1]; gm = orc.p5(s - e, want_grad=True)[1]
        np.testing.assert_allclose((gp - gm) / (2 * h), H[a], atol=1e-8)
    np.testing.assert_allclose(H, H.T, atol=0)
