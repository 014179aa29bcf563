"""Pins for the oracle at l_max = 5..8 and with the 5-body term (paper Eq.7 "l = 1, 2, ..., 8"; b_lm of App.B,
P:306-449; five-body terms named at P:65, P:77 and defined by DESIGN.md R41).  The same pins as for l <= 4: Eq.7-8 against
the Legendre double sum (library Legendre as the referee), dimer closed forms, forces / virial against finite
differences of the energy, and the analytic loss gradient against finite differences of the plain loss."""
import numpy as np
from scipy.special import eval_legendre

import gnep_synth as gs
from cases import labelled_case
from oracle import gnep_oracle as orc

HIGH = {"l_max": 8, "use_4body": True, "use_5body": True, "n_angular": 3, "n_basis_angular": 4, "n_radial": 3,
        "n_basis_radial": 4, "n_neurons": 6}


def test_qnl_equals_legendre_double_sum_up_to_l8():
    spec, sp, b, ob, theta, qs, _ = labelled_case(0, n_structs=1, spec_over=HIGH)
    q = orc.descriptors(sp, theta, ob)
    rptr, j, sh, r = ob.neighbors(1)
    T, NA, KA, NR, KR = 2, spec["n_angular"], spec["n_basis_angular"], spec["n_radial"], spec["n_basis_radial"]
    cA = theta[T * T * NR * KR:][:T * T * NA * KA].reshape(T, T, NA, KA)
    for i in (0, 21, 50):
        rr = r[rptr[i]:rptr[i + 1]]; jj = j[rptr[i]:rptr[i + 1]]
        d = np.linalg.norm(rr, axis=1)
        g = np.array([cA[b["types"][i], b["types"][jx]] @ orc.basis(spec["rc_angular"], KA, dx)[0] for jx, dx in zip(jj, d)])
        cosm = np.clip((rr @ rr.T) / np.outer(d, d), -1, 1)
        for l in range(1, 9):
            Pl = eval_legendre(l, cosm)
            for n in range(NA):
                ref = (2 * l + 1) / (4 * np.pi) * g[:, n] @ Pl @ g[:, n]
                assert abs(q[i, NR + (l - 1) * NA + n] - ref) < 1e-10 * max(1, abs(ref))
        # many-body blocks: 4-body after the 8 three-body blocks, then 5-body = q_{l=1}^2 / 3
        q1 = q[i, NR:NR + NA]
        np.testing.assert_allclose(q[i, NR + 9 * NA:NR + 10 * NA], q1 ** 2 / 3, rtol=1e-12)
    assert q.shape[1] == NR + 10 * NA == gs.n_descriptors(spec)


def test_dimer_closed_forms_with_l8_and_5body():
    spec = dict(gs.MODEL_SPECS[1], **{k: HIGH[k] for k in ("l_max", "use_5body")}); sp = orc.make_spec(spec)
    theta = gs.draw_params(spec, 1)
    d0, dirv = 3.1, np.array([-0.6, 0.2, 0.7]); dirv /= np.linalg.norm(dirv)
    pos = np.array([[10.0, 10.0, 10.0], [10.0, 10.0, 10.0] + d0 * dirv])
    ob = orc.Batch(sp, [0, 2], pos, (np.eye(3) * 30).reshape(1, 9), np.zeros(2, np.int32))
    q = orc.descriptors(sp, theta, ob)
    NR, KR, NA, KA = spec["n_radial"], spec["n_basis_radial"], spec["n_angular"], spec["n_basis_angular"]
    cA = theta[4 * NR * KR:][:4 * NA * KA].reshape(2, 2, NA, KA)
    gA = cA[0, 0] @ orc.basis(spec["rc_angular"], KA, d0)[0]
    for l in range(1, 9):
        np.testing.assert_allclose(q[0, NR + (l - 1) * NA: NR + l * NA], (2 * l + 1) / (4 * np.pi) * gA ** 2, atol=1e-12)
    np.testing.assert_allclose(q[0, NR + 8 * NA:NR + 9 * NA], 8 * orc.kappa4() * gA ** 3, atol=1e-12)
    np.testing.assert_allclose(q[0, NR + 9 * NA:], orc.kappa5() * gA ** 4, atol=1e-12)


def test_forces_virial_and_loss_gradient_fd_at_l8_with_5body():
    spec, sp, b, ob, theta, qs, (E, F, W) = labelled_case(0, n_structs=1, spec_over=HIGH)
    Ep, Fp, Wp = orc.predict(sp, theta, qs, ob)
    assert np.max(np.abs(Fp.sum(axis=0))) < 1e-12
    pos0 = b["positions"].copy(); cell = b["cells"]; off = b["atom_offsets"]; types = b["types"]
    h = 1e-5
    for (i, ax) in ((3, 0), (17, 2), (40, 1)):
        e = []
        for sgn in (1, -1):
            p = pos0.copy(); p[i, ax] += sgn * h
            e.append(orc.predict(sp, theta, qs, orc.Batch(sp, off, p, cell, types))[0][0])
        assert abs(-(e[0] - e[1]) / (2 * h) - Fp[i, ax]) < 1e-7 * max(1, abs(Fp[i, ax]))
    # virial xx and xy: W_ab = -dE/d eps_ab under r'_b += r_a eps_ab (R17)
    for c, (aa, bb) in ((0, (0, 0)), (3, (0, 1))):
        e = []
        for sgn in (1, -1):
            eps = np.eye(3); eps[aa, bb] += sgn * h
            e.append(orc.predict(sp, theta, qs, orc.Batch(sp, off, pos0 @ eps, (cell.reshape(3, 3) @ eps).reshape(1, 9), types))[0][0])
        assert abs(-(e[0] - e[1]) / (2 * h) - Wp[0, c]) < 1e-6 * max(1, abs(Wp[0, c]))
    t, g = orc.loss_and_grad(sp, theta, qs, ob)
    rng = np.random.default_rng(2)
    nA0 = 4 * 3 * 4
    idx = np.concatenate([rng.choice(nA0, 6, replace=False), nA0 + rng.choice(4 * 3 * 4, 14, replace=False),
                          2 * nA0 + rng.choice(len(theta) - 2 * nA0, 16, replace=False)])
    for p in idx:
        tp = theta.copy(); tm = theta.copy(); tp[p] += h; tm[p] -= h
        fd = (orc.loss(sp, tp, qs, ob)[0] - orc.loss(sp, tm, qs, ob)[0]) / (2 * h)
        assert abs(fd - g[p]) <= 2e-6 * max(abs(g[p]), 1e-5), (p, fd, g[p])


def test_intermediate_l_max_blocks_are_prefixes():
    """l_max = 6 is the l_max = 8 model without the l = 7, 8 blocks: same three-body descriptors for l <= 6."""
    s8, sp8, b, ob8, th8, _, _ = labelled_case(0, n_structs=1, spec_over=dict(HIGH, use_4body=False, use_5body=False))
    s6 = dict(s8, l_max=6); sp6 = orc.make_spec(s6)
    ob6 = orc.Batch(sp6, b["atom_offsets"], b["positions"], b["cells"], b["types"])
    ncoef = 4 * (3 * 4 + 3 * 4)
    q8 = orc.descriptors(sp8, th8, ob8)
    th6 = np.concatenate([th8[:ncoef], np.zeros(orc.num_params(sp6) - ncoef)])
    q6 = orc.descriptors(sp6, th6, ob6)
    np.testing.assert_allclose(q6, q8[:, :q6.shape[1]], rtol=1e-13, atol=1e-15)
