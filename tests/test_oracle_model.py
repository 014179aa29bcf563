"""Pins for descriptors, network, energy, forces and virial of the oracle."""
import numpy as np
from scipy.special import eval_legendre

import gnep_synth as gs
from cases import labelled_case, random_rotation
from oracle import gnep_oracle as orc


def _case(config=0, n=2, four=None):
    over = None if four is None else {"use_4body": four}
    return labelled_case(config, n_structs=n, spec_over=over)


def test_qnl_equals_legendre_double_sum():
    """Eq.7-8 collapse, by the addition theorem, to (2l+1)/(4pi) sum_jk g_n(d_ij) g_n(d_ik) P_l(cos jik)."""
    spec, sp, b, ob, theta, qs, _ = _case(0, 1)
    q = orc.descriptors(sp, theta, ob)
    rptr, j, sh, r = ob.neighbors(1)
    T, NA, KA, NR, KR = 2, spec["n_angular"], spec["n_basis_angular"], spec["n_radial"], spec["n_basis_radial"]
    cA = theta[T * T * NR * KR:][:T * T * NA * KA].reshape(T, T, NA, KA)
    for i in (0, 17, 40):
        rr = r[rptr[i]:rptr[i + 1]]; jj = j[rptr[i]:rptr[i + 1]]
        d = np.linalg.norm(rr, axis=1)
        g = np.array([cA[b["types"][i], b["types"][jx]] @ orc.basis(spec["rc_angular"], KA, dx)[0]
                      for jx, dx in zip(jj, d)])                       # [pairs, NA]
        cosm = (rr @ rr.T) / np.outer(d, d)
        for l in range(1, 5):
            Pl = eval_legendre(l, np.clip(cosm, -1, 1))
            for n in range(NA):
                ref = (2 * l + 1) / (4 * np.pi) * g[:, n] @ Pl @ g[:, n]
                assert abs(q[i, NR + (l - 1) * NA + n] - ref) < 1e-10 * max(1, abs(ref))


def test_radial_descriptor_plain_sum():
    spec, sp, b, ob, theta, qs, _ = _case(0, 1)
    q = orc.descriptors(sp, theta, ob)
    rptr, j, sh, r = ob.neighbors(0)
    T, NR, KR = 2, spec["n_radial"], spec["n_basis_radial"]
    cR = theta[:T * T * NR * KR].reshape(T, T, NR, KR)
    for i in (3, 33):
        acc = np.zeros(NR)
        for p in range(rptr[i], rptr[i + 1]):
            acc += cR[b["types"][i], b["types"][j[p]]] @ orc.basis(spec["rc_radial"], KR, np.linalg.norm(r[p]))[0]
        np.testing.assert_allclose(q[i, :NR], acc, atol=1e-12)


def test_dimer_closed_forms():
    """Single neighbour: q_nl = (2l+1)/(4pi) g^2, q4 = 8 kappa4 g^3, E = 2F(G), |F| = 2|sum E'_nu dq_nu/dd|."""
    spec = dict(gs.MODEL_SPECS[1]); sp = orc.make_spec(spec)
    theta = gs.draw_params(spec, 1)
    d0 = 2.9
    dirv = np.array([0.3, -0.5, 0.8]); dirv /= np.linalg.norm(dirv)
    pos = np.array([[10.0, 10.0, 10.0], [10.0, 10.0, 10.0] + d0 * dirv])
    cell = (np.eye(3) * 30).reshape(1, 9)
    types = np.zeros(2, np.int32)
    ob = orc.Batch(sp, [0, 2], pos, cell, types)
    q = orc.descriptors(sp, theta, ob)
    NR, KR, NA, KA = spec["n_radial"], spec["n_basis_radial"], spec["n_angular"], spec["n_basis_angular"]
    cR = theta[:4 * NR * KR].reshape(2, 2, NR, KR); cA = theta[4 * NR * KR:][:4 * NA * KA].reshape(2, 2, NA, KA)
    fR, fRp = orc.basis(spec["rc_radial"], KR, d0); fA, fAp = orc.basis(spec["rc_angular"], KA, d0)
    gR, gA = cR[0, 0] @ fR, cA[0, 0] @ fA
    np.testing.assert_allclose(q[0, :NR], gR, atol=1e-13)
    for l in range(1, 5):
        np.testing.assert_allclose(q[0, NR + (l - 1) * NA: NR + l * NA], (2 * l + 1) / (4 * np.pi) * gA ** 2, atol=1e-12)
    np.testing.assert_allclose(q[0, NR + 4 * NA:], 8 * orc.kappa4() * gA ** 3, atol=1e-12)
    np.testing.assert_allclose(q[0], q[1], atol=1e-12)
    E, F, W = orc.predict(sp, theta, None, ob)
    Ei, Ep = orc.network(sp, theta, None, 0, q[0])
    assert abs(E[0] - 2 * Ei) < 1e-12
    dq = np.concatenate([cR[0, 0] @ fRp] + [(2 * l + 1) / (4 * np.pi) * 2 * gA * (cA[0, 0] @ fAp) for l in range(1, 5)]
                        + [8 * orc.kappa4() * 3 * gA ** 2 * (cA[0, 0] @ fAp)])
    fmag = 2 * (Ep @ dq)
    np.testing.assert_allclose(F[0], fmag * dirv, atol=1e-10)      # F_0 = +dE_i/dr_ij - dE_j/dr_ji
    np.testing.assert_allclose(F[1], -fmag * dirv, atol=1e-10)


def test_invariances_q_E():
    """Translation (with rewrap), rotation of positions + cell, permutation leave q_i, E unchanged."""
    spec, sp, b, ob, theta, qs, _ = _case(1, 1)
    rng = np.random.default_rng(11)
    q0 = orc.descriptors(sp, theta, ob); E0, F0, W0 = orc.predict(sp, theta, qs, ob)
    cell = b["cells"][0].reshape(3, 3)
    # translation
    ob1 = orc.Batch(sp, b["atom_offsets"], b["positions"] + np.array([1.234, -7.7, 3.21]), b["cells"], b["types"])
    np.testing.assert_allclose(orc.descriptors(sp, theta, ob1), q0, atol=1e-9)
    E1, F1, W1 = orc.predict(sp, theta, qs, ob1)
    np.testing.assert_allclose(E1, E0, atol=1e-9); np.testing.assert_allclose(F1, F0, atol=1e-9)
    # rotation
    R = random_rotation(rng)
    ob2 = orc.Batch(sp, b["atom_offsets"], b["positions"] @ R.T, (cell @ R.T).reshape(1, 9), b["types"])
    np.testing.assert_allclose(orc.descriptors(sp, theta, ob2), q0, atol=1e-9)
    E2, F2, W2 = orc.predict(sp, theta, qs, ob2)
    np.testing.assert_allclose(E2, E0, atol=1e-9)
    np.testing.assert_allclose(F2, F0 @ R.T, atol=1e-9)
    Wm = lambda w: np.array([[w[0], w[3], w[5]], [w[3], w[1], w[4]], [w[5], w[4], w[2]]])
    np.testing.assert_allclose(Wm(W2[0]), R @ Wm(W0[0]) @ R.T, atol=1e-8)
    # permutation
    perm = rng.permutation(ob.N)
    ob3 = orc.Batch(sp, b["atom_offsets"], b["positions"][perm], b["cells"], b["types"][perm])
    np.testing.assert_allclose(orc.descriptors(sp, theta, ob3), q0[perm], atol=1e-10)
    E3, F3, _ = orc.predict(sp, theta, qs, ob3)
    np.testing.assert_allclose(E3, E0, atol=1e-10); np.testing.assert_allclose(F3, F0[perm], atol=1e-10)


def test_forces_sum_to_zero_and_fd():
    """sum F = 0 per structure and F = -dE/dr by central differences, 3- and 4-body."""
    for config, four in ((0, False), (1, True)):
        spec, sp, b, ob, theta, qs, _ = _case(config, 1, four)
        E, F, W = orc.predict(sp, theta, qs, ob)
        assert np.max(np.abs(F.sum(0))) < 1e-11
        rng = np.random.default_rng(12); h = 1e-5
        for i in rng.integers(0, ob.N, 4):
            for ax in range(3):
                pp = b["positions"].copy(); pp[i, ax] += h
                pm = b["positions"].copy(); pm[i, ax] -= h
                Ep = orc.predict(sp, theta, qs, orc.Batch(sp, b["atom_offsets"], pp, b["cells"], b["types"]))[0][0]
                Em = orc.predict(sp, theta, qs, orc.Batch(sp, b["atom_offsets"], pm, b["cells"], b["types"]))[0][0]
                assert abs(F[i, ax] + (Ep - Em) / (2 * h)) < 2e-8 * max(1, np.abs(F).max())


def test_virial_is_minus_dE_dstrain():
    spec, sp, b, ob, theta, qs, _ = _case(1, 1)
    E, F, W = orc.predict(sp, theta, qs, ob)
    cell = b["cells"][0].reshape(3, 3); h = 1e-6
    comps = [(0, 0), (1, 1), (2, 2), (0, 1), (1, 2), (2, 0)]
    for c, (a, bb) in enumerate(comps):
        vals = []
        for sgn in (1, -1):
            eps = np.zeros((3, 3)); eps[a, bb] = sgn * h        # r'_b += r_a eps_ab
            dfm = np.eye(3) + eps
            obx = orc.Batch(sp, b["atom_offsets"], b["positions"] @ dfm, (cell @ dfm).reshape(1, 9), b["types"])
            vals.append(orc.predict(sp, theta, qs, obx)[0][0])
        assert abs(W[0, c] + (vals[0] - vals[1]) / (2 * h)) < 1e-6 * max(1, np.abs(W).max())
    # symmetric up to rounding: compare xy with the transposed strain
    eps = np.zeros((3, 3)); vals = []
    for sgn in (1, -1):
        eps[:] = 0; eps[1, 0] = sgn * h; dfm = np.eye(3) + eps
        obx = orc.Batch(sp, b["atom_offsets"], b["positions"] @ dfm, (cell @ dfm).reshape(1, 9), b["types"])
        vals.append(orc.predict(sp, theta, qs, obx)[0][0])
    assert abs(W[0, 3] + (vals[0] - vals[1]) / (2 * h)) < 1e-6 * max(1, np.abs(W).max())


def test_perfect_lattice_special_case():
    """Single-species perfect simple-cubic lattice: l=1,2,3 and 4-body descriptors vanish, F = 0, W ~ identity."""
    spec = dict(gs.MODEL_SPECS[1]); sp = orc.make_spec(spec)
    a, n = 3.05, 6
    g = np.stack(np.meshgrid(*[np.arange(n)] * 3, indexing="ij"), -1).reshape(-1, 3) * a + 0.5
    ob = orc.Batch(sp, [0, len(g)], g, (np.eye(3) * n * a).reshape(1, 9), np.zeros(len(g), np.int32))
    theta = gs.draw_params(spec, 1)
    q = orc.descriptors(sp, theta, ob)
    NR, NA = spec["n_radial"], spec["n_angular"]
    assert np.max(np.abs(q[:, NR:NR + 3 * NA])) < 1e-18 + 1e-12
    assert np.max(np.abs(q[:, NR + 4 * NA:])) < 1e-12
    assert np.max(np.abs(q - q[0])) < 1e-10
    E, F, W = orc.predict(sp, theta, None, ob)
    assert np.max(np.abs(F)) < 1e-10
    assert np.max(np.abs(W[0, 3:])) < 1e-8 and abs(W[0, 0] - W[0, 1]) < 1e-8 and abs(W[0, 0] - W[0, 2]) < 1e-8


def test_network_derivatives_fd():
    """E' (D1.5) and E''D (D1.6) against central differences of D1.1, with input scaling."""
    spec = dict(gs.MODEL_SPECS[0]); sp = orc.make_spec(spec)
    theta = gs.draw_params(spec, 0)
    rng = np.random.default_rng(13)
    nd = gs.n_descriptors(spec)
    q = rng.normal(size=nd); qs = rng.uniform(0.5, 1.5, size=nd); D = rng.normal(size=nd)
    for t in (0, 1):
        E, Ep, hv = orc.network(sp, theta, qs, t, q, D)
        h = 1e-6
        for v in range(nd):
            e = np.zeros(nd); e[v] = h
            fd = (orc.network(sp, theta, qs, t, q + e)[0] - orc.network(sp, theta, qs, t, q - e)[0]) / (2 * h)
            assert abs(Ep[v] - fd) < 1e-8
        fdh = (orc.network(sp, theta, qs, t, q + h * D)[1] - orc.network(sp, theta, qs, t, q - h * D)[1]) / (2 * h)
        np.testing.assert_allclose(hv, fdh, atol=1e-8)
    assert abs(orc.network(sp, theta, qs, 0, q)[0] - orc.network(sp, theta, qs, 1, q)[0]) > 1e-6   # per-species nets
