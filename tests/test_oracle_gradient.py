"""Pins for the oracle's loss (Eq.9-12), analytic gradient (Eq.13-16, App.C/D) and Adam."""
import numpy as np

import gnep_synth as gs
from cases import labelled_case, random_rotation
from oracle import gnep_oracle as orc


def _fd_grad(sp, theta, qs, ob, idx, h=1e-5):
    out = np.zeros(len(idx))
    for k, p in enumerate(idx):
        tp = theta.copy(); tp[p] += h
        tm = theta.copy(); tm[p] -= h
        out[k] = (orc.loss(sp, tp, qs, ob)[0] - orc.loss(sp, tm, qs, ob)[0]) / (2 * h)
    return out


def test_full_fd_sweep_config0():
    """Central finite differences of the PLAIN loss over all 822 parameters of config 0."""
    spec, sp, b, ob, theta, qs, _ = labelled_case(0)
    terms, g = orc.loss_and_grad(sp, theta, qs, ob)
    np.testing.assert_allclose(terms, orc.loss(sp, theta, qs, ob), rtol=1e-14)
    assert len(g) == 822
    fd = _fd_grad(sp, theta, qs, ob, np.arange(len(theta)))
    assert np.linalg.norm(g - fd) / np.linalg.norm(fd) < 1e-8
    assert np.max(np.abs(g - fd)) < 1e-8 * max(1.0, np.abs(fd).max())
    # every parameter group individually
    T, NR, KR, NA, KA = 2, spec["n_radial"], spec["n_basis_radial"], spec["n_angular"], spec["n_basis_angular"]
    o1 = T * T * NR * KR; o2 = o1 + T * T * NA * KA
    for sl in (slice(0, o1), slice(o1, o2), slice(o2, None)):
        assert np.linalg.norm(g[sl] - fd[sl]) / np.linalg.norm(fd[sl]) < 1e-8


def test_fd_sample_with_4body():
    spec, sp, b, ob, theta, qs, _ = labelled_case(1, n_structs=2)
    _, g = orc.loss_and_grad(sp, theta, qs, ob)
    rng = np.random.default_rng(21)
    idx = np.concatenate([rng.integers(0, len(theta), 60), np.arange(432, 432 + 224, 9)])   # incl. c^A block
    fd = _fd_grad(sp, theta, qs, ob, idx)
    assert np.linalg.norm(g[idx] - fd) / np.linalg.norm(fd) < 1e-7


def test_each_loss_term_alone():
    """lambda_f = lambda_v = 0 isolates the first-order terms (C3.5, D1.7-D1.10); then force-only, virial-only."""
    rng = np.random.default_rng(22)
    for lam in ((1, 0, 0), (0, 1, 0), (0, 0, 1)):
        over = {"lambda_e": lam[0], "lambda_f": lam[1], "lambda_v": lam[2], "lambda_2": 0.0}
        spec, sp, b, ob, theta, qs, _ = labelled_case(0, n_structs=2, spec_over=over)
        terms, g = orc.loss_and_grad(sp, theta, qs, ob)
        assert abs(terms[0] - terms[1 + lam.index(1)]) < 1e-15
        idx = rng.integers(0, len(theta), 80)
        fd = _fd_grad(sp, theta, qs, ob, idx)
        assert np.linalg.norm(g[idx] - fd) / np.linalg.norm(fd) < 1e-7


def test_zero_residual_gives_pure_regulariser():
    """theta = teacher, no noise: L = lambda_2 t_2 and grad = 2 lambda_2 theta / P exactly."""
    spec = dict(gs.MODEL_SPECS[0]); sp = orc.make_spec(spec)
    b = gs.make_batch(0, n_structs=2)
    ob = orc.Batch(sp, b["atom_offsets"], b["positions"], b["cells"], b["types"])
    theta = gs.draw_params(spec, 0)
    ob.set_refs(*orc.predict(sp, theta, None, ob))
    terms, g = orc.loss_and_grad(sp, theta, None, ob)
    P = len(theta)
    assert terms[1] == 0 and terms[2] == 0 and terms[3] == 0
    assert abs(terms[0] - spec["lambda_2"] * np.mean(theta ** 2)) < 1e-18
    np.testing.assert_allclose(g, 2 * spec["lambda_2"] * theta / P, rtol=1e-13, atol=1e-20)


def test_rmse_mode_and_missing_refs():
    spec, sp, b, ob, theta, qs, (E, F, W) = labelled_case(0, n_structs=2, spec_over={"loss_mode": 1})
    terms, g = orc.loss_and_grad(sp, theta, qs, ob)
    lam = [spec["lambda_e"], spec["lambda_f"], spec["lambda_v"], spec["lambda_2"]]
    assert abs(terms[0] - sum(l * np.sqrt(t) for l, t in zip(lam, terms[1:]))) < 1e-14
    rng = np.random.default_rng(23); idx = rng.integers(0, len(theta), 60)
    fd = _fd_grad(sp, theta, qs, ob, idx)
    assert np.linalg.norm(g[idx] - fd) / np.linalg.norm(fd) < 1e-7
    # missing virial reference: that term is absent
    sp0 = orc.make_spec(dict(spec, loss_mode=0))
    ob.set_refs(E, F, None)
    t2, g2 = orc.loss_and_grad(sp0, theta, qs, ob)
    assert t2[3] == 0.0
    fd = _fd_grad(sp0, theta, qs, ob, idx)
    assert np.linalg.norm(g2[idx] - fd) / np.linalg.norm(fd) < 1e-7


def test_loss_and_gradient_rotation_invariant():
    """Energy and force terms are rotation invariant; Eq.12's 6-component sum counts off-diagonal
    virial components once, so t_v is not (it is not a Frobenius norm): lambda_v = 0 here."""
    spec, sp, b, ob, theta, qs, (E, F, W) = labelled_case(0, n_structs=1, spec_over={"lambda_v": 0.0})
    t0, g0 = orc.loss_and_grad(sp, theta, qs, ob)
    R = random_rotation(np.random.default_rng(24))
    cell = b["cells"][0].reshape(3, 3)
    Wm = np.array([[W[0, 0], W[0, 3], W[0, 5]], [W[0, 3], W[0, 1], W[0, 4]], [W[0, 5], W[0, 4], W[0, 2]]])
    # the teacher virial is symmetric up to rounding, so rotating the symmetric matrix is consistent
    Wr = R @ Wm @ R.T
    W6 = np.array([[Wr[0, 0], Wr[1, 1], Wr[2, 2], Wr[0, 1], Wr[1, 2], Wr[2, 0]]])
    ob2 = orc.Batch(sp, b["atom_offsets"], b["positions"] @ R.T, (cell @ R.T).reshape(1, 9), b["types"], E, F @ R.T, W6)
    t1, g1 = orc.loss_and_grad(sp, theta, qs, ob2)
    np.testing.assert_allclose(t1[[0, 1, 2, 4]], t0[[0, 1, 2, 4]], rtol=1e-7)
    assert np.linalg.norm(g1 - g0) / np.linalg.norm(g0) < 1e-6


def test_adam_sign_step_and_quadratic():
    rng = np.random.default_rng(25)
    g = rng.normal(size=50); th = rng.normal(size=50); th0 = th.copy()
    m = np.zeros(50); v = np.zeros(50)
    orc.adam_step(th, m, v, g, 1, 1e-3)
    np.testing.assert_allclose(th - th0, -1e-3 * g / (np.abs(g) + 1e-8), rtol=1e-12)
    np.testing.assert_allclose(m, 0.1 * g); np.testing.assert_allclose(v, 0.001 * g * g)
    # 1-D quadratic, independent numpy restatement of Kingma & Ba Algorithm 1
    x = np.array([3.0]); m = np.zeros(1); v = np.zeros(1)
    xr, mr, vr = 3.0, 0.0, 0.0
    for t in range(1, 200):
        orc.adam_step(x, m, v, 2 * x, t, 0.05)
        gr = 2 * xr; mr = 0.9 * mr + 0.1 * gr; vr = 0.999 * vr + 0.001 * gr * gr
        xr -= 0.05 * (mr / (1 - 0.9 ** t)) / (np.sqrt(vr / (1 - 0.999 ** t)) + 1e-8)
        assert abs(x[0] - xr) < 1e-12
    assert abs(x[0]) < 0.5
