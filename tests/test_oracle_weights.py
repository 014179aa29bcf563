"""Pins for the per-structure loss weights of the oracle (R40; the paper's training sets mix
structures with and without virial labels, while Eq.10-12, weigh every structure equally).

Reading R40: a weight is the multiplicity of a structure in the training set, so each term is a weighted mean,
sum_s w_s (...)_s / sum_s w_s (forces: / (3 sum_s w_s N_s)).  That fixes everything that is pinned here WITHOUT the
oracle's own weighted formulas: ones = Eq.10-12 as printed; a 0/1 mask = the loss of the sub-batch that holds only the
labelled structures; an integer weight k = the structure listed k times; and the analytic gradient = finite
differences of the weighted plain loss.
"""
import numpy as np

from cases import labelled_case
from oracle import gnep_oracle as orc


def _sub(b, labels, keep):
    off = b["atom_offsets"]
    idx = np.concatenate([np.arange(off[s], off[s + 1]) for s in keep])
    new_off = np.concatenate([[0], np.cumsum([off[s + 1] - off[s] for s in keep])]).astype(np.int32)
    E, F, W = labels
    return new_off, b["positions"][idx], b["cells"][list(keep)], b["types"][idx], E[list(keep)], F[idx], W[list(keep)]


def test_unit_weights_are_eq_10_to_12():
    spec, sp, b, ob, theta, qs, labels = labelled_case(3, n_structs=4)
    t0, g0 = orc.loss_and_grad(sp, theta, qs, ob)
    ob.set_weights(np.ones(4), np.ones(4), np.ones(4))
    t1, g1 = orc.loss_and_grad(sp, theta, qs, ob)
    np.testing.assert_array_equal(t0, t1)
    np.testing.assert_allclose(g0, g1, rtol=1e-11, atol=1e-18)      # (the OpenMP sum over structures is unordered)


def test_mask_equals_the_sub_batch_of_labelled_structures():
    """Half the structures have no virial, one has no energy, one no forces: every term (and, term by term, the
    gradient) equals that of a batch that simply leaves those structures out."""
    spec, sp, b, ob, theta, qs, labels = labelled_case(3, n_structs=5, spec_over={"lambda_2": 0.0})
    we = np.array([1, 1, 0, 1, 1.0]); wf = np.array([1, 0, 1, 1, 1.0]); wv = np.array([1, 0, 1, 0, 0.0])
    ob.set_weights(we, wf, wv)
    t, g = orc.loss_and_grad(sp, theta, qs, ob)
    total = np.zeros_like(g)
    for k, (w, lam_key) in enumerate([(we, "lambda_e"), (wf, "lambda_f"), (wv, "lambda_v")]):
        keep = [s for s in range(5) if w[s] > 0]
        only = dict(spec, lambda_e=0.0, lambda_f=0.0, lambda_v=0.0); only[lam_key] = spec[lam_key]
        spk = orc.make_spec(only)
        sub = _sub(b, labels, keep)
        obk = orc.Batch(spk, *sub[:4]); obk.set_refs(*sub[4:])
        tk, gk = orc.loss_and_grad(spk, theta, qs, obk)                     # unweighted, labelled structures only
        assert abs(t[1 + k] - tk[1 + k]) <= 1e-13 * abs(tk[1 + k])
        total += gk
    np.testing.assert_allclose(g, total, rtol=1e-11, atol=1e-18)


def test_integer_weight_equals_replication():
    spec, sp, b, ob, theta, qs, labels = labelled_case(0, n_structs=3)
    w = np.array([3.0, 1.0, 2.0])
    ob.set_weights(w, w, w)
    t, g = orc.loss_and_grad(sp, theta, qs, ob)
    rep = [0, 0, 0, 1, 2, 2]
    sub = _sub(b, labels, rep)
    ob2 = orc.Batch(sp, *sub[:4]); ob2.set_refs(*sub[4:])
    t2, g2 = orc.loss_and_grad(sp, theta, qs, ob2)
    np.testing.assert_allclose(t, t2, rtol=1e-12)
    np.testing.assert_allclose(g, g2, rtol=1e-10, atol=1e-16)


def test_weighted_terms_numpy_restatement_and_fd_gradient():
    spec, sp, b, ob, theta, qs, (E, F, W) = labelled_case(3, n_structs=3)
    rng = np.random.default_rng(11)
    we, wf, wv = rng.uniform(0.2, 3.0, size=(3, 3))
    wv[1] = 0.0
    ob.set_weights(we, wf, wv)
    off = b["atom_offsets"]; ns = np.diff(off).astype(np.float64)
    Ep, Fp, Wp = orc.predict(sp, theta, qs, ob)
    t_e = np.sum(we * ((Ep - E) / ns) ** 2) / np.sum(we)
    t_f = sum(wf[s] * np.sum((Fp[off[s]:off[s + 1]] - F[off[s]:off[s + 1]]) ** 2) for s in range(3)) / (3 * np.sum(wf * ns))
    t_v = np.sum(wv[:, None] * ((Wp - W) / ns[:, None]) ** 2) / (6 * np.sum(wv))
    t, g = orc.loss_and_grad(sp, theta, qs, ob)
    np.testing.assert_allclose(t[1:4], [t_e, t_f, t_v], rtol=1e-13)
    idx = rng.choice(len(theta), size=24, replace=False)
    h = 1e-5
    for p in idx:
        tp = theta.copy(); tm = theta.copy(); tp[p] += h; tm[p] -= h
        fd = (orc.loss(sp, tp, qs, ob)[0] - orc.loss(sp, tm, qs, ob)[0]) / (2 * h)
        assert abs(fd - g[p]) <= 2e-6 * max(abs(g[p]), 1e-4), (p, fd, g[p])


def test_all_zero_weights_drop_the_term():
    spec, sp, b, ob, theta, qs, labels = labelled_case(0, n_structs=2)
    ob.set_weights(None, None, np.zeros(2))
    t, g = orc.loss_and_grad(sp, theta, qs, ob)
    assert t[3] == 0.0
    ob.set_weights(None, None, None); ob.set_refs(labels[0], labels[1], None)
    t2, g2 = orc.loss_and_grad(sp, theta, qs, ob)
    np.testing.assert_array_equal(t, t2)
    np.testing.assert_allclose(g, g2, rtol=1e-11, atol=1e-18)
