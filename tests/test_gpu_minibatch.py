"""Mini-batch training through shared handles + the Eq.17 schedule (paper P:142) against the
oracle: every mini-batch is its own resident batch on a handle that shares the parent's parameters and Adam state; a
step is one graph-replayed epoch of that handle at lr(s)."""
import numpy as np
import pytest

from cases import labelled_case
from oracle import gnep_oracle as orc

pytestmark = pytest.mark.gpu


def _slice(b, labels, lo, hi):
    off = b["atom_offsets"]; a0, a1 = off[lo], off[hi]
    E, F, W = labels
    return ((off[lo:hi + 1] - a0).astype(off.dtype), b["positions"][a0:a1], b["cells"][lo:hi], b["types"][a0:a1],
            E[lo:hi], F[a0:a1], W[lo:hi])


@pytest.mark.parametrize("config,n_structs,bs", [(1, 6, 2), (0, 4, 1)])
def test_minibatch_trajectory_matches_oracle(config, n_structs, bs):
    from paper_2507_00528_b200 import Gnep, lr_schedule
    spec, sp, b, ob, theta, qs, labels = labelled_case(config, n_structs=n_structs)
    nb = n_structs // bs
    epochs, n_warm = 2, 2
    n_total = epochs * nb
    parent = Gnep(dict(spec, q_scale=qs))
    parent.set_params(theta.astype(np.float32))
    handles, obatches = [], []
    for k in range(nb):
        off, pos, cells, types, E, F, W = _slice(b, labels, k * bs, (k + 1) * bs)
        h = parent if k == 0 else parent.create_shared()
        h.load_batch(off, pos, cells, types, E, F, W)
        handles.append(h)
        o = orc.Batch(sp, off, pos, cells, types); o.set_refs(E, F, W)
        obatches.append(o)
    th = theta.copy(); m = np.zeros_like(th); v = np.zeros_like(th)
    s = 0
    for _ in range(epochs):
        for k in range(nb):
            lr = orc.lr_schedule(s, n_warm, n_total, 1e-3, 1e-5)
            assert lr_schedule(s, n_warm, n_total, 1e-3, 1e-5) == pytest.approx(lr, rel=1e-14)
            t_ref, g_ref = orc.loss_and_grad(sp, th, qs, obatches[k])
            orc.adam_step(th, m, v, g_ref, s + 1, lr)
            th_seen = handles[k].get_params().astype(np.float64)         # the parameters this step's loss is evaluated at
            terms = handles[k].train_epochs(1, lr)
            # loss parity at 1e-5 on IDENTICAL parameters (the two trajectories drift apart at the 1e-6 level, which the
            # final parameter check bounds; the loss of the oracle's own trajectory agrees to 1e-4)
            assert abs(terms[0] - orc.loss(sp, th_seen, qs, obatches[k])[0]) <= 1e-5 * abs(t_ref[0])
            assert abs(terms[0] - t_ref[0]) <= 1e-4 * abs(t_ref[0])
            s += 1
    for h in handles:                                                    # every handle sees the same shared state
        th_gpu = h.get_params().astype(np.float64)
        assert np.linalg.norm(th_gpu - th) / np.linalg.norm(th) < 1e-4
        assert h.get_opt_state()[2] == n_total
    for h in handles[1:]:
        h.destroy()
    parent.destroy()


def test_held_out_evaluation_on_a_shared_handle(kernel_set):
    """gnep_evaluate: RMSEs of a test batch held by a shared handle, with and without a virial reference."""
    from paper_2507_00528_b200 import Gnep
    spec, sp, b, ob, theta, qs, labels = labelled_case(1, n_structs=5)
    parent = Gnep(dict(spec, q_scale=qs))
    off, pos, cells, types, E, F, W = _slice(b, labels, 0, 3)
    parent.load_batch(off, pos, cells, types, E, F, W)
    parent.set_params(theta.astype(np.float32))
    test = parent.create_shared()
    off, pos, cells, types, E, F, W = _slice(b, labels, 3, 5)
    test.load_batch(off, pos, cells, types, E, F, W)
    o = orc.Batch(sp, off, pos, cells, types); o.set_refs(E, F, W)
    t_ref, _ = orc.loss_and_grad(sp, theta, qs, o)
    np.testing.assert_allclose(test.evaluate(), np.sqrt(t_ref[1:4]), rtol=1e-5)
    # independent restatement from the oracle's predictions: RMSE over structures / atoms x 3 / structures x 6
    Ep, Fp, Wp = orc.predict(sp, theta, qs, o)
    ns = np.diff(off)
    want = [np.sqrt(np.mean(((Ep - E) / ns) ** 2)), np.sqrt(np.mean((Fp - F) ** 2)), np.sqrt(np.mean(((Wp - W) / ns[:, None]) ** 2))]
    np.testing.assert_allclose(test.evaluate(), want, rtol=1e-5)
    test.set_targets(E, F, None)
    r = test.evaluate()
    assert r[2] == 0.0 and r[0] == pytest.approx(want[0], rel=1e-5)
    parent.train_epochs(1, 1e-3)                      # training on the parent moves the shared parameters ...
    assert not np.allclose(test.evaluate()[:2], want[:2], rtol=1e-6)   # ... and the held-out errors with them
    test.destroy(); parent.destroy()


def test_shared_handle_and_evaluate_error_paths():
    import ctypes as C
    from paper_2507_00528_b200 import Gnep, GnepError, load_library
    import gnep_synth as gs
    L = load_library()
    out = C.c_void_p()
    assert L.gnep_create_shared(None, C.byref(out)) == -1              # EINVAL: no parent
    g = Gnep(dict(gs.MODEL_SPECS[0]))
    child = g.create_shared()
    with pytest.raises(GnepError) as e:
        child.evaluate()                                                # ESTATE: the shared handle has no batch yet
    assert e.value.code == -2
    theta = gs.draw_params(dict(gs.MODEL_SPECS[0]), 0).astype(np.float32)
    child.set_params(theta)                                             # parameters are one device buffer for both
    np.testing.assert_array_equal(g.get_params(), theta)
    child.destroy(); g.destroy()
