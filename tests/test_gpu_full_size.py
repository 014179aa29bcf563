"""GPU parity at BASELINE.json's full sizes (configs 3 and 4), in the launch configuration bench.py times
(`gnep_train_epochs`: the CUDA graph of loss + gradient + Adam over the whole resident batch).

The fp64 oracle is fast enough (OpenMP over structures) to evaluate the whole batch once, so the comparison is the
real one, not a sample: loss terms, the full gradient, per-structure energies / virials and all forces, and the
parameters after one graph-replayed Adam epoch.  Labels come from the oracle teacher.  Also checked at full size:
properties that hold at any size (sum of forces per structure, bit-identical repeat evaluations).
"""
import numpy as np
import pytest

from cases import labelled_case
from oracle import gnep_oracle as orc

pytestmark = pytest.mark.gpu


def _rel(a, ref):
    return float(np.max(np.abs(np.asarray(a, dtype=np.float64) - ref)) / max(np.max(np.abs(ref)), 1e-300))


def _full(config):
    from paper_2507_00528_b200 import Gnep
    spec, sp, b, ob, theta, qs, (E, F, W) = labelled_case(config)
    off = b["atom_offsets"]
    g = Gnep(dict(spec, q_scale=qs))
    g.load_batch(off, b["positions"], b["cells"], b["types"], E, F, W)
    g.set_params(theta.astype(np.float32))
    info = g.batch_info()
    assert info["n_atoms"] == off[-1] and info["n_structs"] == len(off) - 1
    assert info["n_pairs_radial"] == ob.num_pairs(0) and info["n_pairs_angular"] == ob.num_pairs(1)
    # predictions of every structure
    Eg, Fg, Wg = g.predict()
    E_ref, F_ref, W_ref = orc.predict(sp, theta, qs, ob)
    assert _rel(Eg, E_ref) < 1e-5 and _rel(Fg, F_ref) < 1e-5 and _rel(Wg, W_ref) < 1e-5
    fsum = np.add.reduceat(np.asarray(Fg, dtype=np.float64), off[:-1], axis=0)
    assert np.max(np.abs(fsum)) < 1e-3 * np.max(np.abs(F_ref)) * np.sqrt(np.diff(off).max())   # Newton's third law
    # loss and the full gradient
    t_ref, g_ref = orc.loss_and_grad(sp, theta, qs, ob)
    terms, grad = g.loss_and_grad(want_grad=True)
    terms2, grad2 = g.loss_and_grad(want_grad=True)
    assert np.array_equal(grad, grad2) and np.array_equal(terms, terms2)                           # fixed-order sums
    for a, r in zip(terms, t_ref):
        assert abs(a - r) <= 1e-5 * abs(r) + 1e-12
    assert np.linalg.norm(grad - g_ref) / np.linalg.norm(g_ref) < 1e-4
    big = np.abs(g_ref) > 1e-6
    assert np.max(np.abs(grad[big] - g_ref[big]) / np.abs(g_ref[big])) < 1e-3
    if (~big).any():
        assert np.max(np.abs(grad[~big] - g_ref[~big])) < 1e-6
    # one epoch through the CUDA graph (the timed configuration)
    th = theta.copy(); m = np.zeros_like(th); v = np.zeros_like(th)
    orc.adam_step(th, m, v, g_ref, 1, 1e-3)
    g.train_epochs(1, 1e-3)
    th_gpu = g.get_params().astype(np.float64)
    assert np.linalg.norm(th_gpu - th) / np.linalg.norm(th) < 1e-4
    g.destroy()


def test_full_size_config3_mixed_1000():
    _full(3)


def test_full_size_config4_liquid_2000():
    _full(4)
