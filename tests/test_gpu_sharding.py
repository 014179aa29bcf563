"""GPU parity of the structure-sharded epoch (every sum of paper Eq.10-16, runs over
structures / atoms): a batch is split over TWO handles on the one GPU exactly as two ranks would hold it
(`sharding.shard_bounds`), each handle is told the job-wide normalisation (`gnep_set_global_norm`), the two partial
gradients and loss-term vectors are summed on the host (what the all-reduce does) and compared with the single-batch
oracle; the summed gradient goes back through `gnep_set_grad` and both handles take the same Adam step.
The two handles do not wait on one another: they are independent models evaluated one after the other."""
import numpy as np
import pytest

from cases import labelled_case
from oracle import gnep_oracle as orc
from paper_2507_00528_b200 import sharding

pytestmark = pytest.mark.gpu


def _shard(b, labels, lo, hi):
    off = b["atom_offsets"]; a0, a1 = off[lo], off[hi]
    E, F, W = labels
    return ((off[lo:hi + 1] - a0).astype(off.dtype), b["positions"][a0:a1], b["cells"][lo:hi], b["types"][a0:a1],
            E[lo:hi], F[a0:a1], W[lo:hi])


@pytest.mark.parametrize("config,n_structs,world", [(1, 6, 2), (3, 7, 3)])
def test_sharded_epoch_matches_single_batch_oracle(config, n_structs, world, kernel_set):
    from paper_2507_00528_b200 import Gnep
    spec, sp, b, ob, theta, qs, labels = labelled_case(config, n_structs=n_structs)
    off = b["atom_offsets"]
    bounds = sharding.shard_bounds(np.diff(off), world)
    assert bounds[0] == 0 and bounds[-1] == n_structs and all(bounds[r] < bounds[r + 1] for r in range(world))
    ranks = []
    for r in range(world):
        g = Gnep(dict(spec, q_scale=qs))
        g.load_batch(*_shard(b, labels, bounds[r], bounds[r + 1]))
        g.set_params(theta.astype(np.float32))
        g.set_global_norm(int(off[-1]), n_structs, 1.0 / world)
        ranks.append(g)
    th = theta.copy(); m = np.zeros_like(th); v = np.zeros_like(th)
    for step in range(1, 4):
        t_ref, g_ref = orc.loss_and_grad(sp, th, qs, ob)
        parts = [g.loss_and_grad(want_grad=True) for g in ranks]
        terms = np.sum([np.asarray(p[0], dtype=np.float64) for p in parts], axis=0)     # the all-reduce, on the host
        grad = np.sum([np.asarray(p[1], dtype=np.float64) for p in parts], axis=0)
        if step == 1:                                                                   # identical parameters
            np.testing.assert_allclose(terms, t_ref, rtol=1e-5, atol=1e-12)
            assert np.linalg.norm(grad - g_ref) / np.linalg.norm(g_ref) < 1e-4
            big = np.abs(g_ref) > 1e-6
            assert np.max(np.abs(grad[big] - g_ref[big]) / np.abs(g_ref[big])) < 1e-3
        orc.adam_step(th, m, v, g_ref, step, 1e-3)
        for g in ranks:
            g.set_grad(grad.astype(np.float32))
            g.adam_step(1e-3)
    thetas = [g.get_params() for g in ranks]
    for t in thetas[1:]:
        np.testing.assert_array_equal(t, thetas[0])                                     # replicas stay bit-identical
    assert np.linalg.norm(thetas[0].astype(np.float64) - th) / np.linalg.norm(th) < 1e-4
    # a held-out evaluation is normalised by the resident batch itself, whatever the job-wide norm says
    lo, hi = bounds[0], bounds[1]
    o0 = orc.Batch(sp, *_shard(b, labels, lo, hi)[:4]); o0.set_refs(*_shard(b, labels, lo, hi)[4:])
    t0 = orc.loss(sp, thetas[0].astype(np.float64), qs, o0)
    np.testing.assert_allclose(ranks[0].evaluate(), np.sqrt(t0[1:4]), rtol=1e-5)
    # RMSE mode cannot be sharded with one exchange (the seeds need the global terms first): refused
    from paper_2507_00528_b200 import GnepError
    g1 = Gnep(dict(spec, q_scale=qs, loss_mode=1))
    with pytest.raises(GnepError) as e:
        g1.set_global_norm(int(off[-1]), n_structs, 0.5)
    assert e.value.code == -1
    g1.destroy()
    for g in ranks:
        g.destroy()
