"""N > 1 host logic (structure sharding + one gradient all-reduce + replicated Adam) on CPU: two gloo ranks.

The CUDA engine cannot run here, so each rank drives `paper_2507_00528_b200.sharding` with a stand-in engine that
answers the same calls from the fp64 oracle on the rank's own structures.  Under `set_global_norm` a rank's loss
terms and gradient are partial sums of the job-wide ones: the stand-in builds them from the
oracle's per-term gradients, t_e and t_v weighted by S_loc/S_job, t_f by N_loc/N_job, the L2 term by its share.
The test checks that the sharded epoch reproduces the single-process oracle epoch (summed gradient, parameters
after Adam on every rank) and that the shard bounds are a deterministic, balanced, gap-free partition.
"""
import os
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import gnep_synth as gs  # noqa: E402
from oracle import gnep_oracle as orc  # noqa: E402
from paper_2507_00528_b200 import sharding  # noqa: E402

LR = 1e-3


class OracleEngine:
    """The `Gnep` calls used by sharding.py, answered by the oracle on a subset of config 0's structures."""

    def __init__(self, spec, batch, lo, hi, theta, qs, labels):
        self.spec, self.qs = dict(spec), qs
        off = batch["atom_offsets"]
        a0, a1 = off[lo], off[hi]
        self.offsets = (off[lo:hi + 1] - a0).astype(off.dtype)
        self.pos, self.cells, self.types = batch["positions"][a0:a1], batch["cells"][lo:hi], batch["types"][a0:a1]
        E, F, W = labels
        self.refs = (E[lo:hi], F[a0:a1], W[lo:hi])
        self.theta = theta.copy()
        self.m = np.zeros_like(theta); self.v = np.zeros_like(theta); self.step = 0
        self.n_atoms, self.n_structs = int(a1 - a0), hi - lo
        self.weights = None
        self.zjob, self.share = self.loss_norms(), 1.0
        self.grad = None

    def set_weights(self, we, wf, wv):
        self.weights = (np.asarray(we, float), np.asarray(wf, float), np.asarray(wv, float))
        self.zjob = self.loss_norms()

    def loss_norms(self):
        """{Z_E, Z_F, Z_V} of this rank's structures (R40): sum w_e, sum w_f N_s, sum w_v."""
        ns = np.diff(self.offsets).astype(float)
        we, wf, wv = self.weights if self.weights is not None else (np.ones_like(ns),) * 3
        return np.array([we.sum(), (wf * ns).sum(), wv.sum()])

    def set_global_norm(self, n_job, s_job, l2_share):
        self.zjob, self.share = np.array([s_job, n_job, s_job], float), l2_share

    def set_global_norms(self, z, l2_share):
        self.zjob, self.share = np.asarray(z, float), l2_share

    def _term(self, which):
        lam = dict(lambda_e=0.0, lambda_f=0.0, lambda_v=0.0, lambda_2=0.0)
        lam[which] = self.spec[which]
        sp = orc.make_spec(dict(self.spec, **lam))
        ob = orc.Batch(sp, self.offsets, self.pos, self.cells, self.types)
        ob.set_refs(*self.refs)
        if self.weights is not None:
            ob.set_weights(*self.weights)
        t, g = orc.loss_and_grad(sp, self.theta, self.qs, ob)
        return t[0], g

    def loss_and_grad(self, want_terms=False, grad=None):
        zl, zj = self.loss_norms(), self.zjob
        w = dict(lambda_e=zl[0] / zj[0], lambda_f=zl[1] / zj[1], lambda_v=zl[2] / zj[2], lambda_2=self.share)
        tot, g = 0.0, np.zeros_like(self.theta)
        for k, wk in w.items():
            t, gk = self._term(k)
            tot += wk * t; g += wk * gk
        self.grad = g
        if grad is not None:
            grad.copy_(torch.from_numpy(g.astype(np.float32)))
        return tot

    def set_grad(self, grad):
        self.grad = grad.numpy().astype(np.float64)

    def adam_step(self, lr, **kw):
        self.step += 1
        orc.adam_step(self.theta, self.m, self.v, self.grad, self.step, lr)


def _case():
    spec = dict(gs.MODEL_SPECS[0])
    b = gs.make_batch(0)
    sp = orc.make_spec(spec)
    ob = orc.Batch(sp, b["atom_offsets"], b["positions"], b["cells"], b["types"])
    theta = gs.draw_params(spec, 0, "student")
    teacher = gs.draw_params(spec, 0, "teacher")
    qs = gs.q_scale_from(orc.descriptors(sp, theta, ob))
    labels = gs.add_label_noise(0, b["atom_offsets"], *orc.predict(sp, teacher, qs, ob))
    ob.set_refs(*labels)
    return spec, sp, b, ob, theta, qs, labels


WEIGHTS = (np.array([1.0, 0.5, 2.0, 1.5]), np.array([2.0, 1.0, 0.0, 1.0]), np.array([1.0, 0.0, 0.0, 3.0]))


def _rank_main(rank, world, port, out_dir, weighted=False):
    os.environ["MASTER_ADDR"] = "127.0.0.1"; os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        spec, sp, b, ob, theta, qs, labels = _case()
        n_s = len(b["atom_offsets"]) - 1
        bounds = sharding.shard_bounds(np.diff(b["atom_offsets"]), world)
        eng = OracleEngine(spec, b, bounds[rank], bounds[rank + 1], theta, qs, labels)
        if weighted:
            eng.set_weights(*[w[bounds[rank]:bounds[rank + 1]] for w in WEIGHTS])
            z = sharding.setup_sharded_weighted(eng, dist)
            ns = np.diff(b["atom_offsets"])
            np.testing.assert_allclose(z, [WEIGHTS[0].sum(), (WEIGHTS[1] * ns).sum(), WEIGHTS[2].sum()], rtol=1e-14)
        else:
            n_job, s_job = sharding.setup_sharded(eng, dist, eng.n_atoms, eng.n_structs)
            assert (n_job, s_job) == (int(b["atom_offsets"][-1]), n_s)
        grad = torch.empty(len(theta), dtype=torch.float32)
        part = eng.loss_and_grad(grad=grad)
        total = sharding.reduce_loss_terms(dist, [part])[0]
        for _ in range(2):
            sharding.sharded_step(eng, dist, grad, LR)
        np.savez(os.path.join(out_dir, "rank%d.npz" % rank), theta=eng.theta, grad=eng.grad, loss=total)
    finally:
        dist.destroy_process_group()


def test_two_rank_epoch_matches_single_process(tmp_path):
    world, port = 2, 29500 + os.getpid() % 2000
    mp.spawn(_rank_main, args=(world, port, str(tmp_path)), nprocs=world, join=True)
    spec, sp, b, ob, theta, qs, labels = _case()
    th = theta.copy(); m = np.zeros_like(th); v = np.zeros_like(th)
    t0, _ = orc.loss_and_grad(sp, th, qs, ob)
    for step in (1, 2):
        _, g = orc.loss_and_grad(sp, th, qs, ob)
        orc.adam_step(th, m, v, g, step, LR)
    r0 = np.load(tmp_path / "rank0.npz"); r1 = np.load(tmp_path / "rank1.npz")
    assert abs(float(r0["loss"]) - t0[0]) <= 1e-6 * abs(t0[0])            # partial loss terms sum to the job's loss
    assert np.array_equal(r0["theta"], r1["theta"])                         # replicas stay identical
    assert np.linalg.norm(r0["grad"] - g) <= 1e-5 * np.linalg.norm(g)       # fp32 all-reduce of the partial gradients
    assert np.linalg.norm(r0["theta"] - th) <= 1e-6 * np.linalg.norm(th)


def test_two_rank_weighted_epoch_matches_single_process(tmp_path):
    """Per-structure weights (R40): every rank contributes its normalisers, the job-wide ones come from one all-reduce."""
    world, port = 2, 31500 + os.getpid() % 2000
    mp.spawn(_rank_main, args=(world, port, str(tmp_path), True), nprocs=world, join=True)
    spec, sp, b, ob, theta, qs, labels = _case()
    ob.set_weights(*WEIGHTS)
    th = theta.copy(); m = np.zeros_like(th); v = np.zeros_like(th)
    t0, _ = orc.loss_and_grad(sp, th, qs, ob)
    for step in (1, 2):
        _, g = orc.loss_and_grad(sp, th, qs, ob)
        orc.adam_step(th, m, v, g, step, LR)
    r0 = np.load(tmp_path / "rank0.npz"); r1 = np.load(tmp_path / "rank1.npz")
    assert abs(float(r0["loss"]) - t0[0]) <= 1e-6 * abs(t0[0])
    assert np.array_equal(r0["theta"], r1["theta"])
    assert np.linalg.norm(r0["grad"] - g) <= 1e-5 * np.linalg.norm(g)
    assert np.linalg.norm(r0["theta"] - th) <= 1e-6 * np.linalg.norm(th)


@pytest.mark.parametrize("world", [1, 2, 3, 8])
def test_shard_bounds_partition(world):
    rng = np.random.default_rng(7)
    w = rng.integers(64, 513, size=40)
    b = sharding.shard_bounds(w, world)
    assert b[0] == 0 and b[-1] == len(w) and len(b) == world + 1
    assert all(b[i] < b[i + 1] for i in range(world))                        # no empty shard
    loads = [w[b[i]:b[i + 1]].sum() for i in range(world)]
    assert max(loads) <= w.sum() / world + w.max()                          # balanced to within one structure
    assert b == sharding.shard_bounds(w, world)                             # deterministic
    assert sharding.shard_bounds([1, 1], 4) == [0, 0, 1, 1, 2]              # fewer structures than ranks
