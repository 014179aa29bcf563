"""Structure sharding of the GNEP epoch over ranks.

Every sum of the loss (paper Eq.10-12) and of its gradient (Eq.13-16) runs over structures / atoms, and neighbours
never cross structures, so the path shards by structure with ONE exchange per epoch: the all-reduce of the P-float
gradient.  Each rank loads its own structures; `set_global_norm(N_job, S_job, 1/world)` makes the rank's loss terms
and gradient *partial sums* of the job-wide ones (the L2 term is shared out evenly), the gradients are summed over
ranks, handed back with `set_grad`, and every rank applies the same Adam step, so parameters stay replicated.

This module is host logic only (which rank gets which structures, the order of the calls, the collective); it is
backend-agnostic (`torch.distributed`: nccl on GPUs, gloo in the CPU tests) and never computes any physics.  The
`engine` argument is anything with the `Gnep` methods used below.
"""
import numpy as np


def shard_bounds(weights, world):
    """Contiguous partition of the structures into `world` shards balanced by `weights` (e.g. atoms or pairs per
    structure).  Returns world+1 offsets; shard r owns structures [b[r], b[r+1]).  Deterministic, every rank computes
    the same answer; no shard is empty while there are at least `world` structures."""
    w = np.asarray(weights, dtype=np.float64)
    n = len(w)
    if world < 1:
        raise ValueError("world must be >= 1")
    if np.any(w < 0):
        raise ValueError("negative weight")
    cum = np.concatenate([[0.0], np.cumsum(w)])
    b = [0]
    for r in range(1, world):
        if n >= world:
            lo, hi = b[-1] + 1, n - (world - r)      # every shard keeps at least one structure
        else:
            lo, hi = b[-1], n
        k = lo + int(np.argmin(np.abs(cum[lo:hi + 1] - cum[-1] * r / world)))
        b.append(k)
    b.append(n)
    return b


def global_counts(dist, n_atoms_local, n_structs_local, device=None):
    """(N_job, S_job): atoms and structures of the whole job (one small all-reduce at load time)."""
    import torch
    t = torch.tensor([int(n_atoms_local), int(n_structs_local)], dtype=torch.int64, device=device)
    dist.all_reduce(t)
    return int(t[0]), int(t[1])


def setup_sharded(engine, dist, n_atoms_local, n_structs_local, device=None):
    """Tell the engine the job-wide normalisation.  Returns (N_job, S_job)."""
    world = dist.get_world_size()
    n_job, s_job = global_counts(dist, n_atoms_local, n_structs_local, device)
    engine.set_global_norm(n_job, s_job, 1.0 / world)
    return n_job, s_job


def setup_sharded_weighted(engine, dist, device=None):
    """The same when per-structure loss weights are set: every rank contributes its normalisers {Z_E, Z_F, Z_V}
    (`loss_norms`), their sums over ranks are the job-wide ones.  Returns them."""
    import torch
    world = dist.get_world_size()
    z = torch.tensor(np.asarray(engine.loss_norms(), dtype=np.float64), device=device)
    dist.all_reduce(z)
    z = z.cpu().numpy()
    engine.set_global_norms(z, 1.0 / world)
    return z


def sharded_step(engine, dist, grad, lr, **adam):
    """One epoch on every rank: partial loss+gradient, all-reduce (sum) of the gradient, identical Adam step.
    `grad` is a float32 torch tensor of P entries on the engine's device, reused every step."""
    engine.loss_and_grad(want_terms=False, grad=grad)      # returns after the engine's stream has written `grad`
    dist.all_reduce(grad)
    if getattr(grad, "is_cuda", False):
        # the collective is ordered on torch's current stream, gnep_set_grad copies on the ENGINE's stream: finish the
        # reduction before handing the buffer over (P floats, latency-bound; correct for any pairing of streams)
        import torch
        torch.cuda.current_stream(grad.device).synchronize()
    engine.set_grad(grad)
    engine.adam_step(lr, **adam)


def reduce_loss_terms(dist, terms, device=None):
    """Job-wide loss terms from the ranks' partial ones (they are partial sums under set_global_norm)."""
    import torch
    t = torch.tensor(np.asarray(terms, dtype=np.float64), device=device)
    dist.all_reduce(t)
    return t.cpu().numpy()
