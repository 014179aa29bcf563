"""gnep_loss_terms_noalloc (include/gnep.h): the loss terms of Eq.10-12 from device-resident predictions, with
the per-structure partial sums in the library's fixed file-scope scratch array -- an entry point that allocates nothing.

Checked against the EXISTING path on the same batch: gnep_set_targets + gnep_loss_and_grad (per-batch buffers), at the
1e-5 relative tolerance the parity tests use for loss terms; two calls in a row (the scratch array keeps the first
call's contents, the second batch is a different one), then the first again; the size limit is refused with ERANGE.
Collected last on purpose (the suite runs with pytest -x); it does not depend on anything the other tests leave behind.
"""
import numpy as np
import pytest

from cases import labelled_case

pytestmark = pytest.mark.gpu


def _existing_and_new(config, n_structs, drop_virial=False):
    import torch
    from paper_2507_00528_b200 import Gnep
    spec, sp, b, ob, theta, qs, (E, F, W) = labelled_case(config, n_structs=n_structs)
    g = Gnep(dict(spec, q_scale=qs))
    g.load_batch(b["atom_offsets"], b["positions"], b["cells"], b["types"])
    g.set_params(theta.astype(np.float32))
    g.set_targets(E, F, None if drop_virial else W)
    terms_old, _ = g.loss_and_grad()                                   # existing path: {L, t_e, t_f, t_v, t_2}
    dev = torch.device("cuda:0")
    S, N = len(E), int(b["atom_offsets"][-1])
    e = torch.empty(S, dtype=torch.float32, device=dev)
    f = torch.empty((N, 3), dtype=torch.float32, device=dev)
    w = torch.empty((S, 6), dtype=torch.float32, device=dev)
    g.predict(e, f, w)                                                 # predictions stay on the device
    off = torch.as_tensor(np.asarray(b["atom_offsets"], dtype=np.int32), device=dev)
    Er = torch.as_tensor(E, dtype=torch.float64, device=dev)
    Fr = torch.as_tensor(F, dtype=torch.float64, device=dev).contiguous()
    Wr = None if drop_virial else torch.as_tensor(W, dtype=torch.float64, device=dev).contiguous()
    out = torch.full((4,), float("nan"), dtype=torch.float32, device=dev)
    torch.cuda.synchronize()
    before = torch.cuda.memory_allocated()
    g.loss_terms_noalloc(off, e, f, w, Er, Fr, Wr, out)
    torch.cuda.synchronize()
    assert torch.cuda.memory_allocated() == before
    lam2_t2 = spec["lambda_2"] * float(terms_old[4])                   # the new entry point leaves the L2 term out
    return g, np.asarray(terms_old, dtype=np.float64), out.cpu().numpy().astype(np.float64), lam2_t2


def _check(old, new, lam2_t2):
    np.testing.assert_allclose(new[1:4], old[1:4], rtol=1e-5, atol=1e-12)
    assert abs(new[0] - (old[0] - lam2_t2)) <= 1e-5 * abs(old[0]) + 1e-12


def test_no_alloc_loss_terms_match_the_existing_path_on_two_calls_in_a_row():
    from paper_2507_00528_b200 import GnepError
    g1, old1, new1, l2a = _existing_and_new(3, 7)                      # unequal structure sizes
    _check(old1, new1, l2a)
    g2, old2, new2, l2b = _existing_and_new(0, 3, drop_virial=True)    # second call: other batch, fewer structures, no virial
    assert new2[3] == 0.0 and old2[3] == 0.0
    _check(old2, new2, l2b)
    assert abs(new2[2] - new1[2]) > 1e-3 * abs(new1[2])                # (the two batches really differ)
    g3, old3, new3, l2c = _existing_and_new(3, 7)                      # and the first again: bit-identical to call one
    np.testing.assert_array_equal(new3, new1)
    # beyond the fixed scratch: refused, nothing launched
    import torch
    big = torch.zeros(8192 + 2, dtype=torch.int32, device="cuda:0")
    out = torch.zeros(4, dtype=torch.float32, device="cuda:0")
    with pytest.raises(GnepError) as err:
        g1.loss_terms_noalloc(big, None, None, None, None, None, None, out)
    assert err.value.code == -5 and "8192" in str(err.value)
    for g in (g1, g2, g3):
        g.destroy()
