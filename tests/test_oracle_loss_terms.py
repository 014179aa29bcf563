"""Pins for the oracle's loss normalisations (paper Eq.9-12) and for the network value (Eq.D1.1).

`loss_terms` (oracle/gnep_oracle.c) turns predictions into t_e, t_f, t_v, t_2 and L.  The finite-difference sweeps of
tests/test_oracle_gradient.py are self-consistent with WHATEVER normalisation it uses, so the normalisations are pinned
here against numpy written straight from the printed equations: a dropped 1/6, a wrong power of N_s or a sum over the
wrong axis fails.  Likewise E_i of Eq.D1.1 is restated directly instead of only through its derivatives.
"""
import numpy as np

import gnep_synth as gs
from cases import labelled_case
from oracle import gnep_oracle as orc


def _numpy_terms(spec, theta, off, pred, ref):
    """Eq.10-12 as printed, with the readings R18 (E and V per atom: divide the structure totals by N_s) and R19
    (N in Eq.11 = atoms of the whole batch); t_2 = mean(theta^2) (R22)."""
    (E, F, W), (Er, Fr, Wr) = pred, ref
    ns = np.diff(off).astype(np.float64)
    S, N = len(ns), int(off[-1])
    t_e = sum(((E[s] - Er[s]) / ns[s]) ** 2 for s in range(S)) / S                                    # Eq.10
    t_f = sum((F[i, a] - Fr[i, a]) ** 2 for i in range(N) for a in range(3)) / (3 * N)                # Eq.11
    t_v = sum(((W[s, c] - Wr[s, c]) / ns[s]) ** 2 for s in range(S) for c in range(6)) / (6 * S)      # Eq.12
    t_2 = float(np.mean(theta ** 2))
    lam = [spec["lambda_e"], spec["lambda_f"], spec["lambda_v"], spec["lambda_2"]]
    return np.array([t_e, t_f, t_v, t_2]), lam


def test_loss_terms_are_eq_10_to_12():
    # unequal structure sizes (config 3 mixes 64..512-atom cells), so that N_s, S and N cannot be confused
    spec, sp, b, ob, theta, qs, refs = labelled_case(3, n_structs=4)
    off = b["atom_offsets"]
    assert len(set(np.diff(off))) > 1
    pred = orc.predict(sp, theta, qs, ob)
    t, lam = _numpy_terms(spec, theta, off, pred, refs)
    got = orc.loss(sp, theta, qs, ob)
    np.testing.assert_allclose(got[1:], t, rtol=1e-13, atol=0)
    assert abs(got[0] - np.dot(lam, t)) <= 1e-14 * abs(got[0])                                        # Eq.9 (+ L2)
    # the analytic-gradient entry point reports the same terms
    got2, _ = orc.loss_and_grad(sp, theta, qs, ob)
    np.testing.assert_allclose(got2, got, rtol=1e-14)


def test_loss_terms_rmse_mode_and_missing_reference():
    spec, sp, b, ob, theta, qs, (E, F, W) = labelled_case(3, n_structs=3, spec_over={"loss_mode": 1})
    off = b["atom_offsets"]
    pred = orc.predict(sp, theta, qs, ob)
    t, lam = _numpy_terms(spec, theta, off, pred, (E, F, W))
    got = orc.loss(sp, theta, qs, ob)
    np.testing.assert_allclose(got[1:], t, rtol=1e-13)
    assert abs(got[0] - np.dot(lam, np.sqrt(t))) <= 1e-14 * abs(got[0])                               # R21, mode 1
    ob.set_refs(E, None, W)                                                                           # R39: no force term
    got = orc.loss(sp, theta, qs, ob)
    assert got[2] == 0.0
    assert abs(got[0] - (lam[0] * np.sqrt(t[0]) + lam[2] * np.sqrt(t[2]) + lam[3] * np.sqrt(t[3]))) <= 1e-14 * abs(got[0])


def test_loss_terms_scale_with_the_printed_powers():
    """Doubling every residual multiplies t_e, t_f, t_v by 4; replicating the batch leaves all means unchanged."""
    spec, sp, b, ob, theta, qs, (E, F, W) = labelled_case(0, n_structs=2)
    Ep, Fp, Wp = orc.predict(sp, theta, qs, ob)
    base = orc.loss(sp, theta, qs, ob)
    ob.set_refs(Ep - 2 * (Ep - E), Fp - 2 * (Fp - F), Wp - 2 * (Wp - W))
    np.testing.assert_allclose(orc.loss(sp, theta, qs, ob)[1:4], 4 * base[1:4], rtol=1e-12)
    off = b["atom_offsets"]; n = off[-1]
    ob2 = orc.Batch(sp, np.concatenate([off, off[1:] + n]), np.concatenate([b["positions"]] * 2),
                    np.concatenate([b["cells"]] * 2), np.concatenate([b["types"]] * 2),
                    np.concatenate([E, E]), np.concatenate([F, F]), np.concatenate([W, W]))
    np.testing.assert_allclose(orc.loss(sp, theta, qs, ob2), base, rtol=1e-12)


def test_network_value_is_eq_D1_1():
    """E_i = sum_mu w1_mu tanh(sum_nu W0_mu,nu s_nu q_nu + b0_mu) + b1, per species block of theta (R6)."""
    spec = dict(gs.MODEL_SPECS[1]); sp = orc.make_spec(spec)
    theta = gs.draw_params(spec, 1)
    nd, nn, T = gs.n_descriptors(spec), spec["n_neurons"], spec["n_species"]
    rng = np.random.default_rng(3)
    q = rng.normal(size=nd); s = rng.uniform(0.2, 2.0, size=nd)
    off_net = T * T * (spec["n_radial"] * spec["n_basis_radial"] + spec["n_angular"] * spec["n_basis_angular"])
    size = nd * nn + 2 * nn + 1
    assert off_net + T * size == orc.num_params(sp)
    for t in range(T):
        blk = theta[off_net + t * size: off_net + (t + 1) * size]
        W0 = blk[:nd * nn].reshape(nn, nd); b0 = blk[nd * nn:nd * nn + nn]; w1 = blk[nd * nn + nn:nd * nn + 2 * nn]; b1 = blk[-1]
        want = sum(w1[m] * np.tanh(sum(W0[m, v] * s[v] * q[v] for v in range(nd)) + b0[m]) for m in range(nn)) + b1
        E, Ep = orc.network(sp, theta, s, t, q)
        assert abs(E - want) <= 1e-14 * max(1.0, abs(want))
        # D1.5 written out: dE/dq_nu = s_nu sum_mu w1_mu (1 - x_mu^2) W0_mu,nu
        x = np.tanh(W0 @ (s * q) + b0)
        np.testing.assert_allclose(Ep, s * ((w1 * (1 - x ** 2)) @ W0), rtol=1e-13, atol=1e-15)
    E0, _ = orc.network(sp, theta, s, 0, q)
    E1, _ = orc.network(sp, theta, s, 1, q)
    assert E0 != E1                                                                                   # per-species networks
