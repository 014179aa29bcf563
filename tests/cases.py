"""Shared small cases for the tests (inputs only; labels come from the oracle teacher)."""
import numpy as np

import gnep_synth as gs
from oracle import gnep_oracle as orc


def golden(name):
    import os
    path = os.path.join(os.path.dirname(__file__), "golden", "closed_forms.txt")
    for line in open(path):
        if line.startswith("#") or not line.strip():
            continue
        k, *v = line.split()
        if k == name:
            return [float(x) for x in v]
    raise KeyError(name)


def labelled_case(config, n_structs=None, spec_over=None, noise=True):
    """Oracle-side view of a config: (spec dict, orc spec, batch dict, orc batch with teacher labels,
    student theta, q_scale, labels (E,F,W))."""
    spec = dict(gs.MODEL_SPECS[config])
    if spec_over:
        spec.update(spec_over)
    sp = orc.make_spec(spec)
    b = gs.make_batch(config, n_structs=n_structs)
    if spec["n_species"] != 2:
        b["types"] = gs.relabel_species(b["types"], spec["n_species"], config)
    ob = orc.Batch(sp, b["atom_offsets"], b["positions"], b["cells"], b["types"])
    theta = gs.draw_params(spec, config, "student")
    teacher = gs.draw_params(spec, config, "teacher")
    qs = gs.q_scale_from(orc.descriptors(sp, theta, ob))
    E, F, W = orc.predict(sp, teacher, qs, ob)
    if noise:
        E, F, W = gs.add_label_noise(config, b["atom_offsets"], E, F, W)
    ob.set_refs(E, F, W)
    return spec, sp, b, ob, theta, qs, (E, F, W)


def random_rotation(rng):
    q, r = np.linalg.qr(rng.normal(size=(3, 3)))
    q = q * np.sign(np.diag(r))
    if np.linalg.det(q) < 0:
        q[:, 0] = -q[:, 0]
    return q
