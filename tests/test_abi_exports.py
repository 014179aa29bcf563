"""The C-ABI library loads and exports every symbol include/gnep.h declares (no compute without a GPU)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "gnep.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(gnep_[a-z0-9_]+)\s*\(", src)))


def test_header_symbols_exported_and_bound():
    from paper_2507_00528_b200 import EXPORTS, build
    lib = ctypes.CDLL(build.build())
    names = _declared()
    assert len(names) >= 20
    for n in names:
        assert hasattr(lib, n), n
    assert sorted(EXPORTS) == names


def test_create_fails_loudly_without_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    import gnep_synth as gs
    from paper_2507_00528_b200 import Gnep, GnepError
    with pytest.raises(GnepError) as e:
        Gnep(dict(gs.MODEL_SPECS[0]))
    assert e.value.code == -3          # GNEP_ECUDA: no CPU fallback


def test_bad_spec_rejected_before_touching_the_device():
    import gnep_synth as gs
    from paper_2507_00528_b200 import Gnep, GnepError
    for over in ({"l_max": 9}, {"n_species": 9}, {"rc_angular": 9.0}, {"n_neurons": 0}, {"loss_mode": 3},
                 {"use_4body": True, "l_max": 1}):
        with pytest.raises(GnepError) as e:
            Gnep(dict(gs.MODEL_SPECS[0], **over))
        assert e.value.code == -1
