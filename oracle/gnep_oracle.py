"""ctypes front-end of the fp64 CPU oracle (oracle/gnep_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference leg may import this module.  It never imports the CUDA package.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gnep_oracle.c")
_LIB = os.path.join(_HERE, "libgnep_oracle.so")


def build(force=False):
    """Compile the oracle with gcc (fp64, no FMA contraction, OpenMP over structures)."""
    if (not force) and os.path.exists(_LIB) and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC):
        return _LIB
    cmd = ["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-std=gnu11", _SRC,
           "-o", _LIB, "-lm"]
    subprocess.check_call(cmd)
    return _LIB


class Spec(C.Structure):
    _fields_ = [("T", C.c_int32), ("NR", C.c_int32), ("KR", C.c_int32), ("NA", C.c_int32),
                ("KA", C.c_int32), ("L", C.c_int32), ("use4", C.c_int32), ("use5", C.c_int32),
                ("Nn", C.c_int32),
                ("loss_mode", C.c_int32), ("rcR", C.c_double), ("rcA", C.c_double),
                ("lam_e", C.c_double), ("lam_f", C.c_double), ("lam_v", C.c_double),
                ("lam_2", C.c_double)]


def make_spec(d):
    """d: dict with the keys of gnep_synth.MODEL_SPECS entries."""
    return Spec(T=d["n_species"], NR=d["n_radial"], KR=d["n_basis_radial"], NA=d["n_angular"],
                KA=d["n_basis_angular"], L=d["l_max"], use4=int(d["use_4body"]), use5=int(d.get("use_5body", False)),
                Nn=d["n_neurons"],
                loss_mode=d.get("loss_mode", 0), rcR=d["rc_radial"], rcA=d["rc_angular"],
                lam_e=d["lambda_e"], lam_f=d["lambda_f"], lam_v=d["lambda_v"], lam_2=d["lambda_2"])


NLM = 80            # (l,m) slots for l = 1..8, slot lm = l*l - 1 + m
_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        dp = C.POINTER(C.c_double)
        L.orc_ndes.restype = C.c_int
        L.orc_num_params.restype = C.c_int64
        L.orc_max_threads.restype = C.c_int
        L.orc_batch_create.restype = C.c_void_p
        L.orc_batch_create.argtypes = [C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                       C.c_double, C.c_double, C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_batch_destroy.argtypes = [C.c_void_p]
        L.orc_batch_num_pairs.restype = C.c_int64
        L.orc_batch_num_pairs.argtypes = [C.c_void_p, C.c_int]
        L.orc_batch_get_neighbors.argtypes = [C.c_void_p, C.c_int] + [C.c_void_p] * 4
        L.orc_batch_get_positions.argtypes = [C.c_void_p, C.c_void_p]
        L.orc_batch_set_refs.argtypes = [C.c_void_p] * 4
        L.orc_batch_set_weights.argtypes = [C.c_void_p] * 4
        L.orc_basis.argtypes = [C.c_double, C.c_int, C.c_double, C.c_void_p, C.c_void_p]
        L.orc_blm.argtypes = [C.c_double] * 3 + [C.c_void_p] * 2
        L.orc_blm_raw.argtypes = [C.c_double] * 3 + [C.c_void_p] * 2
        L.orc_clm.argtypes = [C.c_void_p]
        L.orc_kappa4.restype = C.c_double
        L.orc_p4.restype = C.c_double
        L.orc_p4.argtypes = [C.c_void_p] * 3
        L.orc_kappa5.restype = C.c_double
        L.orc_p5.restype = C.c_double
        L.orc_p5.argtypes = [C.c_void_p] * 3
        L.orc_descriptors.argtypes = [C.c_void_p] * 4
        L.orc_network.restype = C.c_double
        L.orc_network.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int] + [C.c_void_p] * 4
        L.orc_predict.argtypes = [C.c_void_p] * 7
        L.orc_loss.argtypes = [C.c_void_p] * 5
        L.orc_loss_and_grad.argtypes = [C.c_void_p] * 6
        L.orc_adam_step.argtypes = [C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                    C.c_int64, C.c_double, C.c_double, C.c_double, C.c_double]
        _lib = L
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _f64(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64)


def ndes(spec):
    return lib().orc_ndes(C.byref(spec))


def num_params(spec):
    return int(lib().orc_num_params(C.byref(spec)))


def max_threads():
    return int(lib().orc_max_threads())


def basis(rc, K, d):
    f = np.zeros(K); fp = np.zeros(K)
    lib().orc_basis(float(rc), int(K), float(d), _p(f), _p(fp))
    return f, fp


def blm(x, y, z):
    B = np.zeros(NLM); dB = np.zeros((NLM, 3))
    lib().orc_blm(float(x), float(y), float(z), _p(B), _p(dB))
    return B, dB


def blm_raw(x, y, z):
    b = np.zeros(NLM); g = np.zeros((NLM, 3))
    lib().orc_blm_raw(float(x), float(y), float(z), _p(b), _p(g))
    return b, g


def clm():
    c = np.zeros(NLM)
    lib().orc_clm(_p(c))
    return c


def kappa5():
    return float(lib().orc_kappa5())


def p5(s, want_grad=False):
    s = _f64(s)
    if not want_grad:
        return float(lib().orc_p5(_p(s), None, None))
    g = np.zeros(3); H = np.zeros((3, 3))
    v = float(lib().orc_p5(_p(s), _p(g), _p(H)))
    return v, g, H


def kappa4():
    return float(lib().orc_kappa4())


def p4(s, want_grad=False):
    s = _f64(s)
    if not want_grad:
        return float(lib().orc_p4(_p(s), None, None))
    g = np.zeros(5); H = np.zeros((5, 5))
    v = float(lib().orc_p4(_p(s), _p(g), _p(H)))
    return v, g, H


class Batch:
    """A resident batch: wrapped positions and both neighbour lists (built once, like the GPU path)."""

    def __init__(self, spec, atom_offsets, positions, cells, types, ref_energy=None, ref_force=None,
                 ref_virial=None):
        self.spec = spec
        self.aoff = np.ascontiguousarray(atom_offsets, dtype=np.int32)
        self.S = len(self.aoff) - 1
        self.N = int(self.aoff[-1])
        pos = _f64(positions).reshape(-1); cell = _f64(cells).reshape(-1)
        typ = np.ascontiguousarray(types, dtype=np.int32)
        assert pos.size == 3 * self.N and cell.size == 9 * self.S and typ.size == self.N
        E, F, W = _f64(ref_energy), _f64(ref_force), _f64(ref_virial)
        self.h = lib().orc_batch_create(self.S, _p(self.aoff), _p(pos), _p(cell), _p(typ),
                                        float(spec.rcR), float(spec.rcA), _p(E), _p(F), _p(W))
        if not self.h:
            raise ValueError("degenerate cell")

    def __del__(self):
        if getattr(self, "h", None):
            lib().orc_batch_destroy(self.h)
            self.h = None

    def set_refs(self, E, F, W):
        E, F, W = _f64(E), _f64(F), _f64(W)
        lib().orc_batch_set_refs(self.h, _p(E), _p(F), _p(W))

    def set_weights(self, we=None, wf=None, wv=None):
        """Per-structure weights of the energy / force / virial terms (R40); None = ones, 0 = no label."""
        we, wf, wv = _f64(we), _f64(wf), _f64(wv)
        for w in (we, wf, wv):
            assert w is None or w.size == self.S
        lib().orc_batch_set_weights(self.h, _p(we), _p(wf), _p(wv))

    def num_pairs(self, which):
        return int(lib().orc_batch_num_pairs(self.h, which))

    def positions(self):
        p = np.zeros((self.N, 3))
        lib().orc_batch_get_positions(self.h, _p(p))
        return p

    def neighbors(self, which):
        n = self.num_pairs(which)
        rptr = np.zeros(self.N + 1, dtype=np.int64)
        j = np.zeros(n, dtype=np.int32); sh = np.zeros((n, 3), dtype=np.int32); r = np.zeros((n, 3))
        lib().orc_batch_get_neighbors(self.h, which, _p(rptr), _p(j), _p(sh), _p(r))
        return rptr, j, sh, r


def _qs(spec, q_scale):
    return np.ones(ndes(spec)) if q_scale is None else _f64(q_scale)


def descriptors(spec, theta, batch):
    theta = _f64(theta)
    q = np.zeros((batch.N, ndes(spec)))
    lib().orc_descriptors(C.byref(spec), _p(theta), batch.h, _p(q))
    return q


def network(spec, theta, q_scale, t, q, D=None):
    theta = _f64(theta); qs = _qs(spec, q_scale); q = _f64(q)
    Ep = np.zeros(ndes(spec))
    if D is None:
        E = lib().orc_network(C.byref(spec), _p(theta), _p(qs), int(t), _p(q), _p(Ep), None, None)
        return float(E), Ep
    D = _f64(D); h = np.zeros(ndes(spec))
    E = lib().orc_network(C.byref(spec), _p(theta), _p(qs), int(t), _p(q), _p(Ep), _p(D), _p(h))
    return float(E), Ep, h


def predict(spec, theta, q_scale, batch):
    theta = _f64(theta); qs = _qs(spec, q_scale)
    E = np.zeros(batch.S); F = np.zeros((batch.N, 3)); W = np.zeros((batch.S, 6))
    lib().orc_predict(C.byref(spec), _p(theta), _p(qs), batch.h, _p(E), _p(F), _p(W))
    return E, F, W


def loss(spec, theta, q_scale, batch):
    theta = _f64(theta); qs = _qs(spec, q_scale)
    t = np.zeros(5)
    lib().orc_loss(C.byref(spec), _p(theta), _p(qs), batch.h, _p(t))
    return t


def loss_and_grad(spec, theta, q_scale, batch):
    theta = _f64(theta); qs = _qs(spec, q_scale)
    t = np.zeros(5); g = np.zeros(num_params(spec))
    lib().orc_loss_and_grad(C.byref(spec), _p(theta), _p(qs), batch.h, _p(t), _p(g))
    return t, g


def adam_step(theta, m, v, grad, step, lr, beta1=0.9, beta2=0.999, eps=1e-8):
    """In place on theta, m, v (float64 contiguous arrays)."""
    for a in (theta, m, v):
        assert a.dtype == np.float64 and a.flags.c_contiguous
    grad = _f64(grad)
    lib().orc_adam_step(theta.size, _p(theta), _p(m), _p(v), _p(grad), int(step), float(lr),
                        float(beta1), float(beta2), float(eps))


def lr_schedule(step, n_warmup, n_total, lr_start, lr_stop):
    """Paper Eq.17 written out: linear warm-up from lr_stop to lr_start over n_warmup steps, then cosine
    decay back to lr_stop at n_total.  Pinned in tests/test_oracle_schedule.py by its end points, the warm-up slope,
    the cosine mid-point and monotonicity."""
    s = min(max(int(step), 0), int(n_total))
    if s < n_warmup:
        return lr_stop + s / n_warmup * (lr_start - lr_stop)
    if n_total == n_warmup:
        return lr_start
    return lr_stop + (lr_start - lr_stop) * 0.5 * (1.0 + np.cos(np.pi * (s - n_warmup) / (n_total - n_warmup)))
