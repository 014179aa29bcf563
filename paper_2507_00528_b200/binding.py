"""Thin ctypes binding of libgnep_b200.so (include/gnep.h): argument marshalling only.

Every step of the hot path runs in the CUDA kernels of csrc/; there is no CPU fallback and this module
never imports oracle/.  Arrays may be numpy arrays (host) or torch CUDA tensors (device pointers are passed
through unchanged).
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libgnep_b200.so")

EXPORTS = ["gnep_create", "gnep_destroy", "gnep_num_params", "gnep_num_descriptors", "gnep_set_params",
           "gnep_get_params", "gnep_set_q_scale", "gnep_load_batch", "gnep_set_targets", "gnep_neighbor_list",
           "gnep_descriptors", "gnep_predict", "gnep_loss_and_grad", "gnep_adam_step", "gnep_train_epochs",
           "gnep_get_opt_state", "gnep_set_opt_state", "gnep_batch_info", "gnep_launch_count",
           "gnep_set_profiling", "gnep_phase_times", "gnep_last_error", "gnep_set_global_norm", "gnep_set_grad",
           "gnep_create_shared", "gnep_lr_schedule", "gnep_evaluate", "gnep_measure_fp32_peak", "gnep_set_weights",
           "gnep_loss_norms", "gnep_set_global_norms", "gnep_loss_terms_noalloc"]

ERRORS = {-1: "GNEP_EINVAL", -2: "GNEP_ESTATE", -3: "GNEP_ECUDA", -4: "GNEP_ENOMEM", -5: "GNEP_ERANGE",
          -6: "GNEP_ENONFINITE"}


class GnepError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("%s: %s" % (ERRORS.get(code, code), msg))
        self.code = code


class ModelSpec(C.Structure):
    _fields_ = [("n_species", C.c_int32), ("n_radial", C.c_int32), ("n_basis_radial", C.c_int32),
                ("rc_radial", C.c_double), ("n_angular", C.c_int32), ("n_basis_angular", C.c_int32),
                ("rc_angular", C.c_double), ("l_max", C.c_int32), ("use_4body", C.c_int32),
                ("use_5body", C.c_int32), ("n_neurons", C.c_int32), ("lambda_e", C.c_double), ("lambda_f", C.c_double),
                ("lambda_v", C.c_double), ("lambda_2", C.c_double), ("loss_mode", C.c_int32),
                ("q_scale", C.POINTER(C.c_float))]


_lib = None


def load_library(build_if_missing=True):
    """dlopen the library; fails loudly (no fallback) when it cannot be built or loaded."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        if not build_if_missing:
            raise OSError("libgnep_b200.so is missing: run __graft_entry__.build()")
        _build.build()
    L = C.CDLL(LIB_PATH)
    vp = C.c_void_p
    L.gnep_last_error.restype = C.c_char_p
    L.gnep_last_error.argtypes = [vp]
    L.gnep_create.argtypes = [C.POINTER(ModelSpec), vp, C.POINTER(vp)]
    L.gnep_destroy.argtypes = [vp]
    L.gnep_num_params.argtypes = [vp, C.POINTER(C.c_int64)]
    L.gnep_num_descriptors.argtypes = [vp, C.POINTER(C.c_int32)]
    L.gnep_set_params.argtypes = [vp, vp, C.c_int]
    L.gnep_get_params.argtypes = [vp, vp, C.c_int]
    L.gnep_set_q_scale.argtypes = [vp, vp]
    L.gnep_load_batch.argtypes = [vp, C.c_int32] + [vp] * 7 + [C.c_int]
    L.gnep_set_targets.argtypes = [vp, vp, vp, vp, C.c_int]
    L.gnep_neighbor_list.argtypes = [vp, C.c_int, C.POINTER(C.c_int64), vp, vp, vp, C.c_int64, C.c_int]
    L.gnep_descriptors.argtypes = [vp, vp, C.c_int]
    L.gnep_predict.argtypes = [vp, vp, vp, vp, C.c_int]
    L.gnep_loss_and_grad.argtypes = [vp, vp, vp, C.c_int]
    L.gnep_adam_step.argtypes = [vp, C.c_float, C.c_float, C.c_float, C.c_float]
    L.gnep_train_epochs.argtypes = [vp, C.c_int32, C.c_float, C.c_float, C.c_float, C.c_float, vp]
    L.gnep_get_opt_state.argtypes = [vp, vp, vp, C.POINTER(C.c_int64), C.c_int]
    L.gnep_set_opt_state.argtypes = [vp, vp, vp, C.c_int64, C.c_int]
    L.gnep_batch_info.argtypes = [vp] + [C.POINTER(C.c_int64)] * 4
    L.gnep_set_global_norm.argtypes = [vp, C.c_int64, C.c_int64, C.c_double]
    L.gnep_set_grad.argtypes = [vp, vp, C.c_int]
    L.gnep_set_weights.argtypes = [vp, vp, vp, vp, C.c_int]
    L.gnep_loss_norms.argtypes = [vp, C.POINTER(C.c_double)]
    L.gnep_set_global_norms.argtypes = [vp, C.POINTER(C.c_double), C.c_double]
    L.gnep_create_shared.argtypes = [vp, C.POINTER(vp)]
    L.gnep_evaluate.argtypes = [vp, C.POINTER(C.c_float)]
    L.gnep_lr_schedule.argtypes = [C.c_int64, C.c_int64, C.c_int64, C.c_double, C.c_double, C.POINTER(C.c_double)]
    L.gnep_launch_count.argtypes = [vp, C.POINTER(C.c_int64)]
    L.gnep_measure_fp32_peak.argtypes = [vp, C.c_double] + [C.POINTER(C.c_double)] * 3
    L.gnep_set_profiling.argtypes = [vp, C.c_int]
    L.gnep_loss_terms_noalloc.argtypes = [vp, C.c_int32] + [vp] * 8
    L.gnep_phase_times.argtypes = [vp, C.POINTER(C.c_char_p), C.POINTER(C.c_float), C.c_int32, C.POINTER(C.c_int32)]
    for name in EXPORTS:
        if name != "gnep_last_error":
            getattr(L, name).restype = C.c_int
    _lib = L
    return L


def _is_torch(a):
    return type(a).__module__.startswith("torch")


def _ptr(a, dtype):
    """(pointer, is_device, keepalive) of a numpy array / torch tensor / None."""
    if a is None:
        return None, None, None
    if _is_torch(a):
        import torch
        want = {np.float32: torch.float32, np.float64: torch.float64, np.int32: torch.int32,
                np.int64: torch.int64, np.int8: torch.int8}[dtype]
        if a.dtype != want or not a.is_contiguous():
            a = a.to(want).contiguous()
        if a.is_cuda:
            return C.c_void_p(a.data_ptr()), 1, a
        a = a.numpy()
    a = np.ascontiguousarray(a, dtype=dtype)
    return a.ctypes.data_as(C.c_void_p), 0, a


def _out_ptr(a, dtype):
    """Like _ptr for an OUTPUT buffer: the library writes into the caller's memory, so a buffer that would have to be
    converted or copied (wrong dtype, non-contiguous, read-only) is an error, never a silent temporary."""
    if a is None:
        return None, None, None
    if _is_torch(a):
        import torch
        want = {np.float32: torch.float32, np.float64: torch.float64, np.int32: torch.int32,
                np.int64: torch.int64, np.int8: torch.int8}[dtype]
        if a.dtype != want or not a.is_contiguous():
            raise TypeError("output tensor must be contiguous %s" % want)
        if a.is_cuda:
            return C.c_void_p(a.data_ptr()), 1, a
        a = a.numpy()
    if not isinstance(a, np.ndarray) or a.dtype != np.dtype(dtype) or not a.flags.c_contiguous or not a.flags.writeable:
        raise TypeError("output array must be a writeable C-contiguous numpy array of %s" % np.dtype(dtype))
    return a.ctypes.data_as(C.c_void_p), 0, a


def _same_side(flags):
    f = [x for x in flags if x is not None]
    if f and any(x != f[0] for x in f):
        raise ValueError("all arrays of one call must live on the same side (host or device)")
    return f[0] if f else 0


class Gnep:
    """One model + one resident batch.  Method names follow include/gnep.h without the gnep_ prefix."""

    def __init__(self, spec, stream=None):
        """spec: dict with the field names of gnep_model_spec (q_scale optional numpy float32)."""
        self._L = load_library()
        self._h = C.c_void_p()
        qs = spec.get("q_scale")
        self._qs = None if qs is None else np.ascontiguousarray(qs, dtype=np.float32)
        ms = ModelSpec(**{k: (int(v) if isinstance(v, (bool, np.bool_)) else v) for k, v in spec.items()
                          if k != "q_scale"})
        if self._qs is not None:
            ms.q_scale = self._qs.ctypes.data_as(C.POINTER(C.c_float))
        sp = None
        if stream is not None:
            sp = C.c_void_p(stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream))
        rc = self._L.gnep_create(C.byref(ms), sp, C.byref(self._h))
        if rc != 0:
            raise GnepError(rc, (self._L.gnep_last_error(None) or b"").decode())
        self.spec = dict(spec)

    def _ck(self, rc):
        if rc != 0:
            raise GnepError(rc, (self._L.gnep_last_error(self._h) or b"").decode())

    def destroy(self):
        if getattr(self, "_h", None) and self._h.value:
            self._L.gnep_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    # ---- sizes ----
    def num_params(self):
        v = C.c_int64()
        self._ck(self._L.gnep_num_params(self._h, C.byref(v)))
        return v.value

    def num_descriptors(self):
        v = C.c_int32()
        self._ck(self._L.gnep_num_descriptors(self._h, C.byref(v)))
        return v.value

    def batch_info(self):
        v = [C.c_int64() for _ in range(4)]
        self._ck(self._L.gnep_batch_info(self._h, *[C.byref(x) for x in v]))
        return dict(n_atoms=v[0].value, n_structs=v[1].value, n_pairs_radial=v[2].value, n_pairs_angular=v[3].value)

    def launch_count(self):
        v = C.c_int64()
        self._ck(self._L.gnep_launch_count(self._h, C.byref(v)))
        return v.value

    # ---- parameters ----
    def set_params(self, theta):
        p, dev, _k = _ptr(theta, np.float32)
        assert np.prod(theta.shape) == self.num_params()
        self._ck(self._L.gnep_set_params(self._h, p, dev))

    def get_params(self, out=None):
        out = np.empty(self.num_params(), dtype=np.float32) if out is None else out
        p, dev, _k = _out_ptr(out, np.float32)
        self._ck(self._L.gnep_get_params(self._h, p, dev))
        return out

    def set_q_scale(self, q_scale):
        q = np.ascontiguousarray(q_scale, dtype=np.float32)
        assert q.size == self.num_descriptors()
        self._ck(self._L.gnep_set_q_scale(self._h, q.ctypes.data_as(C.c_void_p)))

    def get_opt_state(self):
        P = self.num_params()
        m = np.empty(P, dtype=np.float32); v = np.empty(P, dtype=np.float32); s = C.c_int64()
        self._ck(self._L.gnep_get_opt_state(self._h, m.ctypes.data_as(C.c_void_p), v.ctypes.data_as(C.c_void_p), C.byref(s), 0))
        return m, v, s.value

    def set_opt_state(self, m, v, step):
        pm, d1, _k1 = _ptr(m, np.float32); pv, d2, _k2 = _ptr(v, np.float32)
        self._ck(self._L.gnep_set_opt_state(self._h, pm, pv, int(step), _same_side([d1, d2])))

    # ---- batch ----
    def load_batch(self, atom_offsets, positions, cells, types, ref_energy=None, ref_force=None, ref_virial=None):
        off = np.ascontiguousarray(atom_offsets, dtype=np.int32)
        pp, d1, k1 = _ptr(positions, np.float64); pc, d2, k2 = _ptr(cells, np.float64); pt, d3, k3 = _ptr(types, np.int32)
        pe, d4, k4 = _ptr(ref_energy, np.float64); pf, d5, k5 = _ptr(ref_force, np.float64); pw, d6, k6 = _ptr(ref_virial, np.float64)
        dev = _same_side([d1, d2, d3, d4, d5, d6])
        self._ck(self._L.gnep_load_batch(self._h, len(off) - 1, off.ctypes.data_as(C.c_void_p), pp, pc, pt, pe, pf, pw, dev))
        self._n_atoms = int(off[-1]); self._n_structs = len(off) - 1

    def set_targets(self, ref_energy=None, ref_force=None, ref_virial=None):
        pe, d4, k4 = _ptr(ref_energy, np.float64); pf, d5, k5 = _ptr(ref_force, np.float64); pw, d6, k6 = _ptr(ref_virial, np.float64)
        self._ck(self._L.gnep_set_targets(self._h, pe, pf, pw, _same_side([d4, d5, d6])))

    def set_weights(self, w_e=None, w_f=None, w_v=None):
        """Per-structure weights of the energy / force / virial terms (None = ones, 0 = structure has no such label)."""
        pe, d1, _a = _ptr(w_e, np.float64); pf, d2, _b = _ptr(w_f, np.float64); pv, d3, _c = _ptr(w_v, np.float64)
        for w in (_a, _b, _c):
            assert w is None or int(np.prod(w.shape)) == self._n_structs
        self._ck(self._L.gnep_set_weights(self._h, pe, pf, pv, _same_side([d1, d2, d3])))

    def loss_norms(self):
        z = (C.c_double * 3)()
        self._ck(self._L.gnep_loss_norms(self._h, z))
        return np.array(z[:], dtype=np.float64)

    def neighbor_list(self, which):
        n = C.c_int64()
        self._ck(self._L.gnep_neighbor_list(self._h, which, C.byref(n), None, None, None, 0, 0))
        rp = np.empty(self._n_atoms + 1, dtype=np.int64); j = np.empty(n.value, dtype=np.int32)
        sh = np.empty((n.value, 3), dtype=np.int8)
        self._ck(self._L.gnep_neighbor_list(self._h, which, C.byref(n), rp.ctypes.data_as(C.c_void_p),
                                            j.ctypes.data_as(C.c_void_p), sh.ctypes.data_as(C.c_void_p), n.value, 0))
        return rp, j, sh

    # ---- the hot path ----
    def descriptors(self, out=None):
        out = np.empty((self._n_atoms, self.num_descriptors()), dtype=np.float32) if out is None else out
        p, dev, _k = _out_ptr(out, np.float32)
        self._ck(self._L.gnep_descriptors(self._h, p, dev))
        return out

    def predict(self, energy=None, force=None, virial=None):
        if energy is None and force is None and virial is None:
            energy = np.empty(self._n_structs, dtype=np.float32)
            force = np.empty((self._n_atoms, 3), dtype=np.float32)
            virial = np.empty((self._n_structs, 6), dtype=np.float32)
        pe, d1, _a = _out_ptr(energy, np.float32); pf, d2, _b = _out_ptr(force, np.float32); pw, d3, _c = _out_ptr(virial, np.float32)
        self._ck(self._L.gnep_predict(self._h, pe, pf, pw, _same_side([d1, d2, d3])))
        return energy, force, virial

    def loss_and_grad(self, want_terms=True, grad=None, want_grad=False):
        terms = np.empty(5, dtype=np.float32) if want_terms else None
        if want_grad and grad is None:
            grad = np.empty(self.num_params(), dtype=np.float32)
        pg, dev, _k = _out_ptr(grad, np.float32)
        pt = None if terms is None else terms.ctypes.data_as(C.c_void_p)
        self._ck(self._L.gnep_loss_and_grad(self._h, pt, pg, dev or 0))
        return terms, grad

    def adam_step(self, lr, beta1=0.9, beta2=0.999, eps=1e-8):
        self._ck(self._L.gnep_adam_step(self._h, lr, beta1, beta2, eps))

    def train_epochs(self, n_epochs, lr, beta1=0.9, beta2=0.999, eps=1e-8, want_terms=True):
        terms = np.empty(5, dtype=np.float32) if want_terms else None
        pt = None if terms is None else terms.ctypes.data_as(C.c_void_p)
        self._ck(self._L.gnep_train_epochs(self._h, int(n_epochs), lr, beta1, beta2, eps, pt))
        return terms

    # ---- structure sharding over ranks ----
    def set_global_norm(self, n_atoms_global, n_structs_global, l2_share):
        self._ck(self._L.gnep_set_global_norm(self._h, int(n_atoms_global), int(n_structs_global), float(l2_share)))

    def set_global_norms(self, z, l2_share):
        zz = (C.c_double * 3)(*[float(x) for x in z])
        self._ck(self._L.gnep_set_global_norms(self._h, zz, float(l2_share)))

    def set_grad(self, grad):
        p, dev, _k = _ptr(grad, np.float32)
        self._ck(self._L.gnep_set_grad(self._h, p, dev))

    # ---- mini-batches: handles that share this model's parameters and optimiser state ----
    def create_shared(self):
        """A handle with its own resident batch that shares this model's theta, gradient, Adam state and q_scale
        (gnep_create_shared).  Keep the parent alive while its shared handles are in use."""
        child = object.__new__(Gnep)
        child._L, child._h, child._qs, child.spec = self._L, C.c_void_p(), self._qs, dict(self.spec)
        child._parent = self
        self._ck(self._L.gnep_create_shared(self._h, C.byref(child._h)))
        return child

    def evaluate(self):
        """(rmse_energy eV/atom, rmse_force eV/A, rmse_virial eV/atom) of the resident batch against its references."""
        out = (C.c_float * 3)()
        self._ck(self._L.gnep_evaluate(self._h, out))
        return np.array(out[:], dtype=np.float32)

    # ---- profiling ----
    def measure_fp32_peak(self, min_ms=60.0):
        """dict(tflops, ms, implied_sm_mhz) of the FP32 FMA microbenchmark (gnep_measure_fp32_peak)."""
        v = [C.c_double() for _ in range(3)]
        self._ck(self._L.gnep_measure_fp32_peak(self._h, float(min_ms), *[C.byref(x) for x in v]))
        return dict(tflops=v[0].value, ms=v[1].value, implied_sm_mhz=v[2].value)

    def loss_terms_noalloc(self, atom_offsets, energy, force, virial, Eref, Fref, Wref, terms):
        """gnep_loss_terms_noalloc: {L, t_e, t_f, t_v} of device-resident predictions against device-resident references
        into the 4-float device tensor `terms`; allocates nothing and does not synchronise.  Every argument must already
        be a contiguous CUDA tensor of the right dtype (int32 offsets, float32 predictions, float64 references) or None:
        nothing is converted or copied here."""
        def dev(a, dtype):
            if a is None:
                return None
            p, d, _k = _out_ptr(a, dtype)            # (raises on a dtype / contiguity mismatch instead of copying)
            if d != 1:
                raise TypeError("gnep_loss_terms_noalloc takes CUDA tensors only")
            return p
        n_structs = int(atom_offsets.numel()) - 1
        self._ck(self._L.gnep_loss_terms_noalloc(self._h, n_structs, dev(atom_offsets, np.int32), dev(energy, np.float32),
                                                 dev(force, np.float32), dev(virial, np.float32), dev(Eref, np.float64),
                                                 dev(Fref, np.float64), dev(Wref, np.float64), dev(terms, np.float32)))
        return terms

    def set_profiling(self, on):
        self._ck(self._L.gnep_set_profiling(self._h, int(on)))

    def phase_times(self):
        cap = 64
        names = (C.c_char_p * cap)(); ms = (C.c_float * cap)(); n = C.c_int32()
        self._ck(self._L.gnep_phase_times(self._h, names, ms, cap, C.byref(n)))
        return [(names[i].decode(), float(ms[i])) for i in range(min(n.value, cap))]


def lr_schedule(step, n_warmup, n_total, lr_start, lr_stop):
    """Paper Eq.17 (linear warm-up, cosine decay) through the library's host function gnep_lr_schedule."""
    L = load_library()
    out = C.c_double()
    rc = L.gnep_lr_schedule(int(step), int(n_warmup), int(n_total), float(lr_start), float(lr_stop), C.byref(out))
    if rc != 0:
        raise GnepError(rc, "gnep_lr_schedule: bad arguments")
    return out.value
