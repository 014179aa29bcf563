"""Algorithmic flop / byte counts of the hot-path phases; FMA = 2 flop.

Host bookkeeping for bench.py's roofline only: no method arithmetic happens here.  Every count is what the
phase's algorithm needs once, given the phase's inputs (no credit for padding lanes, idle lanes, or the
second evaluation of something the same kernel already has).
"""

NLM = 24            # (l,m) slots, l = 1..4
HARM_B = 70         # the 24 harmonics b_lm of a unit vector
HARM_BG = 250       # harmonics and their 72 gradient components
FP32_LANES_PER_SM = 128
N_SM = 148
SM_MAX_HZ = 1.965e9


def fp32_peak_tflops(sm_hz=SM_MAX_HZ):
    """Plain FP32 ALU peak: 148 SMs x 128 FMA lanes x 2 flop x clock (B200_PROFILING.md unit counts)."""
    return N_SM * FP32_LANES_PER_SM * 2 * sm_hz / 1e12


def _basis_f(K):
    return 4 * K + 20          # T_k recurrence, f_k, cos


def _basis_ffp(K):
    return 11 * K + 40         # T_k, T_k', f_k, f_k', sincos


def phase_flops(spec, n_atoms, n_pairs_radial, n_pairs_angular):
    """dict phase name (as reported by gnep_phase_times) -> algorithmic flops of one epoch."""
    T, NR, KR, NA, KA, Nn = (spec["n_species"], spec["n_radial"], spec["n_basis_radial"], spec["n_angular"],
                             spec["n_basis_angular"], spec["n_neurons"])
    L = spec["l_max"]
    Nd = NR + NA * L + (NA if spec["use_4body"] else 0)
    N, nR, nA = n_atoms, n_pairs_radial, n_pairs_angular
    geom = 12                                      # d, 1/d, rhat
    f = {}
    f["a1_radial_descriptor"] = nR * (geom + _basis_f(KR) + KR) + N * 2 * T * KR * NR
    moments = 2 * T * KA * NA * NLM                  # S = c.A1 / T = c.A2 per atom (moment form)
    f["a1_angular_descriptor"] = nA * (geom + _basis_f(KA) + HARM_B + 2 * KA * NLM) + N * (moments + 3 * NA * NLM + 60 * NA)
    f["a2_network_forward"] = N * (4 * Nn * Nd + 2 * T * KR * NR + 12 * Nn)
    f["a3_radial_force"] = nR * (geom + _basis_ffp(KR) + 4 * KR + 30)
    f["a3_angular_force"] = nA * (geom + _basis_ffp(KA) + 4 * NA * KA + 4 * NA * NLM + HARM_BG + 9 * NLM + 40) + N * 3 * NA * NLM
    f["a3_radial_force"] += nA * 3          # + the gather of the angular pair forces, done by the same kernel
    f["a4_loss_and_seeds"] = N * 20
    f["a5_radial_adjoint"] = nR * (geom + _basis_ffp(KR) + 2 * KR + 30) + N * 2 * T * KR * NR
    f["a5_angular_adjoint"] = nA * (geom + _basis_ffp(KA) + 2 * KA + HARM_BG + 8 * NLM + 4 * KA * NLM + 30) + N * (moments + 3 * NA * NLM)
    f["a6_network_backward"] = N * (4 * Nn * Nd + 16 * Nn + 2 * Nd)
    f["a6_w0_gradient"] = N * 4 * Nn * Nd
    f["a7_radial_cgrad"] = N * 4 * NR * T * KR
    f["a7_angular_cgrad"] = N * (2 * moments + 12 * NA * NLM)     # sum_lm alpha A1 + beta A2; no pair sweep
    f["a8_grad_reduce"] = 0
    f["a9_adam"] = 0
    return f


def phase_bytes(spec, n_atoms, n_pairs_radial, n_pairs_angular):
    """dict phase -> algorithmic HBM bytes of one epoch (each array read or written once by its phase)."""
    T, NR, KR, NA, Nn = spec["n_species"], spec["n_radial"], spec["n_basis_radial"], spec["n_angular"], spec["n_neurons"]
    L = spec["l_max"]
    Nd = NR + NA * L + (NA if spec["use_4body"] else 0)
    N, nR, nA = n_atoms, n_pairs_radial, n_pairs_angular
    S_ = 4 * NA * NLM                 # bytes of S or T per atom
    M_ = 4 * T * KR                   # bytes of a radial moment row per atom
    A_ = 4 * T * spec["n_basis_angular"] * NLM   # bytes of A1 or A2 per atom
    b = {}
    b["a1_radial_descriptor"] = 16 * nR + N * (M_ + 4 * NR)
    b["a1_angular_descriptor"] = 16 * nA + N * (S_ + A_ + 4 * (Nd - NR))
    b["a2_network_forward"] = N * (4 * Nd + 4 * Nn + 4 + 4 * Nd + M_)
    b["a3_radial_force"] = (16 + 4 * KR) * nR + N * (M_ + 16 + 24)
    b["a3_angular_force"] = (16 + 4 + 16) * nA + N * (S_ + 4 * Nd)
    b["a3_radial_force"] += (4 + 16 + 16 + 16) * nA
    b["a4_loss_and_seeds"] = N * (4 + 16 + 24 + 12 + 16)
    b["a5_radial_adjoint"] = (16 + 16) * nR + N * (M_ + 4 * NR + 16)
    b["a5_angular_adjoint"] = (16 + 4 + 16) * nA + N * (2 * S_ + A_ + 4 * (Nd - NR) + 16)
    b["a6_network_backward"] = N * (4 * Nd * 3 + 4 * Nn * 3)
    b["a6_w0_gradient"] = N * (8 * Nn + 8 * Nd)
    b["a7_radial_cgrad"] = N * (8 * NR + 2 * M_)
    b["a7_angular_cgrad"] = N * (2 * S_ + 2 * A_ + 8 * Nd)
    b["a8_grad_reduce"] = 0
    b["a9_adam"] = 0
    return b


def path_flops_per_atom(spec, n_atoms, n_pairs_radial, n_pairs_angular):
    return sum(phase_flops(spec, n_atoms, n_pairs_radial, n_pairs_angular).values()) / max(n_atoms, 1)
