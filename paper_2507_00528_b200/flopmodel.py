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


# Which unit bounds each phase, from the ncu captures under profiles/ (issue slots / FP32 pipe: "alu"; DRAM: "hbm";
# neither: "latency").  bench.py reports the bound of the dominant phase from this table, never from a max() of fractions.
PHASE_BOUND = {
    "a1_radial_descriptor": "alu", "a1_angular_descriptor": "alu", "a1_descriptor_contraction": "hbm", "a2_network_forward": "alu", "a3_angular_force": "alu",
    "a3_radial_force": "alu", "a4_loss_and_seeds": "latency", "a5_radial_adjoint": "alu", "a5_angular_adjoint": "alu",
    "a6_network_backward": "alu", "a6_w0_gradient": "alu", "a7_radial_cgrad": "hbm", "a7_angular_cgrad": "hbm",
    "a8_grad_reduce": "latency", "a9_adam": "latency",
}


def method_flops(spec, n_atoms, n_pairs_radial, n_pairs_angular):
    """dict phase -> METHOD-algorithmic flops of one epoch: SURVEY.md 8(d).3 as written, in the paper's direct (per-pair
    g_n) form -- what the method needs whatever the implementation does (the moment-form counts of this design are
    `phase_flops`).  Per radial pair 2 NR KR for each of the three pair passes (g_n, g_n' for the force, g_n' for the
    adjoint) plus the shared 14 KR + 5 NR + 60 (basis, geometry) split over them; the radial c-gradient as its moment
    minimum 4 NR T KR per atom.  Per angular pair S 2 NA NLM, force 8 NA NLM, T 4 NA NLM, U/V 4 NA NLM plus the shared
    8 NA KA + 14 KA + 6 NLM + 360 (g_n, basis, harmonics with gradients) split over the four passes.  Network
    12 Nn N_des + 20 Nn per atom (z, E', p, h: 2 Nn N_des each; W0 gradient 4 Nn N_des)."""
    T, NR, KR, NA, KA, Nn = (spec["n_species"], spec["n_radial"], spec["n_basis_radial"], spec["n_angular"],
                             spec["n_basis_angular"], spec["n_neurons"])
    L = spec["l_max"]
    nlm = L * (L + 2)
    Nd = NR + NA * L + (NA if spec["use_4body"] else 0) + (NA if spec.get("use_5body") else 0)
    N, nR, nA = n_atoms, n_pairs_radial, n_pairs_angular
    rs = (14 * KR + 5 * NR + 60) / 3.0
    as_ = (8 * NA * KA + 14 * KA + 6 * nlm + 360) / 4.0
    f = {}
    f["a1_radial_descriptor"] = nR * (2 * NR * KR + rs)
    f["a1_angular_descriptor"] = nA * (2 * NA * nlm + as_) + N * 3 * NA * nlm
    f["a2_network_forward"] = N * (4 * Nn * Nd + 10 * Nn)
    f["a3_radial_force"] = nR * (2 * NR * KR + rs)
    f["a3_angular_force"] = nA * (8 * NA * nlm + as_)
    f["a4_loss_and_seeds"] = N * 20
    f["a5_radial_adjoint"] = nR * (2 * NR * KR + rs)
    f["a5_angular_adjoint"] = nA * (4 * NA * nlm + as_) + N * 3 * NA * nlm
    f["a6_network_backward"] = N * (4 * Nn * Nd + 10 * Nn)
    f["a6_w0_gradient"] = N * 4 * Nn * Nd
    f["a7_radial_cgrad"] = N * 4 * NR * T * KR
    f["a7_angular_cgrad"] = nA * (4 * NA * nlm + as_)
    f["a8_grad_reduce"] = 0
    f["a9_adam"] = 0
    return f


def method_bytes(spec, n_atoms, n_pairs_radial, n_pairs_angular):
    """dict phase -> METHOD-algorithmic HBM bytes: the 16-byte pair record once per pair pass, the 12-byte
    u_j gather in the adjoint passes, the 12-byte force scatter, and the per-atom rows q, E', D, gbar (4 N_des bytes each,
    written and read once), targets and forces -- no moment arrays, no S / T rows."""
    NR, NA, Nn = spec["n_radial"], spec["n_angular"], spec["n_neurons"]
    L = spec["l_max"]
    Nd = NR + NA * L + (NA if spec["use_4body"] else 0) + (NA if spec.get("use_5body") else 0)
    N, nR, nA = n_atoms, n_pairs_radial, n_pairs_angular
    b = {}
    b["a1_radial_descriptor"] = 16 * nR + N * 4 * NR
    b["a1_angular_descriptor"] = 16 * nA + N * 4 * (Nd - NR)
    b["a2_network_forward"] = N * (8 * Nd + 4)
    b["a3_radial_force"] = (16 + 12) * nR + N * (4 * NR + 16 + 24)
    b["a3_angular_force"] = (16 + 12) * nA + N * 4 * (Nd - NR)
    b["a4_loss_and_seeds"] = N * (4 + 16 + 24 + 12 + 16)
    b["a5_radial_adjoint"] = (16 + 12) * nR + N * (4 * NR + 16)
    b["a5_angular_adjoint"] = (16 + 12) * nA + N * (4 * (Nd - NR) + 16)
    b["a6_network_backward"] = N * 12 * Nd
    b["a6_w0_gradient"] = N * 8 * Nd
    b["a7_radial_cgrad"] = 16 * nR + N * 8 * NR
    b["a7_angular_cgrad"] = (16 + 12) * nA + N * 8 * (Nd - NR)
    b["a8_grad_reduce"] = 0
    b["a9_adam"] = 0
    return b


def phase_flops(spec, n_atoms, n_pairs_radial, n_pairs_angular):
    """dict phase name (as reported by gnep_phase_times) -> DESIGN flops of one epoch (moment form)."""
    T, NR, KR, NA, KA, Nn = (spec["n_species"], spec["n_radial"], spec["n_basis_radial"], spec["n_angular"],
                             spec["n_basis_angular"], spec["n_neurons"])
    L = spec["l_max"]
    Nd = NR + NA * L + (NA if spec["use_4body"] else 0) + (NA if spec.get("use_5body") else 0)
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


def contraction_phase(spec, n_atoms):
    """(flops, bytes) of `a1_descriptor_contraction`: with the geometry-only moments M1, A1 resident (built once per loaded
    batch) the epoch's descriptor pass is q_n = c.M1, S = c.A1, q_nl, 4-body per atom -- no pair work.  Counted as such in
    BOTH the method and the design columns: the pair sweeps it replaces are not credited to the epoch."""
    T, NR, KR, NA, KA = spec["n_species"], spec["n_radial"], spec["n_basis_radial"], spec["n_angular"], spec["n_basis_angular"]
    L = spec["l_max"]
    nlm = L * (L + 2)
    Nd = NR + NA * L + (NA if spec["use_4body"] else 0) + (NA if spec.get("use_5body") else 0)
    flops = n_atoms * (2 * T * KR * NR + 2 * T * KA * NA * nlm + 3 * NA * nlm + 60 * NA)
    byts = n_atoms * (4 * T * KR + 4 * T * KA * nlm + 4 * NA * nlm + 4 * Nd)
    return flops, byts
