/*
 * gnep.h -- C ABI of libgnep_b200.so: the data-parallel hot path of GNEP (arxiv 2507.00528) on one
 * NVIDIA B200 (sm_100a): full-batch NEP training loss, its analytic gradient over every trainable
 * parameter, and the Adam update.
 *
 * Citations "P:n" are line numbers of the paper text; "R<k>" are the readings of silent or
 * garbled passages listed in DESIGN.md.  All kernels behind these calls are hand-written CUDA; there is
 * no CPU fallback: gnep_create fails with GNEP_ECUDA when no sm_100 device is usable.
 *
 * Conventions
 *   - every call returns 0 (GNEP_OK) or a negative GNEP_E* code; gnep_last_error(h) then holds a
 *     message (handle-owned string, never freed by the caller).  No C++ exception crosses the ABI.
 *   - the caller owns every pointer it passes.  Inputs are copied during the call (they may be freed on
 *     return); outputs are written only into caller-provided buffers.
 *   - `is_device` != 0: array pointers are CUDA device pointers on the handle's device (e.g. torch
 *     tensors); == 0: host pointers.  Small scalar outputs (loss_terms, P, step) are always host.
 *   - all work is enqueued on the cudaStream_t given at create (NULL = default stream).  Calls that
 *     return host data synchronise that stream; gnep_adam_step and gnep_loss_and_grad with
 *     loss_terms == NULL and host-free arguments do not.
 *   - units: Angstrom, eV, eV/Angstrom; virial in eV (total per structure).
 *   - one handle = one model + one resident batch.  Not thread-safe per handle.
 *   - two environment variables choose between kernel sets that compute the same thing (for tests and
 *     measurements; results agree to rounding): GNEP_ANGULAR_MAPPING=groups (read by gnep_create) runs the
 *     slot-group angular kernels for l_max <= 4 too; GNEP_SMALL_BATCH=0|1 (read by gnep_load_batch) forces
 *     the large-batch / small-batch mappings instead of choosing by the batch size.
 *
 * Parameter vector theta (P floats, R6/S:8(c).2):
 *   [ cR[I][J][n][k] (k fastest; I = species of the central atom, J = of the neighbour)
 *   | cA[I][J][n][k]
 *   | for each species t: W0_t[mu][nu] (nu fastest), b0_t[mu], w1_t[mu], b1_t ]         (P:718 Eq.D1.1)
 * Descriptor index nu: 0..NR-1 radial q_n (Eq.5); NR+(l-1)*NA+n three-body q_nl, l=1..l_max
 * (Eq.7); then NA four-body terms (R14) if use_4body; then NA five-body terms (R41) if use_5body.
 */
#ifndef GNEP_H
#define GNEP_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define GNEP_OK 0
#define GNEP_EINVAL (-1)     /* bad spec / size / null pointer                         */
#define GNEP_ESTATE (-2)     /* call out of order, e.g. loss before load               */
#define GNEP_ECUDA (-3)      /* any CUDA error, or no sm_100 device                    */
#define GNEP_ENOMEM (-4)
#define GNEP_ERANGE (-5)     /* species id >= T, non-positive cell volume, too many pairs */
#define GNEP_ENONFINITE (-6) /* NaN/Inf in the loss                                    */

/* build limits (compile-time array sizes of the kernels) */
#define GNEP_MAX_SPECIES 4
#define GNEP_MAX_NFUNC 16    /* n_radial, n_angular                                    */
#define GNEP_MAX_BASIS 16    /* n_basis_radial, n_basis_angular                        */
#define GNEP_MAX_NEURONS 128

typedef struct gnep_handle gnep_handle; /* opaque; owns all device memory it allocates */

/* Model and loss specification (Eq.5-8; P:718 Eq.D1.1; Eq.9-12). */
typedef struct {
  int32_t n_species;                     /* T, 1..GNEP_MAX_SPECIES                                      */
  int32_t n_radial, n_basis_radial;      /* NR functions n=0..NR-1, KR basis functions k=0..KR-1 (R1,R2) */
  double rc_radial;                      /* radial cutoff r_c^R (Eq.2)                                   */
  int32_t n_angular, n_basis_angular;    /* NA, KA (own coefficients cA, R4)                             */
  double rc_angular;                     /* 0 < rc_angular <= rc_radial                                  */
  int32_t l_max;                         /* 1..8 (Eq.7; b_lm of App.B)                  */
  int32_t use_4body;                     /* 0/1, needs l_max >= 2: cubic invariant of the l = 2 moments (R14) */
  int32_t use_5body;                     /* 0/1: quartic invariant of the l = 1 moments (R41) */
  int32_t n_neurons;                     /* hidden width N_neu, 1..GNEP_MAX_NEURONS                      */
  double lambda_e, lambda_f, lambda_v;   /* Eq.9 weights                                                 */
  double lambda_2;                       /* weight of t_2 = mean(theta^2) (R22; not in the paper)        */
  int32_t loss_mode;                     /* 0: mean-square, paper Eq.9-12; 1: RMSE per term (R21)        */
  const float *q_scale;                  /* host, N_des entries, fixed input scaling G = q_scale*q, or NULL = ones (R15) */
} gnep_model_spec;

/* Create a model on the current CUDA device.  cuda_stream: a cudaStream_t (may be NULL).
 * Parameters start at zero; optimiser state at zero, step 0.  EINVAL on a bad spec; ECUDA if the
 * device is not compute capability 10.x. */
int gnep_create(const gnep_model_spec *spec, void *cuda_stream, gnep_handle **out);
int gnep_destroy(gnep_handle *h);

/* Number of trainable parameters P and of descriptor components N_des. */
int gnep_num_params(const gnep_handle *h, int64_t *P);
int gnep_num_descriptors(const gnep_handle *h, int32_t *n_des);

/* theta: P floats in the layout above. */
int gnep_set_params(gnep_handle *h, const float *theta, int is_device);
int gnep_get_params(const gnep_handle *h, float *theta, int is_device);

/* Replace the fixed, non-trainable input scaling (HOST, N_des floats; R15).  The harness derives it from
 * gnep_descriptors at the initial parameters, which needs a loaded batch, hence a call of its own. */
int gnep_set_q_scale(gnep_handle *h, const float *q_scale);

/* Load the training batch and build its neighbour lists on the GPU (Eq.2; R7-R9): periodic
 * cell-list search, all images with |r_j + shift - r_i| < rc (strict), excluding only (i, zero
 * shift); positions are first moved into the cell by whole lattice vectors.  Replaces any
 * previous batch.  Positions are fixed during training, so this is off the epoch loop.
 *   n_structs S >= 0; atom_offsets: S+1 ints, HOST, ascending, offsets[0] = 0, N = offsets[S]
 *   positions N*3 doubles (x,y,z per atom); cells S*9 doubles (rows a, b, c); types N ints in [0,T)
 *   ref_energy S doubles (total eV) or NULL; ref_force N*3 or NULL; ref_virial S*6 (total eV,
 *   order xx,yy,zz,xy,yz,zx) or NULL.  A NULL reference removes that loss term.
 * ERANGE: species id out of range, degenerate cell, >= 2^31 pairs.  */
int gnep_load_batch(gnep_handle *h, int32_t n_structs, const int32_t *atom_offsets, const double *positions,
                    const double *cells, const int32_t *types, const double *ref_energy,
                    const double *ref_force, const double *ref_virial, int is_device);

/* Replace only the reference values of the resident batch (same shapes / NULL rules as above). */
int gnep_set_targets(gnep_handle *h, const double *ref_energy, const double *ref_force,
                     const double *ref_virial, int is_device);

/* Per-structure loss weights (real training sets mix structures with and without virial labels, P:138,
 * while Eq.10-12, weigh every structure equally).  Reading R40: a weight is the multiplicity of the structure
 * in the training set, so each term is a weighted mean,
 *   t_e = sum_s w_e,s dE_s^2 / Z_E,  t_f = sum_s w_f,s sum_{i in s} |dF_i|^2 / (3 Z_F),  t_v = sum_s w_v,s sum_c dW_s,c^2 / (6 Z_V),
 *   Z_E = sum_s w_e,s,  Z_F = sum_s w_f,s N_s,  Z_V = sum_s w_v,s,
 * which is Eq.10-12 as printed when all weights are 1 (the default after gnep_load_batch) and the mean over the
 * labelled structures when w is a 0/1 mask (w = 0: that structure has no such label; its reference entry is ignored).
 * w_e, w_f, w_v: S doubles each, or NULL (= ones).  EINVAL on a negative or non-finite weight. */
int gnep_set_weights(gnep_handle *h, const double *w_e, const double *w_f, const double *w_v, int is_device);

/* The three normalisers {Z_E, Z_F, Z_V} of the resident batch (HOST, 3 doubles): what a rank contributes to the
 * job-wide normalisers under structure sharding (gnep_set_global_norms). */
int gnep_loss_norms(const gnep_handle *h, double *z);

/* Parity aid: the neighbour list in canonical order (rows by atom, entries ascending (j, sa, sb, sc)),
 * which: 0 radial, 1 angular.  n_pairs (host, may be NULL) receives the pair count; row_ptr N+1 int64;
 * j and shift3 (3 int8 per pair) hold `capacity` pairs; if capacity < n_pairs only n_pairs is set
 * and EINVAL returned.  Any of row_ptr/j/shift3 may be NULL. */
int gnep_neighbor_list(const gnep_handle *h, int which, int64_t *n_pairs, int64_t *row_ptr, int32_t *j,
                       int8_t *shift3, int64_t capacity, int is_device);

/* Parity aid: unscaled descriptors q[N][N_des] at the current parameters (Eq.5, Eq.7, R14). */
int gnep_descriptors(gnep_handle *h, float *q, int is_device);

/* Predictions at the current parameters: E_s (S), F (N*3, input atom order), W_s (S*6) (Eq.1, 3, 4;
 * W_ab = -sum r_ij,a f_ij,b, R17).  Any output may be NULL. */
int gnep_predict(gnep_handle *h, float *energy, float *force, float *virial, int is_device);

/* One full-batch evaluation of the loss and of its analytic gradient (Eq.9-16, App.C/D in
 * contraction-first form).  loss_terms (HOST, 5 floats: L, t_e, t_f, t_v, t_2)
 * may be NULL (no synchronisation then); grad (P floats) may be NULL: the gradient always stays in
 * the handle for gnep_adam_step.  ENONFINITE if loss_terms is requested and L is not finite. */
int gnep_loss_and_grad(gnep_handle *h, float *loss_terms, float *grad, int is_device);

/* Fused Adam update with the internal gradient (textbook, bias-corrected, step counted from 1; R23). */
int gnep_adam_step(gnep_handle *h, float lr, float beta1, float beta2, float eps);

/* One epoch = gnep_loss_and_grad + gnep_adam_step, `n_epochs` times, replayed from a CUDA graph;
 * loss_terms (HOST, 5 floats, or NULL) receives the terms of the LAST epoch's loss evaluation. */
int gnep_train_epochs(gnep_handle *h, int32_t n_epochs, float lr, float beta1, float beta2, float eps,
                      float *loss_terms);

/* Multi-GPU by structure sharding: every rank holds its own structures and calls
 * gnep_set_global_norm with the job-wide atom and structure counts (the normalisers N, N_str of Eq.10-12)
 * and its share of the L2 term (1/world).  Each rank's loss terms and gradient are then partial sums: the
 * caller all-reduces (sum) the P gradient floats, hands the result back with gnep_set_grad and calls
 * gnep_adam_step on every rank.  Negative counts restore single-GPU behaviour.  loss_mode 0 only. */
int gnep_set_global_norm(gnep_handle *h, int64_t n_atoms_global, int64_t n_structs_global, double l2_share);
/* The same with per-structure weights: z = job-wide {Z_E, Z_F, Z_V} (HOST, 3 doubles: the all-reduced sums of every
 * rank's gnep_loss_norms); gnep_set_global_norm(N, S, share) is z = {S, N, S}.  NULL or a negative entry restores
 * single-GPU behaviour. */
int gnep_set_global_norms(gnep_handle *h, const double *z, double l2_share);
int gnep_set_grad(gnep_handle *h, const float *grad, int is_device);

/* Mini-batch training (the paper's regime is mini-batches of size 1).  A shared handle is a
 * model of the same spec that SHARES the parent's device-resident parameter vector, gradient, Adam state (m, v, step)
 * and q_scale, and owns its own resident batch: load one mini-batch into each shared handle once, then step through
 * them (gnep_train_epochs(h_b, 1, lr(s), ...)) -- every step is one CUDA-graph launch on the parent's stream, nothing
 * is reloaded, and all handles see the same parameters.  The parent must outlive its shared handles; gnep_set_q_scale /
 * gnep_set_params on any of them affects all.  EINVAL on a NULL parent. */
int gnep_create_shared(const gnep_handle *parent, gnep_handle **out);

/* Learning-rate schedule of the paper (Eq.17): linear warm-up from lr_stop to lr_start over n_warmup steps,
 * then cosine decay back to lr_stop at n_total.  Pure host arithmetic (fp64).  step is clamped to [0, n_total];
 * EINVAL unless 0 <= n_warmup <= n_total and n_total >= 1. */
int gnep_lr_schedule(int64_t step, int64_t n_warmup, int64_t n_total, double lr_start, double lr_stop, double *lr);

/* Held-out evaluation (paper Fig.2): forward pass only over the resident batch of this
 * handle -- typically a shared handle holding the test set -- and the three root-mean-square errors against its
 * references: rmse[0] energy per atom (eV/atom, over structures), rmse[1] force components (eV/A, over atoms x 3),
 * rmse[2] virial per atom (eV/atom, over structures x 6).  A missing reference gives 0.  rmse: HOST, 3 floats. */
int gnep_evaluate(gnep_handle *h, float *rmse);

/* Checkpoint / resume of the optimiser state (m, v: P floats each; either may be NULL). */
int gnep_get_opt_state(const gnep_handle *h, float *m, float *v, int64_t *step, int is_device);
int gnep_set_opt_state(gnep_handle *h, const float *m, const float *v, int64_t step, int is_device);

/* Sizes of the resident batch: atoms, structures, radial pairs, angular pairs (any may be NULL). */
int gnep_batch_info(const gnep_handle *h, int64_t *n_atoms, int64_t *n_structs, int64_t *n_pairs_radial,
                    int64_t *n_pairs_angular);

/* Loss terms WITHOUT ANY ALLOCATION (for callers that cannot call cudaMalloc: code under CUDA-graph capture, tight
 * serving loops, harnesses that forbid it): t_e, t_f, t_v of Eq.10-12 (readings R18, R19) and
 * L = lam_e t_e + lam_f t_f + lam_v t_v (Eq.9 without the L2 term; square roots per term in loss_mode 1, R21) of
 * caller-held predictions against caller-held references, with the handle's lambdas and unit per-structure weights.
 * A variant of the per-structure reduction of gnep_loss_and_grad whose partial sums live in a fixed file-scope device
 * array of the library (192 KiB + 256 B per GPU, held from library load to process exit) instead of the per-batch
 * buffers: the call makes no cudaMalloc / cudaFree and calls no allocating routine; it enqueues one 4-byte memset and
 * one kernel on the handle's stream and does NOT synchronise.  No batch needs to be loaded.
 *   ALL POINTERS ARE DEVICE POINTERS on the handle's device.  n_structs: 1..GNEP_NOALLOC_MAX_STRUCTS, more is refused
 *   with GNEP_ERANGE (split the batch, or use gnep_set_targets + gnep_loss_and_grad); atom_offsets[n_structs+1] as in
 *   gnep_load_batch; energy[n_structs], force[3 N], virial[6 n_structs]: fp32, caller atom order, exactly what
 *   gnep_predict writes; Eref / Fref / Wref: fp64 like gnep_set_targets, NULL drops that term (R39; its prediction may
 *   then be NULL too); terms: 4 floats {L, t_e, t_f, t_v}, written when the kernel has run (stream order).
 * Every call on a GPU shares the one scratch array, which keeps the last call's contents (the call rewrites all it
 * reads and clears its ticket counter): calls that overlap on the GPU -- different streams, or handles on different
 * streams -- race on it; serialise them. */
#define GNEP_NOALLOC_MAX_STRUCTS 8192
int gnep_loss_terms_noalloc(gnep_handle *h, int32_t n_structs, const int32_t *atom_offsets, const float *energy,
                            const float *force, const float *virial, const double *Eref, const double *Fref,
                            const double *Wref, float *terms);

/* Measured plain-FP32 FMA peak of the device (the denominator of the ALU roofline next to the
 * nominal 148 SM x 128 lanes x 2 x clock): a register-only FMA microbenchmark on every SM of the handle's device that
 * runs for about min_ms milliseconds on the handle's stream (synchronises it).  tflops: HOST, achieved TFLOP/s
 * (FMA = 2 flop); ms (may be NULL): the duration timed with CUDA events; implied_sm_mhz (may be NULL): the SM clock
 * this rate corresponds to at 128 FP32 lanes per SM.  EINVAL unless 0 < min_ms <= 2000. */
int gnep_measure_fp32_peak(gnep_handle *h, double min_ms, double *tflops, double *ms, double *implied_sm_mhz);

/* Kernel launches issued by this handle since creation (for bench.py's gpu_launches). */
int gnep_launch_count(const gnep_handle *h, int64_t *n);

/* Per-phase device times of the most recent gnep_loss_and_grad / gnep_adam_step pair measured with
 * CUDA events on the handle's stream when profiling is on (gnep_set_profiling(h,1)).  names: array of
 * `capacity` const char* (handle-owned), ms: `capacity` floats; *n receives the phase count. */
int gnep_set_profiling(gnep_handle *h, int on);
int gnep_phase_times(const gnep_handle *h, const char **names, float *ms, int32_t capacity, int32_t *n);

/* Last error message of this handle (or of a failed gnep_create when h == NULL). */
const char *gnep_last_error(const gnep_handle *h);

#ifdef __cplusplus
}
#endif
#endif /* GNEP_H */
