// reduce_kernels.cuh -- per-structure sums, loss terms and adjoint seeds (row a4), block->grid reduction of
// the partial gradients (row a8), fused Adam (row a9), and the output un-permutation kernels.
// All cross-CTA sums run in a fixed order with fp64 accumulators: no global atomics, bit-reproducible.
#pragma once
#include "common.cuh"

struct LossCfg {
  int S, N, T, P;
  int hasE, hasF, hasV, loss_mode;
  double lam_e, lam_f, lam_v, lam_2;
  // normalisers of Eq.10-12 over the WHOLE job: Z_E = sum_s w_e,s, Z_F = sum_s w_f,s N_s, Z_V = sum_s w_v,s
  // (= S, N, S without per-structure weights on one GPU; R40)
  double ZE, ZF, ZV;
  double rZE, rZF3, rZV6, rP;   // 1/Z_E, 1/(3 Z_F), 1/(6 Z_V), 1/P from the host (0 where Z = 0): no fp64 division on the device
  double l2_share;    // this rank's share of the L2 term (1 on one GPU, 1/world when structures are sharded)
};

template <int NV>
__device__ __forceinline__ void block_reduce_d(double (&v)[NV], double *sh /*[NV][nwarps]*/) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
#pragma unroll
  for (int i = 0; i < NV; ++i) {
    double x = v[i];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
    if (lane == 0) sh[i * nw + warp] = x;
  }
  __syncthreads();
  if (nw == 4) {                     // the usual 128-thread CTA: independent chains, no loop
#pragma unroll
    for (int i = 0; i < NV; ++i) v[i] = (sh[i * 4] + sh[i * 4 + 1]) + (sh[i * 4 + 2] + sh[i * 4 + 3]);
  } else {
#pragma unroll
    for (int i = 0; i < NV; ++i) {
      double x = 0.0;
      for (int w = 0; w < nw; ++w) x += sh[i * nw + w];
      v[i] = x;
    }
  }
  __syncthreads();
}

// Adam bookkeeping folded into the epoch's kernels when a whole training step is enqueued (gnep_train_epochs): the last
// CTA of k_struct_reduce advances the step counter and writes the two bias corrections (fp64 pow, once per step), and
// k_grad_reduce applies the update to the parameter it has just reduced.  `on == 0`: plain loss / gradient evaluation.
// lnb1, lnb2 = log(beta) from the host in fp64: 1 - beta^t = -expm1(t log beta), whose fp32 evaluation is accurate to
// ~1e-7 RELATIVE also where beta^t is close to 1 (a float pow would lose the difference; a double pow costs a
// microsecond of dependent fp64 instructions at the end of a kernel that one thread runs alone).
struct AdamPre { long long *step; float *bc; float beta1, beta2; double lnb1, lnb2; int on; };
struct AdamFuse { float *m, *v; const float *bc, *lr; float beta1, beta2, eps; int on; };

// a4: loss terms {L, t_e, t_f, t_v, t_2} (Eq.9-12 + L2) and the per-term seed multipliers, by ONE CTA (any size)
// scales = {se, sf, sv, s2}: all 1 in mean-square mode, 1/(2 sqrt t_x) in RMSE mode (0 if t_x = 0).
// `parts` was written by other CTAs of the same launch: read around L1.
#define LOSS_T2_CTAS 8      // extra CTAs of k_struct_reduce that sum theta^2 (the L2 term) in slices

// sum of theta[p]^2 over p = first, first + stride, ... (float4 groups), fp64, fixed order per thread
__device__ __forceinline__ double theta_sq(const float *__restrict__ theta, int P, int first, int stride) {
  double w[4] = {0, 0, 0, 0};
  const int P4 = P >> 2;
  for (int p = first; p < P4; p += stride) {
    const float4 x = ((const float4 *)theta)[p];
    w[0] += (double)x.x * x.x; w[1] += (double)x.y * x.y; w[2] += (double)x.z * x.z; w[3] += (double)x.w * x.w;
  }
  for (int p = 4 * P4 + first; p < P; p += stride) { double x = theta[p]; w[0] += x * x; }
  return (w[0] + w[1]) + (w[2] + w[3]);
}

// The loss terms {L, t_e, t_f, t_v, t_2} (Eq.9-12 + L2) and the per-term seed multipliers from the four batch sums, by
// thread 0 (thread 32 writes the Adam bias corrections of this step next to it).  scales = {se, sf, sv, s2}: all 1 in
// mean-square mode, 1/(2 sqrt t_x) in RMSE mode (0 if t_x = 0).
__device__ __forceinline__ void loss_write(const LossCfg &lc, double se, double sf, double sv, double s2, long long step0,
                                           float *__restrict__ terms, float *__restrict__ scales, const AdamPre &ap) {
  const long long t = step0 + 1;
  if (ap.on && threadIdx.x == 32) {                    // bias corrections 1 - beta^t
    ap.bc[0] = -expm1f((float)((double)t * ap.lnb1));
    ap.bc[1] = -expm1f((float)((double)t * ap.lnb2));
  }
  if (threadIdx.x == 0) {
    const double te = se * lc.rZE, tf = sf * lc.rZF3, tv = sv * lc.rZV6, t2 = lc.l2_share * s2 * lc.rP;
    double L, sc[4] = {1, 1, 1, 1};
    if (lc.loss_mode == 0) L = lc.lam_e * te + lc.lam_f * tf + lc.lam_v * tv + lc.lam_2 * t2;
    else {
      L = lc.lam_e * sqrt(te) + lc.lam_f * sqrt(tf) + lc.lam_v * sqrt(tv) + lc.lam_2 * sqrt(t2);
      sc[0] = te > 0 ? 0.5 / sqrt(te) : 0; sc[1] = tf > 0 ? 0.5 / sqrt(tf) : 0;
      sc[2] = tv > 0 ? 0.5 / sqrt(tv) : 0; sc[3] = t2 > 0 ? 0.5 / sqrt(t2) : 0;
    }
    terms[0] = (float)L; terms[1] = (float)te; terms[2] = (float)tf; terms[3] = (float)tv; terms[4] = (float)t2;
    for (int i = 0; i < 4; ++i) scales[i] = (float)sc[i];
    if (ap.on) *ap.step = t;
  }
}

// nt2 > 0: theta^2 arrives as nt2 slices; nt2 == 0: the CTA sums it here; nt2 < 0: this thread's share is t2_own.
// step0 = the step counter as read at the top of the kernel (its load is off the critical path there).
__device__ __forceinline__ void loss_final(const LossCfg &lc, const double *parts, const double *t2parts, int nt2, double t2_own,
                                           long long step0, const float *__restrict__ theta, float *__restrict__ terms,
                                           float *__restrict__ scales, const AdamPre &ap, double *sh) {
  double v[4] = {0, 0, 0, 0};
  for (int s = threadIdx.x; s < lc.S; s += blockDim.x) { v[0] += __ldcg(parts + s * 3); v[1] += __ldcg(parts + s * 3 + 1); v[2] += __ldcg(parts + s * 3 + 2); }
  if (nt2 > 0) { if (threadIdx.x == 0) for (int i = 0; i < nt2; ++i) v[3] += __ldcg(t2parts + i); }
  else if (nt2 == 0) v[3] = theta_sq(theta, lc.P, threadIdx.x, blockDim.x);
  else v[3] = t2_own;
  block_reduce_d<4>(v, sh);
  loss_write(lc, v[0], v[1], v[2], v[3], step0, terms, scales, ap);
}

// a4: one CTA per structure.  E_s = sum E_i, W_s = sum W_i (Eq.1, Eq.4), residuals of Eq.10-12 and the
// seeds e_s = 2 lam_e w_e,s dE_s/(Z_E N_s), u_i = 2 lam_f w_f,s (F_i - Fref_i)/(3 Z_F), omega_s = 2 lam_v w_v,s dW_s/(6 Z_V N_s)
// (w = per-structure weights, all ones by default: then Z_E = Z_V = S, Z_F = N and these are the seeds of Eq.10-12).
// CTAs S .. S + LOSS_T2_CTAS - 1 each sum a slice of theta^2 instead.  The CTA that finishes last (a ticket counter,
// reset for the next launch) adds the per-structure parts in structure order and the theta^2 slices in slice order --
// a fixed order whichever CTA it is -- and writes the loss terms: no second launch.
__global__ void __launch_bounds__(128)
k_struct_reduce(LossCfg lc, const int *__restrict__ srange /*[S][T][2]*/, const float *__restrict__ Ei,
                const float4 *__restrict__ Fat, const float *__restrict__ Wat, const double *__restrict__ Eref,
                const float *__restrict__ Fref_s, const double *__restrict__ Wref,
                const double *__restrict__ wgt /*[3][S]: w_e, w_f, w_v*/, double *__restrict__ Es,
                double *__restrict__ Ws, float *__restrict__ e_s, float4 *__restrict__ u,
                float *__restrict__ omega, double *parts /*[S][3] + [LOSS_T2_CTAS]*/, unsigned *ticket,
                const float *__restrict__ theta, float *__restrict__ terms, float *__restrict__ scales, AdamPre ap) {
  __shared__ double sh[9 * 4];
  __shared__ int last;
  double solo_sum[4] = {0, 0, 0, 0};       // thread 0, solo: the batch sums stay in registers
  // A batch of a few structures (size-1 mini-batches) is launched as ONE CTA that walks all structures and then
  // writes the loss terms itself: no ticket, no fences, no tail of a second CTA in the chain of dependent launches.
  const bool solo = gridDim.x == 1;
  double *t2parts = parts + (size_t)lc.S * 3;
  const long long step0 = ap.on ? *ap.step : 0;         // (every CTA reads it before the last one advances it)
  const double t2_own = solo ? theta_sq(theta, lc.P, threadIdx.x, blockDim.x) : 0.0;   // loads overlap the first structure's
  for (int s = blockIdx.x; s < (solo ? lc.S : blockIdx.x + 1); ++s) {
  if (s >= lc.S) {                          // a theta^2 slice
    double w[1] = {theta_sq(theta, lc.P, (s - lc.S) * blockDim.x + threadIdx.x, LOSS_T2_CTAS * blockDim.x)};
    block_reduce_d<1>(w, sh);
    if (threadIdx.x == 0) {
      t2parts[s - lc.S] = w[0];
      __threadfence();
      last = atomicAdd(ticket, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (!last) return;
    __threadfence();
    loss_final(lc, parts, t2parts, LOSS_T2_CTAS, 0.0, step0, theta, terms, scales, ap, sh);
    if (threadIdx.x == 0) *ticket = 0u;
    return;
  }
  double v[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0};   // E, W[6], sum |dF|^2, and (solo, first structure) this thread's share of theta^2
  if (solo && s == 0) v[8] = t2_own;
  int Ns = 0;
  const double we = wgt[s], wf = wgt[lc.S + s], wv = wgt[2 * lc.S + s];
  const float cu = lc.hasF && lc.ZF > 0 ? (float)(2.0 * lc.lam_f * wf / (3.0 * lc.ZF)) : 0.f;
  double eref = 0.0, wref[6] = {0, 0, 0, 0, 0, 0};      // requested now, used by thread 0 after the reduction
  if (threadIdx.x == 0) {
    if (lc.hasE) eref = Eref[s];
    if (lc.hasV)
#pragma unroll
      for (int c = 0; c < 6; ++c) wref[c] = Wref[s * 6 + c];
  }
  for (int t = 0; t < lc.T; ++t) {
    int b = srange[(s * lc.T + t) * 2], e = srange[(s * lc.T + t) * 2 + 1];
    Ns += e - b;
    for (int a = b + threadIdx.x; a < e; a += blockDim.x) {
      v[0] += (double)Ei[a];
#pragma unroll
      for (int c = 0; c < 6; ++c) v[1 + c] += (double)Wat[(size_t)a * 6 + c];
      float4 F = Fat[a];
      float dx = 0.f, dy = 0.f, dz = 0.f;
      if (lc.hasF) { dx = F.x - Fref_s[3 * (size_t)a]; dy = F.y - Fref_s[3 * (size_t)a + 1]; dz = F.z - Fref_s[3 * (size_t)a + 2]; }
      v[7] += (double)dx * dx + (double)dy * dy + (double)dz * dz;
      u[a] = make_float4(cu * dx, cu * dy, cu * dz, 0.f);
    }
  }
  block_reduce_d<9>(v, sh);
  if (threadIdx.x == 0) {
    Es[s] = v[0];
    // per-atom residuals through ONE reciprocal of N_s (an fp64 division is ~40 dependent instructions on this one thread)
    const double inv_ns = Ns > 0 ? 1.0 / (double)Ns : 0.0;
    double pe = 0.0, pv = 0.0, es = 0.0;
    if (lc.hasE && Ns > 0 && lc.ZE > 0) {
      const double dE = (v[0] - eref) * inv_ns;
      pe = we * dE * dE;
      es = 2.0 * lc.lam_e * we * lc.rZE * inv_ns * dE;
    }
    e_s[s] = (float)es;
    const bool onV = lc.hasV && Ns > 0 && lc.ZV > 0;
    const double k_om = onV ? 2.0 * lc.lam_v * wv * lc.rZV6 * inv_ns : 0.0;
#pragma unroll
    for (int c = 0; c < 6; ++c) {
      Ws[s * 6 + c] = v[1 + c];
      double om = 0.0;
      if (onV) {
        const double dW = (v[1 + c] - wref[c]) * inv_ns;
        pv += wv * dW * dW;
        om = k_om * dW;
      }
      omega[s * 6 + c] = (float)om;
    }
    parts[s * 3 + 0] = pe; parts[s * 3 + 1] = wf * v[7]; parts[s * 3 + 2] = pv;
    solo_sum[0] += pe; solo_sum[1] += wf * v[7]; solo_sum[2] += pv; solo_sum[3] += v[8];
    if (!solo) {
      __threadfence();                                         // parts visible before the ticket is taken
      last = atomicAdd(ticket, 1u) == gridDim.x - 1;
    }
  }
  __syncthreads();
  }   // structures of this CTA
  if (solo) {                               // thread 0 holds every sum
    loss_write(lc, solo_sum[0], solo_sum[1], solo_sum[2], solo_sum[3], step0, terms, scales, ap);
    return;
  }
  if (!last) return;
  __threadfence();
  loss_final(lc, parts, t2parts, LOSS_T2_CTAS, 0.0, step0, theta, terms, scales, ap, sh);
  if (threadIdx.x == 0) *ticket = 0u;
}

// a4 without structures (an empty batch still has its L2 term): the loss terms alone
__global__ void __launch_bounds__(128)
k_loss_final(LossCfg lc, const double *parts, const float *__restrict__ theta, float *__restrict__ terms,
             float *__restrict__ scales, AdamPre ap) {
  __shared__ double sh[8 * 4];
  loss_final(lc, parts, nullptr, 0, 0.0, ap.on ? *ap.step : 0, theta, terms, scales, ap, sh);
}

// a8: grad[p] = sum over the partial buffers that cover p (fixed order, fp64) + 2 lam_2 s2 theta_p / P.
// a[i] of a small array inside a kernel-parameter struct through static indices (a dynamic index would make the
// compiler copy the whole struct to local memory)
template <int NMAX>
__device__ __forceinline__ int pick(const int (&a)[NMAX], int i) {
  int v = a[0];
#pragma unroll
  for (int j = 1; j < NMAX; ++j) v = i == j ? a[j] : v;
  return v;
}
struct ReduceMap {
  int chunk_base[GNEP_MAX_SPECIES_C + 1];   // K-chunks (W0, cR partials) per species
  int gw_base[GNEP_MAX_SPECIES_C + 1];      // k_gradw_tc CTAs (W0, b0, w1, b1 partials) per species
  int n_warps_ca;                           // partial rows of the angular c-gradient
};
// Block = 8 consecutive parameters x 32 row lanes: every lane sums rows lane, lane+32, ... of its parameter's partial
// buffer in fp64, the 32 lane sums are added in lane order by one thread (fixed order -> bit-reproducible).
__global__ void __launch_bounds__(256)
k_grad_reduce(DevSpec sp, ReduceMap rm, float l2_share, float *theta, const float *__restrict__ scales,
              const float *__restrict__ partialCR, const float *__restrict__ partialCA,
              const float *__restrict__ partialW, const float *__restrict__ partialB, float *__restrict__ grad,
              AdamFuse af) {
  __shared__ double sh[32][9];
  const int tx = threadIdx.x & 7, ty = threadIdx.x >> 3;
  const int p = blockIdx.x * 8 + tx;
  double s = 0.0;
  if (p < sp.P) {
    const float *base; size_t stride; int r0, r1;
    if (p < sp.offA) {                       // cR[I][J][n][k]
      int k = p % sp.KR, r = p / sp.KR;
      int n = r % sp.NR; r /= sp.NR;
      int J = r % sp.T, I = r / sp.T;
      stride = (size_t)sp.NR * sp.T * sp.KRp;
      base = partialCR + n * sp.T * sp.KRp + J * sp.KRp + k;
      r0 = pick(rm.chunk_base, I); r1 = pick(rm.chunk_base, I + 1);
    } else if (p < sp.offNet) {              // cA[I][J][n][k]
      int x = p - sp.offA;
      int k = x % sp.KA, r = x / sp.KA;      // r = (I*T+J)*NA + n
      stride = (size_t)sp.T * sp.T * sp.NA * sp.KAp;
      base = partialCA + r * sp.KAp + k;
      r0 = 0; r1 = rm.n_warps_ca;
    } else {
      int x = p - sp.offNet;
      int t = x / sp.netSize, y = x - t * sp.netSize;
      int nW = sp.Nn * sp.Ndes;
      r0 = pick(rm.gw_base, t); r1 = pick(rm.gw_base, t + 1);
      if (y < nW) { stride = nW; base = partialW + y; }
      else { stride = 2 * sp.Nn + 1; base = partialB + (y - nW); }
    }
    for (int r = r0 + ty; r < r1; r += 32) s += (double)base[(size_t)r * stride];
  }
  sh[ty][tx] = s;
  __syncthreads();
  if (ty == 0 && p < sp.P) {
    double t = 0.0;
#pragma unroll
    for (int r = 0; r < 32; ++r) t += sh[r][tx];
    const float th = theta[p];
    t += 2.0 * (double)l2_share * (double)sp.lam_2 * (double)scales[3] * (double)th / (double)sp.P;
    const float g = (float)t;
    grad[p] = g;
    if (af.on) {                             // a9 on the parameter just reduced (same arithmetic as k_adam)
      const float c1 = af.bc[0], c2 = af.bc[1], lr = *af.lr;
      const float mm = af.beta1 * af.m[p] + (1.f - af.beta1) * g;
      const float vv = af.beta2 * af.v[p] + (1.f - af.beta2) * g * g;
      af.m[p] = mm; af.v[p] = vv;
      theta[p] = th - lr * (mm / c1) / (sqrtf(vv / c2) + af.eps);
    }
  }
}

// a9: textbook Adam with bias correction (Kingma & Ba Alg.1); step counter on the device (graph-safe).
__global__ void __launch_bounds__(256)
k_adam(int P, float *__restrict__ theta, float *__restrict__ m, float *__restrict__ v,
       const float *__restrict__ grad, const long long *__restrict__ step, const float *__restrict__ lr_p, float beta1,
       float beta2, float eps) {
  __shared__ float sc[2];
  if (threadIdx.x == 0) {          // the bias corrections need fp64 pow: once per block, not once per parameter
    const double t = (double)(*step + 1);
    sc[0] = (float)(1.0 - pow((double)beta1, t)); sc[1] = (float)(1.0 - pow((double)beta2, t));
  }
  __syncthreads();
  int p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= P) return;
  const float lr = *lr_p;          // device scalar: a learning-rate schedule changes it without re-building the epoch graph
  const float c1 = sc[0], c2 = sc[1];
  float g = grad[p];
  float mm = beta1 * m[p] + (1.f - beta1) * g;
  float vv = beta2 * v[p] + (1.f - beta2) * g * g;
  m[p] = mm; v[p] = vv;
  theta[p] -= lr * (mm / c1) / (sqrtf(vv / c2) + eps);
}
__global__ void k_step_inc(long long *step) { *step += 1; }
__global__ void k_set_scalar(float *dst, float v) { *dst = v; }

// outputs back to the caller's atom order
__global__ void k_unpermute_force(int N, const int *__restrict__ perm, const float4 *__restrict__ Fat, float *__restrict__ out) {
  int a = blockIdx.x * blockDim.x + threadIdx.x;
  if (a >= N) return;
  float4 f = Fat[a];
  size_t i = perm[a];
  out[3 * i] = f.x; out[3 * i + 1] = f.y; out[3 * i + 2] = f.z;
}
__global__ void k_unpermute_rows(int N, int W, const int *__restrict__ perm, const float *__restrict__ in, float *__restrict__ out) {
  size_t x = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (x >= (size_t)N * W) return;
  size_t a = x / W, c = x - a * W;
  out[(size_t)perm[a] * W + c] = in[x];
}
__global__ void k_permute_fref(int N, const int *__restrict__ perm, const double *__restrict__ in, float *__restrict__ out) {
  int a = blockIdx.x * blockDim.x + threadIdx.x;
  if (a >= N) return;
  size_t i = perm[a];
  out[3 * (size_t)a] = (float)in[3 * i]; out[3 * (size_t)a + 1] = (float)in[3 * i + 1]; out[3 * (size_t)a + 2] = (float)in[3 * i + 2];
}
__global__ void k_d2f(int n, const double *__restrict__ in, float *__restrict__ out) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) out[i] = (float)in[i];
}
