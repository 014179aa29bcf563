// pair_kernels.cuh -- sweeps over the neighbour lists (rows a1, a3, a5, a7 of DESIGN.md section 2).
// One warp per atom.  Atoms are sorted by species (index "a"); pair records are
// float4(r_ij.x, r_ij.y, r_ij.z, bits(a_j)).  Radial rows are split in species segments segR[a][J..J+1]
// so that the neighbour species is warp-uniform; angular rows are processed in chunks of 32 pairs.
#pragma once
#include "common.cuh"

// per-warp dynamic shared memory helper
__device__ __forceinline__ float *warp_smem(float *base, int per_warp_floats) {
  return base + (threadIdx.x >> 5) * per_warp_floats;
}

// ------------------------------------------------------------------------------------------------
// a1 (radial):  M1[a][J][k] = sum_{j in seg J} f_k(d_ij)  ;  q_n = sum_{J,k} cR[I][J][n][k] M1[J][k]
// (paper Eq.5-6, in moment-factored form: g_n is linear in f_k)
// ------------------------------------------------------------------------------------------------
template <int KT>
__global__ void __launch_bounds__(GNEP_WARPS * 32)
k_radial_fwd(DevSpec sp, int N, const int *__restrict__ type_s, const int *__restrict__ segR,
             const float4 *__restrict__ pairR, const float *__restrict__ theta, float *__restrict__ q,
             float *__restrict__ M1) {
  extern __shared__ __align__(16) float smem[];
  float *cs = smem;                                          // [T*T*NR][KT]
  int ncs = sp.T * sp.T * sp.NR * KT;
  float *wbuf = warp_smem(smem + ncs, KT * 33 + KT);          // reduce buffer + moment row
  float *mrow = wbuf + KT * 33;
  stage_coeff(cs, theta, sp.T * sp.T * sp.NR, sp.KR, KT);
  __syncthreads();
  int lane = threadIdx.x & 31;
  int a = blockIdx.x * GNEP_WARPS + (threadIdx.x >> 5);
  if (a >= N) return;
  int I = type_s[a];
  float qn = 0.f;
  for (int J = 0; J < sp.T; ++J) {
    int p0 = segR[a * (sp.T + 1) + J], p1 = segR[a * (sp.T + 1) + J + 1];
    float acc[KT];
#pragma unroll
    for (int k = 0; k < KT; ++k) acc[k] = 0.f;
    for (int p = p0 + lane; p < p1; p += 32) {
      float4 r = pairR[p];
      float d = sqrtf(r.x * r.x + r.y * r.y + r.z * r.z);
      float f[KT];
      cheb_f<KT>(d, sp.rcRinv, f);
#pragma unroll
      for (int k = 0; k < KT; ++k) acc[k] += f[k];
    }
    float s = warp_transpose_reduce<KT>(acc, wbuf, lane);
    if (lane < KT) { M1[(size_t)a * sp.T * KT + J * KT + lane] = s; mrow[lane] = s; }
    __syncwarp();
    if (lane < sp.NR) {
      const float *c = cs + ((I * sp.T + J) * sp.NR + lane) * KT;
#pragma unroll
      for (int k = 0; k < KT; ++k) qn += c[k] * mrow[k];
    }
    __syncwarp();
  }
  if (lane < sp.NR) q[(size_t)a * sp.Ndes + lane] = qn;
}

// ------------------------------------------------------------------------------------------------
// a1 (angular): S_nlm = sum_j g_n(d_ij) B_lm(rhat_ij)  (Eq.8), q_nl = sum_m C_lm S_nlm^2 (Eq.7), 4-body
// phase 1: lane = pair, stages g_n and B_lm in shared memory; phase 2: lane = (n, 8 lm) register tile.
// ------------------------------------------------------------------------------------------------
template <int KT>
__global__ void __launch_bounds__(GNEP_WARPS * 32)
k_angular_fwd(DevSpec sp, int N, const int *__restrict__ type_s, const int *__restrict__ rowA,
              const float4 *__restrict__ pairA, const float *__restrict__ theta, float *__restrict__ q,
              float *__restrict__ S) {
  extern __shared__ __align__(16) float smem[];
  float *cs = smem;                                          // [T*T*NA][KT]
  int ncs = (sp.T * sp.T * sp.NA * KT + 3) & ~3;
  int per_warp = (sp.NA + GNEP_NLM) * 32 + sp.NA * GNEP_NLM;
  float *sg = warp_smem(smem + ncs, per_warp);               // [NA][32]
  float *sB = sg + sp.NA * 32;                               // [24][32]
  float *sS = sB + GNEP_NLM * 32;                            // [NA][24]
  stage_coeff(cs, theta + sp.offA, sp.T * sp.T * sp.NA, sp.KA, KT);
  __syncthreads();
  int lane = threadIdx.x & 31;
  int a = blockIdx.x * GNEP_WARPS + (threadIdx.x >> 5);
  if (a >= N) return;
  int I = type_s[a];
  int r0 = rowA[a], r1 = rowA[a + 1];
  const bool act = lane < 30;
  const int n1 = lane / 3, grp = lane - 3 * n1, n2 = n1 + 10;
  const bool on1 = act && n1 < sp.NA, on2 = act && n2 < sp.NA;
  float acc1[8], acc2[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) { acc1[i] = 0.f; acc2[i] = 0.f; }
  for (int c0 = r0; c0 < r1; c0 += 32) {
    int p = c0 + lane;
    if (p < r1) {
      float4 r = pairA[p];
      float d = sqrtf(r.x * r.x + r.y * r.y + r.z * r.z);
      float rinv = 1.f / d;
      int J = type_s[__float_as_int(r.w)];
      float f[KT];
      cheb_f<KT>(d, sp.rcAinv, f);
      const float *c = cs + (I * sp.T + J) * sp.NA * KT;
      for (int n = 0; n < sp.NA; ++n) {
        float g = 0.f;
#pragma unroll
        for (int k = 0; k < KT; ++k) g += c[n * KT + k] * f[k];
        sg[n * 32 + lane] = g;
      }
      blm_unit(r.x * rinv, r.y * rinv, r.z * rinv,
               [&](int lm, int, float b, float, float, float) { sB[lm * 32 + lane] = b; });
    } else {
      for (int n = 0; n < sp.NA; ++n) sg[n * 32 + lane] = 0.f;
#pragma unroll
      for (int lm = 0; lm < GNEP_NLM; ++lm) sB[lm * 32 + lane] = 0.f;
    }
    __syncwarp();
    int ng4 = (min(32, r1 - c0) + 3) >> 2;
    for (int g4 = 0; g4 < ng4; ++g4) {
      float4 ga = on1 ? *(const float4 *)(sg + n1 * 32 + 4 * g4) : make_float4(0, 0, 0, 0);
      float4 gb = on2 ? *(const float4 *)(sg + n2 * 32 + 4 * g4) : make_float4(0, 0, 0, 0);
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        float4 b = *(const float4 *)(sB + (grp * 8 + i) * 32 + 4 * g4);
        acc1[i] += ga.x * b.x + ga.y * b.y + ga.z * b.z + ga.w * b.w;
        acc2[i] += gb.x * b.x + gb.y * b.y + gb.z * b.z + gb.w * b.w;
      }
    }
    __syncwarp();
  }
  float *Sa = S + (size_t)a * sp.NA * GNEP_NLM;
  if (on1) {
#pragma unroll
    for (int i = 0; i < 8; ++i) { sS[n1 * GNEP_NLM + grp * 8 + i] = acc1[i]; Sa[n1 * GNEP_NLM + grp * 8 + i] = acc1[i]; }
  }
  if (on2) {
#pragma unroll
    for (int i = 0; i < 8; ++i) { sS[n2 * GNEP_NLM + grp * 8 + i] = acc2[i]; Sa[n2 * GNEP_NLM + grp * 8 + i] = acc2[i]; }
  }
  __syncwarp();
  float *qa = q + (size_t)a * sp.Ndes + sp.NR;
  for (int o = lane; o < sp.NA * sp.L; o += 32) {
    int l = o / sp.NA + 1, n = o - (l - 1) * sp.NA;
    int lm0 = l * l - 1;
    float v = 0.f;
    for (int m = 0; m <= 2 * l; ++m) { float s = sS[n * GNEP_NLM + lm0 + m]; v += 0.5f * c_C2[lm0 + m] * s * s; }
    qa[o] = v;
  }
  if (sp.use4 && lane < sp.NA) qa[sp.NA * sp.L + lane] = c_kappa4 * p4_value(sS + lane * GNEP_NLM + 3);
}

// ------------------------------------------------------------------------------------------------
// a3 (radial): F_i += sum_j [ sum_k (etil_i[J][k] + etil_j[I][k]) f_k'(d) ] rhat_ij   (Eq.3 with C3.6),
// per-atom virial  W_ab -= r_a f_ij,b  with f_ij = (sum_k etil_i[J][k] f_k') rhat   (Eq.4, R17).
// etil_i[J][k] = sum_n E'_in cR[I][J][n][k] is produced by the network forward kernel.
// ------------------------------------------------------------------------------------------------
template <int KT>
__global__ void __launch_bounds__(GNEP_WARPS * 32)
k_radial_force(DevSpec sp, int N, const int *__restrict__ type_s, const int *__restrict__ segR,
               const float4 *__restrict__ pairR, const float *__restrict__ etil, float4 *__restrict__ Fat,
               float *__restrict__ Wat) {
  int lane = threadIdx.x & 31;
  int a = blockIdx.x * GNEP_WARPS + (threadIdx.x >> 5);
  if (a >= N) return;
  int I = type_s[a];
  float F[3] = {0.f, 0.f, 0.f}, W[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
  const int TK = sp.T * KT;
  for (int J = 0; J < sp.T; ++J) {
    int p0 = segR[a * (sp.T + 1) + J], p1 = segR[a * (sp.T + 1) + J + 1];
    float ei[KT];
#pragma unroll
    for (int k = 0; k < KT; ++k) ei[k] = __ldg(etil + (size_t)a * TK + J * KT + k);
    for (int p = p0 + lane; p < p1; p += 32) {
      float4 r = pairR[p];
      int j = __float_as_int(r.w);
      float d = sqrtf(r.x * r.x + r.y * r.y + r.z * r.z);
      float rinv = 1.f / d;
      float f[KT], fp[KT];
      cheb_ffp<KT>(d, sp.rcRinv, f, fp);
      const float *ej = etil + (size_t)j * TK + I * KT;
      float si = 0.f, sj = 0.f;
#pragma unroll
      for (int k = 0; k < KT; ++k) { si += ei[k] * fp[k]; sj += __ldg(ej + k) * fp[k]; }
      float hx = r.x * rinv, hy = r.y * rinv, hz = r.z * rinv;
      float tot = si + sj;
      F[0] += tot * hx; F[1] += tot * hy; F[2] += tot * hz;
      float fx = si * hx, fy = si * hy, fz = si * hz;
      W[0] -= r.x * fx; W[1] -= r.y * fy; W[2] -= r.z * fz;
      W[3] -= r.x * fy; W[4] -= r.y * fz; W[5] -= r.z * fx;
    }
  }
#pragma unroll
  for (int c = 0; c < 3; ++c) F[c] = warp_sum(F[c]);
#pragma unroll
  for (int c = 0; c < 6; ++c) W[c] = warp_sum(W[c]);
  if (lane == 0) {
    Fat[a] = make_float4(F[0], F[1], F[2], 0.f);
#pragma unroll
    for (int c = 0; c < 6; ++c) Wat[(size_t)a * 6 + c] = W[c];
  }
}

// beta_nlm = sum_{nu in n} E'_nu dq_nu/dS_nlm  for one atom, into per-warp shared memory [NA][24]
__device__ __forceinline__ void make_beta(const DevSpec &sp, const float *__restrict__ Ep_a,
                                          const float *__restrict__ S_a, float *beta, int lane) {
  for (int o = lane; o < sp.NA * GNEP_NLM; o += 32) {
    int n = o / GNEP_NLM, lm = o - n * GNEP_NLM;
    int l = l_of_lm(lm);
    float be = 0.f;
    if (l <= sp.L) be = Ep_a[sp.NR + (l - 1) * sp.NA + n] * c_C2[lm] * S_a[o];
    if (sp.use4 && lm >= 3 && lm < 8) {
      float s5[5], g4[5];
#pragma unroll
      for (int m = 0; m < 5; ++m) s5[m] = S_a[n * GNEP_NLM + 3 + m];
      p4_grad(s5, g4);
      float g = lm == 3 ? g4[0] : lm == 4 ? g4[1] : lm == 5 ? g4[2] : lm == 6 ? g4[3] : g4[4];
      be += Ep_a[sp.NR + sp.L * sp.NA + n] * c_kappa4 * g;
    }
    beta[o] = be;
  }
}

// ------------------------------------------------------------------------------------------------
// a3 (angular): f_ij = sum_n sum_lm beta_nlm (g_n' B_lm rhat + g_n grad B_lm)   (C3.6 with C2.1-C2.3)
// lane = pair.  gam_lm = sum_n g_n beta_nlm, gamp_lm = sum_n g_n' beta_nlm, then one harmonic sweep.
// Writes f_ij per pair (for the reverse gather), adds own-row sums to Fat / Wat.
// ------------------------------------------------------------------------------------------------
template <int KT>
__global__ void __launch_bounds__(GNEP_WARPS * 32)
k_angular_force(DevSpec sp, int N, const int *__restrict__ type_s, const int *__restrict__ rowA,
                const float4 *__restrict__ pairA, const float *__restrict__ theta, const float *__restrict__ Ep,
                const float *__restrict__ S, float4 *__restrict__ fpair, float4 *__restrict__ Fat,
                float *__restrict__ Wat) {
  extern __shared__ __align__(16) float smem[];
  float *cs = smem;
  int ncs = (sp.T * sp.T * sp.NA * KT + 3) & ~3;
  float *beta = warp_smem(smem + ncs, sp.NA * GNEP_NLM);
  stage_coeff(cs, theta + sp.offA, sp.T * sp.T * sp.NA, sp.KA, KT);
  __syncthreads();
  int lane = threadIdx.x & 31;
  int a = blockIdx.x * GNEP_WARPS + (threadIdx.x >> 5);
  if (a >= N) return;
  int I = type_s[a];
  int r0 = rowA[a], r1 = rowA[a + 1];
  make_beta(sp, Ep + (size_t)a * sp.Ndes, S + (size_t)a * sp.NA * GNEP_NLM, beta, lane);
  __syncwarp();
  float F[3] = {0.f, 0.f, 0.f}, W[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
  for (int p = r0 + lane; p < r1; p += 32) {
    float4 r = pairA[p];
    float d = sqrtf(r.x * r.x + r.y * r.y + r.z * r.z);
    float rinv = 1.f / d;
    int J = type_s[__float_as_int(r.w)];
    float f[KT], fp[KT];
    cheb_ffp<KT>(d, sp.rcAinv, f, fp);
    const float *c = cs + (I * sp.T + J) * sp.NA * KT;
    float gam[GNEP_NLM], gamp[GNEP_NLM];
#pragma unroll
    for (int lm = 0; lm < GNEP_NLM; ++lm) { gam[lm] = 0.f; gamp[lm] = 0.f; }
    for (int n = 0; n < sp.NA; ++n) {
      float g = 0.f, gp = 0.f;
#pragma unroll
      for (int k = 0; k < KT; ++k) { float cv = c[n * KT + k]; g += cv * f[k]; gp += cv * fp[k]; }
#pragma unroll
      for (int v = 0; v < GNEP_NLM / 4; ++v) {
        float4 b4 = *(const float4 *)(beta + n * GNEP_NLM + 4 * v);
        gam[4 * v] += g * b4.x; gam[4 * v + 1] += g * b4.y; gam[4 * v + 2] += g * b4.z; gam[4 * v + 3] += g * b4.w;
        gamp[4 * v] += gp * b4.x; gamp[4 * v + 1] += gp * b4.y; gamp[4 * v + 2] += gp * b4.z; gamp[4 * v + 3] += gp * b4.w;
      }
    }
    float hx = r.x * rinv, hy = r.y * rinv, hz = r.z * rinv;
    float sB = 0.f, sl = 0.f, vx = 0.f, vy = 0.f, vz = 0.f;
    blm_unit(hx, hy, hz, [&](int lm, int l, float b, float gx, float gy, float gz) {
      sB += gamp[lm] * b;
      sl += (float)l * gam[lm] * b;
      vx += gam[lm] * gx; vy += gam[lm] * gy; vz += gam[lm] * gz;
    });
    float fx = hx * sB + rinv * (vx - hx * sl);
    float fy = hy * sB + rinv * (vy - hy * sl);
    float fz = hz * sB + rinv * (vz - hz * sl);
    fpair[p] = make_float4(fx, fy, fz, 0.f);
    F[0] += fx; F[1] += fy; F[2] += fz;
    W[0] -= r.x * fx; W[1] -= r.y * fy; W[2] -= r.z * fz;
    W[3] -= r.x * fy; W[4] -= r.y * fz; W[5] -= r.z * fx;
  }
#pragma unroll
  for (int c = 0; c < 3; ++c) F[c] = warp_sum(F[c]);
#pragma unroll
  for (int c = 0; c < 6; ++c) W[c] = warp_sum(W[c]);
  if (lane == 0) {
    float4 o = Fat[a];
    Fat[a] = make_float4(o.x + F[0], o.y + F[1], o.z + F[2], 0.f);
#pragma unroll
    for (int c = 0; c < 6; ++c) Wat[(size_t)a * 6 + c] += W[c];
  }
}

// F_i -= sum_{p in row i} f_{rev(p)}   (the -dE_j/dr_ji half of Eq.3 for the angular part; no atomics)
__global__ void __launch_bounds__(GNEP_WARPS * 32)
k_force_gather(int N, const int *__restrict__ rowA, const int *__restrict__ revA,
               const float4 *__restrict__ fpair, float4 *__restrict__ Fat) {
  int lane = threadIdx.x & 31;
  int a = blockIdx.x * GNEP_WARPS + (threadIdx.x >> 5);
  if (a >= N) return;
  float x = 0.f, y = 0.f, z = 0.f;
  for (int p = rowA[a] + lane; p < rowA[a + 1]; p += 32) {
    float4 f = fpair[revA[p]];
    x += f.x; y += f.y; z += f.z;
  }
  x = warp_sum(x); y = warp_sum(y); z = warp_sum(z);
  if (lane == 0) { float4 o = Fat[a]; Fat[a] = make_float4(o.x - x, o.y - y, o.z - z, 0.f); }
}

// pair adjoint a_ij = dL/df_ij = sf (u_i - u_j) - sv omega_s . r_ij   (DESIGN.md section 3 step 2)
struct AdjCtx { float ux, uy, uz, o0, o1, o2, o3, o4, o5, sf; };
__device__ __forceinline__ AdjCtx make_adj(const float4 *__restrict__ u, const float *__restrict__ omega,
                                           const float *__restrict__ scales, int a, int s) {
  AdjCtx c;
  float4 ui = u[a];
  float sv = scales[2];
  c.sf = scales[1];
  c.ux = ui.x; c.uy = ui.y; c.uz = ui.z;
  c.o0 = sv * omega[s * 6 + 0]; c.o1 = sv * omega[s * 6 + 1]; c.o2 = sv * omega[s * 6 + 2];
  c.o3 = sv * omega[s * 6 + 3]; c.o4 = sv * omega[s * 6 + 4]; c.o5 = sv * omega[s * 6 + 5];
  return c;
}
__device__ __forceinline__ void pair_adjoint(const AdjCtx &c, const float4 &uj, const float4 &r, float &ax,
                                             float &ay, float &az) {
  ax = c.sf * (c.ux - uj.x) - (c.o0 * r.x + c.o5 * r.z);
  ay = c.sf * (c.uy - uj.y) - (c.o1 * r.y + c.o3 * r.x);
  az = c.sf * (c.uz - uj.z) - (c.o2 * r.z + c.o4 * r.y);
}

// ------------------------------------------------------------------------------------------------
// a5 (radial): M2[a][J][k] = sum_j f_k'(d_ij) (a_ij . rhat_ij) ;  D_n = sum_{J,k} cR[I][J][n][k] M2[J][k]
// ------------------------------------------------------------------------------------------------
template <int KT>
__global__ void __launch_bounds__(GNEP_WARPS * 32)
k_radial_adj(DevSpec sp, int N, const int *__restrict__ type_s, const int *__restrict__ struct_s,
             const int *__restrict__ segR, const float4 *__restrict__ pairR, const float *__restrict__ theta,
             const float4 *__restrict__ u, const float *__restrict__ omega, const float *__restrict__ scales,
             float *__restrict__ D, float *__restrict__ M2) {
  extern __shared__ __align__(16) float smem[];
  float *cs = smem;
  int ncs = sp.T * sp.T * sp.NR * KT;
  float *wbuf = warp_smem(smem + ncs, KT * 33 + KT);
  float *mrow = wbuf + KT * 33;
  stage_coeff(cs, theta, sp.T * sp.T * sp.NR, sp.KR, KT);
  __syncthreads();
  int lane = threadIdx.x & 31;
  int a = blockIdx.x * GNEP_WARPS + (threadIdx.x >> 5);
  if (a >= N) return;
  int I = type_s[a];
  AdjCtx ac = make_adj(u, omega, scales, a, struct_s[a]);
  float Dn = 0.f;
  for (int J = 0; J < sp.T; ++J) {
    int p0 = segR[a * (sp.T + 1) + J], p1 = segR[a * (sp.T + 1) + J + 1];
    float acc[KT];
#pragma unroll
    for (int k = 0; k < KT; ++k) acc[k] = 0.f;
    for (int p = p0 + lane; p < p1; p += 32) {
      float4 r = pairR[p];
      float4 uj = u[__float_as_int(r.w)];
      float d = sqrtf(r.x * r.x + r.y * r.y + r.z * r.z);
      float rinv = 1.f / d;
      float ax, ay, az;
      pair_adjoint(ac, uj, r, ax, ay, az);
      float ar = (ax * r.x + ay * r.y + az * r.z) * rinv;
      float f[KT], fp[KT];
      cheb_ffp<KT>(d, sp.rcRinv, f, fp);
#pragma unroll
      for (int k = 0; k < KT; ++k) acc[k] += fp[k] * ar;
    }
    float s = warp_transpose_reduce<KT>(acc, wbuf, lane);
    if (lane < KT) { M2[(size_t)a * sp.T * KT + J * KT + lane] = s; mrow[lane] = s; }
    __syncwarp();
    if (lane < sp.NR) {
      const float *c = cs + ((I * sp.T + J) * sp.NR + lane) * KT;
#pragma unroll
      for (int k = 0; k < KT; ++k) Dn += c[k] * mrow[k];
    }
    __syncwarp();
  }
  if (lane < sp.NR) D[(size_t)a * sp.Ndes + lane] = Dn;
}

// ------------------------------------------------------------------------------------------------
// a5 (angular): T_nlm = sum_j [ g_n' B_lm (a.rhat) + g_n (grad B_lm . a) ]  (second-order factors of
// C3.9-C3.16 after contraction with the residuals), then D_(n,l) = sum_m 2 C_lm S_nlm T_nlm and the 4-body D.
// ------------------------------------------------------------------------------------------------
template <int KT>
__global__ void __launch_bounds__(GNEP_WARPS * 32)
k_angular_adj(DevSpec sp, int N, const int *__restrict__ type_s, const int *__restrict__ struct_s,
              const int *__restrict__ rowA, const float4 *__restrict__ pairA, const float *__restrict__ theta,
              const float4 *__restrict__ u, const float *__restrict__ omega, const float *__restrict__ scales,
              const float *__restrict__ S, float *__restrict__ Tn, float *__restrict__ D) {
  extern __shared__ __align__(16) float smem[];
  float *cs = smem;
  int ncs = (sp.T * sp.T * sp.NA * KT + 3) & ~3;
  int per_warp = (2 * sp.NA + 2 * GNEP_NLM) * 32 + 2 * sp.NA * GNEP_NLM;
  float *sg1 = warp_smem(smem + ncs, per_warp);     // [NA][32]  g_n' (a.rhat)
  float *sg2 = sg1 + sp.NA * 32;                    // [NA][32]  g_n
  float *sX = sg2 + sp.NA * 32;                     // [24][32]  B_lm
  float *sY = sX + GNEP_NLM * 32;                   // [24][32]  grad B_lm . a
  float *sS = sY + GNEP_NLM * 32;                   // [NA][24]
  float *sT = sS + sp.NA * GNEP_NLM;                // [NA][24]
  stage_coeff(cs, theta + sp.offA, sp.T * sp.T * sp.NA, sp.KA, KT);
  __syncthreads();
  int lane = threadIdx.x & 31;
  int a = blockIdx.x * GNEP_WARPS + (threadIdx.x >> 5);
  if (a >= N) return;
  int I = type_s[a];
  int r0 = rowA[a], r1 = rowA[a + 1];
  AdjCtx ac = make_adj(u, omega, scales, a, struct_s[a]);
  const bool act = lane < 30;
  const int n1 = lane / 3, grp = lane - 3 * n1, n2 = n1 + 10;
  const bool on1 = act && n1 < sp.NA, on2 = act && n2 < sp.NA;
  float acc1[8], acc2[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) { acc1[i] = 0.f; acc2[i] = 0.f; }
  for (int c0 = r0; c0 < r1; c0 += 32) {
    int p = c0 + lane;
    if (p < r1) {
      float4 r = pairA[p];
      int j = __float_as_int(r.w);
      float4 uj = u[j];
      float d = sqrtf(r.x * r.x + r.y * r.y + r.z * r.z);
      float rinv = 1.f / d;
      int J = type_s[j];
      float ax, ay, az;
      pair_adjoint(ac, uj, r, ax, ay, az);
      float hx = r.x * rinv, hy = r.y * rinv, hz = r.z * rinv;
      float ar = ax * hx + ay * hy + az * hz;
      float f[KT], fp[KT];
      cheb_ffp<KT>(d, sp.rcAinv, f, fp);
      const float *c = cs + (I * sp.T + J) * sp.NA * KT;
      for (int n = 0; n < sp.NA; ++n) {
        float g = 0.f, gp = 0.f;
#pragma unroll
        for (int k = 0; k < KT; ++k) { float cv = c[n * KT + k]; g += cv * f[k]; gp += cv * fp[k]; }
        sg1[n * 32 + lane] = gp * ar;
        sg2[n * 32 + lane] = g;
      }
      blm_unit(hx, hy, hz, [&](int lm, int l, float b, float gx, float gy, float gz) {
        sX[lm * 32 + lane] = b;
        sY[lm * 32 + lane] = rinv * ((gx * ax + gy * ay + gz * az) - (float)l * b * ar);
      });
    } else {
      for (int n = 0; n < sp.NA; ++n) { sg1[n * 32 + lane] = 0.f; sg2[n * 32 + lane] = 0.f; }
#pragma unroll
      for (int lm = 0; lm < GNEP_NLM; ++lm) { sX[lm * 32 + lane] = 0.f; sY[lm * 32 + lane] = 0.f; }
    }
    __syncwarp();
    int ng4 = (min(32, r1 - c0) + 3) >> 2;
    for (int g4 = 0; g4 < ng4; ++g4) {
      const float4 z4 = make_float4(0, 0, 0, 0);
      float4 ga1 = on1 ? *(const float4 *)(sg1 + n1 * 32 + 4 * g4) : z4;
      float4 ga2 = on1 ? *(const float4 *)(sg2 + n1 * 32 + 4 * g4) : z4;
      float4 gb1 = on2 ? *(const float4 *)(sg1 + n2 * 32 + 4 * g4) : z4;
      float4 gb2 = on2 ? *(const float4 *)(sg2 + n2 * 32 + 4 * g4) : z4;
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        float4 X = *(const float4 *)(sX + (grp * 8 + i) * 32 + 4 * g4);
        float4 Y = *(const float4 *)(sY + (grp * 8 + i) * 32 + 4 * g4);
        acc1[i] += ga1.x * X.x + ga1.y * X.y + ga1.z * X.z + ga1.w * X.w + ga2.x * Y.x + ga2.y * Y.y + ga2.z * Y.z + ga2.w * Y.w;
        acc2[i] += gb1.x * X.x + gb1.y * X.y + gb1.z * X.z + gb1.w * X.w + gb2.x * Y.x + gb2.y * Y.y + gb2.z * Y.z + gb2.w * Y.w;
      }
    }
    __syncwarp();
  }
  float *Ta = Tn + (size_t)a * sp.NA * GNEP_NLM;
  const float *Sa = S + (size_t)a * sp.NA * GNEP_NLM;
  if (on1) {
#pragma unroll
    for (int i = 0; i < 8; ++i) { sT[n1 * GNEP_NLM + grp * 8 + i] = acc1[i]; Ta[n1 * GNEP_NLM + grp * 8 + i] = acc1[i]; }
  }
  if (on2) {
#pragma unroll
    for (int i = 0; i < 8; ++i) { sT[n2 * GNEP_NLM + grp * 8 + i] = acc2[i]; Ta[n2 * GNEP_NLM + grp * 8 + i] = acc2[i]; }
  }
  for (int o = lane; o < sp.NA * GNEP_NLM; o += 32) sS[o] = Sa[o];
  __syncwarp();
  float *Da = D + (size_t)a * sp.Ndes + sp.NR;
  for (int o = lane; o < sp.NA * sp.L; o += 32) {
    int l = o / sp.NA + 1, n = o - (l - 1) * sp.NA;
    int lm0 = l * l - 1;
    float v = 0.f;
    for (int m = 0; m <= 2 * l; ++m) v += c_C2[lm0 + m] * sS[n * GNEP_NLM + lm0 + m] * sT[n * GNEP_NLM + lm0 + m];
    Da[o] = v;
  }
  if (sp.use4 && lane < sp.NA) {
    float g4[5];
    p4_grad(sS + lane * GNEP_NLM + 3, g4);
    float v = 0.f;
#pragma unroll
    for (int m = 0; m < 5; ++m) v += g4[m] * sT[lane * GNEP_NLM + 3 + m];
    Da[sp.NA * sp.L + lane] = c_kappa4 * v;
  }
}

// ------------------------------------------------------------------------------------------------
// a7 (angular): dL/dcA[I][J][n][k] += U_n f_k(d) + V_n f_k'(d),
//   U_n = sum_lm [alpha_nlm B_lm + beta_nlm (grad B_lm . a)],  V_n = (a.rhat) sum_lm beta_nlm B_lm
// (C2.5-C2.10 with Alg.1's inner loop collapsed into T_nlm; C3.12-C3.20).  Each warp keeps a full
// [T][T][NA][KT] accumulator in shared memory over the atoms it visits and writes one partial at the end.
// ------------------------------------------------------------------------------------------------
template <int KT>
__global__ void __launch_bounds__(GNEP_WARPS * 32)
k_cgrad_angular(DevSpec sp, int N, const int *__restrict__ type_s, const int *__restrict__ struct_s,
                const int *__restrict__ rowA, const float4 *__restrict__ pairA, const float4 *__restrict__ u,
                const float *__restrict__ omega, const float *__restrict__ scales, const float *__restrict__ Ep,
                const float *__restrict__ gbar, const float *__restrict__ S, const float *__restrict__ Tn,
                float *__restrict__ partial) {
  extern __shared__ __align__(16) float smem[];
  const int NAp = sp.NA | 1, KTp = KT + 1;
  const int nacc = sp.T * sp.T * sp.NA * KT;
  int per_warp = ((nacc + 3) & ~3) + 4 * sp.NA * GNEP_NLM + 32 * (2 * NAp + 2 * KTp);
  float *accS = warp_smem(smem, per_warp);
  float *sS = accS + ((nacc + 3) & ~3);             // [NA][24]
  float *sT = sS + sp.NA * GNEP_NLM;
  float *sAl = sT + sp.NA * GNEP_NLM;               // alpha [NA][24]
  float *sBe = sAl + sp.NA * GNEP_NLM;              // beta  [NA][24]
  float *sU = sBe + sp.NA * GNEP_NLM;               // [32][NAp]
  float *sV = sU + 32 * NAp;
  float *sf = sV + 32 * NAp;                        // [32][KTp]
  float *sfp = sf + 32 * KTp;
  int lane = threadIdx.x & 31;
  int gw = blockIdx.x * GNEP_WARPS + (threadIdx.x >> 5);
  int nw = gridDim.x * GNEP_WARPS;
  for (int o = lane; o < nacc; o += 32) accS[o] = 0.f;
  __syncwarp();
  for (int a = gw; a < N; a += nw) {
    int I = type_s[a];
    int r0 = rowA[a], r1 = rowA[a + 1];
    const float *Sa = S + (size_t)a * sp.NA * GNEP_NLM, *Ta = Tn + (size_t)a * sp.NA * GNEP_NLM;
    const float *Epa = Ep + (size_t)a * sp.Ndes, *gba = gbar + (size_t)a * sp.Ndes;
    for (int o = lane; o < sp.NA * GNEP_NLM; o += 32) { sS[o] = Sa[o]; sT[o] = Ta[o]; }
    __syncwarp();
    for (int o = lane; o < sp.NA * GNEP_NLM; o += 32) {
      int n = o / GNEP_NLM, lm = o - n * GNEP_NLM;
      int l = l_of_lm(lm);
      float al = 0.f, be = 0.f;
      if (l <= sp.L) {
        int v = sp.NR + (l - 1) * sp.NA + n;
        float e1 = Epa[v];
        al = c_C2[lm] * (gba[v] * sS[o] + e1 * sT[o]);
        be = c_C2[lm] * e1 * sS[o];
      }
      if (sp.use4 && lm >= 3 && lm < 8) {
        int v4 = sp.NR + sp.L * sp.NA + n;
        float g4[5], hv[5];
        p4_grad(sS + n * GNEP_NLM + 3, g4);
        p4_hess_vec(sS + n * GNEP_NLM + 3, sT + n * GNEP_NLM + 3, hv);
        int m = lm - 3;
        float g = m == 0 ? g4[0] : m == 1 ? g4[1] : m == 2 ? g4[2] : m == 3 ? g4[3] : g4[4];
        float h = m == 0 ? hv[0] : m == 1 ? hv[1] : m == 2 ? hv[2] : m == 3 ? hv[3] : hv[4];
        float e4 = Epa[v4];
        al += c_kappa4 * (gba[v4] * g + e4 * h);
        be += c_kappa4 * e4 * g;
      }
      sAl[o] = al; sBe[o] = be;
    }
    __syncwarp();
    AdjCtx ac = make_adj(u, omega, scales, a, struct_s[a]);
    for (int c0 = r0; c0 < r1; c0 += 32) {
      int p = c0 + lane;
      int J = -1;
      if (p < r1) {
        float4 r = pairA[p];
        int j = __float_as_int(r.w);
        float4 uj = u[j];
        J = type_s[j];
        float d = sqrtf(r.x * r.x + r.y * r.y + r.z * r.z);
        float rinv = 1.f / d;
        float ax, ay, az;
        pair_adjoint(ac, uj, r, ax, ay, az);
        float hx = r.x * rinv, hy = r.y * rinv, hz = r.z * rinv;
        float ar = ax * hx + ay * hy + az * hz;
        float f[KT], fp[KT];
        cheb_ffp<KT>(d, sp.rcAinv, f, fp);
#pragma unroll
        for (int k = 0; k < KT; ++k) { sf[lane * KTp + k] = f[k]; sfp[lane * KTp + k] = fp[k]; }
        float B[GNEP_NLM], Y[GNEP_NLM];
        blm_unit(hx, hy, hz, [&](int lm, int l, float b, float gx, float gy, float gz) {
          B[lm] = b;
          Y[lm] = rinv * ((gx * ax + gy * ay + gz * az) - (float)l * b * ar);
        });
        for (int n = 0; n < sp.NA; ++n) {
          float U = 0.f, V = 0.f;
#pragma unroll
          for (int v = 0; v < GNEP_NLM / 4; ++v) {
            float4 al4 = *(const float4 *)(sAl + n * GNEP_NLM + 4 * v);
            float4 be4 = *(const float4 *)(sBe + n * GNEP_NLM + 4 * v);
            U += al4.x * B[4 * v] + al4.y * B[4 * v + 1] + al4.z * B[4 * v + 2] + al4.w * B[4 * v + 3];
            U += be4.x * Y[4 * v] + be4.y * Y[4 * v + 1] + be4.z * Y[4 * v + 2] + be4.w * Y[4 * v + 3];
            V += be4.x * B[4 * v] + be4.y * B[4 * v + 1] + be4.z * B[4 * v + 2] + be4.w * B[4 * v + 3];
          }
          sU[lane * NAp + n] = U;
          sV[lane * NAp + n] = V * ar;
        }
      }
      unsigned mJ[GNEP_MAX_SPECIES_C];
#pragma unroll
      for (int t = 0; t < GNEP_MAX_SPECIES_C; ++t) mJ[t] = __ballot_sync(0xffffffffu, J == t);
      __syncwarp();
      const int nJ = sp.NA * KT;
      for (int o = lane; o < sp.T * nJ; o += 32) {
        int Jo = o / nJ, rem = o - Jo * nJ;
        int n = rem / KT, k = rem - n * KT;
        unsigned m = Jo == 0 ? mJ[0] : Jo == 1 ? mJ[1] : Jo == 2 ? mJ[2] : mJ[3];
        float s = 0.f;
        while (m) {
          int pl = __ffs(m) - 1;
          m &= m - 1;
          s += sU[pl * NAp + n] * sf[pl * KTp + k] + sV[pl * NAp + n] * sfp[pl * KTp + k];
        }
        accS[I * sp.T * nJ + o] += s;
      }
      __syncwarp();
    }
  }
  __syncwarp();
  for (int o = lane; o < nacc; o += 32) partial[(size_t)gw * nacc + o] = accS[o];
}
