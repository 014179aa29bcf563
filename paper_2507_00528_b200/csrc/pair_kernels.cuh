// pair_kernels.cuh -- radial sweeps over the neighbour list (rows a1, a3, a5) and helpers shared with angular_kernels.cuh.
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
  extern __shared__ __align__(128) float smem[];
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
      float ejv[KT];
      if (KT % 4 == 0) {
#pragma unroll
        for (int k = 0; k < KT / 4; ++k) {
          float4 v = __ldg((const float4 *)ej + k);
          ejv[4 * k] = v.x; ejv[4 * k + 1] = v.y; ejv[4 * k + 2] = v.z; ejv[4 * k + 3] = v.w;
        }
      } else {
#pragma unroll
        for (int k = 0; k < KT / 2; ++k) { float2 v = __ldg((const float2 *)ej + k); ejv[2 * k] = v.x; ejv[2 * k + 1] = v.y; }
      }
      float si = 0.f, sj = 0.f;
#pragma unroll
      for (int k = 0; k < KT; ++k) { si += ei[k] * fp[k]; sj += ejv[k] * fp[k]; }
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
  extern __shared__ __align__(128) float smem[];
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
