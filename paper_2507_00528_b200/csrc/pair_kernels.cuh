// pair_kernels.cuh -- radial sweeps over the neighbour list (rows a1, a3, a5) and helpers shared with angular_kernels.cuh.
// Atoms are sorted by species (index "a"); pair records are float4(r_ij.x, r_ij.y, r_ij.z, bits(a_j)); a radial row is
// ordered by neighbour species, segR[a][J..J+1] bounding the species segments.
// Mapping: ONE THREAD PER ATOM.  Everything a radial sweep produces is a per-atom sum over the row (moments M1/M2, F_i,
// W_i), so a thread that walks its own row needs no cross-lane reduction at all, every lane is busy (rows of
// neighbouring atoms have nearly equal lengths) and the per-pair work is the ~70-110 instructions of the basis
// functions.  The 16-byte pair loads of a warp touch 32 different rows: each 32-byte sector is fetched once and its
// second half is an L1 hit in the next iteration.  (Handing the atoms to the threads sorted by row length, so that the
// rows of a warp end together, was measured and dropped: a global sort loses the locality of the gathers, +60 % on the
// force sweep, and a sort inside each 128-atom window still costs 2-10 %: the lanes' rows are no longer adjacent.)
#pragma once
#include "common.cuh"

#define RAD_THREADS 128
#define RAD_PF 4        // pairs per prefetch group: the loads of a group are issued one whole group ahead

// Walk the row [p, pend) of one atom RAD_PF pairs at a time, the next group's records (64 contiguous bytes per lane)
// already in flight; g = gather(r), the per-pair gather of neighbour data (e.g. u_j), is issued one pair ahead of its
// use.  next_seg(J) is called whenever the walk leaves species segment J, body(r, g) for every pair.
template <class Seg, class Gather, class Body>
__device__ __forceinline__ void walk_row(const float4 *__restrict__ pairR, const int *__restrict__ sg, int T, Seg next_seg,
                                         Gather gather, Body body) {
  int p = sg[0], J = 0, jend = sg[1];
  const int pend = sg[T];
  const float4 dum = make_float4(1.f, 0.f, 0.f, 0.f);      // w = bits(0): a valid atom index for the gather
  float4 nb[RAD_PF];
  // rows start at even record indices and p advances by RAD_PF: two records per 256-bit load.  The second may lie past
  // the row's end -- in the row's pad slot (zeroed at load: w = bits(0), a valid index) or in the next row -- its body
  // is skipped, but gather() still runs on it one pair ahead, so its w must always be a valid atom index
  auto load2 = [&](int q, float4 &r0, float4 &r1) {
    if (q < pend) { const float8 v = ldg256_stream((const float *)(pairR + q)); r0 = v.lo; r1 = v.hi; }
    else { r0 = dum; r1 = dum; }
  };
#pragma unroll
  for (int i = 0; i < RAD_PF; i += 2) load2(p + i, nb[i], nb[i + 1]);
  auto gn = gather(nb[0]);
  while (p < pend) {
    float4 cb[RAD_PF];
#pragma unroll
    for (int i = 0; i < RAD_PF; ++i) cb[i] = nb[i];
#pragma unroll
    for (int i = 0; i < RAD_PF; i += 2) load2(p + RAD_PF + i, nb[i], nb[i + 1]);
#pragma unroll
    for (int i = 0; i < RAD_PF; ++i) {
      const auto gc = gn;
      gn = gather(i + 1 < RAD_PF ? cb[i + 1 < RAD_PF ? i + 1 : 0] : nb[0]);
      if (p + i < pend) {
        while (p + i >= jend) { next_seg(J); ++J; jend = sg[J + 1]; }
        body(cb[i], gc);
      }
    }
    p += RAD_PF;
  }
  for (; J < T; ++J) next_seg(J);
}

template <int KT>
struct RowRegs { float v[KT]; };

template <int KT>
__device__ __forceinline__ void store_row(float *__restrict__ dst, const float (&v)[KT]) {
  if (KT % 4 == 0) {
#pragma unroll
    for (int k = 0; k < KT; k += 4) *(float4 *)(dst + k) = make_float4(v[k], v[k + 1], v[k + 2], v[k + 3]);
  } else {
#pragma unroll
    for (int k = 0; k < KT; k += 2) *(float2 *)(dst + k) = make_float2(v[k], v[k + 1]);
  }
}
template <int KT>
__device__ __forceinline__ void load_row(const float *__restrict__ src, float (&v)[KT]) {
  if (KT % 4 == 0) {
#pragma unroll
    for (int k = 0; k < KT; k += 4) { float4 t = *(const float4 *)(src + k); v[k] = t.x; v[k + 1] = t.y; v[k + 2] = t.z; v[k + 3] = t.w; }
  } else {
#pragma unroll
    for (int k = 0; k < KT; k += 2) { float2 t = *(const float2 *)(src + k); v[k] = t.x; v[k + 1] = t.y; }
  }
}
// out_n = sum_{J,k} cs[I][J][n][k] M[J][k] for n < NR, written to out[n] (row of q or D); M is the atom's moment row
template <int KT>
__device__ __forceinline__ void radial_contract(const DevSpec &sp, const float *cs, int I, const float *__restrict__ Mrow,
                                                float *__restrict__ out) {
  float o[16];
#pragma unroll
  for (int n = 0; n < 16; ++n) o[n] = 0.f;
  for (int J = 0; J < sp.T; ++J) {
    float m[KT];
    load_row<KT>(Mrow + J * KT, m);
    const float *c = cs + (size_t)(I * sp.T + J) * sp.NR * KT;
#pragma unroll
    for (int n = 0; n < 16; ++n)
      if (n < sp.NR) {
        float cv[KT];
        load_row<KT>(c + n * KT, cv);
#pragma unroll
        for (int k = 0; k < KT; ++k) o[n] += cv[k] * m[k];
      }
  }
#pragma unroll
  for (int n = 0; n < 16; ++n)
    if (n < sp.NR) out[n] = o[n];
}

// ------------------------------------------------------------------------------------------------
// a1 (radial):  M1[a][J][k] = sum_{j in seg J} f_k(d_ij)  ;  q_n = sum_{J,k} cR[I][J][n][k] M1[J][k]
// (paper Eq.5-6, in moment-factored form: g_n is linear in f_k)
// ------------------------------------------------------------------------------------------------
template <int KT>
__global__ void __launch_bounds__(RAD_THREADS)
k_radial_fwd(DevSpec sp, int N, const int *__restrict__ type_s, const int *__restrict__ segR,
             const float4 *__restrict__ pairR, const float *__restrict__ theta, float *__restrict__ q,
             float *__restrict__ M1) {
  extern __shared__ __align__(128) float smem[];
  float *cs = smem;                                          // [T*T*NR][KT]
  stage_coeff(cs, theta, sp.T * sp.T * sp.NR, sp.KR, KT);
  __syncthreads();
  const int a = blockIdx.x * RAD_THREADS + threadIdx.x;
  if (a >= N) return;
  const int *sg = segR + (size_t)a * (sp.T + 1);
  float *Mrow = M1 + (size_t)a * sp.T * KT;
  // accumulated per Chebyshev term: acc[k] = sum hfc T_k (k >= 1), acc[0] = sum hfc;  f_0 = 2 hfc, f_k = hfc T_k + hfc
  float acc[KT];
#pragma unroll
  for (int k = 0; k < KT; ++k) acc[k] = 0.f;
  walk_row(pairR, sg, sp.T,
           [&](int J) {                                     // species segment J complete
             float m[KT];
             m[0] = 2.f * acc[0];
#pragma unroll
             for (int k = 1; k < KT; ++k) m[k] = acc[k] + acc[0];
             store_row<KT>(Mrow + J * KT, m);
#pragma unroll
             for (int k = 0; k < KT; ++k) acc[k] = 0.f;
           },
           [](const float4 &) { return 0; },
           [&](const float4 &r, int) {
             float d, rinv, Tk[KT], hfc;
             pair_len(r.x * r.x + r.y * r.y + r.z * r.z, d, rinv);
             cheb_T<KT>(d, sp.rcRinv, Tk, hfc);
             acc[0] += hfc;
#pragma unroll
             for (int k = 1; k < KT; ++k) acc[k] = fmaf(hfc, Tk[k], acc[k]);
           });
  radial_contract<KT>(sp, cs, type_s[a], Mrow, q + (size_t)a * sp.Ndes);
}

// a1 (radial), per epoch: q_n = sum_{J,k} cR[I][J][n][k] M1[J][k] from the resident moments.  M1 depends on the geometry
// only (positions are fixed during training), so the pair sweep above runs once per loaded batch.
template <int KT>
__global__ void __launch_bounds__(RAD_THREADS)
k_radial_q(DevSpec sp, int N, const int *__restrict__ type_s, const float *__restrict__ theta, const float *__restrict__ M1,
           float *__restrict__ q) {
  extern __shared__ __align__(128) float smem[];
  float *cs = smem;                                          // [T*T*NR][KT]
  stage_coeff(cs, theta, sp.T * sp.T * sp.NR, sp.KR, KT);
  __syncthreads();
  const int a = blockIdx.x * RAD_THREADS + threadIdx.x;
  if (a >= N) return;
  radial_contract<KT>(sp, cs, type_s[a], M1 + (size_t)a * sp.T * KT, q + (size_t)a * sp.Ndes);
}

// ------------------------------------------------------------------------------------------------
// a3 (radial): F_i += sum_j [ sum_k (etil_i[J][k] + etil_j[I][k]) f_k'(d) ] rhat_ij   (Eq.3 with C3.6),
// virial W_ab -= r_a f_ij,b with f_ij = (sum_k etil_i[J][k] f_k') rhat (Eq.4, R17), booked per atom as half of the pair's
// symmetric total (only the per-structure sum of W_i is ever used; see the kernel body).
// etil_i[J][k] = sum_n E'_in cR[I][J][n][k] is produced by the network forward kernel.
// ------------------------------------------------------------------------------------------------
template <int KT>
__global__ void __launch_bounds__(RAD_THREADS)
k_radial_force(DevSpec sp, int N, const int *__restrict__ type_s, const int *__restrict__ segR,
               const float4 *__restrict__ pairR, const float *__restrict__ etil, const int *__restrict__ segA,
               const int *__restrict__ revA, const float4 *__restrict__ pairA, const float4 *__restrict__ fpair,
               float4 *__restrict__ Fat, float *__restrict__ Wat) {
  const int a = blockIdx.x * RAD_THREADS + threadIdx.x;
  if (a >= N) return;
  const int I = type_s[a];
  const int TK = sp.T * KT;
  const int *sg = segR + (size_t)a * (sp.T + 1);
  float F[3] = {0.f, 0.f, 0.f}, W[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
  float ei[KT];
  load_row<KT>(etil + (size_t)a * TK, ei);
  walk_row(pairR, sg, sp.T,
           [&](int J) { if (J + 1 < sp.T) load_row<KT>(etil + (size_t)a * TK + (J + 1) * KT, ei); },
           [](const float4 &) { return 0; },
           [&](const float4 &r, int) {
             RowRegs<KT> ej;                              // requested first, used after the basis functions
             load_row<KT>(etil + (size_t)__float_as_int(r.w) * TK + I * KT, ej.v);
             float d, rinv, Tk[KT], Dk[KT], hfc, hfcp, hdf;
             pair_len(r.x * r.x + r.y * r.y + r.z * r.z, d, rinv);
             cheb_TD<KT>(d, sp.rcRinv, Tk, Dk, hfc, hfcp, hdf);
             // tot = sum_k (etil_i[J][k] + etil_j[I][k]) f_k',  f_0' = 2 hfcp, f_k' = D_k hdf + (T_k + 1) hfcp
             float sD = 0.f, sT = 2.f * (ei[0] + ej.v[0]);
#pragma unroll
             for (int k = 1; k < KT; ++k) {
               const float es = ei[k] + ej.v[k];
               sD = fmaf(es, Dk[k], sD);
               sT = fmaf(es, Tk[k] + 1.f, sT);
             }
             const float tot = sD * hdf + sT * hfcp;
             const float hx = r.x * rinv, hy = r.y * rinv, hz = r.z * rinv;
             F[0] += tot * hx; F[1] += tot * hy; F[2] += tot * hz;
             // virial: sum_i W_i only enters per structure, and there sum_(i,j) r (x) rhat s_ij = 1/2 sum_(i,j) r (x) rhat
             // (s_ij + s_ji) because (j,i) carries the same dyad -- so the atom books half of the pair's total
             const float hf = 0.5f * tot;
             const float fx = hf * hx, fy = hf * hy, fz = hf * hz;
             W[0] -= r.x * fx; W[1] -= r.y * fy; W[2] -= r.z * fz;
             W[3] -= r.x * fy; W[4] -= r.y * fz; W[5] -= r.z * fx;
           });
  // angular part (Eq.3, Eq.4): F_i += sum_{p in row i} (f_p - f_rev(p)),  W_i -= sum_p r_p (x) f_p with the pair forces
  // f_p written by k_angular_force; the reverse forces are a dependent gather, so four pairs go through the two load
  // levels together
  if (fpair) {
    const int q0 = segA[(size_t)a * (sp.T + 1)], q1 = segA[(size_t)a * (sp.T + 1) + sp.T];
    for (int pb = q0; pb < q1; pb += 4) {
      int rv[4];
      float4 f[4], x[4], g[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        const bool ok = pb + i < q1;
        rv[i] = ok ? revA[pb + i] : q0;
        f[i] = ok ? fpair[pb + i] : make_float4(0.f, 0.f, 0.f, 0.f);
        x[i] = ok ? pairA[pb + i] : make_float4(0.f, 0.f, 0.f, 0.f);
      }
#pragma unroll
      for (int i = 0; i < 4; ++i) g[i] = pb + i < q1 ? fpair[rv[i]] : make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        F[0] += f[i].x - g[i].x; F[1] += f[i].y - g[i].y; F[2] += f[i].z - g[i].z;
        W[0] -= x[i].x * f[i].x; W[1] -= x[i].y * f[i].y; W[2] -= x[i].z * f[i].z;
        W[3] -= x[i].x * f[i].y; W[4] -= x[i].y * f[i].z; W[5] -= x[i].z * f[i].x;
      }
    }
  }
  Fat[a] = make_float4(F[0], F[1], F[2], 0.f);
#pragma unroll
  for (int c = 0; c < 6; c += 2) *(float2 *)(Wat + (size_t)a * 6 + c) = make_float2(W[c], W[c + 1]);
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
__global__ void __launch_bounds__(RAD_THREADS, KT <= 12 ? 6 : 4)
k_radial_adj(DevSpec sp, int N, const int *__restrict__ type_s, const int *__restrict__ struct_s,
             const int *__restrict__ segR, const float4 *__restrict__ pairR, const float *__restrict__ theta,
             const float4 *__restrict__ u, const float *__restrict__ omega, const float *__restrict__ scales,
             float *__restrict__ D, float *__restrict__ M2) {
  extern __shared__ __align__(128) float smem[];
  float *cs = smem;
  stage_coeff(cs, theta, sp.T * sp.T * sp.NR, sp.KR, KT);
  __syncthreads();
  const int a = blockIdx.x * RAD_THREADS + threadIdx.x;
  if (a >= N) return;
  const AdjCtx ac = make_adj(u, omega, scales, a, struct_s[a]);
  const int *sg = segR + (size_t)a * (sp.T + 1);
  float *Mrow = M2 + (size_t)a * sp.T * KT;
  // M2[k] = sum (a.rhat) f_k'(d),  f_k' = D_k hdf + (T_k + 1) hfcp for every k (T_0 = 1, D_0 = 0); accumulated per
  // Chebyshev term as in k_radial_fwd: acc[k] = sum w1 D_k + w2 T_k, acc[0] = sum w2, M2[k] = acc[k] + acc[0] when the
  // segment ends (one accumulator per k keeps the kernel at 6 resident CTAs per SM; the walk lives on occupancy)
  float acc[KT];
#pragma unroll
  for (int k = 0; k < KT; ++k) acc[k] = 0.f;
  walk_row(pairR, sg, sp.T,
           [&](int J) {                                     // M2[k] = acc[k] + acc[0]  (the "+ 1" of T_k + 1; T_0 = 1)
             float m[KT];
             m[0] = 2.f * acc[0];
#pragma unroll
             for (int k = 1; k < KT; ++k) m[k] = acc[k] + acc[0];
             store_row<KT>(Mrow + J * KT, m);
#pragma unroll
             for (int k = 0; k < KT; ++k) acc[k] = 0.f;
           },
           [&](const float4 &r) { return u[__float_as_int(r.w)]; },
           [&](const float4 &r, const float4 &uj) {
             float d, rinv, Tk[KT], Dk[KT], hfc, hfcp, hdf;
             pair_len(r.x * r.x + r.y * r.y + r.z * r.z, d, rinv);
             float ax, ay, az;
             pair_adjoint(ac, uj, r, ax, ay, az);
             const float ar = (ax * r.x + ay * r.y + az * r.z) * rinv;
             cheb_TD<KT>(d, sp.rcRinv, Tk, Dk, hfc, hfcp, hdf);
             const float w1 = ar * hdf, w2 = ar * hfcp;
             acc[0] += w2;
#pragma unroll
             for (int k = 1; k < KT; ++k) acc[k] = fmaf(w1, Dk[k], fmaf(w2, Tk[k], acc[k]));
           });
  radial_contract<KT>(sp, cs, type_s[a], Mrow, D + (size_t)a * sp.Ndes);
}

// ------------------------------------------------------------------------------------------------
// Small-batch variants of a3 / a5 (radial): RAD_SPLIT LANES PER ATOM.  A mini-batch of a few hundred atoms (the paper
// trains with batch size 1) gives the thread-per-atom kernels a handful of warps, each walking 60-odd pairs one
// after the other: pure latency.  Here the lanes of an atom take every RAD_SPLIT-th pair of a species segment (eight
// consecutive records = 128 contiguous bytes per atom and round) and add their sums by butterflies.  Same arithmetic
// per pair as the kernels above; chosen by the host when the batch cannot fill the SMs with one thread per atom.
// ------------------------------------------------------------------------------------------------
#define RAD_SPLIT 8          // lanes per atom ...
#define RAD_SPLIT_WIDE 32    // ... and for batches so small that even that leaves SMs idle: one warp per atom
template <int SPLIT>
__device__ __forceinline__ float split_sum(float x) {
#pragma unroll
  for (int o = 1; o < SPLIT; o <<= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
  return x;
}

template <int KT, int SPLIT>
__global__ void __launch_bounds__(RAD_THREADS)
k_radial_force_split(DevSpec sp, int N, const int *__restrict__ type_s, const int *__restrict__ segR,
                     const float4 *__restrict__ pairR, const float *__restrict__ etil, const int *__restrict__ segA,
                     const int *__restrict__ revA, const float4 *__restrict__ pairA, const float4 *__restrict__ fpair,
                     float4 *__restrict__ Fat, float *__restrict__ Wat) {
  const int gt = blockIdx.x * RAD_THREADS + threadIdx.x;
  const int a = gt / SPLIT, sub = gt % SPLIT;
  const bool on = a < N;                          // whole warps stay in the butterflies
  float F[3] = {0.f, 0.f, 0.f}, W[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
  if (on) {
    const int I = type_s[a];
    const int TK = sp.T * KT;
    const int *sg = segR + (size_t)a * (sp.T + 1);
    for (int J = 0; J < sp.T; ++J) {
      float ei[KT];
      load_row<KT>(etil + (size_t)a * TK + J * KT, ei);
      for (int p = sg[J] + sub; p < sg[J + 1]; p += SPLIT) {
        const float4 r = pairR[p];
        float ej[KT];
        load_row<KT>(etil + (size_t)__float_as_int(r.w) * TK + I * KT, ej);
        float d, rinv, Tk[KT], Dk[KT], hfc, hfcp, hdf;
        pair_len(r.x * r.x + r.y * r.y + r.z * r.z, d, rinv);
        cheb_TD<KT>(d, sp.rcRinv, Tk, Dk, hfc, hfcp, hdf);
        float sD = 0.f, sT = 2.f * (ei[0] + ej[0]);
#pragma unroll
        for (int k = 1; k < KT; ++k) {
          const float es = ei[k] + ej[k];
          sD = fmaf(es, Dk[k], sD);
          sT = fmaf(es, Tk[k] + 1.f, sT);
        }
        const float tot = sD * hdf + sT * hfcp;
        const float hx = r.x * rinv, hy = r.y * rinv, hz = r.z * rinv;
        F[0] += tot * hx; F[1] += tot * hy; F[2] += tot * hz;
        const float hf = 0.5f * tot;              // half of the pair's symmetric total, as in k_radial_force
        const float fx = hf * hx, fy = hf * hy, fz = hf * hz;
        W[0] -= r.x * fx; W[1] -= r.y * fy; W[2] -= r.z * fz;
        W[3] -= r.x * fy; W[4] -= r.y * fz; W[5] -= r.z * fx;
      }
    }
    if (fpair) {
      const int q0 = segA[(size_t)a * (sp.T + 1)], q1 = segA[(size_t)a * (sp.T + 1) + sp.T];
      for (int p = q0 + sub; p < q1; p += SPLIT) {
        const float4 f = fpair[p], x = pairA[p], g = fpair[revA[p]];
        F[0] += f.x - g.x; F[1] += f.y - g.y; F[2] += f.z - g.z;
        W[0] -= x.x * f.x; W[1] -= x.y * f.y; W[2] -= x.z * f.z;
        W[3] -= x.x * f.y; W[4] -= x.y * f.z; W[5] -= x.z * f.x;
      }
    }
  }
#pragma unroll
  for (int c = 0; c < 3; ++c) F[c] = split_sum<SPLIT>(F[c]);
#pragma unroll
  for (int c = 0; c < 6; ++c) W[c] = split_sum<SPLIT>(W[c]);
  if (on && sub == 0) {
    Fat[a] = make_float4(F[0], F[1], F[2], 0.f);
#pragma unroll
    for (int c = 0; c < 6; c += 2) *(float2 *)(Wat + (size_t)a * 6 + c) = make_float2(W[c], W[c + 1]);
  }
}

template <int KT, int SPLIT>
__global__ void __launch_bounds__(RAD_THREADS)
k_radial_adj_split(DevSpec sp, int N, const int *__restrict__ type_s, const int *__restrict__ struct_s,
                   const int *__restrict__ segR, const float4 *__restrict__ pairR, const float *__restrict__ theta,
                   const float4 *__restrict__ u, const float *__restrict__ omega, const float *__restrict__ scales,
                   float *__restrict__ D, float *__restrict__ M2) {
  extern __shared__ __align__(128) float smem[];
  float *cs = smem;
  stage_coeff(cs, theta, sp.T * sp.T * sp.NR, sp.KR, KT);
  __syncthreads();
  const int gt = blockIdx.x * RAD_THREADS + threadIdx.x;
  const int a = gt / SPLIT, sub = gt % SPLIT;
  const bool on = a < N;
  const int ac = on ? a : 0;
  const int I = N > 0 ? type_s[ac] : 0;
  AdjCtx ctx = {};
  if (on) ctx = make_adj(u, omega, scales, a, struct_s[a]);
  const int *sg = segR + (size_t)ac * (sp.T + 1);
  float o[2] = {0.f, 0.f};                        // D_n of the lane's two functions n = sub, sub + SPLIT
  for (int J = 0; J < sp.T; ++J) {
    float acc[KT];
#pragma unroll
    for (int k = 0; k < KT; ++k) acc[k] = 0.f;
    if (on)
      for (int p = sg[J] + sub; p < sg[J + 1]; p += SPLIT) {
        const float4 r = pairR[p];
        const float4 uj = u[__float_as_int(r.w)];
        float d, rinv, Tk[KT], Dk[KT], hfc, hfcp, hdf;
        pair_len(r.x * r.x + r.y * r.y + r.z * r.z, d, rinv);
        float ax, ay, az;
        pair_adjoint(ctx, uj, r, ax, ay, az);
        const float ar = (ax * r.x + ay * r.y + az * r.z) * rinv;
        cheb_TD<KT>(d, sp.rcRinv, Tk, Dk, hfc, hfcp, hdf);
        const float w1 = ar * hdf, w2 = ar * hfcp;
        acc[0] += w2;
#pragma unroll
        for (int k = 1; k < KT; ++k) acc[k] = fmaf(w1, Dk[k], fmaf(w2, Tk[k], acc[k]));
      }
#pragma unroll
    for (int k = 0; k < KT; ++k) acc[k] = split_sum<SPLIT>(acc[k]);
#pragma unroll
    for (int k = 1; k < KT; ++k) acc[k] += acc[0];                        // the "+ 1" of T_k + 1 (as in k_radial_adj)
    acc[0] *= 2.f;                                                        // every lane of the atom now holds M2[J][.]
    if (on && sub == 0) store_row<KT>(M2 + (size_t)a * sp.T * KT + J * KT, acc);
    const float *c = cs + (size_t)(I * sp.T + J) * sp.NR * KT;
#pragma unroll
    for (int i = 0; i < 2; ++i) {
      const int n = sub + i * SPLIT;
      if (n < sp.NR) {
        float cv[KT];
        load_row<KT>(c + n * KT, cv);
#pragma unroll
        for (int k = 0; k < KT; ++k) o[i] = fmaf(cv[k], acc[k], o[i]);
      }
    }
  }
  if (on) {
#pragma unroll
    for (int i = 0; i < 2; ++i) {
      const int n = sub + i * SPLIT;
      if (n < sp.NR) D[(size_t)a * sp.Ndes + n] = o[i];
    }
  }
}
