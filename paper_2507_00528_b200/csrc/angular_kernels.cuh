// angular_kernels.cuh -- sweeps over the angular neighbour list (rows a1, a3, a5, a7 of DESIGN.md).
//
// Moment form.  g_n(d) = sum_k c[I][J][n][k] f_k(d) is linear in the basis, so with
//   A1[J][k][lm] = sum_{j in J} f_k(d_ij) B_lm(rhat_ij)
//   A2[J][k][lm] = sum_{j in J} f_k'(d_ij) (a_ij.rhat_ij) B_lm + f_k(d_ij) (grad B_lm . a_ij)
// one has S_nlm = sum_{J,k} c A1 (Eq.8), T_nlm = sum_{J,k} c A2 (the summed factors of C3.9-C3.16) and
//   dL/dcA[I][J][n][k] = sum_atoms sum_lm alpha_nlm A1[J][k][lm] + beta_nlm A2[J][k][lm]   (C2.5-C2.10, C3.12-C3.20)
// so the coefficient gradient needs no pair sweep of its own, and the beta.A2 half is contracted inside the adjoint sweep
// while A2 is still in registers (A2 never goes to memory).
//
// Mapping of the moment kernels: ONE THREAD PER (ATOM, GROUP OF ANG_GS (l,m) SLOTS).  The contraction index of every sum
// above is the pair, so a thread that walks its atom's row keeps its K x 6 moment block in registers, needs no cross-lane
// traffic and no shared-memory hand-off between a "pair phase" and an "outer-product phase"; the c-contraction of a
// finished species segment is thread-local as well.  The price is that the ceil(NLM / 6) threads of an atom each
// evaluate the pair's radial basis (they run in different warps of the CTA: warp w = group w, lane = atom, so the code
// of a warp is uniform and the unused harmonics are removed at compile time).  A CTA works on a TILE of 32 atoms of one
// central species; tiles list atoms sorted by their per-species neighbour counts (k_nbr tiles, built at load time), so
// the 32 rows of a warp have equal lengths.
#pragma once
#include "common.cuh"
#include "pair_kernels.cuh"

#define ANG_GS 6          // (l,m) slots per thread
#define ANG_TILE 32       // atoms per tile (= lanes)
#define FRC_WARPS 4       // warps per CTA of the pair-force kernel
#define FRC_TA 8          // atoms per warp of the pair-force kernel

// number of slot groups of a model with l_max = L
__host__ __device__ constexpr int ang_groups(int L) { return (L * (L + 2) + ANG_GS - 1) / ANG_GS; }

// E'-like value of descriptor (n, l) of one atom row (0 when l > l_max)
__device__ __forceinline__ float desc_of(const DevSpec &sp, const float *__restrict__ row, int l, int n) {
  return l <= sp.L ? row[sp.NR + (l - 1) * sp.NA + n] : 0.f;
}
__device__ __forceinline__ void ld6(const float *__restrict__ p, float (&v)[6]) {   // 8-byte aligned
  const float2 a = *(const float2 *)p, b = *(const float2 *)(p + 2), c = *(const float2 *)(p + 4);
  v[0] = a.x; v[1] = a.y; v[2] = b.x; v[3] = b.y; v[4] = c.x; v[5] = c.y;
}
__device__ __forceinline__ void st6(float *__restrict__ p, const float (&v)[6]) {
  *(float2 *)p = make_float2(v[0], v[1]); *(float2 *)(p + 2) = make_float2(v[2], v[3]); *(float2 *)(p + 4) = make_float2(v[4], v[5]);
}

// Per-warp sum over lanes of per-lane values, KT at a time, into the warp's accumulator row accw[]: the values of
// 32 / KT functions are parked in a [32][33] scratch (one row per value, one column per lane), then lane v adds up row v
// in column order (fixed order: bit-reproducible) and adds the sum to its own accumulator slot.
template <int KT>
struct LaneSum {
  static constexpr int NPC = 32 / KT;     // functions n per chunk
  float *scratch, *accw;
  int lane;
  __device__ __forceinline__ void put(int nn, const float (&g)[KT]) {
#pragma unroll
    for (int k = 0; k < KT; ++k) scratch[(nn * KT + k) * 33 + lane] = g[k];
  }
  __device__ __forceinline__ void flush(int chunk, int nv) {   // nv = NA * KT valid values in all
    __syncwarp();
    const float *row = scratch + lane * 33;
    float s0 = 0.f, s1 = 0.f, s2 = 0.f, s3 = 0.f;
#pragma unroll
    for (int j = 0; j < 32; j += 4) { s0 += row[j]; s1 += row[j + 1]; s2 += row[j + 2]; s3 += row[j + 3]; }
    const int v = chunk * 32 + lane;
    if (v < nv) accw[v] += (s0 + s1) + (s2 + s3);
    __syncwarp();
  }
};

// ------------------------------------------------------------------------------------------------
// Memory layouts of the moment kernels.  A row-per-thread access costs one L1 wavefront per lane whatever its width, so
// everything a thread (atom a, slot group G) reads or writes by itself is one contiguous, 32-byte aligned block moved
// with 256-bit accesses ("group-major"):
//   A1g [a][G][J][k][6]      moments of the species segment J               (k_angular_fwd -> k_cgrad_angular)
//   Bg  [a][G][n][6], n < NAp = NA rounded up to 4                           (k_angular_force -> k_angular_adj)
// while the per-atom rows S[a][n][nlmS], T[a][n][nlmS] stay row-major: they are assembled in shared memory by the
// slot-group threads and written (and read) whole by one thread per (atom, n).
// ------------------------------------------------------------------------------------------------
__host__ __device__ inline int ang_nap(int NA) { return (NA + 3) & ~3; }

template <int N8>
__device__ __forceinline__ void st_block(float *__restrict__ p, const float (&v)[8 * N8]) {   // N8 x 8 floats, 32-byte aligned
#pragma unroll
  for (int c = 0; c < N8; ++c)
    stg256(p + 8 * c, make_float4(v[8 * c], v[8 * c + 1], v[8 * c + 2], v[8 * c + 3]),
           make_float4(v[8 * c + 4], v[8 * c + 5], v[8 * c + 6], v[8 * c + 7]));
}
template <int N8>
__device__ __forceinline__ void ld_block(const float *__restrict__ p, float (&v)[8 * N8]) {
#pragma unroll
  for (int c = 0; c < N8; ++c) {
    const float8 t = ldg256(p + 8 * c);
    v[8 * c] = t.lo.x; v[8 * c + 1] = t.lo.y; v[8 * c + 2] = t.lo.z; v[8 * c + 3] = t.lo.w;
    v[8 * c + 4] = t.hi.x; v[8 * c + 5] = t.hi.y; v[8 * c + 6] = t.hi.z; v[8 * c + 7] = t.hi.w;
  }
}

// One (atom, n) row of S or T gathered from the per-thread shared slots part[(n*6 + i) * nthr + G*32 + lane] of the
// ng slot-group threads of the atom (slots of groups that do not exist read as zero)
template <int LMAX>
__device__ __forceinline__ void gather_row(const float *part, int n, int nthr, int ng, int lane, float (&s)[LMAX * (LMAX + 2)]) {
#pragma unroll
  for (int lm = 0; lm < LMAX * (LMAX + 2); ++lm)
    s[lm] = lm / ANG_GS < ng ? part[(n * ANG_GS + lm % ANG_GS) * nthr + (lm / ANG_GS) * 32 + lane] : 0.f;
}
// ... written row-major with 256-bit stores (row stride NS is a multiple of 8 floats; the slots past NLM are zero)
template <int LMAX>
__device__ __forceinline__ void store_row_lm(float *__restrict__ row, const float (&s)[LMAX * (LMAX + 2)], int NS) {
  constexpr int NLM = LMAX * (LMAX + 2);
#pragma unroll
  for (int c = 0; c < NLM / 8; ++c)
    stg256(row + 8 * c, make_float4(s[8 * c], s[8 * c + 1], s[8 * c + 2], s[8 * c + 3]),
           make_float4(s[8 * c + 4], s[8 * c + 5], s[8 * c + 6], s[8 * c + 7]));
  (void)NS;
}
template <int LMAX>
__device__ __forceinline__ void load_row_lm(const float *__restrict__ row, float (&s)[LMAX * (LMAX + 2)]) {
  ld_block<LMAX * (LMAX + 2) / 8>(row, s);
}

// q_nl = sum_m C_lm S_nlm^2 (Eq.7), q4_n = kappa4 P4(S_n2m) (R14), q5_n = kappa5 |S_n1|^4 (R41); out: the atom's angular
// descriptor entries nu - NR
template <int LMAX>
__device__ __forceinline__ void finish_q(const DevSpec &sp, const float (&s)[LMAX * (LMAX + 2)], float *out, int n) {
#pragma unroll
  for (int l = 1; l <= LMAX; ++l) {
    float acc = 0.f;
#pragma unroll
    for (int m = 0; m <= 2 * l; ++m) { const int lm = l * l - 1 + m; acc = fmaf(0.5f * c_C2[lm] * s[lm], s[lm], acc); }
    if (l <= sp.L) out[(l - 1) * sp.NA + n] = acc;
  }
  int o = sp.L * sp.NA;
  if (sp.use4) { out[o + n] = GNEP_KAPPA4 * p4_value(&s[3]); o += sp.NA; }
  if (sp.use5) out[o + n] = p5_value(&s[0]);
}
// D_(n,l) = sum_m 2 C_lm S_nlm T_nlm, D_4 = kappa4 grad P4(S) . T, D_5 = grad q5(S) . T
template <int LMAX>
__device__ __forceinline__ void finish_D(const DevSpec &sp, const float (&s)[LMAX * (LMAX + 2)], const float (&t)[LMAX * (LMAX + 2)],
                                         float *out, int n) {
#pragma unroll
  for (int l = 1; l <= LMAX; ++l) {
    float acc = 0.f;
#pragma unroll
    for (int m = 0; m <= 2 * l; ++m) { const int lm = l * l - 1 + m; acc = fmaf(c_C2[lm] * s[lm], t[lm], acc); }
    if (l <= sp.L) out[(l - 1) * sp.NA + n] = acc;
  }
  int o = sp.L * sp.NA;
  if (sp.use4) {
    float g4[5];
    p4_grad(&s[3], g4);
    out[o + n] = GNEP_KAPPA4 * (g4[0] * t[3] + g4[1] * t[4] + g4[2] * t[5] + g4[3] * t[6] + g4[4] * t[7]);
    o += sp.NA;
  }
  if (sp.use5) {
    float g5[3];
    p5_grad(&s[0], g5);
    out[o + n] = g5[0] * t[0] + g5[1] * t[1] + g5[2] * t[2];
  }
}
// the tile's angular descriptor entries, assembled in shared memory rows[al * stride + nu], go out with coalesced stores
__device__ __forceinline__ void copy_out_rows(const DevSpec &sp, const int *at, const float *rows, int stride, float *__restrict__ dst) {
  const int nqa = sp.Ndes - sp.NR;
  for (int x = threadIdx.x; x < ANG_TILE * nqa; x += blockDim.x) {
    const int al = x / nqa, v = x - al * nqa, a = at[al];
    if (a >= 0) dst[(size_t)a * sp.Ndes + sp.NR + v] = rows[al * stride + v];
  }
}

// ------------------------------------------------------------------------------------------------
// a1 (angular): A1 moments, S_nlm (Eq.8), q_nl (Eq.7), many-body terms (R14, R41)
// ------------------------------------------------------------------------------------------------
template <int KT, int LMAX, int G>
__device__ __forceinline__ void ang_fwd_thread(const DevSpec &sp, const float *cs, float *Spart, int nthr, int ng, int a,
                                               const int *__restrict__ type_s, const int *__restrict__ segA,
                                               const float4 *__restrict__ pairA, float *__restrict__ A1g) {
  const int I = type_s[a];
  const int *sg = segA + (size_t)a * (sp.T + 1);
  float *A1a = A1g + ((size_t)a * ng + G) * sp.T * KT * ANG_GS;
  float *sp_t = Spart + threadIdx.x;
  int pbeg = sg[0];
  for (int J = 0; J < sp.T; ++J) {
    const int pend = sg[J + 1];
    float acc[KT * ANG_GS];
#pragma unroll
    for (int x = 0; x < KT * ANG_GS; ++x) acc[x] = 0.f;
    float4 rn = pbeg < pend ? pairA[pbeg] : make_float4(1.f, 0.f, 0.f, 0.f);
    for (int p = pbeg; p < pend; ++p) {
      const float4 r = rn;
      if (p + 1 < pend) rn = pairA[p + 1];                   // the next record is in flight during this pair
      float d, rinv;
      pair_len(r.x * r.x + r.y * r.y + r.z * r.z, d, rinv);
      float f[KT];
      cheb_f<KT>(d, sp.rcAinv, f);
      float B[ANG_GS];
#pragma unroll
      for (int i = 0; i < ANG_GS; ++i) B[i] = 0.f;
      blm_unit<LMAX>(r.x * rinv, r.y * rinv, r.z * rinv, [&](int lm, int, float b, float, float, float) {
        if (lm >= G * ANG_GS && lm < (G + 1) * ANG_GS) B[lm - G * ANG_GS] = b;
      });
#pragma unroll
      for (int k = 0; k < KT; ++k)
#pragma unroll
        for (int i = 0; i < ANG_GS; ++i) acc[k * ANG_GS + i] = fmaf(f[k], B[i], acc[k * ANG_GS + i]);
    }
    pbeg = pend;
    st_block<KT * ANG_GS / 8>(A1a + (size_t)J * KT * ANG_GS, acc);
    // S += c[I][J] . A1[J]  (thread-local: this thread owns its 6 slots of every n); the running sums live in the
    // thread's shared slots, where the finishing step picks the complete rows up
    const float *c = cs + (size_t)(I * sp.T + J) * sp.NA * KT;
    const bool first = J == 0;
    for (int n = 0; n < sp.NA; ++n) {
      float s[ANG_GS];
#pragma unroll
      for (int i = 0; i < ANG_GS; ++i) s[i] = first ? 0.f : sp_t[(n * ANG_GS + i) * nthr];
#pragma unroll
      for (int k4 = 0; k4 < KT; k4 += 4) {
        const float4 c4 = *(const float4 *)(c + n * KT + k4);
        const float cv[4] = {c4.x, c4.y, c4.z, c4.w};
#pragma unroll
        for (int kk = 0; kk < 4; ++kk)
#pragma unroll
          for (int i = 0; i < ANG_GS; ++i) s[i] = fmaf(cv[kk], acc[(k4 + kk) * ANG_GS + i], s[i]);
      }
#pragma unroll
      for (int i = 0; i < ANG_GS; ++i) sp_t[(n * ANG_GS + i) * nthr] = s[i];
    }
  }
}

// warp w of the CTA runs the code of slot group w (the groups beyond ang_groups(LMAX) are never instantiated)
#define ANG_CASE(LMAX, g, CALL) \
  case g: if constexpr (ang_groups(LMAX) > g) { constexpr int G = g; CALL; } break;
#define ANG_GROUP_SWITCH(LMAX, w, CALL)                                                                        \
  switch (w) {                                                                                                 \
    ANG_CASE(LMAX, 0, CALL) ANG_CASE(LMAX, 1, CALL) ANG_CASE(LMAX, 2, CALL) ANG_CASE(LMAX, 3, CALL)            \
    ANG_CASE(LMAX, 4, CALL) ANG_CASE(LMAX, 5, CALL) ANG_CASE(LMAX, 6, CALL) ANG_CASE(LMAX, 7, CALL)            \
    ANG_CASE(LMAX, 8, CALL) ANG_CASE(LMAX, 9, CALL) ANG_CASE(LMAX, 10, CALL) ANG_CASE(LMAX, 11, CALL)          \
    ANG_CASE(LMAX, 12, CALL) ANG_CASE(LMAX, 13, CALL)                                                          \
    default: break;                                                                                            \
  }

// shared-memory floats: coefficients | per-thread S slots [NA*6][threads] | descriptor rows [32][nqa|1] | atom ids [32]
__host__ __device__ inline int ang_fwd_smem_floats(int T, int NA, int KT, int nwarps, int nqa) {
  return ((T * T * NA * KT + 3) & ~3) + NA * ANG_GS * 32 * nwarps + ANG_TILE * (nqa | 1) + ANG_TILE;
}

template <int KT, int LMAX>
__global__ void __launch_bounds__(32 * ang_groups(LMAX), LMAX <= 4 ? 4 : 1)
k_angular_fwd(DevSpec sp, int n_tiles, const int *__restrict__ tiles, const int *__restrict__ type_s,
              const int *__restrict__ segA, const float4 *__restrict__ pairA, const float *__restrict__ theta,
              float *__restrict__ q, float *__restrict__ S, float *__restrict__ A1g) {
  extern __shared__ __align__(128) float smem[];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nthr = blockDim.x, ng = nthr >> 5;
  const int nqa = sp.Ndes - sp.NR, qst = nqa | 1;
  float *cs = smem;                                             // [T*T*NA][KT]
  float *Spart = smem + ((sp.T * sp.T * sp.NA * KT + 3) & ~3);  // [NA*6][threads]
  float *QS = Spart + sp.NA * ANG_GS * nthr;                    // [32][qst]
  int *at = (int *)(QS + ANG_TILE * qst);
  stage_coeff(cs, theta + sp.offA, sp.T * sp.T * sp.NA, sp.KA, KT);
  const int a = tiles[blockIdx.x * ANG_TILE + lane];
  if (w == 0) at[lane] = a;
  __syncthreads();
  if (a >= 0) {
    ANG_GROUP_SWITCH(LMAX, w, (ang_fwd_thread<KT, LMAX, G>(sp, cs, Spart, nthr, ng, a, type_s, segA, pairA, A1g)));
  }
  __syncthreads();                                              // the S rows of the tile are complete in shared memory
  if (a >= 0)
    for (int n = w; n < sp.NA; n += ng) {
      float s[LMAX * (LMAX + 2)];
      gather_row<LMAX>(Spart, n, nthr, ng, lane, s);
      store_row_lm<LMAX>(S + ((size_t)a * sp.NA + n) * sp.nlmS, s, sp.nlmS);
      finish_q<LMAX>(sp, s, QS + lane * qst, n);
    }
  __syncthreads();
  copy_out_rows(sp, at, QS, qst, q);
}

// ------------------------------------------------------------------------------------------------
// a5 (angular) + the beta half of a7: A2 moments with the pair adjoint a_ij, T_nlm = c.A2, D_(n,l), D_4, D_5, and
// dL/dcA[I][J][n][k] += sum_lm beta_nlm A2[J][k][lm]  (beta = E' dq/dS was written by k_angular_force)
// ------------------------------------------------------------------------------------------------
template <int KT, int LMAX, int G>
__device__ __forceinline__ void ang_adj_thread(const DevSpec &sp, const float *cs, float *Tpart, int nthr, int ng, LaneSum<KT> &ls,
                                               int a, const int *__restrict__ type_s, const int *__restrict__ struct_s,
                                               const int *__restrict__ segA, const float4 *__restrict__ pairA,
                                               const float4 *__restrict__ u, const float *__restrict__ omega,
                                               const float *__restrict__ scales, const float *__restrict__ Bg, bool act) {
  const int I = type_s[a];
  const int *sg = segA + (size_t)a * (sp.T + 1);
  const AdjCtx ac = make_adj(u, omega, scales, a, struct_s[a]);
  const float *Ba = Bg + ((size_t)a * ng + G) * ang_nap(sp.NA) * ANG_GS;
  float *tp_t = Tpart + threadIdx.x;
  float *accw_I = ls.accw;                                      // [T][NA*KT] block of this central species
  int pbeg = act ? sg[0] : 0;
  for (int J = 0; J < sp.T; ++J) {
    const int pend = act ? sg[J + 1] : 0;
    float acc[KT][ANG_GS];
#pragma unroll
    for (int k = 0; k < KT; ++k)
#pragma unroll
      for (int i = 0; i < ANG_GS; ++i) acc[k][i] = 0.f;
    // records two pairs ahead, the gather of u_j one pair ahead
    const float4 rdum = make_float4(1.f, 0.f, 0.f, __int_as_float(a));
    float4 r1 = pbeg < pend ? pairA[pbeg] : rdum;
    float4 r2 = pbeg + 1 < pend ? pairA[pbeg + 1] : rdum;
    float4 uj1 = u[__float_as_int(r1.w)];
    for (int p = pbeg; p < pend; ++p) {
      const float4 r = r1, uj = uj1;
      r1 = r2;
      uj1 = u[__float_as_int(r1.w)];
      r2 = p + 2 < pend ? pairA[p + 2] : rdum;
      float d, rinv, ax, ay, az;
      pair_len(r.x * r.x + r.y * r.y + r.z * r.z, d, rinv);
      pair_adjoint(ac, uj, r, ax, ay, az);
      const float hx = r.x * rinv, hy = r.y * rinv, hz = r.z * rinv;
      const float ar = ax * hx + ay * hy + az * hz;
      float f[KT], fp[KT];
      cheb_ffp<KT>(d, sp.rcAinv, f, fp);
      float X[ANG_GS], Y[ANG_GS];
#pragma unroll
      for (int i = 0; i < ANG_GS; ++i) { X[i] = 0.f; Y[i] = 0.f; }
      blm_unit<LMAX>(hx, hy, hz, [&](int lm, int l, float b, float gx, float gy, float gz) {
        if (lm >= G * ANG_GS && lm < (G + 1) * ANG_GS) {
          X[lm - G * ANG_GS] = b;
          Y[lm - G * ANG_GS] = rinv * ((gx * ax + gy * ay + gz * az) - (float)l * b * ar);
        }
      });
#pragma unroll
      for (int k = 0; k < KT; ++k) {
        const float f1 = fp[k] * ar;
#pragma unroll
        for (int i = 0; i < ANG_GS; ++i) acc[k][i] = fmaf(f1, X[i], fmaf(f[k], Y[i], acc[k][i]));
      }
    }
    pbeg = pend;
    const float *c = cs + (size_t)(I * sp.T + J) * sp.NA * KT;
    const bool first = J == 0;
    // T += c[I][J] . A2[J], running sums in the thread's shared slots
    if (act)
      for (int n = 0; n < sp.NA; ++n) {
        float t[ANG_GS];
#pragma unroll
        for (int i = 0; i < ANG_GS; ++i) t[i] = first ? 0.f : tp_t[(n * ANG_GS + i) * nthr];
#pragma unroll
        for (int k4 = 0; k4 < KT; k4 += 4) {
          const float4 c4 = *(const float4 *)(c + n * KT + k4);
          const float cv[4] = {c4.x, c4.y, c4.z, c4.w};
#pragma unroll
          for (int kk = 0; kk < 4; ++kk)
#pragma unroll
            for (int i = 0; i < ANG_GS; ++i) t[i] = fmaf(cv[kk], acc[k4 + kk][i], t[i]);
        }
#pragma unroll
        for (int i = 0; i < ANG_GS; ++i) tp_t[(n * ANG_GS + i) * nthr] = t[i];
      }
    // dL/dcA[I][J][n][k] += sum_{lm in group} beta_nlm A2[J][k][lm], summed over the 32 atoms of the warp
    ls.accw = accw_I + J * sp.NA * KT;
    constexpr int NPC = LaneSum<KT>::NPC;                       // functions per chunk: their beta slots are one aligned block
    for (int ch = 0; ch * NPC < sp.NA; ++ch) {
      float be[NPC * ANG_GS];
      if (act) {
        if constexpr ((NPC * ANG_GS) % 8 == 0) ld_block<NPC * ANG_GS / 8>(Ba + ch * NPC * ANG_GS, be);
        else {
#pragma unroll
          for (int v = 0; v < NPC * ANG_GS; v += 4) {
            const float4 t4 = *(const float4 *)(Ba + ch * NPC * ANG_GS + v);
            be[v] = t4.x; be[v + 1] = t4.y; be[v + 2] = t4.z; be[v + 3] = t4.w;
          }
        }
      } else {
#pragma unroll
        for (int v = 0; v < NPC * ANG_GS; ++v) be[v] = 0.f;
      }
#pragma unroll
      for (int nn = 0; nn < NPC; ++nn) {
        float g[KT];
#pragma unroll
        for (int k = 0; k < KT; ++k) {
          g[k] = 0.f;
#pragma unroll
          for (int i = 0; i < ANG_GS; ++i) g[k] = fmaf(be[nn * ANG_GS + i], acc[k][i], g[k]);   // (beta rows past NA are zero)
        }
        ls.put(nn, g);
      }
      ls.flush(ch, sp.NA * KT);
    }
  }
  ls.accw = accw_I;
}

// shared-memory floats of k_angular_adj: coefficients | per-thread T slots | D rows [32][nqa|1] | per-warp scratch [32][33]
// | per-warp accumulators [T*T][NA*KT] | atom ids
__host__ __device__ inline int ang_adj_smem_floats(int T, int NA, int KT, int nwarps, int nqa) {
  return ((T * T * NA * KT + 3) & ~3) + NA * ANG_GS * 32 * nwarps + ANG_TILE * (nqa | 1) + nwarps * 32 * 33 +
         nwarps * T * T * NA * KT + ANG_TILE;
}

template <int KT, int LMAX>
__global__ void __launch_bounds__(32 * ang_groups(LMAX), LMAX <= 4 ? 4 : 1)
k_angular_adj(DevSpec sp, int n_tiles, const int *__restrict__ tiles, const int *__restrict__ type_s,
              const int *__restrict__ struct_s, const int *__restrict__ segA, const float4 *__restrict__ pairA,
              const float *__restrict__ theta, const float4 *__restrict__ u, const float *__restrict__ omega,
              const float *__restrict__ scales, const float *__restrict__ S, const float *__restrict__ Bg,
              float *__restrict__ Tn, float *__restrict__ D, float *__restrict__ partial) {
  extern __shared__ __align__(128) float smem[];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nthr = blockDim.x, ng = nthr >> 5;
  const int ncs = (sp.T * sp.T * sp.NA * KT + 3) & ~3, nv = sp.NA * KT, nacc = sp.T * sp.T * nv;
  const int nqa = sp.Ndes - sp.NR, qst = nqa | 1;
  float *cs = smem;
  float *Tpart = cs + ncs;                                      // [NA*6][threads]
  float *DS = Tpart + sp.NA * ANG_GS * nthr;                    // [32][qst]
  float *scr = DS + ANG_TILE * qst + w * 32 * 33;               // per warp [32][33]
  float *accw = DS + ANG_TILE * qst + ng * 32 * 33 + w * nacc;  // per warp [T*T][NA*KT]
  int *at = (int *)(DS + ANG_TILE * qst + ng * 32 * 33 + ng * nacc);
  stage_coeff(cs, theta + sp.offA, sp.T * sp.T * sp.NA, sp.KA, KT);
  for (int o = lane; o < nacc; o += 32) accw[o] = 0.f;
  for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
    const int a = tiles[tile * ANG_TILE + lane];
    const int a0 = tiles[tile * ANG_TILE];                      // lane 0 of a tile is always a real atom
    __syncthreads();                                            // coefficients staged; previous tile's rows copied out
    if (w == 0) at[lane] = a;
    const int I = type_s[a0];
    LaneSum<KT> ls{scr, accw + I * sp.T * nv, lane};
    const bool act = a >= 0;
    const int aa = act ? a : a0;                                // idle lanes walk no pairs but join the lane sums
    ANG_GROUP_SWITCH(LMAX, w, (ang_adj_thread<KT, LMAX, G>(sp, cs, Tpart, nthr, ng, ls, aa, type_s, struct_s, segA, pairA, u, omega,
                                                            scales, Bg, act)));
    __syncthreads();                                            // the T rows of the tile are complete in shared memory
    if (act)
      for (int n = w; n < sp.NA; n += ng) {
        float s[LMAX * (LMAX + 2)], t[LMAX * (LMAX + 2)];
        const size_t row = ((size_t)a * sp.NA + n) * sp.nlmS;
        load_row_lm<LMAX>(S + row, s);
        gather_row<LMAX>(Tpart, n, nthr, ng, lane, t);
        store_row_lm<LMAX>(Tn + row, t, sp.nlmS);
        finish_D<LMAX>(sp, s, t, DS + lane * qst, n);
      }
    __syncthreads();
    copy_out_rows(sp, at, DS, qst, D);
  }
  __syncwarp();
  float *dst = partial + (size_t)(blockIdx.x * ng + w) * nacc;
  for (int o = lane; o < nacc; o += 32) dst[o] = accw[o];
}

// ------------------------------------------------------------------------------------------------
// a3 (angular): f_ij = sum_n sum_lm beta_nlm (g_n' B_lm rhat + g_n grad B_lm)   (C3.6 with C2.1-C2.3)
// lane = pair over the packed pairs of FRC_TA atoms; beta of the tile's atoms lives in shared memory (and is written to
// global memory once for the adjoint sweep).  gam_lm = sum_n g_n beta_nlm, gamp_lm = sum_n g_n' beta_nlm, then one
// harmonic sweep.  Writes f_ij per pair.
// ------------------------------------------------------------------------------------------------
// beta_nlm = E'_(n,l) 2C_lm S_nlm (+ E'_4 kappa4 dP4/ds_m for l = 2, + E'_5 dq5/ds_m for l = 1) of one (atom, n) row
template <int LMAX>
__device__ __forceinline__ void beta_row(const DevSpec &sp, const float *__restrict__ Srow, const float *__restrict__ Epa, int n,
                                         float *__restrict__ out_s) {
  constexpr int NLM = LMAX * (LMAX + 2);
  float s[NLM], b[NLM];
  load_row_lm<LMAX>(Srow, s);
#pragma unroll
  for (int l = 1; l <= LMAX; ++l) {
    const float e = desc_of(sp, Epa, l, n);
#pragma unroll
    for (int m = 0; m <= 2 * l; ++m) { const int lm = l * l - 1 + m; b[lm] = e * c_C2[lm] * s[lm]; }
  }
  int o = sp.NR + sp.L * sp.NA;
  if (sp.use4) {
    float g4[5];
    p4_grad(&s[3], g4);
    const float e4 = GNEP_KAPPA4 * Epa[o + n];
#pragma unroll
    for (int m = 0; m < 5; ++m) b[3 + m] += e4 * g4[m];
    o += sp.NA;
  }
  if (sp.use5) {
    float g5[3];
    p5_grad(&s[0], g5);
    const float e5 = Epa[o + n];
#pragma unroll
    for (int m = 0; m < 3; ++m) b[m] += e5 * g5[m];
  }
#pragma unroll
  for (int v = 0; v < NLM; v += 4) *(float4 *)(out_s + v) = make_float4(b[v], b[v + 1], b[v + 2], b[v + 3]);
}

// contribution of the harmonics lm in [LO, HI) to the pair force: gam_lm = sum_n g_n beta_nlm, gamp_lm = sum_n g_n' beta_nlm
// over that slot range, then the harmonic sweep.  LO and HI - LO are multiples of 4 (16-byte loads of the beta rows).
template <int KT, int LMAX, int LO, int HI>
__device__ __forceinline__ void force_block(const DevSpec &sp, const float *__restrict__ be, int NS, const float *__restrict__ c,
                                            const float (&f)[KT], const float (&fp)[KT], float hx, float hy, float hz,
                                            float &sB, float &sl, float &vx, float &vy, float &vz) {
  constexpr int NB = HI - LO;
  static_assert(LO % 4 == 0 && NB % 4 == 0, "slot blocks are float4-aligned");
  float gam[NB], gamp[NB];
#pragma unroll
  for (int i = 0; i < NB; ++i) { gam[i] = 0.f; gamp[i] = 0.f; }
  for (int n = 0; n < sp.NA; ++n) {
    float g = 0.f, gp = 0.f;
#pragma unroll
    for (int k = 0; k < KT; ++k) { const float cv = c[n * KT + k]; g = fmaf(cv, f[k], g); gp = fmaf(cv, fp[k], gp); }
#pragma unroll
    for (int v = 0; v < NB / 4; ++v) {
      const float4 b4 = *(const float4 *)(be + n * NS + LO + 4 * v);
      gam[4 * v] = fmaf(g, b4.x, gam[4 * v]); gam[4 * v + 1] = fmaf(g, b4.y, gam[4 * v + 1]);
      gam[4 * v + 2] = fmaf(g, b4.z, gam[4 * v + 2]); gam[4 * v + 3] = fmaf(g, b4.w, gam[4 * v + 3]);
      gamp[4 * v] = fmaf(gp, b4.x, gamp[4 * v]); gamp[4 * v + 1] = fmaf(gp, b4.y, gamp[4 * v + 1]);
      gamp[4 * v + 2] = fmaf(gp, b4.z, gamp[4 * v + 2]); gamp[4 * v + 3] = fmaf(gp, b4.w, gamp[4 * v + 3]);
    }
  }
  blm_unit<LMAX>(hx, hy, hz, [&](int lm, int l, float b, float gx, float gy, float gz) {
    if (lm >= LO && lm < HI) {
      sB = fmaf(gamp[lm - LO], b, sB);
      sl = fmaf((float)l * gam[lm - LO], b, sl);
      vx = fmaf(gam[lm - LO], gx, vx); vy = fmaf(gam[lm - LO], gy, vy); vz = fmaf(gam[lm - LO], gz, vz);
    }
  });
}

template <int KT, int LMAX>
__global__ void __launch_bounds__(FRC_WARPS * 32)
k_angular_force(DevSpec sp, int N, const int *__restrict__ type_s, const int *__restrict__ segA,
                const int *__restrict__ atomA, const float4 *__restrict__ pairA, const float *__restrict__ theta,
                const float *__restrict__ Ep, const float *__restrict__ S, float *__restrict__ Bg,
                float4 *__restrict__ fpair) {
  extern __shared__ __align__(128) float smem[];
  float *cs = smem;
  const int ncs = (sp.T * sp.T * sp.NA * KT + 3) & ~3;
  const int NS = sp.nlmS, nb = sp.NA * NS;
  float *beta = smem + ncs + (threadIdx.x >> 5) * FRC_TA * nb;
  stage_coeff(cs, theta + sp.offA, sp.T * sp.T * sp.NA, sp.KA, KT);
  __syncthreads();
  const int lane = threadIdx.x & 31;
  const int a_lo = (blockIdx.x * FRC_WARPS + (threadIdx.x >> 5)) * FRC_TA;
  if (a_lo >= N) return;
  const int a_hi = min(a_lo + FRC_TA, N);
  const int T1 = sp.T + 1;
  const int P_lo = segA[a_lo * T1], P_hi = segA[(a_hi - 1) * T1 + sp.T];
  // beta of the tile's atoms: one (atom, n) row per lane and round, into shared memory ...
  for (int it = lane; it < (a_hi - a_lo) * sp.NA; it += 32) {
    const int al = it / sp.NA, n = it - al * sp.NA;
    beta_row<LMAX>(sp, S + ((size_t)(a_lo + al) * sp.NA + n) * NS, Ep + (size_t)(a_lo + al) * sp.Ndes, n, beta + al * nb + n * NS);
  }
  __syncwarp();
  // ... and out to global memory in the group-major layout of the adjoint sweep, Bg[a][G][n < NAp][6], 32 bytes per
  // lane and store (rows n >= NA are zero)
  {
    const int ng = ang_groups(sp.L), nap = ang_nap(sp.NA), per_atom = ng * nap * ANG_GS / 8;
    for (int it = lane; it < (a_hi - a_lo) * per_atom; it += 32) {
      const int al = it / per_atom, c8 = it - al * per_atom;
      const int G = c8 / (nap * ANG_GS / 8), e0 = (c8 - G * (nap * ANG_GS / 8)) * 8;
      float v[8];
#pragma unroll
      for (int e = 0; e < 8; ++e) {
        const int n = (e0 + e) / ANG_GS, i = (e0 + e) - n * ANG_GS;
        v[e] = n < sp.NA ? beta[al * nb + n * NS + G * ANG_GS + i] : 0.f;
      }
      stg256(Bg + ((size_t)(a_lo + al) * ng + G) * nap * ANG_GS + e0, make_float4(v[0], v[1], v[2], v[3]), make_float4(v[4], v[5], v[6], v[7]));
    }
  }
  if (P_lo == P_hi) return;
  // atomA packs (central atom | neighbour species << 28 | central species << 30); the next chunk's record is in flight
  float4 rn = make_float4(1.f, 0.f, 0.f, 0.f);
  int an = 0;
  if (P_lo + lane < P_hi) { rn = pairA[P_lo + lane]; an = atomA[P_lo + lane]; }
  for (int p = P_lo + lane; p < P_hi; p += 32) {
    const float4 r = rn;
    const unsigned packed = (unsigned)an;
    if (p + 32 < P_hi) { rn = pairA[p + 32]; an = atomA[p + 32]; }
    const int a = (int)(packed & 0x0fffffffu), J = (int)((packed >> 28) & 3u), I = (int)(packed >> 30);
    const float *be = beta + (a - a_lo) * nb;
    float d, rinv;
    pair_len(r.x * r.x + r.y * r.y + r.z * r.z, d, rinv);
    float f[KT], fp[KT];
    cheb_ffp<KT>(d, sp.rcAinv, f, fp);
    const float *c = cs + (I * sp.T + J) * sp.NA * KT;
    const float hx = r.x * rinv, hy = r.y * rinv, hz = r.z * rinv;
    float sB = 0.f, sl = 0.f, vx = 0.f, vy = 0.f, vz = 0.f;
    force_block<KT, LMAX, 0, 24>(sp, be, NS, c, f, fp, hx, hy, hz, sB, sl, vx, vy, vz);              // l = 1..4
    if constexpr (LMAX > 4) {
      if (sp.L >= 5) force_block<KT, LMAX, 24, 48>(sp, be, NS, c, f, fp, hx, hy, hz, sB, sl, vx, vy, vz);   // l = 5, 6
      if (sp.L >= 7) force_block<KT, LMAX, 48, 64>(sp, be, NS, c, f, fp, hx, hy, hz, sB, sl, vx, vy, vz);   // l = 7 and slot 63
      if (sp.L >= 8) force_block<KT, LMAX, 64, 80>(sp, be, NS, c, f, fp, hx, hy, hz, sB, sl, vx, vy, vz);   // rest of l = 8
    }
    fpair[p] = make_float4(hx * sB + rinv * (vx - hx * sl), hy * sB + rinv * (vy - hy * sl),
                           hz * sB + rinv * (vz - hz * sl), 0.f);
  }
}

// (The gather F_i += sum_p (f_p - f_rev(p)), W_i -= sum_p r_p (x) f_p is done by k_radial_force, thread per atom.)

// ------------------------------------------------------------------------------------------------
// a7 (angular), alpha half: dL/dcA[I][J][n][k] += sum_atoms sum_lm alpha_nlm A1[J][k][lm]
//   alpha_nlm = gbar_(n,l) 2C_lm S_nlm + E'_(n,l) 2C_lm T_nlm (+ 4-body: gbar_4 k4 dP4/ds_m + E'_4 k4 (H4 T)_m, 5-body alike)
// No pair sweep (the A1 moments were stored by k_angular_fwd).  Per tile: the E' and gbar rows are staged in shared memory
// with coalesced loads, one thread per (atom, n) builds the alpha row from the S and T rows, then the slot-group threads
// contract their alpha slots with their A1 block and the lane sums go to the per-warp accumulators as in the adjoint sweep.
// ------------------------------------------------------------------------------------------------
template <int LMAX>
__device__ __forceinline__ void alpha_row(const DevSpec &sp, const float (&s)[LMAX * (LMAX + 2)], const float (&t)[LMAX * (LMAX + 2)],
                                          const float *ep, const float *gb, int n, float (&al)[LMAX * (LMAX + 2)]) {
#pragma unroll
  for (int l = 1; l <= LMAX; ++l) {
    const float e1 = l <= sp.L ? ep[(l - 1) * sp.NA + n] : 0.f, g1 = l <= sp.L ? gb[(l - 1) * sp.NA + n] : 0.f;
#pragma unroll
    for (int m = 0; m <= 2 * l; ++m) { const int lm = l * l - 1 + m; al[lm] = c_C2[lm] * (g1 * s[lm] + e1 * t[lm]); }
  }
  int o = sp.L * sp.NA;
  if (sp.use4) {
    float g4[5], hv[5];
    p4_grad(&s[3], g4);
    p4_hess_vec(&s[3], &t[3], hv);
    const float e4 = GNEP_KAPPA4 * ep[o + n], gb4 = GNEP_KAPPA4 * gb[o + n];
#pragma unroll
    for (int m = 0; m < 5; ++m) al[3 + m] += gb4 * g4[m] + e4 * hv[m];
    o += sp.NA;
  }
  if (sp.use5) {
    float g5[3], hv[3];
    p5_grad(&s[0], g5);
    p5_hess_vec(&s[0], &t[0], hv);
    const float e5 = ep[o + n], gb5 = gb[o + n];
#pragma unroll
    for (int m = 0; m < 3; ++m) al[m] += gb5 * g5[m] + e5 * hv[m];
  }
}

template <int KT, int G>
__device__ __forceinline__ void ang_cgrad_thread(const DevSpec &sp, LaneSum<KT> &ls, const float *AL, int nthr, int ng, int a, bool act,
                                                 const float *__restrict__ A1g) {
  const float *A1a = A1g + ((size_t)a * ng + G) * sp.T * KT * ANG_GS;
  const float *al_t = AL + threadIdx.x;                         // alpha slots of this thread: AL[(n*6 + i) * nthr + tid]
  float *accw_I = ls.accw;
  constexpr int NPC = LaneSum<KT>::NPC;
  for (int J = 0; J < sp.T; ++J) {
    float a1[KT * ANG_GS];
    if (act) ld_block<KT * ANG_GS / 8>(A1a + (size_t)J * KT * ANG_GS, a1);
    else {
#pragma unroll
      for (int x = 0; x < KT * ANG_GS; ++x) a1[x] = 0.f;
    }
    ls.accw = accw_I + J * sp.NA * KT;
    for (int ch = 0; ch * NPC < sp.NA; ++ch) {
#pragma unroll
      for (int nn = 0; nn < NPC; ++nn) {
        const int n = ch * NPC + nn;
        float g[KT];
#pragma unroll
        for (int k = 0; k < KT; ++k) g[k] = 0.f;
        if (n < sp.NA) {
          float al[ANG_GS];
#pragma unroll
          for (int i = 0; i < ANG_GS; ++i) al[i] = al_t[(n * ANG_GS + i) * nthr];
#pragma unroll
          for (int k = 0; k < KT; ++k)
#pragma unroll
            for (int i = 0; i < ANG_GS; ++i) g[k] = fmaf(al[i], a1[k * ANG_GS + i], g[k]);
        }
        ls.put(nn, g);
      }
      ls.flush(ch, sp.NA * KT);
    }
  }
  ls.accw = accw_I;
}

// shared-memory floats of k_cgrad_angular: alpha slots [NA*6][threads] | E' and gbar rows 2 x [32][nqa|1] | per-warp scratch
// | per-warp accumulators | atom ids
__host__ __device__ inline int ang_cgrad_smem_floats(int T, int NA, int KT, int nwarps, int nqa) {
  return NA * ANG_GS * 32 * nwarps + 2 * ANG_TILE * (nqa | 1) + nwarps * 32 * 33 + nwarps * T * T * NA * KT + ANG_TILE;
}

template <int KT, int LMAX>
__global__ void __launch_bounds__(32 * ang_groups(LMAX), LMAX <= 4 ? 4 : 1)
k_cgrad_angular(DevSpec sp, int n_tiles, const int *__restrict__ tiles, const int *__restrict__ type_s,
                const float *__restrict__ Ep, const float *__restrict__ gbar, const float *__restrict__ S,
                const float *__restrict__ Tn, const float *__restrict__ A1g, float *__restrict__ partial) {
  extern __shared__ __align__(128) float smem[];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nthr = blockDim.x, ng = nthr >> 5;
  const int nv = sp.NA * KT, nacc = sp.T * sp.T * nv;
  const int nqa = sp.Ndes - sp.NR, qst = nqa | 1;
  float *AL = smem;                                             // [NA*6][threads]
  float *EG = AL + sp.NA * ANG_GS * nthr;                       // E' rows [32][qst], gbar rows [32][qst]
  float *scr = EG + 2 * ANG_TILE * qst + w * 32 * 33;
  float *accw = EG + 2 * ANG_TILE * qst + ng * 32 * 33 + w * nacc;
  int *at = (int *)(EG + 2 * ANG_TILE * qst + ng * 32 * 33 + ng * nacc);
  for (int o = lane; o < nacc; o += 32) accw[o] = 0.f;
  for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
    const int a = tiles[tile * ANG_TILE + lane];
    const int a0 = tiles[tile * ANG_TILE];
    __syncthreads();                                            // the previous tile's alpha slots and rows are no longer read
    if (w == 0) at[lane] = a;
    __syncthreads();
    for (int x = threadIdx.x; x < ANG_TILE * nqa; x += nthr) {  // stage the angular parts of the E' and gbar rows
      const int al = x / nqa, v = x - al * nqa, aa = at[al];
      EG[al * qst + v] = aa >= 0 ? Ep[(size_t)aa * sp.Ndes + sp.NR + v] : 0.f;
      EG[(ANG_TILE + al) * qst + v] = aa >= 0 ? gbar[(size_t)aa * sp.Ndes + sp.NR + v] : 0.f;
    }
    __syncthreads();
    const bool act = a >= 0;
    if (act)
      for (int n = w; n < sp.NA; n += ng) {                     // alpha row of (atom, n) -> the slot owners' shared slots
        float s[LMAX * (LMAX + 2)], t[LMAX * (LMAX + 2)], al[LMAX * (LMAX + 2)];
        const size_t row = ((size_t)a * sp.NA + n) * sp.nlmS;
        load_row_lm<LMAX>(S + row, s);
        load_row_lm<LMAX>(Tn + row, t);
        alpha_row<LMAX>(sp, s, t, EG + lane * qst, EG + (ANG_TILE + lane) * qst, n, al);
#pragma unroll
        for (int lm = 0; lm < LMAX * (LMAX + 2); ++lm)
          if (lm / ANG_GS < ng) AL[(n * ANG_GS + lm % ANG_GS) * nthr + (lm / ANG_GS) * 32 + lane] = al[lm];
      }
    __syncthreads();
    const int I = type_s[a0];
    LaneSum<KT> ls{scr, accw + I * sp.T * nv, lane};
    ANG_GROUP_SWITCH(LMAX, w, (ang_cgrad_thread<KT, G>(sp, ls, AL, nthr, ng, act ? a : a0, act, A1g)));
  }
  __syncwarp();
  float *dst = partial + (size_t)(blockIdx.x * ng + w) * nacc;
  for (int o = lane; o < nacc; o += 32) dst[o] = accw[o];
}
