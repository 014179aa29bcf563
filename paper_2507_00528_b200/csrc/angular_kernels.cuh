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
// Memory traffic of the tile kernels.  A load or store whose 32 lanes touch 32 different lines costs one L1 wavefront
// (about two cycles) per lane whatever its width, and a thread-per-atom kernel that does its own global accesses is bound
// by exactly that.  So the tile kernels move data COOPERATIVELY: consecutive lanes take consecutive 32-byte pieces of
// one atom's rows (S, T, beta: [a][n][nlmS] row-major; q, D, E', gbar: the atom's descriptor row), and the data meets
// the per-thread view in shared memory "slot arrays"  X[(n*6 + i) * SST + G*32 + al],  SST = threads + 1:
//   - the owner thread (atom al, slot group G) reads / updates its 6 slots of every n without bank conflicts,
//   - one thread per (atom, n) gathers a whole (l,m) row across the groups without bank conflicts,
//   - the cooperative copies (lanes along an atom's rows) see only occasional two-way conflicts.
// Pair records are read once per pair (not once per slot group): phase 1 evaluates the radial basis, the unit vector
// and the pair adjoint for a chunk of ANG_PC pairs per atom into shared memory, phase 2 (the slot-group threads) adds
// the harmonics of its group and the K x 6 outer products.  Only the A1 moment blocks, which their own thread reads
// back in k_cgrad_angular, stay thread-private in global memory: A1g[a][G][J][k][6], 256-bit accesses.
// ------------------------------------------------------------------------------------------------
#define ANG_PC 8          // pairs per atom per staged chunk

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
template <int LMAX>
__device__ __forceinline__ void load_row_lm(const float *__restrict__ row, float (&s)[LMAX * (LMAX + 2)]) {
  ld_block<LMAX * (LMAX + 2) / 8>(row, s);
}

// per-tile bookkeeping in shared memory: atom ids (-1 = idle lane), species-segment bounds of each atom's angular row,
// longest segment of the tile per neighbour species
struct TileInfo {
  int at[ANG_TILE];
  int seg[ANG_TILE][GNEP_MAX_SPECIES_C + 1];
  int maxlen[GNEP_MAX_SPECIES_C];
};
// called by every thread; the caller synchronises the CTA afterwards
__device__ __forceinline__ void tile_setup(TileInfo *ti, const DevSpec &sp, const int *__restrict__ tiles, int tile,
                                           const int *__restrict__ segA) {
  if (threadIdx.x < 32) {
    const int lane = threadIdx.x, a = tiles[tile * ANG_TILE + lane];
    ti->at[lane] = a;
    int prev = a >= 0 ? segA[(size_t)a * (sp.T + 1)] : 0;
    ti->seg[lane][0] = prev;
    for (int J = 0; J < sp.T; ++J) {
      const int e = a >= 0 ? segA[(size_t)a * (sp.T + 1) + J + 1] : 0;
      ti->seg[lane][J + 1] = e;
      int m = e - prev;
      prev = e;
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) m = max(m, __shfl_xor_sync(0xffffffffu, m, o));
      if (lane == 0) ti->maxlen[J] = m;
    }
  }
}

// slot of (n, lm) of atom al in a slot array; the stride SST = 32 * ang_groups(LMAX) + 1 is a compile-time constant (also
// for models with l_max < LMAX, which simply leave the upper groups' slots unused), so that slot offsets are immediates
template <int LMAX> struct AngDims {
  static constexpr int NG = ang_groups(LMAX), NTH = 32 * NG, SST = NTH + 1, NLM = LMAX * (LMAX + 2), NS = LMAX <= 4 ? 24 : 88;
};
__host__ __device__ constexpr int ang_sst(int lmax) { return 32 * ang_groups(lmax) + 1; }
__device__ __forceinline__ int slot_of(int n, int lm, int sst, int al) { return (n * ANG_GS + lm % ANG_GS) * sst + (lm / ANG_GS) * 32 + al; }

// cooperative global -> slot array: the tile's rows g[a][n][NS] (NA*NS floats per atom); lanes run along an atom's rows,
// 32 bytes each.  A piece is 8 consecutive slots of one row, so its slot offsets from the row's base are immediates.
template <int LMAX, int PART>
__device__ __forceinline__ void piece_to_slots(float *Xn, const float8 &v8, int ng) {
  constexpr int SST = AngDims<LMAX>::SST;
  const float v[8] = {v8.lo.x, v8.lo.y, v8.lo.z, v8.lo.w, v8.hi.x, v8.hi.y, v8.hi.z, v8.hi.w};
#pragma unroll
  for (int e = 0; e < 8; ++e) {
    constexpr int dummy = 0; (void)dummy;
    const int lm = 8 * PART + e;
    if (lm < AngDims<LMAX>::NG * ANG_GS && lm / ANG_GS < ng) Xn[(lm % ANG_GS) * SST + (lm / ANG_GS) * 32] = v[e];
  }
}
template <int LMAX, int PART>
__device__ __forceinline__ void slots_to_piece(const float *Xn, float (&v)[8], int ng) {
  constexpr int SST = AngDims<LMAX>::SST;
#pragma unroll
  for (int e = 0; e < 8; ++e) {
    const int lm = 8 * PART + e;
    v[e] = (lm < AngDims<LMAX>::NG * ANG_GS && lm / ANG_GS < ng) ? Xn[(lm % ANG_GS) * SST + (lm / ANG_GS) * 32] : 0.f;
  }
}
#define ANG_PART_CASE(LMAX, pt, CALL) case pt: if constexpr (AngDims<LMAX>::NS / 8 > pt) { constexpr int PART = pt; CALL; } break;
#define ANG_PART_SWITCH(LMAX, part, CALL)                                                                       \
  switch (part) {                                                                                               \
    ANG_PART_CASE(LMAX, 0, CALL) ANG_PART_CASE(LMAX, 1, CALL) ANG_PART_CASE(LMAX, 2, CALL) ANG_PART_CASE(LMAX, 3, CALL)   \
    ANG_PART_CASE(LMAX, 4, CALL) ANG_PART_CASE(LMAX, 5, CALL) ANG_PART_CASE(LMAX, 6, CALL) ANG_PART_CASE(LMAX, 7, CALL)   \
    ANG_PART_CASE(LMAX, 8, CALL) ANG_PART_CASE(LMAX, 9, CALL) ANG_PART_CASE(LMAX, 10, CALL)                               \
    default: break;                                                                                             \
  }
template <int LMAX>
__device__ __forceinline__ void coop_load_rows(const DevSpec &sp, const TileInfo *ti, const float *__restrict__ g, float *X, int ng) {
  constexpr int NS = AngDims<LMAX>::NS, P8 = NS / 8, SST = AngDims<LMAX>::SST;
  const int len8 = sp.NA * P8;
  for (int x = threadIdx.x; x < ANG_TILE * len8; x += blockDim.x) {
    const int al = x / len8, c8 = x - al * len8, a = ti->at[al];
    if (a < 0) continue;
    const int n = c8 / P8, part = c8 - n * P8;
    const float8 v8 = ldg256(g + (size_t)a * sp.NA * NS + 8 * c8);
    float *Xn = X + n * ANG_GS * SST + al;
    ANG_PART_SWITCH(LMAX, part, (piece_to_slots<LMAX, PART>(Xn, v8, ng)));
  }
}
// cooperative slot array -> global rows (slots of groups that do not exist are written as zero)
template <int LMAX>
__device__ __forceinline__ void coop_store_rows(const DevSpec &sp, const TileInfo *ti, const float *X, int ng, float *__restrict__ g) {
  constexpr int NS = AngDims<LMAX>::NS, P8 = NS / 8, SST = AngDims<LMAX>::SST;
  const int len8 = sp.NA * P8;
  for (int x = threadIdx.x; x < ANG_TILE * len8; x += blockDim.x) {
    const int al = x / len8, c8 = x - al * len8, a = ti->at[al];
    if (a < 0) continue;
    const int n = c8 / P8, part = c8 - n * P8;
    const float *Xn = X + n * ANG_GS * SST + al;
    float v[8];
    ANG_PART_SWITCH(LMAX, part, (slots_to_piece<LMAX, PART>(Xn, v, ng)));
    stg256(g + (size_t)a * sp.NA * NS + 8 * c8, make_float4(v[0], v[1], v[2], v[3]), make_float4(v[4], v[5], v[6], v[7]));
  }
}
// one (atom, n) row gathered from a slot array
template <int LMAX>
__device__ __forceinline__ void gather_row(const float *X, int n, int ng, int al, float (&s)[LMAX * (LMAX + 2)]) {
  constexpr int SST = AngDims<LMAX>::SST;
  const float *Xn = X + n * ANG_GS * SST + al;
#pragma unroll
  for (int lm = 0; lm < LMAX * (LMAX + 2); ++lm) s[lm] = lm / ANG_GS < ng ? Xn[(lm % ANG_GS) * SST + (lm / ANG_GS) * 32] : 0.f;
}

// the harmonics of slot group G of a unit vector: B[i] = B_lm, lm = 6G + i (and, with the pair adjoint (ax,ay,az), ar =
// a.rhat: Y[i] = grad B_lm . a = ((grad b_lm).a - l b_lm ar) / d).  G is warp-uniform; the unused harmonics of every
// case are removed at compile time.
template <int LMAX, int G>
__device__ __forceinline__ void harm_case(float hx, float hy, float hz, float (&B)[ANG_GS]) {
  blm_unit<LMAX>(hx, hy, hz, [&](int lm, int, float b, float, float, float) {
    if (lm >= G * ANG_GS && lm < (G + 1) * ANG_GS) B[lm - G * ANG_GS] = b;
  });
}
template <int LMAX, int G>
__device__ __forceinline__ void harm_case(float hx, float hy, float hz, float rinv, float ax, float ay, float az, float ar,
                                          float (&X)[ANG_GS], float (&Y)[ANG_GS]) {
  blm_unit<LMAX>(hx, hy, hz, [&](int lm, int l, float b, float gx, float gy, float gz) {
    if (lm >= G * ANG_GS && lm < (G + 1) * ANG_GS) {
      X[lm - G * ANG_GS] = b;
      Y[lm - G * ANG_GS] = rinv * ((gx * ax + gy * ay + gz * az) - (float)l * b * ar);
    }
  });
}
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
__device__ __forceinline__ void copy_out_rows(const DevSpec &sp, const TileInfo *ti, const float *rows, int stride, float *__restrict__ dst) {
  const int nqa = sp.Ndes - sp.NR;
  for (int x = threadIdx.x; x < ANG_TILE * nqa; x += blockDim.x) {
    const int al = x / nqa, v = x - al * nqa, a = ti->at[al];
    if (a >= 0) dst[(size_t)a * sp.Ndes + sp.NR + v] = rows[al * stride + v];
  }
}
// X[n] (+)= c[I][J][n][.] . acc[.][6]: the thread-local contraction of a finished species segment into the thread's slots
template <int KT, int SST>
__device__ __forceinline__ void contract_segment(const DevSpec &sp, const float *c, const float (&acc)[KT * ANG_GS], float *x_t, bool first) {
  for (int n = 0; n < sp.NA; ++n, x_t += ANG_GS * SST, c += KT) {
    float s[ANG_GS];
#pragma unroll
    for (int i = 0; i < ANG_GS; ++i) s[i] = first ? 0.f : x_t[i * SST];
#pragma unroll
    for (int k4 = 0; k4 < KT; k4 += 4) {
      const float4 c4 = *(const float4 *)(c + k4);
      const float cv[4] = {c4.x, c4.y, c4.z, c4.w};
#pragma unroll
      for (int kk = 0; kk < 4; ++kk)
#pragma unroll
        for (int i = 0; i < ANG_GS; ++i) s[i] = fmaf(cv[kk], acc[(k4 + kk) * ANG_GS + i], s[i]);
    }
#pragma unroll
    for (int i = 0; i < ANG_GS; ++i) x_t[i * SST] = s[i];
  }
}

// ------------------------------------------------------------------------------------------------
// a1 (angular): A1 moments, S_nlm (Eq.8), q_nl (Eq.7), many-body terms (R14, R41)
// ------------------------------------------------------------------------------------------------
// shared-memory floats: coefficients | S slots [NA*6][SST] | descriptor rows [32][nqa|1] | pair stage 2 x [PC][32][KT+4] | TileInfo
__host__ __device__ inline int ang_fwd_smem_floats(int T, int NA, int KT, int lmax, int nqa) {
  return ((T * T * NA * KT + 3) & ~3) + ((NA * ANG_GS * ang_sst(lmax) + 3) & ~3) + ((ANG_TILE * (nqa | 1) + 3) & ~3) +
         2 * ANG_PC * 32 * (KT + 4) + (int)(sizeof(TileInfo) / 4);
}

template <int KT, int LMAX>
__global__ void __launch_bounds__(32 * ang_groups(LMAX), LMAX <= 4 ? 3 : 1)
k_angular_fwd(DevSpec sp, int n_tiles, const int *__restrict__ tiles, const int *__restrict__ type_s,
              const int *__restrict__ segA, const float4 *__restrict__ pairA, const float *__restrict__ theta,
              float *__restrict__ q, float *__restrict__ S, float *__restrict__ A1g) {
  extern __shared__ __align__(128) float smem[];
  constexpr int SST = AngDims<LMAX>::SST, NF4 = KT / 4 + 1, PSZ = ANG_PC * 32 * NF4;
  // the CTA always has ang_groups(LMAX) warps; those beyond the model's ng slot groups (l_max < LMAX) only help with phase 1
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5, ng = ang_groups(sp.L);
  const bool grp = w < ng;
  const int nqa = sp.Ndes - sp.NR, qst = nqa | 1;
  float *cs = smem;                                             // [T*T*NA][KT]
  float *Sst = cs + ((sp.T * sp.T * sp.NA * KT + 3) & ~3);      // S slots
  float *QS = Sst + ((sp.NA * ANG_GS * SST + 3) & ~3);          // [32][qst]
  float4 *PS = (float4 *)(QS + ((ANG_TILE * qst + 3) & ~3));    // 2 x [KT/4 + 1][PC][32]: f_k, then (hx, hy, hz, -)
  TileInfo *ti = (TileInfo *)(PS + 2 * PSZ);
  stage_coeff(cs, theta + sp.offA, sp.T * sp.T * sp.NA, sp.KA, KT);
  tile_setup(ti, sp, tiles, blockIdx.x, segA);
  __syncthreads();
  const int a = ti->at[lane];
  const int I = type_s[ti->at[0]];
  float *s_t = Sst + threadIdx.x;
  float *A1a = A1g + ((size_t)max(a, 0) * ng + w) * sp.T * KT * ANG_GS;
  int buf = 0;
  for (int J = 0; J < sp.T; ++J) {
    float acc[KT * ANG_GS];
#pragma unroll
    for (int x = 0; x < KT * ANG_GS; ++x) acc[x] = 0.f;
    const int lo = ti->seg[lane][J], len = ti->seg[lane][J + 1] - lo, mlen = ti->maxlen[J];
    for (int c0 = 0; c0 < mlen; c0 += ANG_PC, buf ^= 1) {
      float4 *ps = PS + buf * PSZ + lane;
      // phase 1: radial basis and unit vector, once per pair (warp w takes the pairs w, w + ng, ... of the chunk).  The
      // stage is double-buffered: the barrier below also orders this chunk's writes after everybody's reads of the chunk
      // before the previous one.
      for (int p = w; p < ANG_PC; p += nw)
        if (c0 + p < len) {
          const float4 r = pairA[lo + c0 + p];
          float d, rinv, f[KT];
          pair_len(r.x * r.x + r.y * r.y + r.z * r.z, d, rinv);
          cheb_f<KT>(d, sp.rcAinv, f);
#pragma unroll
          for (int k4 = 0; k4 < KT / 4; ++k4) ps[(k4 * ANG_PC + p) * 32] = make_float4(f[4 * k4], f[4 * k4 + 1], f[4 * k4 + 2], f[4 * k4 + 3]);
          ps[((KT / 4) * ANG_PC + p) * 32] = make_float4(r.x * rinv, r.y * rinv, r.z * rinv, 0.f);
        }
      __syncthreads();
      const int np = grp ? min(ANG_PC, len - c0) : 0;           // phase 2: harmonics of this group, K x 6 outer products
      const float4 *pp = ps;
      for (int p = 0; p < np; ++p, pp += 32) {
        float f[KT], B[ANG_GS];
#pragma unroll
        for (int k4 = 0; k4 < KT / 4; ++k4) {
          const float4 f4 = pp[k4 * ANG_PC * 32];
          f[4 * k4] = f4.x; f[4 * k4 + 1] = f4.y; f[4 * k4 + 2] = f4.z; f[4 * k4 + 3] = f4.w;
        }
        const float4 h = pp[(KT / 4) * ANG_PC * 32];
#pragma unroll
        for (int i = 0; i < ANG_GS; ++i) B[i] = 0.f;
        ANG_GROUP_SWITCH(LMAX, w, (harm_case<LMAX, G>(h.x, h.y, h.z, B)));
#pragma unroll
        for (int k = 0; k < KT; ++k)
#pragma unroll
          for (int i = 0; i < ANG_GS; ++i) acc[k * ANG_GS + i] = fmaf(f[k], B[i], acc[k * ANG_GS + i]);
      }
    }
    if (a >= 0 && grp) {
      st_block<KT * ANG_GS / 8>(A1a + (size_t)J * KT * ANG_GS, acc);
      contract_segment<KT, SST>(sp, cs + (size_t)(I * sp.T + J) * sp.NA * KT, acc, s_t, J == 0);
    }
  }
  __syncthreads();                                              // the S rows of the tile are complete in the slot array
  if (a >= 0)
    for (int n = w; n < sp.NA; n += nw) {
      float s[LMAX * (LMAX + 2)];
      gather_row<LMAX>(Sst, n, ng, lane, s);
      finish_q<LMAX>(sp, s, QS + lane * qst, n);
    }
  coop_store_rows<LMAX>(sp, ti, Sst, ng, S);
  __syncthreads();
  copy_out_rows(sp, ti, QS, qst, q);
}

// ------------------------------------------------------------------------------------------------
// a5 (angular) + the beta half of a7: A2 moments with the pair adjoint a_ij, T_nlm = c.A2, D_(n,l), D_4, D_5, and
// dL/dcA[I][J][n][k] += sum_lm beta_nlm A2[J][k][lm]  (beta = E' dq/dS was written by k_angular_force)
// ------------------------------------------------------------------------------------------------
#define ANG_PCA 4         // pairs per atom per staged chunk of the adjoint sweep (its stage holds 2K+8 floats per pair)

// shared-memory floats: coefficients | T slots | beta slots (S slots for the finishing step) | D rows [32][nqa|1] | pair stage
// 2 x [PCA][32][2KT+8] | per-warp scratch [32][33] | per-warp accumulators [T*T][NA*KT] | TileInfo
__host__ __device__ inline int ang_adj_smem_floats(int T, int NA, int KT, int lmax, int nqa) {
  const int nwarps = ang_groups(lmax);
  return ((T * T * NA * KT + 3) & ~3) + 2 * ((NA * ANG_GS * ang_sst(lmax) + 3) & ~3) + ((ANG_TILE * (nqa | 1) + 3) & ~3) +
         2 * ANG_PCA * 32 * (2 * KT + 8) + nwarps * 32 * 33 + ((nwarps * T * T * NA * KT + 3) & ~3) + (int)(sizeof(TileInfo) / 4);
}

template <int KT, int LMAX>
__global__ void __launch_bounds__(32 * ang_groups(LMAX), LMAX <= 4 ? 2 : 1)
k_angular_adj(DevSpec sp, int n_tiles, const int *__restrict__ tiles, const int *__restrict__ type_s,
              const int *__restrict__ struct_s, const int *__restrict__ segA, const float4 *__restrict__ pairA,
              const float *__restrict__ theta, const float4 *__restrict__ u, const float *__restrict__ omega,
              const float *__restrict__ scales, const float *__restrict__ S, const float *__restrict__ Beta,
              float *__restrict__ Tn, float *__restrict__ D, float *__restrict__ partial) {
  extern __shared__ __align__(128) float smem[];
  constexpr int SST = AngDims<LMAX>::SST, NGM = AngDims<LMAX>::NG, NF4 = KT / 2 + 2, PSZ = ANG_PCA * 32 * NF4;
  constexpr int PPT = (ANG_PCA + NGM - 1) / NGM;                 // pairs per thread and chunk in phase 1 (1 with 4 or more warps)
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5, ng = ang_groups(sp.L);   // nw == NGM
  const bool grp = w < ng;
  const int ncs = (sp.T * sp.T * sp.NA * KT + 3) & ~3, nv = sp.NA * KT, nacc = sp.T * sp.T * nv;
  const int nqa = sp.Ndes - sp.NR, qst = nqa | 1, nslot = (sp.NA * ANG_GS * SST + 3) & ~3;
  float *cs = smem;
  float *Tst = cs + ncs;
  float *Bst = Tst + nslot;
  float *DS = Bst + nslot;
  float4 *PS = (float4 *)(DS + ((ANG_TILE * qst + 3) & ~3));    // 2 x [2 KT/4 + 2][PCA][32]: f_k' (a.rhat), f_k, (rhat, 1/d), (a, a.rhat)
  float *scr = (float *)(PS + 2 * PSZ) + w * 32 * 33;
  float *accw = (float *)(PS + 2 * PSZ) + NGM * 32 * 33 + w * nacc;
  TileInfo *ti = (TileInfo *)((float *)(PS + 2 * PSZ) + NGM * 32 * 33 + ((NGM * nacc + 3) & ~3));
  stage_coeff(cs, theta + sp.offA, sp.T * sp.T * sp.NA, sp.KA, KT);
  for (int o = lane; o < nacc; o += 32) accw[o] = 0.f;
  const float sfF = scales[1], svV = scales[2];
  int buf = 0;
  for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
    __syncthreads();                                            // the previous tile is done with every shared array
    tile_setup(ti, sp, tiles, tile, segA);
    __syncthreads();
    const int a = ti->at[lane];
    const bool act = a >= 0;
    const int I = type_s[ti->at[0]];
    // Phase 1 of a chunk belongs to warp w for the pairs w, w + ng, ... < PCA of every atom (lane).  Their records and the
    // gathered u_j are requested one chunk ahead (the first chunk of the next species segment before the flush of the
    // current one), so that no global latency is exposed in the chunk loop.
    float4 rq[PPT], uq[PPT];
    auto request = [&](int J, int c0) {
#pragma unroll
      for (int t = 0; t < PPT; ++t) {
        const int p = w + t * nw;
        const bool on = J < sp.T && p < ANG_PCA && c0 + p < ti->seg[lane][J + 1] - ti->seg[lane][J];
        rq[t] = on ? pairA[ti->seg[lane][J] + c0 + p] : make_float4(1.f, 0.f, 0.f, __int_as_float(max(a, 0)));
        uq[t] = u[__float_as_int(rq[t].w)];
      }
    };
    int Jn = 0;                                                 // first species segment that has pairs in this tile
    while (Jn < sp.T && ti->maxlen[Jn] == 0) ++Jn;
    request(Jn, 0);
    coop_load_rows<LMAX>(sp, ti, Beta, Bst, ng);                // (visible after the first chunk barrier / the flush barrier)
    // this lane's atom: adjoint seed u_i and the structure's omega, used by phase 1
    float4 ui = make_float4(0.f, 0.f, 0.f, 0.f);
    float om[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
    if (act) {
      ui = u[a];
      const float *o6 = omega + (size_t)struct_s[a] * 6;
#pragma unroll
      for (int c = 0; c < 6; ++c) om[c] = svV * o6[c];
    }
    float *t_t = Tst + threadIdx.x;
    const float *b_t = Bst + threadIdx.x;
    LaneSum<KT> ls{scr, accw, lane};
    for (int J = 0; J < sp.T; ++J) {
      float acc[KT * ANG_GS];
#pragma unroll
      for (int x = 0; x < KT * ANG_GS; ++x) acc[x] = 0.f;
      const int len = ti->seg[lane][J + 1] - ti->seg[lane][J], mlen = ti->maxlen[J];
      for (int c0 = 0; c0 < mlen; c0 += ANG_PCA, buf ^= 1) {
        float4 *ps = PS + buf * PSZ + lane;
#pragma unroll
        for (int t = 0; t < PPT; ++t) {                         // phase 1: one record, one gather, one basis evaluation per pair
          const int p = w + t * nw;
          if (p < ANG_PCA && c0 + p < len) {
            const float4 r = rq[t], uj = uq[t];
            float d, rinv, f[KT], fp[KT];
            pair_len(r.x * r.x + r.y * r.y + r.z * r.z, d, rinv);
            const float ax = sfF * (ui.x - uj.x) - (om[0] * r.x + om[5] * r.z);
            const float ay = sfF * (ui.y - uj.y) - (om[1] * r.y + om[3] * r.x);
            const float az = sfF * (ui.z - uj.z) - (om[2] * r.z + om[4] * r.y);
            const float hx = r.x * rinv, hy = r.y * rinv, hz = r.z * rinv;
            const float ar = ax * hx + ay * hy + az * hz;
            cheb_ffp<KT>(d, sp.rcAinv, f, fp);
#pragma unroll
            for (int k4 = 0; k4 < KT / 4; ++k4) {
              ps[(k4 * ANG_PCA + p) * 32] = make_float4(fp[4 * k4] * ar, fp[4 * k4 + 1] * ar, fp[4 * k4 + 2] * ar, fp[4 * k4 + 3] * ar);
              ps[((KT / 4 + k4) * ANG_PCA + p) * 32] = make_float4(f[4 * k4], f[4 * k4 + 1], f[4 * k4 + 2], f[4 * k4 + 3]);
            }
            ps[((KT / 2) * ANG_PCA + p) * 32] = make_float4(hx, hy, hz, rinv);
            ps[((KT / 2 + 1) * ANG_PCA + p) * 32] = make_float4(ax, ay, az, ar);
          }
        }
        if (c0 + ANG_PCA < mlen) request(J, c0 + ANG_PCA);      // next chunk of this segment, or the next segment's first
        else {
          Jn = J + 1;
          while (Jn < sp.T && ti->maxlen[Jn] == 0) ++Jn;
          request(Jn, 0);
        }
        __syncthreads();
        const int np = grp ? min(ANG_PCA, len - c0) : 0;
        const float4 *pp = ps;
        for (int p = 0; p < np; ++p, pp += 32) {                // phase 2
          float f1[KT], f2[KT], X[ANG_GS], Y[ANG_GS];
#pragma unroll
          for (int k4 = 0; k4 < KT / 4; ++k4) {
            const float4 u4 = pp[k4 * ANG_PCA * 32], v4 = pp[(KT / 4 + k4) * ANG_PCA * 32];
            f1[4 * k4] = u4.x; f1[4 * k4 + 1] = u4.y; f1[4 * k4 + 2] = u4.z; f1[4 * k4 + 3] = u4.w;
            f2[4 * k4] = v4.x; f2[4 * k4 + 1] = v4.y; f2[4 * k4 + 2] = v4.z; f2[4 * k4 + 3] = v4.w;
          }
          const float4 h = pp[(KT / 2) * ANG_PCA * 32], av = pp[(KT / 2 + 1) * ANG_PCA * 32];
#pragma unroll
          for (int i = 0; i < ANG_GS; ++i) { X[i] = 0.f; Y[i] = 0.f; }
          ANG_GROUP_SWITCH(LMAX, w, (harm_case<LMAX, G>(h.x, h.y, h.z, h.w, av.x, av.y, av.z, av.w, X, Y)));
#pragma unroll
          for (int k = 0; k < KT; ++k)
#pragma unroll
            for (int i = 0; i < ANG_GS; ++i) acc[k * ANG_GS + i] = fmaf(f1[k], X[i], fmaf(f2[k], Y[i], acc[k * ANG_GS + i]));
        }
      }
      if (J == 0) __syncthreads();                              // beta slots are loaded (also when the first segment is empty)
      if (!grp) continue;
      if (act) contract_segment<KT, SST>(sp, cs + (size_t)(I * sp.T + J) * sp.NA * KT, acc, t_t, J == 0);
      // dL/dcA[I][J][n][k] += sum_{lm in group} beta_nlm A2[J][k][lm], summed over the 32 atoms of the warp
      ls.accw = accw + (I * sp.T + J) * nv;
      constexpr int NPC = LaneSum<KT>::NPC;
      const float *bn = b_t;
      for (int ch = 0; ch * NPC < sp.NA; ++ch) {
#pragma unroll
        for (int nn = 0; nn < NPC; ++nn, bn += ANG_GS * SST) {
          const int n = ch * NPC + nn;
          float g[KT];
#pragma unroll
          for (int k = 0; k < KT; ++k) g[k] = 0.f;
          if (act && n < sp.NA) {
            float be[ANG_GS];
#pragma unroll
            for (int i = 0; i < ANG_GS; ++i) be[i] = bn[i * SST];
#pragma unroll
            for (int k = 0; k < KT; ++k)
#pragma unroll
              for (int i = 0; i < ANG_GS; ++i) g[k] = fmaf(be[i], acc[k * ANG_GS + i], g[k]);
          }
          ls.put(nn, g);
        }
        ls.flush(ch, nv);
      }
    }
    __syncthreads();                                            // T slots complete, beta slots no longer needed
    coop_load_rows<LMAX>(sp, ti, S, Bst, ng);                   // S rows for D = sum_m 2C S T
    __syncthreads();
    if (act)
      for (int n = w; n < sp.NA; n += nw) {
        float s[LMAX * (LMAX + 2)], t[LMAX * (LMAX + 2)];
        gather_row<LMAX>(Bst, n, ng, lane, s);
        gather_row<LMAX>(Tst, n, ng, lane, t);
        finish_D<LMAX>(sp, s, t, DS + lane * qst, n);
      }
    coop_store_rows<LMAX>(sp, ti, Tst, ng, Tn);
    __syncthreads();
    copy_out_rows(sp, ti, DS, qst, D);
  }
  __syncwarp();
  float *dst = partial + (size_t)(blockIdx.x * nw + w) * nacc;
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
  constexpr int NS = LMAX <= 4 ? 24 : 88;                       // the row's padding slots are zero
#pragma unroll
  for (int v = NLM; v < NS; v += 4) *(float4 *)(out_s + v) = make_float4(0.f, 0.f, 0.f, 0.f);
}

// contribution of the harmonics lm in [LO, HI) to the pair force: gam_lm = sum_n g_n beta_nlm, gamp_lm = sum_n g_n' beta_nlm
// over that slot range, then the harmonic sweep.  LO and HI - LO are multiples of 4 (16-byte loads of the beta rows).
template <int KT, int LMAX, int LO, int HI>
__device__ __forceinline__ void force_block(const DevSpec &sp, const float *__restrict__ be, int NS, const float *__restrict__ c,
                                            const float2 (&ffp)[KT], float hx, float hy, float hz,
                                            float &sB, float &sl, float &vx, float &vy, float &vz) {
  constexpr int NB = HI - LO;
  static_assert(LO % 4 == 0 && NB % 4 == 0, "slot blocks are float4-aligned");
  // (gam, gamp) and (g_n, g_n') live in register pairs: every FMA of the two sums is one packed FP32 FMA (FFMA2) with
  // the coefficient / the beta entry as the broadcast operand -- half the issue slots of the scalar form
  float2 gg[NB];
#pragma unroll
  for (int i = 0; i < NB; ++i) gg[i] = make_float2(0.f, 0.f);
  for (int n = 0; n < sp.NA; ++n) {
    float2 g2 = make_float2(0.f, 0.f);
#pragma unroll
    for (int k = 0; k < KT; ++k) { const float cv = c[n * KT + k]; g2 = __ffma2_rn(make_float2(cv, cv), ffp[k], g2); }
#pragma unroll
    for (int v = 0; v < NB / 4; ++v) {
      const float4 b4 = *(const float4 *)(be + n * NS + LO + 4 * v);
      gg[4 * v] = __ffma2_rn(g2, make_float2(b4.x, b4.x), gg[4 * v]);
      gg[4 * v + 1] = __ffma2_rn(g2, make_float2(b4.y, b4.y), gg[4 * v + 1]);
      gg[4 * v + 2] = __ffma2_rn(g2, make_float2(b4.z, b4.z), gg[4 * v + 2]);
      gg[4 * v + 3] = __ffma2_rn(g2, make_float2(b4.w, b4.w), gg[4 * v + 3]);
    }
  }
  float2 slB = make_float2(sl, sB), vxy = make_float2(vx, vy);
  blm_unit<LMAX>(hx, hy, hz, [&](int lm, int l, float b, float gx, float gy, float gz) {
    if (lm >= LO && lm < HI) {
      const float2 g = gg[lm - LO];                                  // (gam, gamp)
      slB = __ffma2_rn(g, make_float2((float)l * b, b), slB);        // sl += l gam b,  sB += gamp b
      vxy = __ffma2_rn(make_float2(g.x, g.x), make_float2(gx, gy), vxy);
      vz = fmaf(g.x, gz, vz);
    }
  });
  sl = slB.x; sB = slB.y; vx = vxy.x; vy = vxy.y;
}

template <int KT, int LMAX>
__global__ void __launch_bounds__(FRC_WARPS * 32)
k_angular_force(DevSpec sp, int N, int ta /* atoms per warp, <= FRC_TA */, const int *__restrict__ type_s, const int *__restrict__ segA,
                const int *__restrict__ atomA, const float4 *__restrict__ pairA, const float *__restrict__ theta,
                const float *__restrict__ Ep, const float *__restrict__ S, float *__restrict__ Beta,
                float4 *__restrict__ fpair) {
  extern __shared__ __align__(128) float smem[];
  float *cs = smem;
  const int ncs = (sp.T * sp.T * sp.NA * KT + 3) & ~3;
  const int NS = sp.nlmS, nb = sp.NA * NS;
  float *beta = smem + ncs + (threadIdx.x >> 5) * FRC_TA * nb;
  stage_coeff(cs, theta + sp.offA, sp.T * sp.T * sp.NA, sp.KA, KT);
  __syncthreads();
  const int lane = threadIdx.x & 31;
  const int a_lo = (blockIdx.x * FRC_WARPS + (threadIdx.x >> 5)) * ta;
  if (a_lo >= N) return;
  const int a_hi = min(a_lo + ta, N);
  const int T1 = sp.T + 1;
  const int P_lo = segA[a_lo * T1], P_hi = segA[(a_hi - 1) * T1 + sp.T];
  // beta of the warp's atoms: one (atom, n) row per lane and round, into shared memory ...
  for (int it = lane; it < (a_hi - a_lo) * sp.NA; it += 32) {
    const int al = it / sp.NA, n = it - al * sp.NA;
    beta_row<LMAX>(sp, S + ((size_t)(a_lo + al) * sp.NA + n) * NS, Ep + (size_t)(a_lo + al) * sp.Ndes, n, beta + al * nb + n * NS);
  }
  __syncwarp();
  // ... and out to global memory, row-major like S, for the adjoint sweep (32 bytes per lane and store)
  if (Beta)                                      // (only the slot-group adjoint sweep reads it: nullptr on the warp-tile path)
    for (int it = lane; it < (a_hi - a_lo) * (nb / 8); it += 32) {
      const float4 *src = (const float4 *)(beta + 8 * it);
      stg256(Beta + (size_t)a_lo * nb + 8 * it, src[0], src[1]);
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
    float2 ffp[KT];                                  // (f_k, f_k') pairs
    cheb_ffp2<KT>(d, sp.rcAinv, ffp);
    const float *c = cs + (I * sp.T + J) * sp.NA * KT;
    const float hx = r.x * rinv, hy = r.y * rinv, hz = r.z * rinv;
    float sB = 0.f, sl = 0.f, vx = 0.f, vy = 0.f, vz = 0.f;
    force_block<KT, LMAX, 0, 24>(sp, be, NS, c, ffp, hx, hy, hz, sB, sl, vx, vy, vz);              // l = 1..4
    if constexpr (LMAX > 4) {
      if (sp.L >= 5) force_block<KT, LMAX, 24, 48>(sp, be, NS, c, ffp, hx, hy, hz, sB, sl, vx, vy, vz);   // l = 5, 6
      if (sp.L >= 7) force_block<KT, LMAX, 48, 64>(sp, be, NS, c, ffp, hx, hy, hz, sB, sl, vx, vy, vz);   // l = 7 and slot 63
      if (sp.L >= 8) force_block<KT, LMAX, 64, 80>(sp, be, NS, c, ffp, hx, hy, hz, sB, sl, vx, vy, vz);   // rest of l = 8
    }
    fpair[p] = make_float4(hx * sB + rinv * (vx - hx * sl), hy * sB + rinv * (vy - hy * sl),
                           hz * sB + rinv * (vz - hz * sl), 0.f);
  }
}

// (The gather F_i += sum_p (f_p - f_rev(p)), W_i -= sum_p r_p (x) f_p is done by k_radial_force, thread per atom.)

// ------------------------------------------------------------------------------------------------
// a7 (angular), alpha half: dL/dcA[I][J][n][k] += sum_atoms sum_lm alpha_nlm A1[J][k][lm]
//   alpha_nlm = gbar_(n,l) 2C_lm S_nlm + E'_(n,l) 2C_lm T_nlm (+ 4-body: gbar_4 k4 dP4/ds_m + E'_4 k4 (H4 T)_m, 5-body alike)
// No pair sweep (the A1 moments were stored by k_angular_fwd).  Per tile: the S, T rows and the E', gbar rows are staged in
// shared memory with coalesced loads, one thread per (atom, n) builds the alpha row, then the slot-group threads contract
// their alpha slots with their A1 block and the lane sums go to the per-warp accumulators as in the adjoint sweep.
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

// shared-memory floats of k_cgrad_angular: S slots | T slots (then alpha) | E' and gbar rows 2 x [32][nqa|1] | per-warp
// scratch | per-warp accumulators | TileInfo
__host__ __device__ inline int ang_cgrad_smem_floats(int T, int NA, int KT, int lmax, int nqa) {
  const int nwarps = ang_groups(lmax);
  return 2 * ((NA * ANG_GS * ang_sst(lmax) + 3) & ~3) + ((2 * ANG_TILE * (nqa | 1) + 3) & ~3) + nwarps * 32 * 33 +
         ((nwarps * T * T * NA * KT + 3) & ~3) + (int)(sizeof(TileInfo) / 4);
}

template <int KT, int LMAX>
__global__ void __launch_bounds__(32 * ang_groups(LMAX), LMAX <= 4 ? 2 : 1)
k_cgrad_angular(DevSpec sp, int n_tiles, const int *__restrict__ tiles, const int *__restrict__ type_s,
                const int *__restrict__ segA, const float *__restrict__ Ep, const float *__restrict__ gbar,
                const float *__restrict__ S, const float *__restrict__ Tn, const float *__restrict__ A1g,
                float *__restrict__ partial) {
  extern __shared__ __align__(128) float smem[];
  constexpr int SST = AngDims<LMAX>::SST;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nthr = blockDim.x, nw = nthr >> 5, ng = ang_groups(sp.L);
  const bool grp = w < ng;
  const int nv = sp.NA * KT, nacc = sp.T * sp.T * nv;
  const int nqa = sp.Ndes - sp.NR, qst = nqa | 1, nslot = (sp.NA * ANG_GS * SST + 3) & ~3;
  float *Sst = smem;
  float *Tst = Sst + nslot;                                     // T, then alpha
  float *EG = Tst + nslot;                                      // E' rows [32][qst], gbar rows [32][qst]
  float *scr = EG + ((2 * ANG_TILE * qst + 3) & ~3) + w * 32 * 33;
  float *accw = EG + ((2 * ANG_TILE * qst + 3) & ~3) + nw * 32 * 33 + w * nacc;
  TileInfo *ti = (TileInfo *)(EG + ((2 * ANG_TILE * qst + 3) & ~3) + nw * 32 * 33 + ((nw * nacc + 3) & ~3));
  for (int o = lane; o < nacc; o += 32) accw[o] = 0.f;
  for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
    __syncthreads();                                            // the previous tile is done with every shared array
    tile_setup(ti, sp, tiles, tile, segA);
    __syncthreads();
    const int a = ti->at[lane];
    const bool act = a >= 0;
    const int I = type_s[ti->at[0]];
    // this thread's A1 blocks are requested first: their latency hides behind the alpha rows
    const float *A1a = A1g + ((size_t)max(a, 0) * ng + w) * sp.T * KT * ANG_GS;
    coop_load_rows<LMAX>(sp, ti, S, Sst, ng);
    coop_load_rows<LMAX>(sp, ti, Tn, Tst, ng);
    for (int x = threadIdx.x; x < ANG_TILE * nqa; x += nthr) {  // the angular parts of the E' and gbar rows
      const int al = x / nqa, v = x - al * nqa, aa = ti->at[al];
      EG[al * qst + v] = aa >= 0 ? Ep[(size_t)aa * sp.Ndes + sp.NR + v] : 0.f;
      EG[(ANG_TILE + al) * qst + v] = aa >= 0 ? gbar[(size_t)aa * sp.Ndes + sp.NR + v] : 0.f;
    }
    __syncthreads();
    if (act)
      for (int n = w; n < sp.NA; n += nw) {                     // alpha row of (atom, n) overwrites the T slots of that row
        float s[LMAX * (LMAX + 2)], t[LMAX * (LMAX + 2)], al[LMAX * (LMAX + 2)];
        gather_row<LMAX>(Sst, n, ng, lane, s);
        gather_row<LMAX>(Tst, n, ng, lane, t);
        alpha_row<LMAX>(sp, s, t, EG + lane * qst, EG + (ANG_TILE + lane) * qst, n, al);
        float *Xn = Tst + n * ANG_GS * SST + lane;
#pragma unroll
        for (int lm = 0; lm < LMAX * (LMAX + 2); ++lm)
          if (lm / ANG_GS < ng) Xn[(lm % ANG_GS) * SST + (lm / ANG_GS) * 32] = al[lm];
      }
    __syncthreads();
    const float *al_t = Tst + threadIdx.x;
    LaneSum<KT> ls{scr, accw, lane};
    constexpr int NPC = LaneSum<KT>::NPC;
    for (int J = 0; J < sp.T && grp; ++J) {
      float a1[KT * ANG_GS];
      if (act) ld_block<KT * ANG_GS / 8>(A1a + (size_t)J * KT * ANG_GS, a1);
      else {
#pragma unroll
        for (int x = 0; x < KT * ANG_GS; ++x) a1[x] = 0.f;
      }
      ls.accw = accw + (I * sp.T + J) * nv;
      for (int ch = 0; ch * NPC < sp.NA; ++ch) {
#pragma unroll
        for (int nn = 0; nn < NPC; ++nn) {
          const int n = ch * NPC + nn;
          float g[KT];
#pragma unroll
          for (int k = 0; k < KT; ++k) g[k] = 0.f;
          if (act && n < sp.NA) {
            float al[ANG_GS];
#pragma unroll
            for (int i = 0; i < ANG_GS; ++i) al[i] = al_t[(n * ANG_GS + i) * SST];
#pragma unroll
            for (int k = 0; k < KT; ++k)
#pragma unroll
              for (int i = 0; i < ANG_GS; ++i) g[k] = fmaf(al[i], a1[k * ANG_GS + i], g[k]);
          }
          ls.put(nn, g);
        }
        ls.flush(ch, nv);
      }
    }
  }
  __syncwarp();
  float *dst = partial + (size_t)(blockIdx.x * nw + w) * nacc;
  for (int o = lane; o < nacc; o += 32) dst[o] = accw[o];
}
