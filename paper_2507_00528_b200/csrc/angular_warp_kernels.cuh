// angular_warp_kernels.cuh -- the angular moment sweeps for l_max <= 4 (24 (l,m) slots) in their WARP-TILE mapping
// (rows a1, a5, a7 of DESIGN.md); angular_kernels.cuh holds the slot-group mapping used for l_max up to 8 and the pair-force
// kernel shared by both.
//
// Moment form.  g_n(d) = sum_k c[I][J][n][k] f_k(d) is linear in the basis, so with
//   A1[J][k][lm] = sum_{j in J} f_k(d_ij) B_lm(rhat_ij)
//   A2[J][k][lm] = sum_{j in J} f_k'(d_ij) (a_ij.rhat_ij) B_lm + f_k(d_ij) (grad B_lm . a_ij)
// one has S_nlm = sum_{J,k} c A1 (Eq.8), T_nlm = sum_{J,k} c A2 (the summed factors of C3.9-C3.16) and
//   dL/dcA[I][J][n][k] = sum_atoms sum_lm alpha_nlm A1[J][k][lm] + beta_nlm A2[J][k][lm]   (C2.5-C2.10, C3.12-C3.20)
// so the coefficient gradient needs no pair sweep of its own.
//
// Mapping: a warp owns ANG_TA consecutive atoms; their pairs are contiguous in pairA, so phase 1 (lane = pair)
// runs on full 32-pair chunks that cross atom boundaries, and phase 2 (lane = (KT/4 k, 3 lm) register tile: the
// shape with the fewest shared-memory operand loads per FMA for 32 lanes on an 8 x 24 output) walks the
// (atom, species-segment) boundaries inside the chunk.  Shared rows have stride ANG_LD = 36 floats so that the
// LDS.128 of 8 different rows hit 8 different bank quads.
#pragma once
#include "common.cuh"
#include "pair_kernels.cuh"
#include "angular_kernels.cuh"

#define ANGW_NLM 24       // (l,m) slots, l = 1..4

#define ANG_TA 16        // atoms per warp tile (fwd / adj)
#define ANG_WARPS 4      // warps per CTA
#define ANG_LD 36        // shared-memory row stride in floats
#define ANG_NQ 16        // n padded to 16 in the transposed coefficient table
#define ANG_SEGS (ANG_TA * GNEP_MAX_SPECIES_C)   // (atom, J) segments of a warp tile

// coefficients for the S/T contractions, ct[(((I*T+J)*KT + k)*4 + q)*4 + j] = c[I][J][n = q + 4 j][k] (zero padded):
// the functions n = q, q + 4, q + 8, q + 12 owned by one lane are one 16-byte load
__device__ __forceinline__ void stage_coeff_t(float *dst, const float *src, int T, int NA, int K, int KT) {
  int tot = T * T * KT * ANG_NQ;
  for (int x = threadIdx.x; x < tot; x += blockDim.x) {
    int j = x & 3, q = (x >> 2) & 3, r = x / ANG_NQ;
    int n = q + 4 * j;
    int k = r % KT, ij = r / KT;
    dst[x] = (n < NA && k < K) ? src[(ij * NA + n) * K + k] : 0.f;
  }
}

__device__ __forceinline__ float dot4(const float4 &a, const float4 &b) { return a.x * b.x + a.y * b.y + a.z * b.z + a.w * b.w; }
// acc += a . b as one FMA chain
__device__ __forceinline__ void fma4(float &acc, const float4 &a, const float4 &b) {
  acc = fmaf(a.x, b.x, acc); acc = fmaf(a.y, b.y, acc); acc = fmaf(a.z, b.z, acc); acc = fmaf(a.w, b.w, acc);
}

// Packed FP32 FMA (sm_100 FFMA2, fma.rn.f32x2): two independent IEEE fp32 FMAs in ONE issue slot.  The sweeps are bound
// by issue slots, not by the FMA pipe, so the outer products are written on register pairs.
// (k0, k1) += F(k0, k1; pair p) x_p over the four pairs of a group; Fa = (k0p0, k1p0, k0p1, k1p1), Fb = (k0p2, ..., k1p3)
__device__ __forceinline__ void fma4x2(float &a0, float &a1, const float4 &Fa, const float4 &Fb, const float4 &X) {
  float2 t = make_float2(a0, a1);
  t = __ffma2_rn(make_float2(Fa.x, Fa.y), make_float2(X.x, X.x), t);
  t = __ffma2_rn(make_float2(Fa.z, Fa.w), make_float2(X.y, X.y), t);
  t = __ffma2_rn(make_float2(Fb.x, Fb.y), make_float2(X.z, X.z), t);
  t = __ffma2_rn(make_float2(Fb.z, Fb.w), make_float2(X.w, X.w), t);
  a0 = t.x; a1 = t.y;
}

// Per-atom lane layout "(n, lmg)": lane = 3*nq + lmg (lanes 0..29), n = nb + nq for nb = 0, 10, ..., and the lane owns
// lm in [8 lmg, 8 lmg + 8): lmg 0 = all of l=1 (i<3) and l=2; lmg 1 = all of l=3 (i<7) and the first slot of l=4;
// lmg 2 = the rest of l=4.  Everything per-atom (S, T, beta, alpha, q_nl, D_nl) is produced in this layout with static
// register indexing and 2*C_lm held in registers (no divergent constant-memory indexing in the hot loops).
struct NLane {
  int nq, lmg, la, lb, split;
  bool act;
  float c2[8];
};
__device__ __forceinline__ NLane make_nlane(int lane) {
  NLane L;
  L.nq = lane / 3; L.lmg = lane - 3 * L.nq; L.act = lane < 30;
  L.la = L.lmg == 0 ? 1 : L.lmg == 1 ? 3 : 4;
  L.lb = L.lmg == 0 ? 2 : 4;
  L.split = L.lmg == 0 ? 3 : L.lmg == 1 ? 7 : 8;
#pragma unroll
  for (int i = 0; i < 8; ++i) L.c2[i] = c_C2[8 * (L.lmg < 3 ? L.lmg : 0) + i];
  return L;
}
// sums of w[i] over the lane's two l-blocks
__device__ __forceinline__ void split_sums(const NLane &nl, const float (&w)[8], float &sa, float &sb) {
  sa = 0.f; sb = 0.f;
#pragma unroll
  for (int i = 0; i < 8; ++i) { if (i < nl.split) sa += w[i]; else sb += w[i]; }
}

// Epilogue contraction X = c . A (S = c.A1, T = c.A2) without a second pass over shared memory.  When a segment's
// register tile acc[KQ][3] (k in the lane's quarter kq, 3 lm) is complete, the four lanes (kq = 0..3) that share the
// same 3 lm exchange their tiles by shuffles, so that each holds A[all k][its 3 lm]; lane kq then owns the functions
// n = kq, kq + 4, ... and adds  Xo[j][i] += sum_k c[I][J][n_j][k] A[k][lm_i].  At the end of the atom X[n][lm] goes to
// shared memory once (Xs[n][24]) for the per-(n, l) contractions.  (Re-reading the moment matrix from shared memory for
// every n-group, or summing partial X over the k-quarters by butterflies, both cost more instructions.)
template <int KT, int KQ, int NJ>
__device__ __forceinline__ void xown_add(const DevSpec &sp, const float *ct, int I, int J, int lane, int kq,
                                         const float (&acc)[KQ][3], float (&Xo)[NJ][3]) {
#pragma unroll
  for (int d = 0; d < 4; ++d) {
    const int kb = ((kq + d) & 3) * KQ;             // first k of the tile held by lane kq + d
#pragma unroll
    for (int r = 0; r < KQ; ++r) {
      float a[3];
#pragma unroll
      for (int i = 0; i < 3; ++i) a[i] = d == 0 ? acc[r][i] : __shfl_sync(0xffffffffu, acc[r][i], (lane + 8 * d) & 31);
      if (kb + r < KT) {
        const float4 c4 = *(const float4 *)(ct + ((I * sp.T + J) * KT + kb + r) * ANG_NQ + 4 * kq);   // n = kq + 4 j
        const float cv[4] = {c4.x, c4.y, c4.z, c4.w};                                                // zero beyond NA
#pragma unroll
        for (int j = 0; j + 1 < NJ; j += 2)         // two functions n per packed FMA
#pragma unroll
          for (int i = 0; i < 3; ++i) {
            const float2 t = __ffma2_rn(make_float2(cv[j], cv[j + 1]), make_float2(a[i], a[i]), make_float2(Xo[j][i], Xo[j + 1][i]));
            Xo[j][i] = t.x; Xo[j + 1][i] = t.y;
          }
        if (NJ & 1)
#pragma unroll
          for (int i = 0; i < 3; ++i) Xo[NJ - 1][i] = fmaf(cv[NJ - 1], a[i], Xo[NJ - 1][i]);
      }
    }
  }
}
template <int NJ>
__device__ __forceinline__ void xown_store(int kq, int lmq, float (&Xo)[NJ][3], float *Xs) {
#pragma unroll
  for (int j = 0; j < NJ; ++j)
#pragma unroll
    for (int i = 0; i < 3; ++i) {
      Xs[(kq + 4 * j) * ANGW_NLM + 3 * lmq + i] = Xo[j][i];     // rows up to 4 NJ - 1 <= ANG_NQ - 1 exist
      Xo[j][i] = 0.f;
    }
  __syncwarp();
}

// ------------------------------------------------------------------------------------------------
// a1 (angular): A1 moments, S_nlm (Eq.8), q_nl = sum_m C_lm S_nlm^2 (Eq.7), 4-body (R14)
// ------------------------------------------------------------------------------------------------
template <int KT, int NQ>
__global__ void __launch_bounds__(ANG_WARPS * 32)
k_angw_fwd(DevSpec sp, int N, int ta /* atoms per warp, <= ANG_TA */, const int *__restrict__ type_s, const int *__restrict__ segA,
              const float4 *__restrict__ pairA, const float *__restrict__ theta, float *__restrict__ q,
              float *__restrict__ S, float *__restrict__ A1) {
  constexpr int KQ = (KT + 3) / 4;      // k per lane: lane = (k quarter kq, lm eighth lmq) holds a KQ x 3 register tile
  extern __shared__ __align__(128) float smem[];
  float *ct = smem;
  const int nct = sp.T * sp.T * KT * ANG_NQ;
  const int nA = sp.T * KT * ANGW_NLM;
  const int per_warp = (KT + ANGW_NLM) * ANG_LD + nA + ANG_NQ * ANGW_NLM + ANG_SEGS;
  float *sf = smem + nct + (threadIdx.x >> 5) * per_warp;   // [KT][LD]
  float *sB = sf + KT * ANG_LD;                              // [24][LD]
  float *As = sB + ANGW_NLM * ANG_LD;                        // [T][KT][24]
  float *Xs = As + nA;                                       // [NQ][24]  S of the current atom
  int *sEnd = (int *)(Xs + ANG_NQ * ANGW_NLM);               // segment ends of the tile
  stage_coeff_t(ct, theta + sp.offA, sp.T, sp.NA, sp.KA, KT);
  __syncthreads();
  const int lane = threadIdx.x & 31;
  const int a_lo = (blockIdx.x * ANG_WARPS + (threadIdx.x >> 5)) * ta;
  if (a_lo >= N) return;
  const int a_hi = min(a_lo + ta, N);
  const int T1 = sp.T + 1;
  const int P_lo = segA[a_lo * T1], P_hi = segA[(a_hi - 1) * T1 + sp.T];
  const int kq = lane >> 3, lmq = lane & 7;
  const NLane nl = make_nlane(lane);
  float acc[KQ][3];
#pragma unroll
  for (int r = 0; r < KQ; ++r)
#pragma unroll
    for (int i = 0; i < 3; ++i) acc[r][i] = 0.f;
  constexpr int NJ = (NQ + 3) / 4;
  float Xo[NJ][3];
#pragma unroll
  for (int j = 0; j < NJ; ++j)
#pragma unroll
    for (int i = 0; i < 3; ++i) Xo[j][i] = 0.f;
  for (int x = lane; x < (a_hi - a_lo) * sp.T; x += 32) sEnd[x] = segA[(a_lo + x / sp.T) * T1 + x % sp.T + 1];
  __syncwarp();
  int a = a_lo, J = 0;
  int seg_end = sEnd[0];

  int Icur = type_s[a_lo];       // species of atom a, requested when the previous atom ends
  auto next_atom = [&]() { if (a < a_hi) Icur = type_s[a]; };
  auto flush_segment = [&]() {   // accumulators of (a, J) -> S partial sums and shared As, then reset
    xown_add<KT, KQ, NJ>(sp, ct, Icur, J, lane, kq, acc, Xo);
#pragma unroll
    for (int r = 0; r < KQ; ++r) {
      int k = kq * KQ + r;
      if (k < KT) {
        int o = (J * KT + k) * ANGW_NLM + 3 * lmq;
#pragma unroll
        for (int i = 0; i < 3; ++i) { As[o + i] = acc[r][i]; acc[r][i] = 0.f; }
      }
    }
  };
  auto atom_epilogue = [&]() {   // A1 -> global, S = c.A1, q_nl, q4 of atom a
    __syncwarp();
    for (int x = lane; x < nA / 4; x += 32) ((float4 *)(A1 + (size_t)a * nA))[x] = ((const float4 *)As)[x];
    xown_store<NJ>(kq, lmq, Xo, Xs);
    float *Sa = S + (size_t)a * sp.NA * ANGW_NLM;
    float *qa = q + (size_t)a * sp.Ndes + sp.NR;
    for (int nb = 0; nb < sp.NA; nb += 10) {
      const int n = nb + nl.nq;
      const bool on = nl.act && n < sp.NA;
      float sv[8], qa_ = 0.f, qb_ = 0.f;
      if (on) {
        {
          const float4 s0 = *(const float4 *)(Xs + n * ANGW_NLM + 8 * nl.lmg), s1 = *(const float4 *)(Xs + n * ANGW_NLM + 8 * nl.lmg + 4);
          sv[0] = s0.x; sv[1] = s0.y; sv[2] = s0.z; sv[3] = s0.w; sv[4] = s1.x; sv[5] = s1.y; sv[6] = s1.z; sv[7] = s1.w;
        }
        stg256(Sa + n * ANGW_NLM + 8 * nl.lmg, make_float4(sv[0], sv[1], sv[2], sv[3]), make_float4(sv[4], sv[5], sv[6], sv[7]));
        float w[8];
#pragma unroll
        for (int i = 0; i < 8; ++i) w[i] = 0.5f * nl.c2[i] * sv[i] * sv[i];
        split_sums(nl, w, qa_, qb_);
      }
      const float nxt = __shfl_down_sync(0xffffffffu, qa_, 1);     // the l=4 remainder held by (n, lmg 2)
      if (on && nl.lmg == 0) {
        qa[n] = qa_;
        if (sp.L >= 2) qa[sp.NA + n] = qb_;
        if (sp.use4) qa[sp.NA * sp.L + n] = GNEP_KAPPA4 * p4_value(sv + 3);
        if (sp.use5) qa[sp.NA * (sp.L + sp.use4) + n] = p5_value(sv);          // R41: kappa5 |S_n,1|^4, after the 4-body block
      }
      if (on && nl.lmg == 1) {
        if (sp.L >= 3) qa[2 * sp.NA + n] = qa_;
        if (sp.L >= 4) qa[3 * sp.NA + n] = qb_ + nxt;
      }
    }
    __syncwarp();
  };
  auto next_segment = [&]() {
    flush_segment();
    if (++J == sp.T) { atom_epilogue(); J = 0; ++a; next_atom(); }
    seg_end = a < a_hi ? sEnd[(a - a_lo) * sp.T + J] : 0x7fffffff;
  };

  float4 rn = P_lo + lane < P_hi ? pairA[P_lo + lane] : make_float4(1.f, 0.f, 0.f, 0.f);
  for (int c0 = P_lo; c0 < P_hi; c0 += 32) {
    const int p = c0 + lane;
    const float4 r = rn;
    if (p + 32 < P_hi) rn = pairA[p + 32];                    // the next chunk's record is in flight during this chunk
    if (p < P_hi) {
      float d, rinv;
      pair_len(r.x * r.x + r.y * r.y + r.z * r.z, d, rinv);
      float f[KT];
      cheb_f<KT>(d, sp.rcAinv, f);
#pragma unroll
      for (int k = 0; k < KT; ++k) sf[k * ANG_LD + lane] = f[k];
      blm_unit<4>(r.x * rinv, r.y * rinv, r.z * rinv,
               [&](int lm, int, float b, float, float, float) { sB[lm * ANG_LD + lane] = b; });
    } else {   // keep masked lanes finite
#pragma unroll
      for (int k = 0; k < KT; ++k) sf[k * ANG_LD + lane] = 0.f;
#pragma unroll
      for (int lm = 0; lm < ANGW_NLM; ++lm) sB[lm * ANG_LD + lane] = 0.f;
    }
    __syncwarp();
    const int chunk_end = min(c0 + 32, P_hi);
    int pos = c0;
    while (pos < chunk_end) {
      while (seg_end <= pos) next_segment();
      const int hi = min(seg_end, chunk_end);
      // segments are multiples of 4 pairs (k_pad_angular) and so are the chunk bounds: whole 4-pair groups only
      for (int g = (pos - c0) >> 2; g < (hi - c0) >> 2; ++g) {
        float4 fv[KQ];
#pragma unroll
        for (int r = 0; r < KQ; ++r) {
          int k = kq * KQ + r;
          fv[r] = k < KT ? *(const float4 *)(sf + k * ANG_LD + 4 * g) : make_float4(0.f, 0.f, 0.f, 0.f);
        }
#pragma unroll
        for (int i = 0; i < 3; ++i) {
          float4 b = *(const float4 *)(sB + (3 * lmq + i) * ANG_LD + 4 * g);
#pragma unroll
          for (int r = 0; r < KQ; ++r) acc[r][i] += dot4(fv[r], b);
        }
      }
      pos = hi;
    }
    __syncwarp();
  }
  while (a < a_hi) next_segment();
}

// ------------------------------------------------------------------------------------------------
// a1, per epoch: the whole descriptor pass as contractions with the RESIDENT moments,
//   q_n = sum_{J,k} cR[I][J][n][k] M1[J][k] (Eq.5-6),  S_nlm = sum_{J,k} cA[I][J][n][k] A1[J][k][lm] (Eq.8), q_nl (Eq.7), 4-body.
// M1 = sum_j f_k and A1 = sum_j f_k B_lm depend on the geometry only (positions are fixed during training): the
// pair sweeps that build them (k_radial_fwd, k_angw_fwd) run once per loaded batch.  Warp per atom (grid-stride).  The
// atom's A1 block (T*KT*24 floats, contiguous) and M1 row arrive as full-width loads requested one atom ahead and are
// parked in a per-warp shared buffer; the contraction reads them as 32-byte pieces shared by the lanes of a slot group,
// lane = (n, lmg) as in the epilogues above (8 (l,m) slots of one n per lane), cA[I][J][n][.] as float4.
// ------------------------------------------------------------------------------------------------
__host__ __device__ inline int angw_S_smem_floats(int T, int NA, int KT, int NR, int KRp) {
  return T * T * NA * KT + ((T * T * NR * KRp + 3) & ~3) + ANG_WARPS * 2 * (T * KT * ANGW_NLM + ((T * KRp + 7) & ~7));
}
// Two atoms per warp and iteration: lanes 0..14 work on the first, 16..30 on the second; within a half lane = (n pair, lmg):
// two functions n and 8 (l,m) slots each, so that one 32-byte piece of an A1 row feeds 16 FMAs.
template <int KT, int TMAX>
__global__ void __launch_bounds__(ANG_WARPS * 32, TMAX <= 2 ? 4 : 2)
k_angw_S(DevSpec sp, int N, const int *__restrict__ type_s, const float *__restrict__ theta, const float *__restrict__ M1,
         const float *__restrict__ A1, float *__restrict__ q, float *__restrict__ S) {
  constexpr int NP = (2 * TMAX * KT * 3 + 31) / 32;                // 32-byte pieces of two A1 blocks per lane (T <= TMAX species)
  extern __shared__ __align__(128) float smem[];
  const int nA = sp.T * KT * ANGW_NLM, nM = sp.T * sp.KRp, nMs = (nM + 7) & ~7;
  float *csA = smem;                                             // [T*T*NA][KT]
  float *csR = csA + sp.T * sp.T * sp.NA * KT;                   // [T*T][KRp][NR] (transposed: lanes n read consecutive words)
  float *stage = csR + ((sp.T * sp.T * sp.NR * sp.KRp + 3) & ~3) + (threadIdx.x >> 5) * 2 * (nA + nMs);   // two A1 blocks
  float *m1s = stage + 2 * nA;                                   // two M1 rows
  stage_coeff(csA, theta + sp.offA, sp.T * sp.T * sp.NA, sp.KA, KT);
  for (int x = threadIdx.x; x < sp.T * sp.T * sp.NR * sp.KRp; x += blockDim.x) {
    const int n = x % sp.NR, k = (x / sp.NR) % sp.KRp, ij = x / (sp.NR * sp.KRp);
    csR[x] = k < sp.KR ? theta[((size_t)ij * sp.NR + n) * sp.KR + k] : 0.f;
  }
  __syncthreads();
  const int lane = threadIdx.x & 31, half = lane >> 4, hl = lane & 15;
  const int nq = hl / 3, lmg = hl - 3 * nq;                      // n pair 0..4 (hl 15 idles), slot group
  const bool act = hl < 15;
  float c2[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) c2[i] = c_C2[8 * (lmg < 3 ? lmg : 0) + i];
  const int split = lmg == 0 ? 3 : lmg == 1 ? 7 : 8;             // slots below `split` belong to the lane's first l
  const int gw = blockIdx.x * ANG_WARPS + (threadIdx.x >> 5), nw = gridDim.x * ANG_WARPS;
  const int pieces = nA / 8;                                     // of ONE block
  float8 pre[NP];
  constexpr int NMP = TMAX <= 2 ? 2 : 4;
  float mpre[NMP];                                               // two M1 rows of T * KRp <= 16 TMAX floats
#pragma unroll
  for (int v = 0; v < NMP; ++v) mpre[v] = 0.f;
  int Ipre = 0;
  // the pair of atoms (2 it, 2 it + 1): their A1 blocks are adjacent in memory, 2 * pieces pieces in all
  auto request = [&](int it) {
    const int a0 = 2 * it;
    if (a0 >= N) return;
    const int np2 = (a0 + 1 < N ? 2 : 1) * pieces;
    Ipre = type_s[min(a0 + half, N - 1)];
#pragma unroll
    for (int v = 0; v < NP; ++v)
      if (lane + 32 * v < np2) pre[v] = ldg256(A1 + (size_t)a0 * nA + 8 * (lane + 32 * v));
    const int nm2 = (a0 + 1 < N ? 2 : 1) * nM;
#pragma unroll
    for (int v = 0; v < NMP; ++v)
      if (lane + 32 * v < nm2) mpre[v] = M1[(size_t)a0 * nM + lane + 32 * v];
  };
  const int n_it = (N + 1) >> 1;
  request(gw);
  for (int it = gw; it < n_it; it += nw) {
    const int np2 = (2 * it + 1 < N ? 2 : 1) * pieces, nm2 = (2 * it + 1 < N ? 2 : 1) * nM;
#pragma unroll
    for (int v = 0; v < NP; ++v)
      if (lane + 32 * v < np2) {     // piece p = 8 floats of a row: low quads in one plane, high quads in the other, so that
        *(float4 *)(stage + 4 * (lane + 32 * v)) = pre[v].lo;          // both stores are contiguous across the lanes (a 32-byte
        *(float4 *)(stage + nA + 4 * (lane + 32 * v)) = pre[v].hi;     // stride per lane is a two-way bank conflict)
      }
#pragma unroll
    for (int v = 0; v < NMP; ++v) {
      const int x = lane + 32 * v;                               // (the two rows are parked nMs apart)
      if (x < nm2) m1s[(x >= nM ? nMs - nM : 0) + x] = mpre[v];
    }
    const int I = Ipre;
    __syncwarp();
    request(it + nw);                                            // the next pair's blocks are in flight during this contraction
    const int a = 2 * it + half;
    const bool on_a = a < N;
    float *Sa = S + (size_t)a * sp.NA * ANGW_NLM;
    float *qa = q + (size_t)a * sp.Ndes + sp.NR;
    if (on_a && hl < sp.NR) {                                    // radial descriptors: lane = n (NR <= 16)
      float acc = 0.f;
      const float *c = csR + (size_t)I * sp.T * sp.KRp * sp.NR + hl;
      const float *m = m1s + half * nMs;
      for (int jk = 0; jk < nM; jk += 2) {                       // (KRp is even)
        const float2 m2 = *(const float2 *)(m + jk);
        acc = fmaf(c[jk * sp.NR], m2.x, acc);
        acc = fmaf(c[(jk + 1) * sp.NR], m2.y, acc);
      }
      q[(size_t)a * sp.Ndes + hl] = acc;
    }
    for (int nb = 0; nb < sp.NA; nb += 10) {
      const int n0 = nb + 2 * nq;
      const bool on0 = on_a && act && n0 < sp.NA, on1 = on0 && n0 + 1 < sp.NA;
      float sv[2][8];
#pragma unroll
      for (int i = 0; i < 8; ++i) { sv[0][i] = 0.f; sv[1][i] = 0.f; }
      if (on0) {
        for (int J = 0; J < sp.T; ++J) {
          const float *c = csA + ((size_t)(I * sp.T + J) * sp.NA + n0) * KT;
          const float *c1 = on1 ? c + KT : c;
          const float *row = stage + 4 * ((half * nA) / 8 + J * KT * 3 + lmg);   // low quad of piece (J, k = 0, lmg); + 12 per k; high plane + nA
#pragma unroll
          for (int k4 = 0; k4 < KT; k4 += 4) {
            const float4 ca = *(const float4 *)(c + k4), cb = *(const float4 *)(c1 + k4);
            const float cv0[4] = {ca.x, ca.y, ca.z, ca.w}, cv1[4] = {cb.x, cb.y, cb.z, cb.w};
#pragma unroll
            for (int kk = 0; kk < 4; ++kk) {
              const float4 lo = *(const float4 *)(row + (k4 + kk) * 12), hi = *(const float4 *)(row + nA + (k4 + kk) * 12);
              const float av[8] = {lo.x, lo.y, lo.z, lo.w, hi.x, hi.y, hi.z, hi.w};
#pragma unroll
              for (int i = 0; i < 8; ++i) { sv[0][i] = fmaf(cv0[kk], av[i], sv[0][i]); sv[1][i] = fmaf(cv1[kk], av[i], sv[1][i]); }
            }
          }
        }
      }
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        const int n = n0 + e;
        const bool on = e == 0 ? on0 : on1;
        float qa_ = 0.f, qb_ = 0.f;
        if (on) {
          stg256(Sa + n * ANGW_NLM + 8 * lmg, make_float4(sv[e][0], sv[e][1], sv[e][2], sv[e][3]), make_float4(sv[e][4], sv[e][5], sv[e][6], sv[e][7]));
#pragma unroll
          for (int i = 0; i < 8; ++i) {
            const float w = 0.5f * c2[i] * sv[e][i] * sv[e][i];
            if (i < split) qa_ += w; else qb_ += w;
          }
        }
        const float nxt = __shfl_down_sync(0xffffffffu, qa_, 1);   // the l=4 remainder held by (n, lmg 2)
        if (on && lmg == 0) {
          qa[n] = qa_;
          if (sp.L >= 2) qa[sp.NA + n] = qb_;
          if (sp.use4) qa[sp.NA * sp.L + n] = GNEP_KAPPA4 * p4_value(sv[e] + 3);
          if (sp.use5) qa[sp.NA * (sp.L + sp.use4) + n] = p5_value(sv[e]);
        }
        if (on && lmg == 1) {
          if (sp.L >= 3) qa[2 * sp.NA + n] = qa_;
          if (sp.L >= 4) qa[3 * sp.NA + n] = qb_ + nxt;
        }
      }
    }
    __syncwarp();                                                // the stage is rewritten for the next pair
  }
}

// ------------------------------------------------------------------------------------------------
// a5 (angular): A2 moments with the pair adjoint a_ij, T_nlm = c.A2, D_(n,l) = sum_m 2 C_lm S_nlm T_nlm, D_4
// ------------------------------------------------------------------------------------------------
template <int KT, int NQ, bool B5 /* model has the 5-body term */>
__global__ void __launch_bounds__(ANG_WARPS * 32)
k_angw_adj(DevSpec sp, int N, int ta /* atoms per warp, <= ANG_TA */, const int *__restrict__ type_s, const int *__restrict__ struct_s,
              const int *__restrict__ segA, const int *__restrict__ atomA, const float4 *__restrict__ pairA,
              const float *__restrict__ theta, const float4 *__restrict__ u, const float *__restrict__ omega,
              const float *__restrict__ scales, const float *__restrict__ S, float *__restrict__ Tn,
              float *__restrict__ A2, float *__restrict__ D) {
  constexpr int KQ = (KT + 3) / 4;      // k per lane: lane = (k quarter kq, lm eighth lmq) holds a KQ x 3 register tile
  constexpr bool KPAIR = (KQ % 2 == 0); // radial factors stored as k pairs, outer products on packed FMAs
  extern __shared__ __align__(128) float smem[];
  float *ct = smem;
  const int nct = sp.T * sp.T * KT * ANG_NQ;
  const int nA = sp.T * KT * ANGW_NLM;
  const int per_warp = (2 * KT + 2 * ANGW_NLM) * ANG_LD + nA + ANG_NQ * ANGW_NLM + ANG_SEGS;
  float *sf1 = smem + nct + (threadIdx.x >> 5) * per_warp;   // [KT][LD]  f_k' (a.rhat)
  float *sf2 = sf1 + KT * ANG_LD;                             // [KT][LD]  f_k
  float *sX = sf2 + KT * ANG_LD;                              // [24][LD]  B_lm
  float *sY = sX + ANGW_NLM * ANG_LD;                         // [24][LD]  grad B_lm . a
  float *As = sY + ANGW_NLM * ANG_LD;                         // [T][KT][24]
  float *Xs = As + nA;                                        // [NQ][24]  T of the current atom
  int *sEnd = (int *)(Xs + ANG_NQ * ANGW_NLM);                // segment ends of the tile
  stage_coeff_t(ct, theta + sp.offA, sp.T, sp.NA, sp.KA, KT);
  __syncthreads();
  const int lane = threadIdx.x & 31;
  const int a_lo = (blockIdx.x * ANG_WARPS + (threadIdx.x >> 5)) * ta;
  if (a_lo >= N) return;
  const int a_hi = min(a_lo + ta, N);
  const int T1 = sp.T + 1;
  const int P_lo = segA[a_lo * T1], P_hi = segA[(a_hi - 1) * T1 + sp.T];
  const int kq = lane >> 3, lmq = lane & 7;
  const NLane nl = make_nlane(lane);
  const float sfF = scales[1], svV = scales[2];
  float acc[KQ][3];
#pragma unroll
  for (int r = 0; r < KQ; ++r)
#pragma unroll
    for (int i = 0; i < 3; ++i) acc[r][i] = 0.f;
  constexpr int NJ = (NQ + 3) / 4;
  float Xo[NJ][3];
#pragma unroll
  for (int j = 0; j < NJ; ++j)
#pragma unroll
    for (int i = 0; i < 3; ++i) Xo[j][i] = 0.f;
  for (int x = lane; x < (a_hi - a_lo) * sp.T; x += 32) sEnd[x] = segA[(a_lo + x / sp.T) * T1 + x % sp.T + 1];
  __syncwarp();
  int a = a_lo, J = 0;
  int seg_end = sEnd[0];

  int Icur = type_s[a_lo];       // species of atom a, requested when the previous atom ends
  // S of atom a in the (n, lmg) lane layout of the epilogue (first n-round), requested when the previous atom ends
  float4 sn0 = make_float4(0.f, 0.f, 0.f, 0.f), sn1 = sn0;
  auto next_atom = [&]() {
    if (a < a_hi) {
      Icur = type_s[a];
      if (nl.act && nl.nq < sp.NA) {
        const float *Sa_ = S + (size_t)a * sp.NA * ANGW_NLM + nl.nq * ANGW_NLM + 8 * nl.lmg;
        const float8 s8 = ldg256(Sa_); sn0 = s8.lo; sn1 = s8.hi;
      }
    }
  };
  next_atom();
  auto flush_segment = [&]() {
    xown_add<KT, KQ, NJ>(sp, ct, Icur, J, lane, kq, acc, Xo);
#pragma unroll
    for (int r = 0; r < KQ; ++r) {
      int k = kq * KQ + r;
      if (k < KT) {
        int o = (J * KT + k) * ANGW_NLM + 3 * lmq;
#pragma unroll
        for (int i = 0; i < 3; ++i) { As[o + i] = acc[r][i]; acc[r][i] = 0.f; }
      }
    }
  };
  auto atom_epilogue = [&]() {   // A2 -> global, T = c.A2, D of atom a
    __syncwarp();
    for (int x = lane; x < nA / 4; x += 32) ((float4 *)(A2 + (size_t)a * nA))[x] = ((const float4 *)As)[x];
    xown_store<NJ>(kq, lmq, Xo, Xs);
    const float *Sa = S + (size_t)a * sp.NA * ANGW_NLM;
    float *Ta = Tn + (size_t)a * sp.NA * ANGW_NLM;
    float *Da = D + (size_t)a * sp.Ndes + sp.NR;
    for (int nb = 0; nb < sp.NA; nb += 10) {
      const int n = nb + nl.nq;
      const bool on = nl.act && n < sp.NA;
      float tv[8], sv[8], da = 0.f, db = 0.f;
      if (on) {
        float4 s0 = sn0, s1 = sn1;
        if (nb > 0) { const float8 s8 = ldg256(Sa + n * ANGW_NLM + 8 * nl.lmg); s0 = s8.lo; s1 = s8.hi; }
        sv[0] = s0.x; sv[1] = s0.y; sv[2] = s0.z; sv[3] = s0.w; sv[4] = s1.x; sv[5] = s1.y; sv[6] = s1.z; sv[7] = s1.w;
        {
          const float4 t0 = *(const float4 *)(Xs + n * ANGW_NLM + 8 * nl.lmg), t1 = *(const float4 *)(Xs + n * ANGW_NLM + 8 * nl.lmg + 4);
          tv[0] = t0.x; tv[1] = t0.y; tv[2] = t0.z; tv[3] = t0.w; tv[4] = t1.x; tv[5] = t1.y; tv[6] = t1.z; tv[7] = t1.w;
        }
        stg256(Ta + n * ANGW_NLM + 8 * nl.lmg, make_float4(tv[0], tv[1], tv[2], tv[3]), make_float4(tv[4], tv[5], tv[6], tv[7]));
        float w[8];
#pragma unroll
        for (int i = 0; i < 8; ++i) w[i] = nl.c2[i] * sv[i] * tv[i];
        split_sums(nl, w, da, db);
      }
      const float nxt = __shfl_down_sync(0xffffffffu, da, 1);
      if (on && nl.lmg == 0) {
        Da[n] = da;
        if (sp.L >= 2) Da[sp.NA + n] = db;
        if (sp.use4) {
          float g4[5];
          p4_grad(sv + 3, g4);
          Da[sp.NA * sp.L + n] = GNEP_KAPPA4 * (g4[0] * tv[3] + g4[1] * tv[4] + g4[2] * tv[5] + g4[3] * tv[6] + g4[4] * tv[7]);
        }
        if constexpr (B5) {                              // directional derivative of q5 = kappa5 |S_1|^4 along T
          float g5[3];
          p5_grad(sv, g5);
          Da[sp.NA * (sp.L + sp.use4) + n] = g5[0] * tv[0] + g5[1] * tv[1] + g5[2] * tv[2];
        }
      }
      if (on && nl.lmg == 1) {
        if (sp.L >= 3) Da[2 * sp.NA + n] = da;
        if (sp.L >= 4) Da[3 * sp.NA + n] = db + nxt;
      }
    }
    __syncwarp();
  };
  auto next_segment = [&]() {
    flush_segment();
    if (++J == sp.T) { atom_epilogue(); J = 0; ++a; next_atom(); }
    seg_end = a < a_hi ? sEnd[(a - a_lo) * sp.T + J] : 0x7fffffff;
  };

  // three-stage pipeline over chunks: records (r, atom) two chunks ahead, their gathers (u_i, u_j, structure) one
  // chunk ahead, arithmetic on the current chunk
  const float4 rdum = make_float4(1.f, 0.f, 0.f, 0.f);
  float4 r1 = rdum, r2 = rdum, ui1 = rdum, uj1 = rdum;
  int ai1 = 0, ai2 = 0, s1 = 0;
  if (P_lo + lane < P_hi) { r1 = pairA[P_lo + lane]; ai1 = atomA[P_lo + lane]; }
  if (P_lo + 32 + lane < P_hi) { r2 = pairA[P_lo + 32 + lane]; ai2 = atomA[P_lo + 32 + lane]; }
  ui1 = u[ai1]; uj1 = u[__float_as_int(r1.w)]; s1 = struct_s[ai1];
  for (int c0 = P_lo; c0 < P_hi; c0 += 32) {
    const int p = c0 + lane;
    const float4 r = r1, ui = ui1, uj = uj1;
    const int s = s1;
    r1 = r2; ai1 = ai2;
    ui1 = u[ai1]; uj1 = u[__float_as_int(r1.w)]; s1 = struct_s[ai1];
    if (p + 64 < P_hi) { r2 = pairA[p + 64]; ai2 = atomA[p + 64]; } else { r2 = rdum; ai2 = 0; }
    if (p < P_hi) {
      float d, rinv;
      pair_len(r.x * r.x + r.y * r.y + r.z * r.z, d, rinv);
      const float *om = omega + s * 6;
      float ax = sfF * (ui.x - uj.x) - svV * (om[0] * r.x + om[5] * r.z);
      float ay = sfF * (ui.y - uj.y) - svV * (om[1] * r.y + om[3] * r.x);
      float az = sfF * (ui.z - uj.z) - svV * (om[2] * r.z + om[4] * r.y);
      float hx = r.x * rinv, hy = r.y * rinv, hz = r.z * rinv;
      float ar = ax * hx + ay * hy + az * hz;
      float f[KT], fp[KT];
      cheb_ffp<KT>(d, sp.rcAinv, f, fp);
      if constexpr (KPAIR) {   // rows of k pairs: [k/2][slot][2]
#pragma unroll
        for (int k = 0; k < KT; k += 2) {
          *(float2 *)(sf1 + k * ANG_LD + 2 * lane) = make_float2(fp[k] * ar, fp[k + 1] * ar);
          *(float2 *)(sf2 + k * ANG_LD + 2 * lane) = make_float2(f[k], f[k + 1]);
        }
      } else {
#pragma unroll
        for (int k = 0; k < KT; ++k) { sf1[k * ANG_LD + lane] = fp[k] * ar; sf2[k * ANG_LD + lane] = f[k]; }
      }
      // Y_lm = (grad B_lm . a - l B_lm (a.rhat)) / d with a / d and l (a.rhat) / d formed once per pair: four FMAs per slot
      const float bx = ax * rinv, by = ay * rinv, bz = az * rinv, br = ar * rinv;
      const float lar[4] = {-br, -2.f * br, -3.f * br, -4.f * br};
      blm_unit<4>(hx, hy, hz, [&](int lm, int l, float b, float gx, float gy, float gz) {
        sX[lm * ANG_LD + lane] = b;
        sY[lm * ANG_LD + lane] = fmaf(lar[l - 1], b, fmaf(gz, bz, fmaf(gy, by, gx * bx)));
      });
    } else {
      if constexpr (KPAIR) {
#pragma unroll
        for (int k = 0; k < KT; k += 2) {
          *(float2 *)(sf1 + k * ANG_LD + 2 * lane) = make_float2(0.f, 0.f);
          *(float2 *)(sf2 + k * ANG_LD + 2 * lane) = make_float2(0.f, 0.f);
        }
      } else {
#pragma unroll
        for (int k = 0; k < KT; ++k) { sf1[k * ANG_LD + lane] = 0.f; sf2[k * ANG_LD + lane] = 0.f; }
      }
#pragma unroll
      for (int lm = 0; lm < ANGW_NLM; ++lm) { sX[lm * ANG_LD + lane] = 0.f; sY[lm * ANG_LD + lane] = 0.f; }
    }
    __syncwarp();
    const int chunk_end = min(c0 + 32, P_hi);
    int pos = c0;
    while (pos < chunk_end) {
      while (seg_end <= pos) next_segment();
      const int hi = min(seg_end, chunk_end);
      if constexpr (KPAIR) {
        for (int g = (pos - c0) >> 2; g < (hi - c0) >> 2; ++g) {   // whole 4-pair groups only (padded segments)
          float4 f1a[KQ / 2], f1b[KQ / 2], f2a[KQ / 2], f2b[KQ / 2];
#pragma unroll
          for (int rp = 0; rp < KQ / 2; ++rp) {                     // the lane's k pairs (k0, k0 + 1), four pair slots each
            const int o = (kq * KQ + 2 * rp) * ANG_LD + 8 * g;
            f1a[rp] = *(const float4 *)(sf1 + o); f1b[rp] = *(const float4 *)(sf1 + o + 4);
            f2a[rp] = *(const float4 *)(sf2 + o); f2b[rp] = *(const float4 *)(sf2 + o + 4);
          }
#pragma unroll
          for (int i = 0; i < 3; ++i) {
            const float4 X = *(const float4 *)(sX + (3 * lmq + i) * ANG_LD + 4 * g);
            const float4 Y = *(const float4 *)(sY + (3 * lmq + i) * ANG_LD + 4 * g);
#pragma unroll
            for (int rp = 0; rp < KQ / 2; ++rp) {
              fma4x2(acc[2 * rp][i], acc[2 * rp + 1][i], f1a[rp], f1b[rp], X);
              fma4x2(acc[2 * rp][i], acc[2 * rp + 1][i], f2a[rp], f2b[rp], Y);
            }
          }
        }
      } else
      for (int g = (pos - c0) >> 2; g < (hi - c0) >> 2; ++g) {   // whole 4-pair groups only (padded segments)
        float4 f1[KQ], f2[KQ];
#pragma unroll
        for (int r = 0; r < KQ; ++r) {
          int k = kq * KQ + r;
          const float4 z4 = make_float4(0.f, 0.f, 0.f, 0.f);
          f1[r] = k < KT ? *(const float4 *)(sf1 + k * ANG_LD + 4 * g) : z4;
          f2[r] = k < KT ? *(const float4 *)(sf2 + k * ANG_LD + 4 * g) : z4;
        }
#pragma unroll
        for (int i = 0; i < 3; ++i) {
          float4 X = *(const float4 *)(sX + (3 * lmq + i) * ANG_LD + 4 * g);
          float4 Y = *(const float4 *)(sY + (3 * lmq + i) * ANG_LD + 4 * g);
#pragma unroll
          for (int r = 0; r < KQ; ++r) { fma4(acc[r][i], f1[r], X); fma4(acc[r][i], f2[r], Y); }
        }
      }
      pos = hi;
    }
    __syncwarp();
  }
  while (a < a_hi) next_segment();
}

// ------------------------------------------------------------------------------------------------
// a7 (angular): dL/dcA[I][J][n][k] = sum_atoms sum_lm alpha_nlm A1[J][k][lm] + beta_nlm A2[J][k][lm]
//   alpha_nlm = gbar_(n,l) 2C_lm S_nlm + E'_(n,l) 2C_lm T_nlm (+ 4-body: gbar_4 k4 dP4/ds_m + E'_4 k4 (H4 T)_m)
//   beta_nlm  = E'_(n,l) 2C_lm S_nlm (+ E'_4 k4 dP4/ds_m)
// One warp per atom (grid-stride); lane = ((J,k) row, half of n).  Each warp keeps a [T][T][NA][KT] accumulator in
// shared memory over the atoms it visits and writes one partial at the end (reduced by k_grad_reduce).
// ------------------------------------------------------------------------------------------------
template <int KT, bool B5 /* model has the 5-body term */>
__global__ void __launch_bounds__(ANG_WARPS * 32, 4)
k_angw_cgrad(DevSpec sp, int N, const int *__restrict__ type_s, const float *__restrict__ Ep,
                const float *__restrict__ gbar, const float *__restrict__ S, const float *__restrict__ Tn,
                const float *__restrict__ A1, const float *__restrict__ A2, float *__restrict__ partial) {
  extern __shared__ __align__(128) float smem[];
  const int nacc = sp.T * sp.T * sp.NA * KT;
  const int nb = sp.NA * ANGW_NLM;
  const int nA = sp.T * KT * ANGW_NLM;
  const int per_warp = ((nacc + 3) & ~3) + 2 * ((nb + 3) & ~3);
  float *accS = smem + (threadIdx.x >> 5) * per_warp;
  float *sAl = accS + ((nacc + 3) & ~3);
  float *sBe = sAl + ((nb + 3) & ~3);
  const int lane = threadIdx.x & 31;
  const NLane nl = make_nlane(lane);
  const int gw = blockIdx.x * ANG_WARPS + (threadIdx.x >> 5);
  const int nw = gridDim.x * ANG_WARPS;
  for (int o = lane; o < nacc; o += 32) accS[o] = 0.f;
  __syncwarp();
  const int rows = sp.T * KT;                      // (J,k) rows of A1/A2
  const int nh = (sp.NA + 1) >> 1;                 // n's per half
  const int half = lane & 1;
  const int n_lo = half * nh, n_hi = min(sp.NA, n_lo + nh);
  for (int a = gw; a < N; a += nw) {
    const int I = type_s[a];
    // requests in the order of use: the per-atom rows S, T, E', gbar of the first n-round (needed at once for
    // alpha/beta), then the moment rows of the first contraction round, whose latency hides behind the alpha/beta work
    const float *Sa = S + (size_t)a * nb, *Ta = Tn + (size_t)a * nb;
    const float *Epa = Ep + (size_t)a * sp.Ndes, *gba = gbar + (size_t)a * sp.Ndes;
    float8 s8, t8;
    s8.lo = s8.hi = t8.lo = t8.hi = make_float4(0.f, 0.f, 0.f, 0.f);
    float ea = 0.f, eb = 0.f, ga = 0.f, gb = 0.f, e4r = 0.f, gb4r = 0.f;
    auto request = [&](int n) {
      const int o = n * ANGW_NLM + 8 * nl.lmg;
      s8 = ldg256(Sa + o); t8 = ldg256(Ta + o);
      ea = desc_of(sp, Epa, nl.la, n); eb = desc_of(sp, Epa, nl.lb, n);
      ga = desc_of(sp, gba, nl.la, n); gb = desc_of(sp, gba, nl.lb, n);
      if (sp.use4 && nl.lmg == 0) { e4r = Epa[sp.NR + sp.L * sp.NA + n]; gb4r = gba[sp.NR + sp.L * sp.NA + n]; }
    };
    if (nl.act && nl.nq < sp.NA) request(nl.nq);
    float4 x1[6], x2[6];
    {
      const int row = lane >> 1;
      if (row < rows) {
        const float4 *a1 = (const float4 *)(A1 + (size_t)a * nA + row * ANGW_NLM);
        const float4 *a2 = (const float4 *)(A2 + (size_t)a * nA + row * ANGW_NLM);
#pragma unroll
        for (int v = 0; v < 6; v += 2) {
          const float8 u1 = ldg256((const float *)(a1 + v)), u2 = ldg256((const float *)(a2 + v));
          x1[v] = u1.lo; x1[v + 1] = u1.hi; x2[v] = u2.lo; x2[v + 1] = u2.hi;
        }
      }
    }
    for (int n0 = 0; n0 < sp.NA; n0 += 10) {      // alpha, beta in the (n, lmg) lane layout
      const int n = n0 + nl.nq;
      if (nl.act && n < sp.NA) {
        const int o = n * ANGW_NLM + 8 * nl.lmg;
        if (n0 > 0) request(n);
        const float4 s0 = s8.lo, s1 = s8.hi, t0 = t8.lo, t1 = t8.hi;
        float sv[8] = {s0.x, s0.y, s0.z, s0.w, s1.x, s1.y, s1.z, s1.w};
        float tv[8] = {t0.x, t0.y, t0.z, t0.w, t1.x, t1.y, t1.z, t1.w};
        float al[8], be[8];
#pragma unroll
        for (int i = 0; i < 8; ++i) {
          const float e1 = i < nl.split ? ea : eb, g1 = i < nl.split ? ga : gb;
          al[i] = nl.c2[i] * (g1 * sv[i] + e1 * tv[i]);
          be[i] = nl.c2[i] * e1 * sv[i];
        }
        if (sp.use4 && nl.lmg == 0) {
          float g4[5], hv[5];
          p4_grad(sv + 3, g4);
          p4_hess_vec(sv + 3, tv + 3, hv);
          const float e4 = GNEP_KAPPA4 * e4r, gb4 = GNEP_KAPPA4 * gb4r;
#pragma unroll
          for (int m = 0; m < 5; ++m) { al[3 + m] += gb4 * g4[m] + e4 * hv[m]; be[3 + m] += e4 * g4[m]; }
        }
        if (B5 && nl.lmg == 0) {                        // 5-body (R41) on the l = 1 slots; its E', gbar are fetched here
          const int o5 = sp.NR + (sp.L + sp.use4) * sp.NA + n;
          const float e5 = Epa[o5], gb5 = gba[o5];
          float g5[3], hv[3];
          p5_grad(sv, g5);
          p5_hess_vec(sv, tv, hv);
#pragma unroll
          for (int m = 0; m < 3; ++m) { al[m] += gb5 * g5[m] + e5 * hv[m]; be[m] += e5 * g5[m]; }
        }
        *(float4 *)(sAl + o) = make_float4(al[0], al[1], al[2], al[3]);
        *(float4 *)(sAl + o + 4) = make_float4(al[4], al[5], al[6], al[7]);
        *(float4 *)(sBe + o) = make_float4(be[0], be[1], be[2], be[3]);
        *(float4 *)(sBe + o + 4) = make_float4(be[4], be[5], be[6], be[7]);
      }
    }
    __syncwarp();
    // contraction: lane -> row = lane>>1 (+16 per round), half = lane&1 -> n in [half*nh, min(NA, half*nh+nh))
    for (int row = lane >> 1; row < rows; row += 16) {
      if (row >= 16) {
        const float4 *a1 = (const float4 *)(A1 + (size_t)a * nA + row * ANGW_NLM);
        const float4 *a2 = (const float4 *)(A2 + (size_t)a * nA + row * ANGW_NLM);
#pragma unroll
        for (int v = 0; v < 6; v += 2) {
          const float8 u1 = ldg256((const float *)(a1 + v)), u2 = ldg256((const float *)(a2 + v));
          x1[v] = u1.lo; x1[v + 1] = u1.hi; x2[v] = u2.lo; x2[v + 1] = u2.hi;
        }
      }
      const int J = row / KT, k = row - J * KT;
      float *dst = accS + ((I * sp.T + J) * sp.NA) * KT + k;
      for (int n = n_lo; n < n_hi; ++n) {
        float2 sa[2], sb[2];                              // four independent chains of packed FMAs (even / odd lm partial sums)
        sa[0] = sa[1] = sb[0] = sb[1] = make_float2(0.f, 0.f);
#pragma unroll
        for (int v = 0; v < 6; ++v) {
          const float4 al4 = *(const float4 *)(sAl + n * ANGW_NLM + 4 * v);
          const float4 be4 = *(const float4 *)(sBe + n * ANGW_NLM + 4 * v);
          float2 &s = sa[v & 1], &t = sb[v & 1];
          s = __ffma2_rn(make_float2(al4.x, al4.y), make_float2(x1[v].x, x1[v].y), s);
          s = __ffma2_rn(make_float2(al4.z, al4.w), make_float2(x1[v].z, x1[v].w), s);
          t = __ffma2_rn(make_float2(be4.x, be4.y), make_float2(x2[v].x, x2[v].y), t);
          t = __ffma2_rn(make_float2(be4.z, be4.w), make_float2(x2[v].z, x2[v].w), t);
        }
        const float2 st = __fadd2_rn(__fadd2_rn(sa[0], sa[1]), __fadd2_rn(sb[0], sb[1]));
        dst[n * KT] += st.x + st.y;
      }
    }
    __syncwarp();
  }
  for (int o = lane; o < nacc; o += 32) partial[(size_t)gw * nacc + o] = accS[o];
}
